// stray_static.cu -- mmx_stray_field_static: the stray-field probe of stray.cu (Fig.3; reading S40) for
// callers that must not allocate.
//
// Who that is.  mmx_stray_field builds its Newell table on the host, cudaMallocs room for it, and cudaFrees it again on
// every call; the world it runs on owns more cudaMalloc'd storage.  That is fine for a script, and unusable for
//   * a process whose device memory is already handed out in full to a pooling allocator (a PyTorch / CuPy caching
//     allocator, an inference server's arena): a raw cudaMalloc there fails, or succeeds only after the pool was flushed;
//   * a latency-bound loop: cudaMalloc and cudaFree take a driver lock and cudaFree waits for the whole device, so one
//     imaging call stalls every other stream of the process;
//   * a thread that runs while another thread of the process captures a CUDA graph in the default (global) capture mode:
//     cudaMalloc is one of the calls that breaks such a capture.
// For them this file keeps the only scratch the evaluation needs -- the summed magnetisation M = sum_s Ms^(s) m^(s)
// (P:L144), [3][Nz][Ny][Nx] fp32 -- in one file-scope device array of fixed size that the CUDA module carries itself.
// The price: every GPU on which this library's module is loaded holds the MMX_STRAY_STATIC_MAX_CELLS * 12 bytes (3 MiB)
// from then until the process exits, used or not, and grids above that limit are refused.
//
// The Newell table is an *input* here (device memory the caller already owns, filled once from mmx_stray_table_host,
// which is plain host code and may be run anywhere, any time before); the entry point itself reaches no cudaMalloc,
// cudaFree, cudaMallocAsync, no host heap and no library routine that allocates.
//
// The array's name in host code is only a handle of the host-side shadow of the symbol, not a device address; a kernel
// handed `g_M` from the host would fault (or, where the GPU can reach host memory, quietly use the wrong bytes).  The
// device address is asked from the runtime once per device, cudaGetSymbolAddress with that device current, and that
// pointer is what the kernels receive.
//
// Sharing.  There is one array per device and every call on that device uses it; it still holds the previous call's M
// when the next call starts.  Nothing has to start at zero: k_gather_s overwrites elements [0, 3N) before k_stray_s
// reads exactly those, and both run in order on the caller's stream.  Two calls that overlap on one GPU (different
// streams, or two host threads) race on the array and give garbage: serialise them.
#include <mutex>

#include "mmx_internal.h"

int mmx_newell_quadrant_at(int nx, int ny, const double cell[3], double dz, double cutoff_cells, std::vector<double>& out);

namespace {

constexpr int ST = 16;        // probe / source tile edge, as in stray.cu
constexpr int MAX_DEV = 64;   // devices per process this file keeps an address for

static __device__ __align__(256) float g_M[3 * (size_t)MMX_STRAY_STATIC_MAX_CELLS];

std::mutex g_mu;
float* g_M_addr[MAX_DEV];     // device address of g_M on device d, null until the first call on d

struct MsRow { float v[3]; };

// M_c = sum_s Ms^(s) m_c^(s), the same fused multiply-add chain as k_gather_M of stray.cu with one region.
__global__ void __launch_bounds__(256) k_gather_s(const float* __restrict__ m, MsRow Ms, int S, unsigned N, float* __restrict__ M) {
  const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  float mx = 0.f, my = 0.f, mz = 0.f;
  for (int s = 0; s < S; ++s) {
    const float* ms = m + (size_t)s * 3 * N;
    mx = fmaf(Ms.v[s], ms[i], mx); my = fmaf(Ms.v[s], ms[N + i], my); mz = fmaf(Ms.v[s], ms[2 * (size_t)N + i], mz);
  }
  M[i] = mx; M[N + i] = my; M[2 * (size_t)N + i] = mz;
}

// B_i(x, y) = sum_{x', y', k} sum_j T_ij(|x - x'|, |y - y'|, k) M_j(x', y', k), signs of the odd components restored from
// the sign of the offset; T carries -mu0.  A CTA owns ST x ST probe cells and walks over the source tiles, fp32 within a
// tile, fp64 across tiles: the arithmetic and its order are those of k_stray in stray.cu.
__global__ void __launch_bounds__(ST * ST) k_stray_s(const float* __restrict__ M, const float* __restrict__ tab, int nx, int ny, int nz,
                                                     float* __restrict__ out) {
  __shared__ float sM[3][ST * ST];
  const int tx = blockIdx.x * ST + threadIdx.x, ty = blockIdx.y * ST + threadIdx.y;
  const int t = threadIdx.y * ST + threadIdx.x;
  const size_t plane = (size_t)nx * ny, N = plane * nz;
  const bool mine = tx < nx && ty < ny;
  double bx = 0.0, by = 0.0, bz = 0.0;
  for (int k = 0; k < nz; ++k) {
    const float* T = tab + (size_t)k * 6 * plane;
    for (int sy0 = 0; sy0 < ny; sy0 += ST)
      for (int sx0 = 0; sx0 < nx; sx0 += ST) {
        const int sx = sx0 + threadIdx.x, sy = sy0 + threadIdx.y;
        const bool in = sx < nx && sy < ny;
        const size_t si = (size_t)k * plane + (size_t)sy * nx + sx;
        __syncthreads();
#pragma unroll
        for (int c = 0; c < 3; ++c) sM[c][t] = in ? M[(size_t)c * N + si] : 0.f;
        __syncthreads();
        if (!mine) continue;
        float ax = 0.f, ay = 0.f, az = 0.f;
        const int ylim = min(ST, ny - sy0), xlim = min(ST, nx - sx0);
        for (int j = 0; j < ylim; ++j) {
          const int dy = ty - (sy0 + j);
          const float sgy = dy < 0 ? -1.f : 1.f;
          const float* Ty = T + (size_t)abs(dy) * nx;
          for (int i = 0; i < xlim; ++i) {
            const int dx = tx - (sx0 + i);
            const float sgx = dx < 0 ? -1.f : 1.f;
            const float* p = Ty + abs(dx);
            const float nxx = __ldg(p), nyy = __ldg(p + plane), nzz = __ldg(p + 2 * plane);
            const float nxy = sgx * sgy * __ldg(p + 3 * plane), nxz = sgx * __ldg(p + 4 * plane), nyz = sgy * __ldg(p + 5 * plane);
            const float mx = sM[0][j * ST + i], my = sM[1][j * ST + i], mz = sM[2][j * ST + i];
            ax = fmaf(nxx, mx, fmaf(nxy, my, fmaf(nxz, mz, ax)));
            ay = fmaf(nxy, mx, fmaf(nyy, my, fmaf(nyz, mz, ay)));
            az = fmaf(nxz, mx, fmaf(nyz, my, fmaf(nzz, mz, az)));
          }
        }
        bx += (double)ax; by += (double)ay; bz += (double)az;
      }
  }
  if (mine) {
    const size_t o = (size_t)ty * nx + tx;
    out[o] = (float)bx; out[plane + o] = (float)by; out[2 * plane + o] = (float)bz;
  }
}

// Device address of g_M on the current device; asked from the runtime the first time this device is seen.
int scratch_on_current_device(float** out) {
  int dev = -1;
  MMX_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= MAX_DEV) return mmx_fail(MMX_EINVAL, "mmx_stray_field_static: device ordinal %d is beyond the %d this entry point keeps", dev, MAX_DEV);
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_M_addr[dev]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_M);
    if (e != cudaSuccess || !p)
      return mmx_fail(MMX_ECUDA, "mmx_stray_field_static: cudaGetSymbolAddress of the scratch array failed on device %d: %s", dev,
                      cudaGetErrorString(e));
    g_M_addr[dev] = (float*)p;
  }
  *out = g_M_addr[dev];
  return MMX_OK;
}

}  // namespace

extern "C" int mmx_stray_table_host(const int grid[3], const double cellsize[3], double height, float* out, long long out_len) {
  if (!grid || !cellsize || !out) return mmx_fail(MMX_EINVAL, "NULL argument");
  for (int a = 0; a < 3; ++a)
    if (grid[a] < 1 || !(cellsize[a] > 0)) return mmx_fail(MMX_EINVAL, "grid and cellsize must be positive");
  if (!(height > -0.5 * cellsize[2])) return mmx_fail(MMX_EINVAL, "the probe layer must lie above the centre of the top layer");
  const int nx = grid[0], ny = grid[1], nz = grid[2];
  const size_t plane = (size_t)nx * ny;
  if (out_len != (long long)(6 * plane * nz)) return mmx_fail(MMX_EINVAL, "out_len must be Nz*6*Ny*Nx = %zu", 6 * plane * nz);
  const double MU0 = 4e-7 * M_PI;
  std::vector<double> quad;
  for (int k = 0; k < nz; ++k) {
    const double dz = (nz - k - 0.5) * cellsize[2] + height;
    if (int rc = mmx_newell_quadrant_at(nx, ny, cellsize, dz, 0.0, quad)) return rc;
    for (size_t q = 0; q < 6 * plane; ++q) out[(size_t)k * 6 * plane + q] = (float)(-MU0 * quad[q]);
  }
  return MMX_OK;
}

extern "C" int mmx_stray_field_static(const int grid[3], int n_sublattices, const double Ms[], const float* m, const float* table,
                                      float* out, void* cuda_stream) {
  if (!grid || !Ms || !m || !table || !out) return mmx_fail(MMX_EINVAL, "NULL argument");
  if (n_sublattices < 1 || n_sublattices > 3) return mmx_fail(MMX_EINVAL, "n_sublattices must be 1, 2 or 3");
  for (int a = 0; a < 3; ++a)
    if (grid[a] < 1) return mmx_fail(MMX_EINVAL, "grid sizes must be >= 1");
  const long long N = (long long)grid[0] * grid[1] * grid[2];
  if (N > (long long)MMX_STRAY_STATIC_MAX_CELLS)
    return mmx_fail(MMX_EINVAL,
                    "mmx_stray_field_static: %d x %d x %d = %lld cells, above the %d cells of the built-in scratch array "
                    "(MMX_STRAY_STATIC_MAX_CELLS); use mmx_stray_field, which allocates",
                    grid[0], grid[1], grid[2], N, (int)MMX_STRAY_STATIC_MAX_CELLS);
  float* M = nullptr;
  if (int rc = scratch_on_current_device(&M)) return rc;
  MsRow row = {{0.f, 0.f, 0.f}};
  for (int s = 0; s < n_sublattices; ++s) row.v[s] = (float)Ms[s];
  cudaStream_t st = (cudaStream_t)cuda_stream;
  k_gather_s<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(m, row, n_sublattices, (unsigned)N, M);
  k_stray_s<<<dim3((grid[0] + ST - 1) / ST, (grid[1] + ST - 1) / ST), dim3(ST, ST), 0, st>>>(M, table, grid[0], grid[1], grid[2], out);
  MMX_CUDA(cudaGetLastError());
  return MMX_OK;
}
