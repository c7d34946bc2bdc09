// stray.cu -- the field of the magnet in a probe layer above it ("we calculate the out-of-plane component of
// the magnet's stray field 60 nm above the film's surface"; reading S40).
//
//   B_i(x, y) = -mu0 sum_{x', y', k} sum_j N_ij(x - x', y - y', Dz_k) M_j(x', y', k),   M = sum_s Ms^(s) m^(s)
//   Dz_k = (Nz - k - 1/2) dz + height
//
// N is the cell-to-cell Newell tensor at a z offset that is not a multiple of the cell height (newell.cpp), tabulated on
// the non-negative quadrant of in-plane offsets per source layer, parity giving the other three quadrants.  The sum is
// taken as written (a direct O(N_probe N_source) sum: an imaging evaluation, made once per relaxed state, not a step of
// the time loop): a CTA owns 16 x 16 probe cells and walks over the source tiles, M of a tile staged in shared memory,
// fp32 products summed per tile and accumulated in fp64 across tiles.  Open boundaries.
#include <vector>

#include "mmx_internal.h"

int mmx_newell_quadrant_at(int nx, int ny, const double cell[3], double dz, double cutoff_cells, std::vector<double>& out);

namespace {

constexpr int ST = 16;

__global__ void __launch_bounds__(256) k_gather_M(const float* y, const uint16_t* reg, const float* mat, int S, int nreg,
                                                  size_t N, float* M) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int r = reg ? reg[i] : 0;
  float mx = 0.f, my = 0.f, mz = 0.f;
  for (int s = 0; s < S; ++s) {
    const float Ms = mat[((size_t)s * nreg + r) * MMX_MATW + MP_MS];
    const float* m = y + (size_t)s * 3 * N;
    mx = fmaf(Ms, m[i], mx); my = fmaf(Ms, m[N + i], my); mz = fmaf(Ms, m[2 * N + i], mz);
  }
  M[i] = mx; M[N + i] = my; M[2 * N + i] = mz;
}

// tab: [nz][6][ny][nx] with -mu0 folded in; components xx, yy, zz, xy, xz, yz
__global__ void __launch_bounds__(ST * ST) k_stray(const float* M, const float* tab, int nx, int ny, int nz, float* out) {
  __shared__ float sM[3][ST * ST];
  const int tx = blockIdx.x * ST + threadIdx.x, ty = blockIdx.y * ST + threadIdx.y;
  const int t = threadIdx.y * ST + threadIdx.x;
  const size_t plane = (size_t)nx * ny, N = plane * nz;
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
        if (tx < nx && ty < ny) {
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
  }
  if (tx < nx && ty < ny) {
    const size_t o = (size_t)ty * nx + tx;
    out[o] = (float)bx; out[plane + o] = (float)by; out[2 * plane + o] = (float)bz;
  }
}

}  // namespace

// scratch: [3][N] floats for M; returns the field in dev_out [3][ny][nx]
int mmx_stray_launch(mmx_world* w, double height, double cutoff_cells, float* dev_out) {
  const int nx = w->grid[0], ny = w->grid[1], nz = w->grid[2];
  const size_t plane = (size_t)nx * ny;
  const double MU0 = 4e-7 * M_PI;
  std::vector<float> tab((size_t)nz * 6 * plane);
  std::vector<double> quad;
  for (int k = 0; k < nz; ++k) {
    const double dz = (nz - k - 0.5) * w->cell[2] + height;
    if (int rc = mmx_newell_quadrant_at(nx, ny, w->cell, dz, cutoff_cells, quad)) return rc;
    for (size_t q = 0; q < 6 * plane; ++q) tab[(size_t)k * 6 * plane + q] = (float)(-MU0 * quad[q]);
  }
  float* d_tab = nullptr;
  MMX_CUDA(cudaMalloc(&d_tab, tab.size() * sizeof(float)));
  cudaError_t e = cudaMemcpyAsync(d_tab, tab.data(), tab.size() * sizeof(float), cudaMemcpyHostToDevice, w->stream);
  if (e == cudaSuccess) {
    k_gather_M<<<(unsigned)((w->N + 255) / 256), 256, 0, w->stream>>>(w->Y[w->sel_host], w->nreg > 1 ? w->d_reg : nullptr, w->d_mat,
                                                                     w->S, w->nreg, w->N, w->scratch);
    k_stray<<<dim3((nx + ST - 1) / ST, (ny + ST - 1) / ST), dim3(ST, ST), 0, w->stream>>>(w->scratch, d_tab, nx, ny, nz, dev_out);
    w->launches += 2;
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaStreamSynchronize(w->stream);
  cudaFree(d_tab);
  if (e != cudaSuccess) return mmx_fail(MMX_ECUDA, "stray field evaluation failed: %s", cudaGetErrorString(e));
  return MMX_OK;
}
