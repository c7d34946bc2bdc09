// demag.cu -- magnetostatic field as a zero-padded FFT convolution.
//
// B_demag = -mu0 sum_r' N(r - r') M(r'), M = sum_s Ms^(s) m^(s) (the vector sum of
// the sublattice moments is formed first).  The convolution is evaluated with
// hand-written shared-memory FFT passes (fft.cuh), pruned for the zero padding:
//
//   x_fwd   rows of M (gathered from m on load), two real rows per complex line, Nx -> Px,
//           split into the two half spectra, kept columns 0..Px/2       -> spec1 [3][Nz][Ny][XP]
//   mid_fwd (3-D only) along y, Ny -> Py, rows y >= Ny never read       -> spec2 [3][Nz][Py][XP]
//   inner   along the last transformed axis (z in 3-D, y in 2-D): forward transform of the
//           three components, multiply by the real symmetric 3x3 kernel spectrum, inverse
//           transform, only the first N planes stored, in place
//   mid_inv along y, only rows y < Ny stored                             -> spec1
//   x_inv   half spectra of two rows -> one complex line -> inverse -> real/imag parts are
//           the two rows of B_demag, only x < Nx stored                  -> B [3][Nz][Ny][Nx]
//
// The kernel spectrum is real (the tensor components are even or odd per axis); only the
// octant kx<=Px/2, ky<=Py/2, kz<=Pz/2 is stored and sign-reflected for the odd components.
#include <cstdio>

#include "fft.cuh"
#include "mmx_internal.h"

using namespace mmxfft;

namespace {

// lines (rows / columns) of a CTA tile: "wide" tiles for grids that fill the GPU anyway, "narrow" ones (an eighth) for
// small grids, where the number of CTAs -- not the width of a CTA's memory accesses -- decides the time of a pass
// (c2's inner pass ran on 9 CTAs with wide tiles)
constexpr int lines_for(int P) {
  return P <= 256 ? 16 : (4096 / P < 2 ? 2 : 4096 / P);
}
constexpr int lines_narrow(int P) { return lines_for(P) / 8 < 1 ? 1 : lines_for(P) / 8; }
constexpr int block_of(int P, int L) { return L * threads_per_line(P); }

struct XArgs {
  int nx, rows, xc, xp, S, nreg, gated;
  size_t N;               // cells
  const float* yin[2];    // state [nvec][3][N]
  const uint16_t* reg;
  const float* mat;
  const MmxCtrl* ctrl;
  const float2* tw;
  float2* spec;           // spec1
  float* bout;            // x_inv output [3][N]
};

struct MidArgs {
  int n_in, n_out, xc, xp, gated;
  size_t in_outer, out_outer;   // elements between consecutive (c, z) slabs
  const float2* in;
  float2* out;
  const float2* tw;
  const MmxCtrl* ctrl;
};

struct InnerArgs {
  int n_valid, xc, xp, gated;
  int p_outer;                  // transform length of the outer axis (1: none)
  size_t line_stride, comp_stride, outer_stride;
  size_t k_inner_stride, k_outer_stride, k_comp_stride;
  unsigned odd_inner, odd_outer;   // bit c set: component c is odd along that axis
  int two_d;                       // xz, yz components vanish
  float2* spec;
  const float* khat;
  const float2* tw;
  const MmxCtrl* ctrl;
};

__device__ __forceinline__ float gather_M(const XArgs& a, const float* y, size_t off, size_t cell) {
  // M = sum_s Ms^(s)(region) m^(s)
  int r = a.reg ? a.reg[cell] : 0;
  float M = 0.f;
  for (int s = 0; s < a.S; ++s)
    M = fmaf(a.mat[((size_t)s * a.nreg + r) * MMX_MATW + MP_MS], y[(size_t)s * 3 * a.N + off], M);
  return M;
}

template <int P, int L>
__global__ void __launch_bounds__(block_of(P, L)) k_x_fwd(XArgs a) {
  constexpr int LP = L | 1, TPL = threads_per_line(P);
  extern __shared__ float2 s[];
  if (a.gated && !a.ctrl->active) return;
  const float* y = a.yin[a.ctrl->sel];
  const int tid = threadIdx.x, T = L * TPL;
  const long long row0 = (long long)blockIdx.x * (2 * L);
  const unsigned rpc = (unsigned)a.rows / 3u;   // rows per component: the cell of element (row r, x) is (r mod rpc) nx + x
#pragma unroll
  for (int idx = tid; idx < L * P; idx += T) {
    const int line = idx / P, x = idx % P;
    float2 v = make_float2(0.f, 0.f);
    if (x < a.nx) {
      const unsigned r0 = (unsigned)row0 + 2u * (unsigned)line;   // (32-bit index arithmetic: rows < 2^31)
      if (r0 < (unsigned)a.rows) v.x = gather_M(a, y, (size_t)r0 * a.nx + x, (size_t)(r0 % rpc) * a.nx + x);
      if (r0 + 1 < (unsigned)a.rows) v.y = gather_M(a, y, (size_t)(r0 + 1) * a.nx + x, (size_t)((r0 + 1) % rpc) * a.nx + x);
    }
    s[x * LP + line] = v;
  }
  __syncthreads();
  InPlace<P, -1>::run(s, LP, tid % L, tid / L, a.tw, true);
  // split  Z = FFT(a + i b)  into  A = FFT(a), B = FFT(b),  columns 0..P/2
  for (int idx = tid; idx < 2 * L * a.xc; idx += T) {
    const int rl = idx / a.xc, k = idx % a.xc;
    const int line = rl >> 1, part = rl & 1;
    const long long r = row0 + rl;
    if (r < a.rows) {
      const float2 zk = s[k * LP + line];
      const float2 zm = s[((P - k) & (P - 1)) * LP + line];
      float2 o;
      if (part == 0) o = make_float2(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y));
      else o = make_float2(0.5f * (zk.y + zm.y), -0.5f * (zk.x - zm.x));
      a.spec[(size_t)r * a.xp + k] = o;
    }
  }
}

template <int P, int L>
__global__ void __launch_bounds__(block_of(P, L)) k_x_inv(XArgs a) {
  constexpr int LP = L | 1, TPL = threads_per_line(P);
  extern __shared__ float2 s[];
  if (a.gated && !a.ctrl->active) return;
  const int tid = threadIdx.x, T = L * TPL;
  const long long row0 = (long long)blockIdx.x * (2 * L);
  for (int idx = tid; idx < L * a.xc; idx += T) {
    const int line = idx / a.xc, k = idx % a.xc;
    const long long r0 = row0 + 2 * line;
    float2 A = make_float2(0.f, 0.f), B = A;
    if (r0 < a.rows) A = a.spec[(size_t)r0 * a.xp + k];
    if (r0 + 1 < a.rows) B = a.spec[(size_t)(r0 + 1) * a.xp + k];
    s[k * LP + line] = make_float2(A.x - B.y, A.y + B.x);           // A + i B
    if (k > 0 && 2 * k < P) s[(P - k) * LP + line] = make_float2(A.x + B.y, B.x - A.y);  // conj A + i conj B
  }
  __syncthreads();
  InPlace<P, +1>::run(s, LP, tid % L, tid / L, a.tw, true);
  for (int idx = tid; idx < 2 * L * a.nx; idx += T) {
    const int rl = idx / a.nx, x = idx % a.nx;
    const long long r = row0 + rl;
    if (r < a.rows) {
      const float2 z = s[x * LP + (rl >> 1)];
      a.bout[(size_t)r * a.nx + x] = (rl & 1) ? z.y : z.x;
    }
  }
}

template <int P, int L, int DIR>
__global__ void __launch_bounds__(block_of(P, L)) k_mid(MidArgs a) {
  constexpr int LP = L, TPL = threads_per_line(P);
  extern __shared__ float2 s[];
  if (a.gated && !a.ctrl->active) return;
  const int tid = threadIdx.x, T = L * TPL;
  const int kx0 = blockIdx.x * L;
  const float2* in = a.in + (size_t)blockIdx.y * a.in_outer;
  float2* out = a.out + (size_t)blockIdx.y * a.out_outer;
  for (int idx = tid; idx < P * L; idx += T) {
    const int pos = idx / L, l = idx % L;
    float2 v = make_float2(0.f, 0.f);
    if (pos < a.n_in && kx0 + l < a.xc) v = in[(size_t)pos * a.xp + kx0 + l];
    s[pos * LP + l] = v;
  }
  __syncthreads();
  InPlace<P, DIR>::run(s, LP, tid % L, tid / L, a.tw, true);
  for (int idx = tid; idx < a.n_out * L; idx += T) {
    const int pos = idx / L, l = idx % L;
    if (kx0 + l < a.xc) out[(size_t)pos * a.xp + kx0 + l] = s[pos * LP + l];
  }
}

template <int P, int L>
__global__ void __launch_bounds__(block_of(P, L)) k_inner(InnerArgs a) {
  constexpr int LP = L, TPL = threads_per_line(P);
  extern __shared__ float2 s[];
  if (a.gated && !a.ctrl->active) return;
  const int tid = threadIdx.x, T = L * TPL;
  const int kx0 = blockIdx.x * L;
  const int ko = blockIdx.y;  // outer wave number (ky in 3-D)
  float2* base = a.spec + (size_t)ko * a.outer_stride;
  for (int c = 0; c < 3; ++c) {
    float2* sc = s + c * (P * LP);
    const float2* in = base + (size_t)c * a.comp_stride;
    for (int idx = tid; idx < P * L; idx += T) {
      const int pos = idx / L, l = idx % L;
      float2 v = make_float2(0.f, 0.f);
      if (pos < a.n_valid && kx0 + l < a.xc) v = in[(size_t)pos * a.line_stride + kx0 + l];
      sc[pos * LP + l] = v;
    }
  }
  __syncthreads();
  if constexpr (P > 1) {
    for (int c = 0; c < 3; ++c) InPlace<P, -1>::run(s + c * (P * LP), LP, tid % L, tid / L, a.tw, true);
  }
  // B^_i = sum_j K^_ij M^_j ; K^ real, 6 unique components, octant + parity
  {
    int kom = ko, so = 0;
    if (a.p_outer > 1 && 2 * ko > a.p_outer) { kom = a.p_outer - ko; so = 1; }
    const float* kb = a.khat + (size_t)kom * a.k_outer_stride;
    for (int idx = tid; idx < P * L; idx += T) {
      const int pos = idx / L, l = idx % L;
      const int kx = kx0 + l;
      if (kx >= a.xc) continue;
      int pm = pos, si = 0;
      if (2 * pos > P) { pm = P - pos; si = 1; }
      const float* kp = kb + (size_t)pm * a.k_inner_stride + kx;
      float K[6];
#pragma unroll
      for (int c = 0; c < 6; ++c) {
        if (a.two_d && c >= 4) { K[c] = 0.f; continue; }
        float v = __ldg(kp + (size_t)c * a.k_comp_stride);
        const int flip = (si & (a.odd_inner >> c)) ^ (so & (a.odd_outer >> c));
        K[c] = (flip & 1) ? -v : v;
      }
      const float2 mx = s[pos * LP + l], my = s[P * LP + pos * LP + l], mz = s[2 * P * LP + pos * LP + l];
      float2 bx, by, bz;
      bx.x = fmaf(K[0], mx.x, fmaf(K[3], my.x, K[4] * mz.x));
      bx.y = fmaf(K[0], mx.y, fmaf(K[3], my.y, K[4] * mz.y));
      by.x = fmaf(K[3], mx.x, fmaf(K[1], my.x, K[5] * mz.x));
      by.y = fmaf(K[3], mx.y, fmaf(K[1], my.y, K[5] * mz.y));
      bz.x = fmaf(K[4], mx.x, fmaf(K[5], my.x, K[2] * mz.x));
      bz.y = fmaf(K[4], mx.y, fmaf(K[5], my.y, K[2] * mz.y));
      s[pos * LP + l] = bx;
      s[P * LP + pos * LP + l] = by;
      s[2 * P * LP + pos * LP + l] = bz;
    }
  }
  __syncthreads();
  if constexpr (P > 1) {
    for (int c = 0; c < 3; ++c) InPlace<P, +1>::run(s + c * (P * LP), LP, tid % L, tid / L, a.tw, true);
  }
  for (int c = 0; c < 3; ++c) {
    const float2* sc = s + c * (P * LP);
    float2* out = base + (size_t)c * a.comp_stride;
    for (int idx = tid; idx < a.n_valid * L; idx += T) {
      const int pos = idx / L, l = idx % L;
      if (kx0 + l < a.xc) out[(size_t)pos * a.line_stride + kx0 + l] = sc[pos * LP + l];
    }
  }
}

#define MMX_SWITCH_P(P_, MIN_, CALL)                        \
  switch (P_) {                                             \
    case 1: if (MIN_ <= 1) { CALL(1); } break;              \
    case 2: CALL(2); break;                                 \
    case 4: CALL(4); break;                                 \
    case 8: CALL(8); break;                                 \
    case 16: CALL(16); break;                               \
    case 32: CALL(32); break;                               \
    case 64: CALL(64); break;                               \
    case 128: CALL(128); break;                             \
    case 256: CALL(256); break;                             \
    case 512: CALL(512); break;                             \
    case 1024: CALL(1024); break;                           \
    case 2048: CALL(2048); break;                           \
    default: return mmx_fail(MMX_EINVAL, "unsupported transform length %d", P_); \
  }

template <typename Kern>
int set_smem(Kern k, size_t bytes) {
  if (bytes > 48 * 1024) MMX_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
  return MMX_OK;
}

int next_pow2(int n) {
  int p = 1;
  while (p < n) p <<= 1;
  return p;
}

}  // namespace

// transform lengths: 2 * pow2(N) on an open axis (zero padding), N on a periodic one (must be
// a power of two), 1 on a single-cell y/z axis.  x is always transformed (Px >= 2).
int mmx_demag_plan_sizes(mmx_world* w) {
  DemagPlan& d = w->dm;
  d.nx = w->grid[0]; d.ny = w->grid[1]; d.nz = w->grid[2];
  int P[3];
  for (int a = 0; a < 3; ++a) {
    const int n = w->grid[a];
    if (w->pbc[a] > 0) {
      if (n & (n - 1)) return mmx_fail(MMX_EINVAL, "periodic axis %d has size %d, not a power of two", a, n);
      P[a] = n;
    } else {
      P[a] = n == 1 ? 1 : 2 * next_pow2(n);
    }
  }
  if (P[0] < 2) P[0] = 2;
  for (int a = 0; a < 3; ++a)
    if (P[a] > 2048) return mmx_fail(MMX_EINVAL, "transform length %d on axis %d exceeds 2048", P[a], a);
  d.px = P[0]; d.py = P[1]; d.pz = P[2];
  d.xc = d.px / 2 + 1;
  d.xp = (d.xc + 15) & ~15;  // rows start on 128-byte boundaries
  d.ky = d.py > 1 ? d.py / 2 + 1 : 1;
  d.kz = d.pz > 1 ? d.pz / 2 + 1 : 1;
  return MMX_OK;
}

int mmx_demag_launch(mmx_world* w, const float* const yin[2], float* bout) {
  DemagPlan& d = w->dm;
  if (!d.ready) return mmx_fail(MMX_ESTATE, "mmx_demag_kernel_init has not been called");
  cudaStream_t st = w->stream;
  // narrow CTA tiles when the wide ones would leave most of the GPU idle.  Measured (c1, c2, c3, c5):
  // the row passes gain whenever the wide grid has fewer CTAs than multiprocessors (c5 x forward 18.4 -> 14.8 us with
  // 48 -> 192 CTAs), the column passes only when it has fewer than a quarter of them (c2 inner 21.0 -> 16.8 us with
  // 9 -> 65 CTAs; c3 with 65 wide CTAs lost 2 us on narrow 32-byte column accesses)
  auto narrow_rows = [&](long long ctas_wide) { return ctas_wide < (long long)w->sm_count; };
  auto narrow = [&](long long ctas_wide) { return 4 * ctas_wide < (long long)w->sm_count; };
  const int rows = 3 * d.nz * d.ny;
  const bool three_d = d.nz > 1;
  XArgs xa;
  xa.nx = d.nx; xa.rows = rows; xa.xc = d.xc; xa.xp = d.xp; xa.S = w->S; xa.nreg = w->nreg; xa.gated = 1;
  xa.N = w->N; xa.yin[0] = yin[0]; xa.yin[1] = yin[1];
  xa.reg = w->nreg > 1 ? w->d_reg : nullptr; xa.mat = w->d_mat; xa.ctrl = w->d_ctrl;
  xa.tw = d.tw[0]; xa.spec = d.spec1; xa.bout = bout;

#define CALL_XF_L(PP, L)                                                                  \
  {                                                                                       \
    size_t sm = sizeof(float2) * PP * (L | 1);                                            \
    if (int rc = set_smem(k_x_fwd<PP, L>, sm)) return rc;                                 \
    ProfScope ps(w, PK_X_FWD);                                                             \
    k_x_fwd<PP, L><<<(rows + 2 * L - 1) / (2 * L), block_of(PP, L), sm, st>>>(xa);        \
  }
#define CALL_XF(PP)                                                                       \
  if (narrow_rows((rows + 2 * lines_for(PP) - 1) / (2 * lines_for(PP)))) CALL_XF_L(PP, lines_narrow(PP)) else CALL_XF_L(PP, lines_for(PP))
  const bool xwarp = mmx_x_warp_ok(w);
  if (xwarp) {
    if (int rc = mmx_x_warp_launch(w, -1, yin, bout)) return rc;
  } else {
    MMX_SWITCH_P(d.px, 2, CALL_XF)
  }
  w->launches++;

  if (three_d && d.py > 1) {
    MidArgs ma;
    ma.n_in = d.ny; ma.n_out = d.py; ma.xc = d.xc; ma.xp = d.xp; ma.gated = 1;
    ma.in_outer = (size_t)d.ny * d.xp; ma.out_outer = (size_t)d.py * d.xp;
    ma.in = d.spec1; ma.out = d.spec2; ma.tw = d.tw[1]; ma.ctrl = w->d_ctrl;
#define CALL_MF_L(PP, L)                                                                  \
  {                                                                                       \
    size_t sm = sizeof(float2) * PP * L;                                                  \
    if (int rc = set_smem(k_mid<PP, L, -1>, sm)) return rc;                               \
    dim3 g((d.xc + L - 1) / L, 3 * d.nz);                                                 \
    ProfScope ps(w, PK_MID_FWD);                                                           \
    k_mid<PP, L, -1><<<g, block_of(PP, L), sm, st>>>(ma);                                 \
  }
#define CALL_MF(PP)                                                                       \
  if (narrow((d.xc + lines_for(PP) - 1) / lines_for(PP) * 3 * d.nz)) CALL_MF_L(PP, lines_narrow(PP)) else CALL_MF_L(PP, lines_for(PP))
    if (mmx_mid_col_ok(d.py, d.ny)) {
      if (int rc = mmx_mid_col_launch(w, d.py, -1, d.spec1, d.spec2, d.ny, d.py, ma.in_outer, ma.out_outer,
                                      3 * d.nz, d.tw[1])) return rc;
    } else {
      MMX_SWITCH_P(d.py, 2, CALL_MF)
    }
    w->launches++;
  }

  {
    InnerArgs ia;
    ia.xc = d.xc; ia.xp = d.xp; ia.gated = 1; ia.khat = d.khat; ia.ctrl = w->d_ctrl;
    ia.k_comp_stride = (size_t)d.kz * d.ky * d.xp;
    int Pin, nouter;
    if (three_d) {
      const bool mid = d.py > 1;
      const int pyy = mid ? d.py : d.ny;  // == 1 when !mid
      ia.spec = mid ? d.spec2 : d.spec1;
      ia.n_valid = d.nz; Pin = d.pz; nouter = pyy; ia.p_outer = d.py;
      ia.line_stride = (size_t)pyy * d.xp; ia.comp_stride = (size_t)d.nz * pyy * d.xp; ia.outer_stride = d.xp;
      ia.k_inner_stride = (size_t)d.ky * d.xp; ia.k_outer_stride = d.xp;
      ia.odd_inner = (1u << 4) | (1u << 5); ia.odd_outer = (1u << 3) | (1u << 5);
      ia.two_d = 0; ia.tw = d.tw[2];
    } else {
      ia.spec = d.spec1;
      ia.n_valid = d.ny; Pin = d.py; nouter = 1; ia.p_outer = 1;
      ia.line_stride = d.xp; ia.comp_stride = (size_t)d.ny * d.xp; ia.outer_stride = 0;
      ia.k_inner_stride = d.xp; ia.k_outer_stride = 0;
      ia.odd_inner = (1u << 3) | (1u << 5); ia.odd_outer = 0;
      ia.two_d = 1; ia.tw = d.tw[1];
    }
#define CALL_IN_L(PP, L)                                                                  \
  {                                                                                       \
    size_t sm = sizeof(float2) * 3 * PP * L;                                              \
    if (int rc = set_smem(k_inner<PP, L>, sm)) return rc;                                 \
    dim3 g((d.xc + L - 1) / L, nouter);                                                   \
    ProfScope ps(w, PK_INNER);                                                             \
    k_inner<PP, L><<<g, block_of(PP, L), sm, st>>>(ia);                                   \
  }
#define CALL_IN(PP)                                                                       \
  if (narrow((d.xc + lines_for(PP) - 1) / lines_for(PP) * nouter)) CALL_IN_L(PP, lines_narrow(PP)) else CALL_IN_L(PP, lines_for(PP))
    if (d.tiled) {
      if (int rc = mmx_inner_tile_launch(w)) return rc;
    } else if (mmx_inner_col_ok(d, Pin, ia.n_valid)) {
      InnerColLaunch L;
      L.spec = ia.spec; L.tw = ia.tw; L.n_valid = ia.n_valid; L.p_outer = ia.p_outer; L.n_outer = nouter;
      L.line_stride = ia.line_stride; L.comp_stride = ia.comp_stride; L.outer_stride = ia.outer_stride;
      L.k_inner_stride = ia.k_inner_stride; L.k_outer_stride = ia.k_outer_stride; L.k_comp_stride = ia.k_comp_stride;
      L.odd_inner = ia.odd_inner; L.odd_outer = ia.odd_outer;
      if (int rc = mmx_inner_col_launch(w, L)) return rc;
    } else {
      MMX_SWITCH_P(Pin, 1, CALL_IN)
    }
    w->launches++;
  }

  if (three_d && d.py > 1) {
    MidArgs ma;
    ma.n_in = d.py; ma.n_out = d.ny; ma.xc = d.xc; ma.xp = d.xp; ma.gated = 1;
    ma.in_outer = (size_t)d.py * d.xp; ma.out_outer = (size_t)d.ny * d.xp;
    ma.in = d.spec2; ma.out = d.spec1; ma.tw = d.tw[1]; ma.ctrl = w->d_ctrl;
#define CALL_MI_L(PP, L)                                                                  \
  {                                                                                       \
    size_t sm = sizeof(float2) * PP * L;                                                  \
    if (int rc = set_smem(k_mid<PP, L, +1>, sm)) return rc;                               \
    dim3 g((d.xc + L - 1) / L, 3 * d.nz);                                                 \
    ProfScope ps(w, PK_MID_INV);                                                           \
    k_mid<PP, L, +1><<<g, block_of(PP, L), sm, st>>>(ma);                                 \
  }
#define CALL_MI(PP)                                                                       \
  if (narrow((d.xc + lines_for(PP) - 1) / lines_for(PP) * 3 * d.nz)) CALL_MI_L(PP, lines_narrow(PP)) else CALL_MI_L(PP, lines_for(PP))
    if (mmx_mid_col_ok(d.py, d.ny)) {
      if (int rc = mmx_mid_col_launch(w, d.py, +1, d.spec2, d.spec1, d.py, d.ny, ma.in_outer, ma.out_outer,
                                      3 * d.nz, d.tw[1])) return rc;
    } else {
      MMX_SWITCH_P(d.py, 2, CALL_MI)
    }
    w->launches++;
  }

#define CALL_XI_L(PP, L)                                                                  \
  {                                                                                       \
    size_t sm = sizeof(float2) * PP * (L | 1);                                            \
    if (int rc = set_smem(k_x_inv<PP, L>, sm)) return rc;                                 \
    ProfScope ps(w, PK_X_INV);                                                             \
    k_x_inv<PP, L><<<(rows + 2 * L - 1) / (2 * L), block_of(PP, L), sm, st>>>(xa);        \
  }
#define CALL_XI(PP)                                                                       \
  if (narrow_rows((rows + 2 * lines_for(PP) - 1) / (2 * lines_for(PP)))) CALL_XI_L(PP, lines_narrow(PP)) else CALL_XI_L(PP, lines_for(PP))
  if (xwarp) {
    if (int rc = mmx_x_warp_launch(w, +1, yin, bout)) return rc;
  } else {
    MMX_SWITCH_P(d.px, 2, CALL_XI)
  }
  w->launches++;
  MMX_CUDA(cudaGetLastError());
  return MMX_OK;
}
