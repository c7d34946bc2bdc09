// demag_col.cu -- register-resident "column" FFT passes of the demag convolution for the
// strided axes, the fast path of demag.cu.
//
// Lanes of a warp are neighbouring kx columns (contiguous in memory, 8 B each), so every
// global access of a warp is one contiguous row segment; the points of a line live in the
// registers of R threads (R points each) and cross threads once per H = R^2 point transform
// through a shared-memory tile [point][lane] (bank-conflict free).  See fft_reg.cuh for the
// index algebra.  Transform length P = 2 R^2; an open (zero-padded) axis is pruned: the upper
// input half is never read, the upper output half of the inverse never formed.
//
//   k_inner_col<8>  P = 128: forward along the innermost transformed axis, multiply by the real
//                   symmetric 3x3 kernel spectrum (octant + parity), inverse, in place.
//   k_mid_col<16>   P = 512 (also <8>: 128, <4>: 32): the y pass of a 3-D world, forward
//                   (n_in rows -> P rows) or inverse (P rows -> n_out rows).
//
// The column kx = Px/2 (Nyquist) would waste a whole lane tile; it is served by separate CTAs
// whose lanes run over the outer index instead (strided, but 1/257 of the data).
#include "fft_reg.cuh"
#include "mmx_internal.h"

using namespace mmxreg;

#ifndef MMX_MID_PERSISTENT
#define MMX_MID_PERSISTENT 1
#endif

namespace {

__device__ __forceinline__ void prefetch_l2(const void* p) {
  asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}

struct InnerColArgs {
  float2* spec;
  const float* khat;
  const float2* tw;      // exp(-2 pi i q / P)
  const MmxCtrl* ctrl;
  int gated, n_valid, xc, p_outer;
  int ntile_main;        // lane tiles over kx
  int xc_main;           // columns served by those tiles
  int nyq;               // 1: an extra tile column serves kx = xc-1 with lanes over the outer index
  size_t line_stride, comp_stride, outer_stride;
  size_t k_inner_stride, k_outer_stride, k_comp_stride;
  unsigned odd_inner, odd_outer;
};

// P = 2 R^2 = 128, R = 8.  CTA = 32 lanes x 8 warps; thread (lane, j) holds points j + 8u.
template <int R>
__global__ void __launch_bounds__(32 * R, 2) k_inner_col(InnerColArgs a) {
  constexpr int H = R * R, P = 2 * H;
  extern __shared__ float2 sm[];  // [6][H][32]
  __shared__ float2 stw[P];
  if (a.gated && !a.ctrl->active) return;
  const int lane = threadIdx.x & 31, j = threadIdx.x >> 5;
  int kx, ko;
  bool ok;
  const bool main_tile = (int)blockIdx.x < a.ntile_main;
  if (main_tile) {
    kx = blockIdx.x * 32 + lane; ko = blockIdx.y; ok = kx < a.xc_main;
  } else {
    if ((int)blockIdx.y * 32 >= a.p_outer) return;
    kx = a.xc - 1; ko = blockIdx.y * 32 + lane; ok = ko < a.p_outer;
  }
  if (!ok) { kx = 0; ko = 0; }
  for (int q = threadIdx.x; q < P; q += 32 * R) stw[q] = a.tw[q];

  // kernel octant rows of this CTA -> L2 (they are needed only after the forward transform)
  int kom = ko, so = 0;
  if (a.p_outer > 1 && 2 * ko > a.p_outer) { kom = a.p_outer - ko; so = 1; }
  const float* kb = a.khat + (size_t)kom * a.k_outer_stride + kx;
  if (main_tile) {
    for (int r = threadIdx.x; r < 6 * (H + 1); r += 32 * R) {
      const int c = r / (H + 1), pm = r % (H + 1);
      const float* p = a.khat + (size_t)kom * a.k_outer_stride + (size_t)blockIdx.x * 32 +
                       (size_t)pm * a.k_inner_stride + (size_t)c * a.k_comp_stride;
      prefetch_l2(p);
      prefetch_l2(p + 31);
    }
  }

  float2* base = a.spec + (size_t)ko * a.outer_stride + kx;
  float2 x[3][R];
#pragma unroll
  for (int c = 0; c < 3; ++c)
#pragma unroll
    for (int u = 0; u < R; ++u) {
      const int n = j + R * u;
      x[c][u] = (ok && n < a.n_valid) ? base[(size_t)c * a.comp_stride + (size_t)n * a.line_stride]
                                      : make_float2(0.f, 0.f);
    }
  __syncthreads();  // stw

  // forward stage 1: both halves of each component
#pragma unroll
  for (int c = 0; c < 3; ++c) {
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      float2 v[R];
#pragma unroll
      for (int u = 0; u < R; ++u) v[u] = h ? cmul(x[c][u], stw[j + R * u]) : x[c][u];
      Dft<R, -1>::run(v);
      float2* t = sm + (size_t)(c * 2 + h) * H * 32 + lane;
      t[(0 * R + j) * 32] = v[0];
#pragma unroll
      for (int q = 1; q < R; ++q) t[(q * R + j) * 32] = cmul(v[q], stw[2 * j * q]);
    }
  }
  __syncthreads();
  // forward stage 2: thread j now owns outputs m = j + R b of each half, wave number 2m + h
  float2 X[3][2][R];
#pragma unroll
  for (int c = 0; c < 3; ++c)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const float2* t = sm + (size_t)(c * 2 + h) * H * 32 + lane;
#pragma unroll
      for (int q = 0; q < R; ++q) X[c][h][q] = t[(j * R + q) * 32];
      Dft<R, -1>::run(X[c][h]);
    }
  // B^_i = sum_j K^_ij M^_j ; K^ real, 6 unique components, octant + parity
#pragma unroll
  for (int h = 0; h < 2; ++h)
#pragma unroll
    for (int b = 0; b < R; ++b) {
      const int kz = 2 * (j + R * b) + h;
      int pm = kz, si = 0;
      if (2 * kz > P) { pm = P - kz; si = 1; }
      const float* kp = kb + (size_t)pm * a.k_inner_stride;
      float K[6];
#pragma unroll
      for (int c = 0; c < 6; ++c) {
        const float v = __ldg(kp + (size_t)c * a.k_comp_stride);
        const int flip = (si & (a.odd_inner >> c)) ^ (so & (a.odd_outer >> c));
        K[c] = (flip & 1) ? -v : v;
      }
      const float2 mx = X[0][h][b], my = X[1][h][b], mz = X[2][h][b];
      X[0][h][b] = make_float2(fmaf(K[0], mx.x, fmaf(K[3], my.x, K[4] * mz.x)),
                               fmaf(K[0], mx.y, fmaf(K[3], my.y, K[4] * mz.y)));
      X[1][h][b] = make_float2(fmaf(K[3], mx.x, fmaf(K[1], my.x, K[5] * mz.x)),
                               fmaf(K[3], mx.y, fmaf(K[1], my.y, K[5] * mz.y)));
      X[2][h][b] = make_float2(fmaf(K[4], mx.x, fmaf(K[5], my.x, K[2] * mz.x)),
                               fmaf(K[4], mx.y, fmaf(K[5], my.y, K[2] * mz.y)));
    }
  // inverse stage 1 (over b); the thread writes the rows it has just read: no barrier needed
#pragma unroll
  for (int c = 0; c < 3; ++c)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      Dft<R, +1>::run(X[c][h]);
      float2* t = sm + (size_t)(c * 2 + h) * H * 32 + lane;
      t[(j * R + 0) * 32] = X[c][h][0];
#pragma unroll
      for (int q = 1; q < R; ++q) t[(j * R + q) * 32] = cmulc(X[c][h][q], stw[2 * j * q]);
    }
  __syncthreads();
  // inverse stage 2 (over the former thread index), combine the halves, store rows n < n_valid
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    float2 g[2][R];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const float2* t = sm + (size_t)(c * 2 + h) * H * 32 + lane;
#pragma unroll
      for (int q = 0; q < R; ++q) g[h][q] = t[(q * R + j) * 32];
      Dft<R, +1>::run(g[h]);
    }
#pragma unroll
    for (int b = 0; b < R; ++b) {
      const int n = j + R * b;
      const float2 o = cadd(g[0][b], cmulc(g[1][b], stw[n]));
      if (ok && n < a.n_valid) base[(size_t)c * a.comp_stride + (size_t)n * a.line_stride] = o;
    }
  }
}

struct MidColArgs {
  const float2* in;
  float2* out;
  const float2* tw;
  const MmxCtrl* ctrl;
  int gated, n_in, n_out, xc, xp, nslab;
  int ntile_main, xc_main, nyq;
  size_t in_outer, out_outer;  // elements between consecutive (component, z) slabs
};

// P = 2 R^2.  CTA = TILE columns x R threads per line x 2 halves; thread (kxl, j, h) transforms
// half h (even / odd wave numbers) of the line of column kxl.
template <int R, int TILE, int DIR>
__global__ void __launch_bounds__(2 * R * TILE, 2) k_mid_col(MidColArgs a) {
  constexpr int H = R * R, P = 2 * H, T = 2 * R * TILE;
  extern __shared__ float2 sm[];  // forward: [2][H][TILE]; inverse: [3][H][TILE]
  __shared__ float2 stw[P];
  if (a.gated && !a.ctrl->active) return;
  const int t = threadIdx.x;
  const int kxl = t % TILE, j = (t / TILE) % R, h = t / (TILE * R);
  int kx, slab;
  bool ok;
  if ((int)blockIdx.x < a.ntile_main) {
    kx = blockIdx.x * TILE + kxl; slab = blockIdx.y; ok = kx < a.xc_main;
  } else {
    if ((int)blockIdx.y * TILE >= a.nslab) return;
    kx = a.xc - 1; slab = blockIdx.y * TILE + kxl; ok = slab < a.nslab;
  }
  if (!ok) { kx = 0; slab = 0; }
  for (int q = t; q < P; q += T) stw[q] = a.tw[q];
  const float2* in = a.in + (size_t)slab * a.in_outer + kx;
  float2* out = a.out + (size_t)slab * a.out_outer + kx;
  float2* ex = sm + (size_t)h * H * TILE + kxl;

  float2 v[R];
  if (DIR < 0) {
#pragma unroll
    for (int u = 0; u < R; ++u) {
      const int n = j + R * u;
      v[u] = (ok && n < a.n_in) ? in[(size_t)n * a.xp] : make_float2(0.f, 0.f);
    }
    __syncthreads();  // stw
    if (h) {
#pragma unroll
      for (int u = 0; u < R; ++u) v[u] = cmul(v[u], stw[j + R * u]);
    }
  } else {
#pragma unroll
    for (int u = 0; u < R; ++u) {
      const int k = 2 * (j + R * u) + h;
      v[u] = ok ? in[(size_t)k * a.xp] : make_float2(0.f, 0.f);
    }
    __syncthreads();  // stw
  }
  Dft<R, DIR>::run(v);
  ex[(0 * R + j) * TILE] = v[0];
#pragma unroll
  for (int q = 1; q < R; ++q) ex[(q * R + j) * TILE] = ctw<DIR>(v[q], stw[2 * j * q]);
  __syncthreads();
#pragma unroll
  for (int q = 0; q < R; ++q) v[q] = ex[(j * R + q) * TILE];
  Dft<R, DIR>::run(v);
  if (DIR < 0) {
    if (ok) {
#pragma unroll
      for (int b = 0; b < R; ++b) out[(size_t)(2 * (j + R * b) + h) * a.xp] = v[b];
    }
  } else {
    // x[n] = g0[n] + conj(w_P^n) g1[n]; the two halves swap half of their rows so that both
    // thread groups store
    float2* sw = sm + (size_t)2 * H * TILE + kxl;
    if (h) {
#pragma unroll
      for (int b = 0; b < R; ++b) v[b] = cmulc(v[b], stw[j + R * b]);
#pragma unroll
      for (int b = 0; b < R / 2; ++b) sw[(j + R * b) * TILE] = v[b];
    } else {
#pragma unroll
      for (int b = R / 2; b < R; ++b) sw[(j + R * b) * TILE] = v[b];
    }
    __syncthreads();
    if (h) {
#pragma unroll
      for (int b = R / 2; b < R; ++b) {
        const int n = j + R * b;
        const float2 o = cadd(v[b], sw[n * TILE]);
        if (ok && n < a.n_out) out[(size_t)n * a.xp] = o;
      }
    } else {
#pragma unroll
      for (int b = 0; b < R / 2; ++b) {
        const int n = j + R * b;
        const float2 o = cadd(v[b], sw[n * TILE]);
        if (ok && n < a.n_out) out[(size_t)n * a.xp] = o;
      }
    }
  }
}

// Persistent variant: one CTA per SM walks over the tiles and loads the points of its next tile
// into registers before it transforms the current one, so that global loads are in flight
// during the whole kernel (the non-persistent CTAs above alternate between a load phase and a
// compute phase and leave HBM idle in between).
template <int R, int TILE, int DIR>
__global__ void __launch_bounds__(2 * R * TILE, 1) k_mid_colp(MidColArgs a) {
  constexpr int H = R * R, P = 2 * H, T = 2 * R * TILE;
  extern __shared__ float2 sm[];  // forward: [2][H][TILE]; inverse: [3][H][TILE]
  __shared__ float2 stw[P];
  if (a.gated && !a.ctrl->active) return;
  const int t = threadIdx.x;
  const int kxl = t % TILE, j = (t / TILE) % R, h = t / (TILE * R);
  const int ntm = a.ntile_main * a.nslab;
  const int nt = ntm + (a.nyq ? (a.nslab + TILE - 1) / TILE : 0);
  for (int q = t; q < P; q += T) stw[q] = a.tw[q];
  float2* ex = sm + (size_t)h * H * TILE + kxl;

  auto locate = [&](int tile, int& kx, int& slab) -> bool {
    bool ok;
    if (tile < ntm) {
      slab = tile / a.ntile_main; kx = (tile - slab * a.ntile_main) * TILE + kxl; ok = kx < a.xc_main;
    } else {
      kx = a.xc - 1; slab = (tile - ntm) * TILE + kxl; ok = slab < a.nslab;
    }
    if (!ok) { kx = 0; slab = 0; }
    return ok;
  };
  auto load = [&](int tile, float2* v) {
    int kx, slab;
    const bool ok = locate(tile, kx, slab);
    const float2* in = a.in + (size_t)slab * a.in_outer + kx;
#pragma unroll
    for (int u = 0; u < R; ++u) {
      const int n = DIR < 0 ? j + R * u : 2 * (j + R * u) + h;
      v[u] = (ok && n < a.n_in) ? in[(size_t)n * a.xp] : make_float2(0.f, 0.f);
    }
  };

  float2 nxt[R];
  int tile = blockIdx.x;
  if (tile < nt) load(tile, nxt);
  __syncthreads();  // stw
  for (; tile < nt; tile += gridDim.x) {
    float2 v[R];
#pragma unroll
    for (int u = 0; u < R; ++u) v[u] = nxt[u];
    if (tile + (int)gridDim.x < nt) load(tile + gridDim.x, nxt);
    int kx, slab;
    const bool ok = locate(tile, kx, slab);
    float2* out = a.out + (size_t)slab * a.out_outer + kx;
    if (DIR < 0 && h) {
#pragma unroll
      for (int u = 0; u < R; ++u) v[u] = cmul(v[u], stw[j + R * u]);
    }
    Dft<R, DIR>::run(v);
    ex[(0 * R + j) * TILE] = v[0];
#pragma unroll
    for (int q = 1; q < R; ++q) ex[(q * R + j) * TILE] = ctw<DIR>(v[q], stw[2 * j * q]);
    __syncthreads();
#pragma unroll
    for (int q = 0; q < R; ++q) v[q] = ex[(j * R + q) * TILE];
    Dft<R, DIR>::run(v);
    if (DIR < 0) {
      if (ok) {
#pragma unroll
        for (int b = 0; b < R; ++b) out[(size_t)(2 * (j + R * b) + h) * a.xp] = v[b];
      }
    } else {
      float2* sw = sm + (size_t)2 * H * TILE + kxl;
      if (h) {
#pragma unroll
        for (int b = 0; b < R; ++b) v[b] = cmulc(v[b], stw[j + R * b]);
#pragma unroll
        for (int b = 0; b < R / 2; ++b) sw[(j + R * b) * TILE] = v[b];
      } else {
#pragma unroll
        for (int b = R / 2; b < R; ++b) sw[(j + R * b) * TILE] = v[b];
      }
      __syncthreads();
      if (h) {
#pragma unroll
        for (int b = R / 2; b < R; ++b) {
          const int n = j + R * b;
          const float2 o = cadd(v[b], sw[n * TILE]);
          if (ok && n < a.n_out) out[(size_t)n * a.xp] = o;
        }
      } else {
#pragma unroll
        for (int b = 0; b < R / 2; ++b) {
          const int n = j + R * b;
          const float2 o = cadd(v[b], sw[n * TILE]);
          if (ok && n < a.n_out) out[(size_t)n * a.xp] = o;
        }
      }
    }
    __syncthreads();  // exchange tiles are rewritten by the next iteration
  }
}

template <typename Kern>
int set_smem_col(Kern k, size_t bytes) {
  if (bytes > 48 * 1024) MMX_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
  return MMX_OK;
}

}  // namespace

// ---- launchers (called by mmx_demag_launch when the shapes fit) ---------------------------------

bool mmx_inner_col_ok(const DemagPlan& d, int P, int n_valid) {
  (void)d;
  return P == 128 && n_valid <= 64;
}

int mmx_inner_col_launch(mmx_world* w, const InnerColLaunch& L) {
  const DemagPlan& d = w->dm;
  InnerColArgs a;
  a.spec = L.spec; a.khat = d.khat; a.tw = L.tw; a.ctrl = w->d_ctrl; a.gated = 1;
  a.n_valid = L.n_valid; a.xc = d.xc; a.p_outer = L.p_outer;
  a.nyq = ((d.xc - 1) % 32 == 0 && d.xc > 1 && L.n_outer >= 32) ? 1 : 0;
  if (a.nyq) { a.ntile_main = (d.xc - 1) / 32; a.xc_main = d.xc - 1; }
  else { a.ntile_main = (d.xc + 31) / 32; a.xc_main = d.xc; }
  a.line_stride = L.line_stride; a.comp_stride = L.comp_stride; a.outer_stride = L.outer_stride;
  a.k_inner_stride = L.k_inner_stride; a.k_outer_stride = L.k_outer_stride; a.k_comp_stride = L.k_comp_stride;
  a.odd_inner = L.odd_inner; a.odd_outer = L.odd_outer;
  const size_t smem = sizeof(float2) * 6 * 64 * 32;
  if (int rc = set_smem_col(k_inner_col<8>, smem)) return rc;
  dim3 g(a.ntile_main + a.nyq, L.n_outer);
  ProfScope ps(w, PK_INNER);
  k_inner_col<8><<<g, 256, smem, w->stream>>>(a);
  return MMX_OK;
}

bool mmx_mid_col_ok(int P, int n) { return (P == 512 || P == 128 || P == 32) && 2 * n <= P; }

template <int R, int TILE>
static int mid_col_launch_t(mmx_world* w, MidColArgs& a, int dir) {
  a.nyq = ((a.xc - 1) % TILE == 0 && a.xc > 1 && a.nslab >= TILE) ? 1 : 0;
  if (a.nyq) { a.ntile_main = (a.xc - 1) / TILE; a.xc_main = a.xc - 1; }
  else { a.ntile_main = (a.xc + TILE - 1) / TILE; a.xc_main = a.xc; }
  dim3 g(a.ntile_main + a.nyq, a.nslab);
  const size_t smem = sizeof(float2) * (dir < 0 ? 2 : 3) * R * R * TILE;
  ProfScope ps(w, dir < 0 ? PK_MID_FWD : PK_MID_INV);
  const int ntiles = a.ntile_main * a.nslab + (a.nyq ? (a.nslab + TILE - 1) / TILE : 0);
  if (MMX_MID_PERSISTENT && ntiles >= 4 * w->sm_count) {
    if (dir < 0) {
      if (int rc = set_smem_col(k_mid_colp<R, TILE, -1>, smem)) return rc;
      k_mid_colp<R, TILE, -1><<<w->sm_count, 2 * R * TILE, smem, w->stream>>>(a);
    } else {
      if (int rc = set_smem_col(k_mid_colp<R, TILE, +1>, smem)) return rc;
      k_mid_colp<R, TILE, +1><<<w->sm_count, 2 * R * TILE, smem, w->stream>>>(a);
    }
    return MMX_OK;
  }
  if (dir < 0) {
    if (int rc = set_smem_col(k_mid_col<R, TILE, -1>, smem)) return rc;
    k_mid_col<R, TILE, -1><<<g, 2 * R * TILE, smem, w->stream>>>(a);
  } else {
    if (int rc = set_smem_col(k_mid_col<R, TILE, +1>, smem)) return rc;
    k_mid_col<R, TILE, +1><<<g, 2 * R * TILE, smem, w->stream>>>(a);
  }
  return MMX_OK;
}

int mmx_mid_col_launch(mmx_world* w, int P, int dir, const float2* in, float2* out, int n_in, int n_out,
                       size_t in_outer, size_t out_outer, int nslab, const float2* tw) {
  const DemagPlan& d = w->dm;
  MidColArgs a;
  a.in = in; a.out = out; a.tw = tw; a.ctrl = w->d_ctrl; a.gated = 1;
  a.n_in = n_in; a.n_out = n_out; a.xc = d.xc; a.xp = d.xp; a.nslab = nslab;
  a.in_outer = in_outer; a.out_outer = out_outer;
  switch (P) {
    case 512: return mid_col_launch_t<16, 16>(w, a, dir);
    case 128: return mid_col_launch_t<8, 32>(w, a, dir);
    case 32: return mid_col_launch_t<4, 32>(w, a, dir);
  }
  return mmx_fail(MMX_EINVAL, "mid column pass: unsupported length %d", P);
}
