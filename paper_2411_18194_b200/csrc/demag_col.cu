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
#define MMX_PACKED_R16 0   // measured on c4: y passes 68.0 / 80.8 us packed, 66.1 / 78.4 us scalar
#include "fft_reg.cuh"
#include "mmx_internal.h"

using namespace mmxreg;

#ifndef MMX_MID_PERSISTENT
#define MMX_MID_PERSISTENT 1
#endif
#ifndef MMX_INNER_TL
#define MMX_INNER_TL 16       // columns per CTA of variant P (16: two 256-thread CTAs per SM, 207 us on c4; 8: four of 128, 272 us)
#endif
#ifndef MMX_MID_PIPE
#define MMX_MID_PIPE 1        // 1: pipelined y pass (cp.async stages) for 512-point lines on large grids
#endif
#ifndef MMX_INNER_VARIANT
#define MMX_INNER_VARIANT 3   // 3: variant Q (kernel rows staged in shared memory, twiddles in registers: 170 us on c4); 2: variant P (persistent, cp.async pipeline, kernel values in registers: 207 us); 0: 32-column tiles (persistent when large), 1: variant W (16 columns, halves in one warp)
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

// Persistent form of k_inner_col: 2 CTAs per SM walk over the (ky, kx-tile) list; before a CTA
// transforms a tile it asks L2 for the rows of its next tile (prefetch.global.L2: no registers,
// no shared memory), so HBM keeps streaming while the SM computes and the loads of the next
// iteration are L2 hits.  Tile order: ky and Py - ky are neighbours (same kernel rows).
template <int R>
__global__ void __launch_bounds__(32 * R, 2) k_inner_colp(InnerColArgs a) {
  constexpr int H = R * R, P = 2 * H;
  extern __shared__ float2 sm[];  // [6][H][32]
  __shared__ float2 stw[P];
  if (a.gated && !a.ctrl->active) return;
  const int lane = threadIdx.x & 31, j = threadIdx.x >> 5;
  for (int q = threadIdx.x; q < P; q += 32 * R) stw[q] = a.tw[q];
  const int ntm = a.ntile_main * a.p_outer;
  const int nt = ntm + (a.nyq ? (a.p_outer + 31) / 32 : 0);

  auto locate = [&](int tile, int& kx, int& ko, bool& main_tile) -> bool {
    bool ok;
    main_tile = tile < ntm;
    if (main_tile) {
      const int yy = tile / a.ntile_main;
      ko = (yy & 1) ? a.p_outer - ((yy + 1) >> 1) : (yy >> 1);
      kx = (tile - yy * a.ntile_main) * 32 + lane; ok = kx < a.xc_main;
    } else {
      kx = a.xc - 1; ko = (tile - ntm) * 32 + lane; ok = ko < a.p_outer;
    }
    if (!ok) { kx = 0; ko = 0; }
    return ok;
  };
  auto prefetch_tile = [&](int tile) {
    if (tile >= ntm) return;  // Nyquist tiles are scattered and tiny
    int kx, ko; bool mt;
    locate(tile, kx, ko, mt);
    const int kx0 = kx - lane;
    const int kom = (2 * ko > a.p_outer) ? a.p_outer - ko : ko;
    // spectrum rows: 3 components x n_valid rows x 256 B (two 128 B lines each)
    for (int r = threadIdx.x; r < 3 * a.n_valid * 2; r += 32 * R) {
      const int c = r / (2 * a.n_valid), rem = r - c * 2 * a.n_valid;
      const int n = rem >> 1, hl = rem & 1;
      prefetch_l2(a.spec + (size_t)ko * a.outer_stride + (size_t)c * a.comp_stride + (size_t)n * a.line_stride + kx0 + hl * 16);
    }
    for (int r = threadIdx.x; r < 6 * (H + 1); r += 32 * R) {
      const int c = r / (H + 1), pm = r - c * (H + 1);
      const float* p = a.khat + (size_t)kom * a.k_outer_stride + kx0 + (size_t)pm * a.k_inner_stride + (size_t)c * a.k_comp_stride;
      prefetch_l2(p);
      prefetch_l2(p + 31);
    }
  };

  int tile = blockIdx.x;
  if (tile < nt) prefetch_tile(tile);
  __syncthreads();  // stw
  for (; tile < nt; tile += gridDim.x) {
    if (tile + (int)gridDim.x < nt) prefetch_tile(tile + gridDim.x);
    int kx, ko; bool main_tile;
    const bool ok = locate(tile, kx, ko, main_tile);
    int kom = ko, so = 0;
    if (a.p_outer > 1 && 2 * ko > a.p_outer) { kom = a.p_outer - ko; so = 1; }
    const float* kb = a.khat + (size_t)kom * a.k_outer_stride + kx;
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
    // sign masks of the odd components: xy is odd along the outer axis, xz along the inner one,
    // yz along both (3-D); the 2-D caller passes its own odd_inner / odd_outer
    const unsigned mo3 = (so & (a.odd_outer >> 3)) << 31, mo4 = (so & (a.odd_outer >> 4)) << 31, mo5 = (so & (a.odd_outer >> 5)) << 31;
    const unsigned mi3 = ((a.odd_inner >> 3) & 1u) << 31, mi4 = ((a.odd_inner >> 4) & 1u) << 31, mi5 = ((a.odd_inner >> 5) & 1u) << 31;
#pragma unroll
    for (int h = 0; h < 2; ++h)
#pragma unroll
      for (int b = 0; b < R; ++b) {
        const int kz = 2 * (j + R * b) + h;
        const bool mir = 2 * kz > P;
        const int pm = mir ? P - kz : kz;
        const float* kp = kb + (size_t)pm * a.k_inner_stride;
        float K[6];
#pragma unroll
        for (int c = 0; c < 6; ++c) K[c] = __ldg(kp + (size_t)c * a.k_comp_stride);
        K[3] = __uint_as_float(__float_as_uint(K[3]) ^ mo3 ^ (mir ? mi3 : 0u));
        K[4] = __uint_as_float(__float_as_uint(K[4]) ^ mo4 ^ (mir ? mi4 : 0u));
        K[5] = __uint_as_float(__float_as_uint(K[5]) ^ mo5 ^ (mir ? mi5 : 0u));
        const float2 mx = X[0][h][b], my = X[1][h][b], mz = X[2][h][b];
        X[0][h][b] = make_float2(fmaf(K[0], mx.x, fmaf(K[3], my.x, K[4] * mz.x)),
                                 fmaf(K[0], mx.y, fmaf(K[3], my.y, K[4] * mz.y)));
        X[1][h][b] = make_float2(fmaf(K[3], mx.x, fmaf(K[1], my.x, K[5] * mz.x)),
                                 fmaf(K[3], mx.y, fmaf(K[1], my.y, K[5] * mz.y)));
        X[2][h][b] = make_float2(fmaf(K[4], mx.x, fmaf(K[5], my.x, K[2] * mz.x)),
                                 fmaf(K[4], mx.y, fmaf(K[5], my.y, K[2] * mz.y)));
      }
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
    __syncthreads();  // the exchange tiles are rewritten by the next iteration
  }
}

// Variant W of the fused inner pass: 16 kx columns per CTA, lane = column + 16 h, so that the
// two halves of a line sit in the same warp (their inputs are one load, their results meet by
// shuffle) and a thread carries one half of three components (48 data registers): three CTAs
// per SM instead of two.  The kernel-spectrum rows of the CTA (6 x (H+1) x 16 floats) are
// copied to shared memory with cp.async at the start and waited for only before the multiply.
__device__ __forceinline__ void cpa16(void* smem, const void* gmem) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gmem) : "memory");
}

#ifndef MMX_INW_MINB
#define MMX_INW_MINB 3
#endif
template <int R>
__global__ void __launch_bounds__(32 * R, MMX_INW_MINB) k_inner_w(InnerColArgs a) {
  constexpr int H = R * R, P = 2 * H, TL = 16;
  extern __shared__ __align__(16) unsigned char smraw[];
  float2* sm = reinterpret_cast<float2*>(smraw);                          // [3][2][H][TL]
  float* ks = reinterpret_cast<float*>(smraw + sizeof(float2) * 6 * H * TL);  // [6][H+1][TL]
  __shared__ float2 stw[P];
  if (a.gated && !a.ctrl->active) return;
  const int lane = threadIdx.x & 31, j = threadIdx.x >> 5;
  const int kxl = lane & 15, h = lane >> 4;
  // blockIdx.y -> outer wave number: ky and p_outer - ky are neighbours in launch order (they
  // read the same kernel rows, the second read hits L2)
  int yy = blockIdx.y;
  int kx, ko;
  bool ok;
  const bool main_tile = (int)blockIdx.x < a.ntile_main;
  if (main_tile) {
    ko = (yy & 1) ? a.p_outer - ((yy + 1) >> 1) : (yy >> 1);
    kx = blockIdx.x * TL + kxl; ok = kx < a.xc_main;
  } else {
    if (yy * TL >= a.p_outer) return;
    kx = a.xc - 1; ko = yy * TL + kxl; ok = ko < a.p_outer;
  }
  if (!ok) { kx = 0; ko = 0; }
  for (int q = threadIdx.x; q < P; q += 32 * R) stw[q] = a.tw[q];
  int kom = ko, so = 0;
  if (a.p_outer > 1 && 2 * ko > a.p_outer) { kom = a.p_outer - ko; so = 1; }
  if (main_tile) {
    const float* kt = a.khat + (size_t)kom * a.k_outer_stride + (size_t)blockIdx.x * TL;
    for (int r = threadIdx.x; r < 6 * (H + 1) * (TL / 4); r += 32 * R) {
      const int row = r / (TL / 4), ch = r % (TL / 4);
      const int c = row / (H + 1), pm = row % (H + 1);
      cpa16(ks + (size_t)row * TL + 4 * ch, kt + (size_t)c * a.k_comp_stride + (size_t)pm * a.k_inner_stride + 4 * ch);
    }
  }
  asm volatile("cp.async.commit_group;" ::: "memory");

  float2* base = a.spec + (size_t)ko * a.outer_stride + kx;
  float2 X[3][R];
#pragma unroll
  for (int c = 0; c < 3; ++c)
#pragma unroll
    for (int u = 0; u < R; ++u) {
      const int n = j + R * u;
      X[c][u] = (ok && n < a.n_valid) ? base[(size_t)c * a.comp_stride + (size_t)n * a.line_stride]
                                      : make_float2(0.f, 0.f);
    }
  __syncthreads();  // stw
  // forward stage 1 of this thread's half
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    if (h) {
#pragma unroll
      for (int u = 0; u < R; ++u) X[c][u] = cmul(X[c][u], stw[j + R * u]);
    }
    Dft<R, -1>::run(X[c]);
    float2* t = sm + (size_t)(c * 2 + h) * H * TL + kxl;
    t[(0 * R + j) * TL] = X[c][0];
#pragma unroll
    for (int q = 1; q < R; ++q) t[(q * R + j) * TL] = cmul(X[c][q], stw[2 * j * q]);
  }
  __syncthreads();
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const float2* t = sm + (size_t)(c * 2 + h) * H * TL + kxl;
#pragma unroll
    for (int q = 0; q < R; ++q) X[c][q] = t[(j * R + q) * TL];
    Dft<R, -1>::run(X[c]);
  }
  // B^_i = sum_j K^_ij M^_j ; K^ real, 6 unique components, octant + parity
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  __syncthreads();  // kernel rows of all threads have landed
  const float* kb = a.khat + (size_t)kom * a.k_outer_stride + kx;
#pragma unroll
  for (int b = 0; b < R; ++b) {
    const int kz = 2 * (j + R * b) + h;
    int pm = kz, si = 0;
    if (2 * kz > P) { pm = P - kz; si = 1; }
    float K[6];
#pragma unroll
    for (int c = 0; c < 6; ++c) {
      const float v = main_tile ? ks[((size_t)c * (H + 1) + pm) * TL + kxl]
                                : __ldg(kb + (size_t)pm * a.k_inner_stride + (size_t)c * a.k_comp_stride);
      const int flip = (si & (a.odd_inner >> c)) ^ (so & (a.odd_outer >> c));
      K[c] = (flip & 1) ? -v : v;
    }
    const float2 mx = X[0][b], my = X[1][b], mz = X[2][b];
    X[0][b] = make_float2(fmaf(K[0], mx.x, fmaf(K[3], my.x, K[4] * mz.x)),
                          fmaf(K[0], mx.y, fmaf(K[3], my.y, K[4] * mz.y)));
    X[1][b] = make_float2(fmaf(K[3], mx.x, fmaf(K[1], my.x, K[5] * mz.x)),
                          fmaf(K[3], mx.y, fmaf(K[1], my.y, K[5] * mz.y)));
    X[2][b] = make_float2(fmaf(K[4], mx.x, fmaf(K[5], my.x, K[2] * mz.x)),
                          fmaf(K[4], mx.y, fmaf(K[5], my.y, K[2] * mz.y)));
  }
  // inverse stage 1 (over b); the thread writes the rows it has read: no barrier needed
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    Dft<R, +1>::run(X[c]);
    float2* t = sm + (size_t)(c * 2 + h) * H * TL + kxl;
    t[(j * R + 0) * TL] = X[c][0];
#pragma unroll
    for (int q = 1; q < R; ++q) t[(j * R + q) * TL] = cmulc(X[c][q], stw[2 * j * q]);
  }
  __syncthreads();
  // inverse stage 2, then x[n] = g0[n] + conj(w_P^n) g1[n]: lanes h = 0 finish rows b < R/2,
  // lanes h = 1 rows b >= R/2, the other half's value arrives by shuffle
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const float2* t = sm + (size_t)(c * 2 + h) * H * TL + kxl;
#pragma unroll
    for (int q = 0; q < R; ++q) X[c][q] = t[(q * R + j) * TL];
    Dft<R, +1>::run(X[c]);
    if (h) {
#pragma unroll
      for (int b = 0; b < R; ++b) X[c][b] = cmulc(X[c][b], stw[j + R * b]);
    }
#pragma unroll
    for (int bb = 0; bb < R / 2; ++bb) {
      const float2 mine = h ? X[c][bb + R / 2] : X[c][bb];
      const float2 send = h ? X[c][bb] : X[c][bb + R / 2];
      float2 recv;
      recv.x = __shfl_xor_sync(0xffffffffu, send.x, 16);
      recv.y = __shfl_xor_sync(0xffffffffu, send.y, 16);
      const int n = j + R * (h ? bb + R / 2 : bb);
      if (ok && n < a.n_valid)
        base[(size_t)c * a.comp_stride + (size_t)n * a.line_stride] = cadd(mine, recv);
    }
  }
}

// Variant P of the fused inner pass: the thread mapping of variant W (16 columns, lane =
// column + 16 h) in a persistent CTA with a two-stage cp.async pipeline.  While a CTA transforms
// tile i out of one shared-memory stage, the rows of tile i+1 stream into the other, and the
// kernel-spectrum values of tile i (48 per thread) are loaded into registers at the top of the
// iteration, long before the multiply: no phase of the CTA waits for HBM.
template <int BYTES>
__device__ __forceinline__ void cpa_zfill(void* smem, const void* gmem, bool valid) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
  const int n = valid ? BYTES : 0;
  if (BYTES == 16)
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(sa), "l"(gmem), "r"(n) : "memory");
  else
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(sa), "l"(gmem), "r"(n) : "memory");
}

template <int R, int TL>
__global__ void __launch_bounds__(2 * TL * R, 32 / TL) k_inner_pipe(InnerColArgs a) {
  constexpr int H = R * R, P = 2 * H, NT = 2 * TL * R;
  constexpr int EXT = H * TL + (TL < 16 ? 8 : 0);  // one exchange tile (+8: the halves of a 64-bit wavefront use different banks)
  extern __shared__ __align__(16) unsigned char smraw[];
  float2* sm = reinterpret_cast<float2*>(smraw);             // exchange [3][2][H][TL]
  float2* stage = sm + (size_t)6 * EXT;                      // input stages [2][3][H][TL]
  __shared__ float2 stw[P];
  if (a.gated && !a.ctrl->active) return;
  // lane = column + TL h (+ 2 TL (j % (16 / TL)) when TL < 16)
  const int lane = threadIdx.x & 31;
  const int kxl = lane % TL, h = (lane / TL) & 1, j = (threadIdx.x >> 5) * (16 / TL) + lane / (2 * TL);
  for (int q = threadIdx.x; q < P; q += NT) stw[q] = a.tw[q];
  const int ntm = a.ntile_main * a.p_outer;
  const int nt = ntm + (a.nyq ? (a.p_outer + TL - 1) / TL : 0);

  // tile -> first column / outer index of lane l
  auto tile_ko = [&](int tile) -> int {
    const int yy = tile / a.ntile_main;
    return (yy & 1) ? a.p_outer - ((yy + 1) >> 1) : (yy >> 1);
  };
  auto issue = [&](int tile, int buf) {
    float2* dst = stage + (size_t)buf * 3 * H * TL;
    if (tile < ntm) {
      const int yy = tile / a.ntile_main;
      const int ko = (yy & 1) ? a.p_outer - ((yy + 1) >> 1) : (yy >> 1);
      const int kx0 = (tile - yy * a.ntile_main) * TL;
      const float2* src = a.spec + (size_t)ko * a.outer_stride + kx0;
      // 3 H rows of TL float2 = 8 chunks of 16 B each; thread t always copies chunk t % 8 of rows
      // t / 8 + (NT / 8) i: the source offsets are two row offsets x three components
      constexpr int RPI = NT / (TL / 2);  // rows per sweep of the CTA
      const int ch = threadIdx.x % (TL / 2), r0 = threadIdx.x / (TL / 2);
#pragma unroll
      for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int i = 0; i < H / RPI; ++i) {
          const int n = r0 + RPI * i;
          cpa_zfill<16>(dst + (c * H + n) * TL + 2 * ch,
                        src + (size_t)c * a.comp_stride + (size_t)n * a.line_stride + 2 * ch, n < a.n_valid);
        }
    } else {
      const int ko0 = (tile - ntm) * TL;
      for (int q = threadIdx.x; q < 3 * H * TL; q += NT) {
        const int row = q / TL, l = q % TL;
        const int c = row / H, n = row % H;
        const bool v = n < a.n_valid && ko0 + l < a.p_outer;
        const int ko = v ? ko0 + l : 0;
        cpa_zfill<8>(dst + (size_t)row * TL + l,
                     a.spec + (size_t)ko * a.outer_stride + (a.xc - 1) + (size_t)c * a.comp_stride + (size_t)n * a.line_stride, v);
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };

  int tile = blockIdx.x;
  if (tile < nt) issue(tile, 0);
#ifdef MMX_INNER_STAGGER_NS
  // the CTAs that share an SM would otherwise run the same phase (butterflies / exchange) at the same
  // time for the whole kernel; delay the second wave by about half a tile
  if (blockIdx.x >= gridDim.x / 2) __nanosleep(MMX_INNER_STAGGER_NS);
#endif
  int buf = 0;
  for (; tile < nt; tile += gridDim.x, buf ^= 1) {
    const int nxt = tile + gridDim.x;
    if (nxt < nt) issue(nxt, buf ^ 1);
    // where this thread's column lives
    int kx, ko;
    bool ok = true;
    const bool main_tile = tile < ntm;
    if (main_tile) {
      ko = tile_ko(tile);
      kx = (tile - (tile / a.ntile_main) * a.ntile_main) * TL + kxl;
      ok = kx < a.xc_main;  // (columns up to the row pitch exist: reads are safe, stores are masked)
    } else {
      kx = a.xc - 1; ko = (tile - ntm) * TL + kxl; ok = ko < a.p_outer;
      if (!ok) ko = 0;
    }
    int kom = ko, so = 0;
    if (a.p_outer > 1 && 2 * ko > a.p_outer) { kom = a.p_outer - ko; so = 1; }
    // kernel spectrum of this thread's 8 wave numbers: issued now, used after the forward transform
    // (32-bit element offsets from the uniform base pointer: the launcher checks that they fit)
    const unsigned kis = (unsigned)a.k_inner_stride, kcs = (unsigned)a.k_comp_stride;
    const unsigned koff = (unsigned)kom * (unsigned)a.k_outer_stride + (unsigned)kx;
    float K[R][6];
#pragma unroll
    for (int b = 0; b < R; ++b) {
      const int kz = 2 * (j + R * b) + h;
      const unsigned pm = 2 * kz > P ? P - kz : kz;
      const unsigned o = koff + pm * kis;
#pragma unroll
      for (int c = 0; c < 6; ++c) K[b][c] = __ldg(a.khat + (o + c * kcs));
    }
    if (nxt < nt) asm volatile("cp.async.wait_group 1;" ::: "memory");
    else asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();  // tile i has landed for every thread; exchange tiles of tile i-1 are free
    const float2* xin = stage + (size_t)buf * 3 * H * TL + kxl;
    float2 X[3][R];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
#pragma unroll
      for (int u = 0; u < R; ++u) {
        const float2 w = h ? stw[j + R * u] : make_float2(1.f, 0.f);  // (both halves share a warp: no branch)
        X[c][u] = cmul(xin[(c * H + j + R * u) * TL], w);
      }
      Dft<R, -1>::run(X[c]);
      float2* t = sm + (c * 2 + h) * EXT + kxl;
      t[(0 * R + j) * TL] = X[c][0];
#pragma unroll
      for (int q = 1; q < R; ++q) t[(q * R + j) * TL] = cmul(X[c][q], stw[2 * j * q]);
    }
    __syncthreads();
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const float2* t = sm + (c * 2 + h) * EXT + kxl;
#pragma unroll
      for (int q = 0; q < R; ++q) X[c][q] = t[(j * R + q) * TL];
      Dft<R, -1>::run(X[c]);
    }
    // B^_i = sum_j K^_ij M^_j ; K^ real, octant + parity (sign bit flips)
    const unsigned mo3 = (so & (a.odd_outer >> 3)) << 31, mo4 = (so & (a.odd_outer >> 4)) << 31, mo5 = (so & (a.odd_outer >> 5)) << 31;
    const unsigned mi3 = ((a.odd_inner >> 3) & 1u) << 31, mi4 = ((a.odd_inner >> 4) & 1u) << 31, mi5 = ((a.odd_inner >> 5) & 1u) << 31;
#pragma unroll
    for (int b = 0; b < R; ++b) {
      const bool mir = 2 * (2 * (j + R * b) + h) > P;
      const float k0 = K[b][0], k1 = K[b][1], k2 = K[b][2];
      const float k3 = __uint_as_float(__float_as_uint(K[b][3]) ^ mo3 ^ (mir ? mi3 : 0u));
      const float k4 = __uint_as_float(__float_as_uint(K[b][4]) ^ mo4 ^ (mir ? mi4 : 0u));
      const float k5 = __uint_as_float(__float_as_uint(K[b][5]) ^ mo5 ^ (mir ? mi5 : 0u));
      const float2 mx = X[0][b], my = X[1][b], mz = X[2][b];
      X[0][b] = make_float2(fmaf(k0, mx.x, fmaf(k3, my.x, k4 * mz.x)), fmaf(k0, mx.y, fmaf(k3, my.y, k4 * mz.y)));
      X[1][b] = make_float2(fmaf(k3, mx.x, fmaf(k1, my.x, k5 * mz.x)), fmaf(k3, mx.y, fmaf(k1, my.y, k5 * mz.y)));
      X[2][b] = make_float2(fmaf(k4, mx.x, fmaf(k5, my.x, k2 * mz.x)), fmaf(k4, mx.y, fmaf(k5, my.y, k2 * mz.y)));
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      Dft<R, +1>::run(X[c]);
      float2* t = sm + (c * 2 + h) * EXT + kxl;
      t[(j * R + 0) * TL] = X[c][0];
#pragma unroll
      for (int q = 1; q < R; ++q) t[(j * R + q) * TL] = cmulc(X[c][q], stw[2 * j * q]);
    }
    __syncthreads();
    const unsigned soff = (unsigned)ko * (unsigned)a.outer_stride + (unsigned)kx;
    const unsigned sls = (unsigned)a.line_stride, scs = (unsigned)a.comp_stride;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const float2* t = sm + (c * 2 + h) * EXT + kxl;
#pragma unroll
      for (int q = 0; q < R; ++q) X[c][q] = t[(q * R + j) * TL];
      Dft<R, +1>::run(X[c]);
#pragma unroll
      for (int b = 0; b < R; ++b) {
        const float2 w = h ? stw[j + R * b] : make_float2(1.f, 0.f);
        X[c][b] = cmulc(X[c][b], w);
      }
#pragma unroll
      for (int bb = 0; bb < R / 2; ++bb) {
        const float2 mine = h ? X[c][bb + R / 2] : X[c][bb];
        const float2 send = h ? X[c][bb] : X[c][bb + R / 2];
        float2 recv;
        recv.x = __shfl_xor_sync(0xffffffffu, send.x, TL);
        recv.y = __shfl_xor_sync(0xffffffffu, send.y, TL);
        const int n = j + R * (h ? bb + R / 2 : bb);
        if (ok && n < a.n_valid) a.spec[soff + c * scs + (unsigned)n * sls] = cadd(mine, recv);
      }
    }
  }
}

// Variant Q of the fused inner pass: as variant P, but the kernel-spectrum rows of a tile are staged
// in shared memory by cp.async (one tile ahead) instead of being held in 48 registers, and the
// registers freed hold the 15 twiddles of the thread for the whole kernel (no per-component reloads,
// no selects).  One spectrum stage (refilled as soon as the tile has been read) + one kernel stage.
template <int R>
__global__ void __launch_bounds__(32 * R, 2) k_inner_q(InnerColArgs a) {
  constexpr int H = R * R, P = 2 * H, TL = 16, NT = 32 * R, EXT = H * TL;
  extern __shared__ __align__(16) unsigned char smraw[];
  float2* sm = reinterpret_cast<float2*>(smraw);             // exchange [3][2][H][TL]
  float2* xst = sm + 6 * EXT;                                // spectrum stage [3][H][TL]
  float* kst = reinterpret_cast<float*>(xst + 3 * H * TL);   // kernel stage [6][H+1][TL]
  const int lane = threadIdx.x & 31, j = threadIdx.x >> 5;
  const int kxl = lane & 15, h = lane >> 4;
  const int ntm = a.ntile_main * a.p_outer;
  const int nt = ntm + (a.nyq ? (a.p_outer + TL - 1) / TL : 0);
  // twiddles of this thread: stage w_H^(j q), half w_P^(j + R u) (identity for the even half)
  float2 tws[R], twp[R];
#pragma unroll
  for (int q = 0; q < R; ++q) {
    tws[q] = a.tw[2 * j * q];
    twp[q] = h ? a.tw[j + R * q] : make_float2(1.f, 0.f);
  }

  pdl_wait();      // the twiddle loads above do not depend on the previous kernel
  pdl_trigger();   // persistent kernel: the next kernel's CTAs take over as ours exit
  if (a.gated && !a.ctrl->active) return;

  auto tile_ko = [&](int tile) -> int {
    const int yy = tile / a.ntile_main;
    return (yy & 1) ? a.p_outer - ((yy + 1) >> 1) : (yy >> 1);
  };
  auto issue_x = [&](int tile) {
    if (tile < ntm) {
      const int ko = tile_ko(tile);
      const int kx0 = (tile - (tile / a.ntile_main) * a.ntile_main) * TL;
      constexpr int RPI = NT / (TL / 2);
      const unsigned ch = threadIdx.x % (TL / 2), r0 = threadIdx.x / (TL / 2);
      const unsigned so = (unsigned)ko * (unsigned)a.outer_stride + (unsigned)kx0 + r0 * (unsigned)a.line_stride + 2 * ch;
#pragma unroll
      for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int i = 0; i < H / RPI; ++i) {
          const int n = r0 + RPI * i;
          cpa_zfill<16>(xst + (c * H + n) * TL + 2 * ch,
                        a.spec + (so + (unsigned)c * (unsigned)a.comp_stride + (unsigned)(RPI * i) * (unsigned)a.line_stride),
                        n < a.n_valid);
        }
    } else {
      const int ko0 = (tile - ntm) * TL;
      for (int q = threadIdx.x; q < 3 * H * TL; q += NT) {
        const int row = q / TL, l = q % TL;
        const int c = row / H, n = row % H;
        const bool v = n < a.n_valid && ko0 + l < a.p_outer;
        const int ko = v ? ko0 + l : 0;
        cpa_zfill<8>(xst + row * TL + l,
                     a.spec + (size_t)ko * a.outer_stride + (a.xc - 1) + (size_t)c * a.comp_stride + (size_t)n * a.line_stride, v);
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  auto issue_k = [&](int tile) {
    if (tile < ntm) {
      const int ko = tile_ko(tile);
      const int kom = (a.p_outer > 1 && 2 * ko > a.p_outer) ? a.p_outer - ko : ko;
      const int kx0 = (tile - (tile / a.ntile_main) * a.ntile_main) * TL;
      const unsigned kb = (unsigned)kom * (unsigned)a.k_outer_stride + (unsigned)kx0;
      for (int q = threadIdx.x; q < 6 * (H + 1) * (TL / 4); q += NT) {
        const int row = q / (TL / 4), ch = q % (TL / 4);
        const int c = row / (H + 1), pm = row - c * (H + 1);
        const unsigned sa = (unsigned)__cvta_generic_to_shared(kst + row * TL + 4 * ch);
        const float* g = a.khat + (kb + (unsigned)c * (unsigned)a.k_comp_stride + (unsigned)pm * (unsigned)a.k_inner_stride + 4 * ch);
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(g) : "memory");
      }
    } else {
      const int ko0 = (tile - ntm) * TL;
      for (int q = threadIdx.x; q < 6 * (H + 1) * TL; q += NT) {
        const int row = q / TL, l = q % TL;
        const int c = row / (H + 1), pm = row - c * (H + 1);
        const bool v = ko0 + l < a.p_outer;
        const int ko = v ? ko0 + l : 0;
        const int kom = (a.p_outer > 1 && 2 * ko > a.p_outer) ? a.p_outer - ko : ko;
        const unsigned sa = (unsigned)__cvta_generic_to_shared(kst + row * TL + l);
        const float* g = a.khat + (size_t)kom * a.k_outer_stride + (a.xc - 1) + (size_t)c * a.k_comp_stride + (size_t)pm * a.k_inner_stride;
        asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(sa), "l"(g) : "memory");
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };

  int tile = blockIdx.x;
  if (tile < nt) { issue_x(tile); issue_k(tile); }
  for (; tile < nt; tile += gridDim.x) {
    const int nxt = tile + gridDim.x;
    int kx, ko;
    bool ok = true;
    if (tile < ntm) {
      ko = tile_ko(tile);
      kx = (tile - (tile / a.ntile_main) * a.ntile_main) * TL + kxl;
      ok = kx < a.xc_main;
    } else {
      kx = a.xc - 1; ko = (tile - ntm) * TL + kxl; ok = ko < a.p_outer;
      if (!ok) ko = 0;
    }
    const int so = (a.p_outer > 1 && 2 * ko > a.p_outer) ? 1 : 0;
    asm volatile("cp.async.wait_group 1;" ::: "memory");  // the spectrum stage (the kernel stage may still fly)
    __syncthreads();  // tile has landed for every thread; exchange tiles of the previous tile are free
    float2 X[3][R];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
#pragma unroll
      for (int u = 0; u < R; ++u) X[c][u] = cmul(xst[(c * H + j + R * u) * TL + kxl], twp[u]);
      Dft<R, -1>::run(X[c]);
      float2* t = sm + (c * 2 + h) * EXT + kxl;
      t[(0 * R + j) * TL] = X[c][0];
#pragma unroll
      for (int q = 1; q < R; ++q) t[(q * R + j) * TL] = cmul(X[c][q], tws[q]);
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");  // kernel stage of this tile
    __syncthreads();
    if (nxt < nt) issue_x(nxt);  // the spectrum stage has been read by everyone
    else asm volatile("cp.async.commit_group;" ::: "memory");
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const float2* t = sm + (c * 2 + h) * EXT + kxl;
#pragma unroll
      for (int q = 0; q < R; ++q) X[c][q] = t[(j * R + q) * TL];
      Dft<R, -1>::run(X[c]);
    }
    // B^_i = sum_j K^_ij M^_j ; K^ real, octant + parity (sign bit flips)
    const unsigned mo3 = (so & (a.odd_outer >> 3)) << 31, mo4 = (so & (a.odd_outer >> 4)) << 31, mo5 = (so & (a.odd_outer >> 5)) << 31;
    const unsigned mi3 = ((a.odd_inner >> 3) & 1u) << 31, mi4 = ((a.odd_inner >> 4) & 1u) << 31, mi5 = ((a.odd_inner >> 5) & 1u) << 31;
#pragma unroll
    for (int b = 0; b < R; ++b) {
      const int kz = 2 * (j + R * b) + h;
      const bool mir = 2 * kz > P;
      const int pm = mir ? P - kz : kz;
      const float* kp = kst + pm * TL + kxl;
      const float k0 = kp[0 * (H + 1) * TL], k1 = kp[1 * (H + 1) * TL], k2 = kp[2 * (H + 1) * TL];
      const float k3 = __uint_as_float(__float_as_uint(kp[3 * (H + 1) * TL]) ^ mo3 ^ (mir ? mi3 : 0u));
      const float k4 = __uint_as_float(__float_as_uint(kp[4 * (H + 1) * TL]) ^ mo4 ^ (mir ? mi4 : 0u));
      const float k5 = __uint_as_float(__float_as_uint(kp[5 * (H + 1) * TL]) ^ mo5 ^ (mir ? mi5 : 0u));
      const float2 mx = X[0][b], my = X[1][b], mz = X[2][b];
      X[0][b] = make_float2(fmaf(k0, mx.x, fmaf(k3, my.x, k4 * mz.x)), fmaf(k0, mx.y, fmaf(k3, my.y, k4 * mz.y)));
      X[1][b] = make_float2(fmaf(k3, mx.x, fmaf(k1, my.x, k5 * mz.x)), fmaf(k3, mx.y, fmaf(k1, my.y, k5 * mz.y)));
      X[2][b] = make_float2(fmaf(k4, mx.x, fmaf(k5, my.x, k2 * mz.x)), fmaf(k4, mx.y, fmaf(k5, my.y, k2 * mz.y)));
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      Dft<R, +1>::run(X[c]);
      float2* t = sm + (c * 2 + h) * EXT + kxl;
      t[(j * R + 0) * TL] = X[c][0];
#pragma unroll
      for (int q = 1; q < R; ++q) t[(j * R + q) * TL] = cmulc(X[c][q], tws[q]);
    }
    __syncthreads();
    if (nxt < nt) issue_k(nxt);  // every thread is past the multiply: the kernel stage is free
    else asm volatile("cp.async.commit_group;" ::: "memory");
    const unsigned soff = (unsigned)ko * (unsigned)a.outer_stride + (unsigned)kx;
    const unsigned sls = (unsigned)a.line_stride, scs = (unsigned)a.comp_stride;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const float2* t = sm + (c * 2 + h) * EXT + kxl;
#pragma unroll
      for (int q = 0; q < R; ++q) X[c][q] = t[(q * R + j) * TL];
      Dft<R, +1>::run(X[c]);
#pragma unroll
      for (int b = 0; b < R; ++b) X[c][b] = cmulc(X[c][b], twp[b]);
#pragma unroll
      for (int bb = 0; bb < R / 2; ++bb) {
        const float2 mine = h ? X[c][bb + R / 2] : X[c][bb];
        const float2 send = h ? X[c][bb] : X[c][bb + R / 2];
        float2 recv;
        recv.x = __shfl_xor_sync(0xffffffffu, send.x, TL);
        recv.y = __shfl_xor_sync(0xffffffffu, send.y, TL);
        const int n = j + R * (h ? bb + R / 2 : bb);
        if (ok && n < a.n_valid) a.spec[soff + c * scs + (unsigned)n * sls] = cadd(mine, recv);
      }
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

// Pipelined y pass (P = 2 R^2): persistent CTAs of 8 columns x R threads per line x 2 halves
// (lane = column + 8 h + 16 (j & 1)), the rows of the next tile stream into shared memory with
// cp.async while the current tile is transformed; the halves of the inverse meet by shuffle.
// Small CTAs (16 R threads, 65-97 KB) so that three (forward) or two (inverse) of them share an SM.
#ifndef MMX_MIDP_TW_REGS
#define MMX_MIDP_TW_REGS 1   // stage twiddles of a thread live in registers for the whole kernel
#endif
#ifndef MMX_MIDP_MINB_F
#define MMX_MIDP_MINB_F 2   // (2 CTAs of 128 registers beat 3 of 80 once the twiddles are register-resident)
#endif
#ifndef MMX_MIDP_MINB_I
#define MMX_MIDP_MINB_I 2
#endif
template <int R, int DIR>
__global__ void __launch_bounds__(16 * R, DIR < 0 ? MMX_MIDP_MINB_F : MMX_MIDP_MINB_I) k_mid_pipe(MidColArgs a) {
  constexpr int H = R * R, P = 2 * H, TL = 8, NT = 16 * R;
  constexpr int ROWS = DIR < 0 ? H : P;   // rows of a staged tile
  constexpr int EXT = H * TL + 8;         // exchange tile of one half (+8: the halves use different banks)
  extern __shared__ __align__(16) unsigned char smraw[];
  float2* exb = reinterpret_cast<float2*>(smraw);   // [2][EXT]
  float2* stage = exb + 2 * EXT;                     // [2][ROWS][TL]
  __shared__ float2 stw[P];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int kxl = lane & 7, h = (lane >> 3) & 1, j = 2 * wid + (lane >> 4);
  for (int q = threadIdx.x; q < P; q += NT) stw[q] = a.tw[q];
  const int ntm = a.ntile_main * a.nslab;
  const int nt = ntm + (a.nyq ? (a.nslab + TL - 1) / TL : 0);
  float2* ex = exb + h * EXT + kxl;
#if MMX_MIDP_TW_REGS
  // stage twiddles w_H^(j q) of this thread, loaded once for all tiles
  float2 tws[R];
#pragma unroll
  for (int q = 0; q < R; ++q) tws[q] = a.tw[2 * j * q];
#define MMX_TWS(q) tws[q]
  // forward pass: also the half twiddles w_P^(j + R u) (identity for the even half)
  float2 twp[DIR < 0 ? R : 1];
  if (DIR < 0) {
#pragma unroll
    for (int u = 0; u < R; ++u) twp[u] = h ? a.tw[j + R * u] : make_float2(1.f, 0.f);
  }
#else
#define MMX_TWS(q) stw[2 * j * (q)]
#endif

  pdl_wait();      // the twiddle loads above do not depend on the previous kernel
  pdl_trigger();   // persistent kernel: the next kernel's CTAs take over as ours exit
  if (a.gated && !a.ctrl->active) return;

  auto issue = [&](int tile, int buf) {
    float2* dst = stage + (size_t)buf * ROWS * TL;
    if (tile < ntm) {
      const int slab = tile / a.ntile_main;
      const int kx0 = (tile - slab * a.ntile_main) * TL;
      // thread t always copies 16-byte chunk t % 4 of rows t / 4 + (NT / 4) i; 32-bit element offsets
      // from the uniform base (the launcher checks that they fit)
      constexpr int RPI = NT / (TL / 2);
      const unsigned ch = threadIdx.x % (TL / 2), r0 = threadIdx.x / (TL / 2);
      const unsigned xp = (unsigned)a.xp;
      const unsigned so = (unsigned)slab * (unsigned)a.in_outer + (unsigned)kx0 + r0 * xp + 2 * ch;
#pragma unroll
      for (int i = 0; i < ROWS / RPI; ++i) {
        const int row = r0 + RPI * i;
        cpa_zfill<16>(dst + row * TL + 2 * ch, a.in + (so + (unsigned)(RPI * i) * xp), row < a.n_in);
      }
    } else {
      const int slab0 = (tile - ntm) * TL;
      for (int q = threadIdx.x; q < ROWS * TL; q += NT) {
        const int row = q / TL, l = q % TL;
        const bool v = row < a.n_in && slab0 + l < a.nslab;
        const int slab = v ? slab0 + l : 0;
        cpa_zfill<8>(dst + row * TL + l, a.in + (size_t)slab * a.in_outer + (size_t)row * a.xp + (a.xc - 1), v);
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };

  int tile = blockIdx.x;
  if (tile < nt) issue(tile, 0);
  int buf = 0;
  for (; tile < nt; tile += gridDim.x, buf ^= 1) {
    const int nxt = tile + gridDim.x;
    if (nxt < nt) {
      issue(nxt, buf ^ 1);
      asm volatile("cp.async.wait_group 1;" ::: "memory");
    } else {
      asm volatile("cp.async.wait_group 0;" ::: "memory");
    }
    __syncthreads();  // tile landed for all threads; exchange tiles of the previous tile are free
    int kx, slab;
    bool ok = true;
    if (tile < ntm) {
      slab = tile / a.ntile_main;
      kx = (tile - slab * a.ntile_main) * TL + kxl;
      ok = kx < a.xc_main;
    } else {
      kx = a.xc - 1; slab = (tile - ntm) * TL + kxl; ok = slab < a.nslab;
      if (!ok) slab = 0;
    }
    const float2* xin = stage + (size_t)buf * ROWS * TL + kxl;
    float2 v[R];
    if (DIR < 0) {
#pragma unroll
      for (int u = 0; u < R; ++u) {
        const float2 x = xin[(j + R * u) * TL];
#if MMX_MIDP_TW_REGS
        v[u] = cmul(x, twp[u]);
#else
        const float2 w = h ? stw[j + R * u] : make_float2(1.f, 0.f);
        v[u] = cmul(x, w);
#endif
      }
    } else {
#pragma unroll
      for (int u = 0; u < R; ++u) v[u] = xin[(2 * (j + R * u) + h) * TL];
    }
    Dft<R, DIR>::run(v);
    ex[(0 * R + j) * TL] = v[0];
#pragma unroll
    for (int q = 1; q < R; ++q) ex[(q * R + j) * TL] = ctw<DIR>(v[q], MMX_TWS(q));
    __syncthreads();
#pragma unroll
    for (int q = 0; q < R; ++q) v[q] = ex[(j * R + q) * TL];
    Dft<R, DIR>::run(v);
    const unsigned xpu = (unsigned)a.xp;
    const unsigned oo = (unsigned)slab * (unsigned)a.out_outer + (unsigned)kx;
    if (DIR < 0) {
      if (ok) {
        const unsigned o0 = oo + (unsigned)(2 * j + h) * xpu;
#pragma unroll
        for (int b = 0; b < R; ++b) a.out[o0 + (unsigned)(2 * R * b) * xpu] = v[b];
      }
    } else {
      // x[n] = g0[n] + conj(w_P^n) g1[n]: lanes h = 0 finish rows b < R/2, lanes h = 1 the others
#pragma unroll
      for (int b = 0; b < R; ++b) {
        const float2 w = h ? stw[j + R * b] : make_float2(1.f, 0.f);
        v[b] = cmulc(v[b], w);
      }
#pragma unroll
      for (int bb = 0; bb < R / 2; ++bb) {
        const float2 mine = h ? v[bb + R / 2] : v[bb];
        const float2 send = h ? v[bb] : v[bb + R / 2];
        float2 recv;
        recv.x = __shfl_xor_sync(0xffffffffu, send.x, 8);
        recv.y = __shfl_xor_sync(0xffffffffu, send.y, 8);
        const int n = j + R * (h ? bb + R / 2 : bb);
        if (ok && n < a.n_out) a.out[oo + (unsigned)n * xpu] = cadd(mine, recv);
      }
    }
  }
}

template <typename Kern>
int set_smem_col(Kern k, size_t bytes) {
  // (the kernels also hold a static twiddle table: the 48 KB default limit counts both)
  if (bytes > 32 * 1024) MMX_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
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
#if MMX_INNER_VARIANT == 3
  constexpr int TL = 16;
#elif MMX_INNER_VARIANT == 2
  constexpr int TL = MMX_INNER_TL;
#elif MMX_INNER_VARIANT == 1
  constexpr int TL = 16;
#else
  constexpr int TL = 32;
#endif
  a.nyq = ((d.xc - 1) % TL == 0 && d.xc > 1 && L.n_outer >= TL && L.p_outer == L.n_outer) ? 1 : 0;
  if (a.nyq) { a.ntile_main = (d.xc - 1) / TL; a.xc_main = d.xc - 1; }
  else { a.ntile_main = (d.xc + TL - 1) / TL; a.xc_main = d.xc; }
  a.line_stride = L.line_stride; a.comp_stride = L.comp_stride; a.outer_stride = L.outer_stride;
  a.k_inner_stride = L.k_inner_stride; a.k_outer_stride = L.k_outer_stride; a.k_comp_stride = L.k_comp_stride;
  a.odd_inner = L.odd_inner; a.odd_outer = L.odd_outer;
  ProfScope ps(w, PK_INNER);
#if MMX_INNER_VARIANT == 3
  const size_t smem = sizeof(float2) * (6 + 3) * 64 * TL + sizeof(float) * 6 * 65 * TL;
  if (int rc = set_smem_col(k_inner_q<8>, smem)) return rc;
  const int nt = a.ntile_main * L.n_outer + (a.nyq ? (L.p_outer + TL - 1) / TL : 0);
  int grid = mmx_persistent_grid(k_inner_q<8>, 256, smem, w->sm_count, 2);
  if (grid > nt) grid = nt;
  if (L.p_outer != L.n_outer) return mmx_fail(MMX_EINVAL, "inner column pass: outer extent mismatch");
  if (3 * L.comp_stride >= (1ull << 31) || 6 * L.k_comp_stride >= (1ull << 31))
    return mmx_fail(MMX_EINVAL, "inner column pass: spectra exceed the 32-bit element offsets of this kernel");
  MMX_CUDA(mmx_launch(k_inner_q<8>, grid, 256, smem, w->stream, a));
#elif MMX_INNER_VARIANT == 2
  const size_t smem = sizeof(float2) * (6 * (64 * TL + (TL < 16 ? 8 : 0)) + 6 * 64 * TL);
  if (int rc = set_smem_col(k_inner_pipe<8, TL>, smem)) return rc;
  const int nt = a.ntile_main * L.n_outer + (a.nyq ? (L.p_outer + TL - 1) / TL : 0);
  int grid = (32 / TL) * w->sm_count;
  if (grid > nt) grid = nt;
  if (L.p_outer != L.n_outer) return mmx_fail(MMX_EINVAL, "inner column pass: outer extent mismatch");
  if (3 * L.comp_stride >= (1ull << 31) || 6 * L.k_comp_stride >= (1ull << 31))
    return mmx_fail(MMX_EINVAL, "inner column pass: spectra exceed the 32-bit element offsets of this kernel");
  k_inner_pipe<8, TL><<<grid, 2 * TL * 8, smem, w->stream>>>(a);
#elif MMX_INNER_VARIANT == 1
  const size_t smem = sizeof(float2) * 6 * 64 * TL + sizeof(float) * 6 * 65 * TL;
  if (int rc = set_smem_col(k_inner_w<8>, smem)) return rc;
  dim3 g(a.ntile_main + a.nyq, L.n_outer);
  k_inner_w<8><<<g, 256, smem, w->stream>>>(a);
#else
  const size_t smem = sizeof(float2) * 6 * 64 * TL;
  const int nt = a.ntile_main * L.n_outer + (a.nyq ? (L.p_outer + 31) / 32 : 0);
  if (L.p_outer == L.n_outer && nt >= 8 * w->sm_count) {
    if (int rc = set_smem_col(k_inner_colp<8>, smem)) return rc;
    k_inner_colp<8><<<2 * w->sm_count, 256, smem, w->stream>>>(a);
  } else {
    if (int rc = set_smem_col(k_inner_col<8>, smem)) return rc;
    dim3 g(a.ntile_main + a.nyq, L.n_outer);
    k_inner_col<8><<<g, 256, smem, w->stream>>>(a);
  }
#endif
  MMX_CUDA(cudaGetLastError());
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
  // measured on c4: the register-prefetching persistent form wins for the inverse pass (89 vs 95 us),
  // the plain grid for the forward pass (80 vs 90 us)
#if MMX_MID_PIPE
  if (R == 16 && ntiles >= 8 * w->sm_count && (size_t)a.nslab * a.out_outer < (1ull << 31) &&
      (size_t)a.nslab * a.in_outer < (1ull << 31)) {
    MidColArgs b = a;
    constexpr int TL = 8;
    b.nyq = ((a.xc - 1) % TL == 0 && a.xc > 1 && a.nslab >= TL) ? 1 : 0;
    if (b.nyq) { b.ntile_main = (a.xc - 1) / TL; b.xc_main = a.xc - 1; }
    else { b.ntile_main = (a.xc + TL - 1) / TL; b.xc_main = a.xc; }
    const int nt = b.ntile_main * a.nslab + (b.nyq ? (a.nslab + TL - 1) / TL : 0);
    const size_t sm = sizeof(float2) * (2 * (R * R * TL + 8) + 2 * (dir < 0 ? R * R : 2 * R * R) * TL);
    if (dir < 0) {
      if (int rc = set_smem_col(k_mid_pipe<16, -1>, sm)) return rc;
      int grid = mmx_persistent_grid(k_mid_pipe<16, -1>, 16 * 16, sm, w->sm_count, MMX_MIDP_MINB_F);
      MMX_CUDA(mmx_launch(k_mid_pipe<16, -1>, grid < nt ? grid : nt, 16 * 16, sm, w->stream, b));
    } else {
      if (int rc = set_smem_col(k_mid_pipe<16, +1>, sm)) return rc;
      int grid = mmx_persistent_grid(k_mid_pipe<16, +1>, 16 * 16, sm, w->sm_count, MMX_MIDP_MINB_I);
      MMX_CUDA(mmx_launch(k_mid_pipe<16, +1>, grid < nt ? grid : nt, 16 * 16, sm, w->stream, b));
    }
    MMX_CUDA(cudaGetLastError());
    return MMX_OK;
  }
#endif
  if (MMX_MID_PERSISTENT && dir > 0 && ntiles >= 4 * w->sm_count) {
    if (dir < 0) {
      if (int rc = set_smem_col(k_mid_colp<R, TILE, -1>, smem)) return rc;
      k_mid_colp<R, TILE, -1><<<w->sm_count, 2 * R * TILE, smem, w->stream>>>(a);
    } else {
      if (int rc = set_smem_col(k_mid_colp<R, TILE, +1>, smem)) return rc;
      k_mid_colp<R, TILE, +1><<<w->sm_count, 2 * R * TILE, smem, w->stream>>>(a);
    }
    MMX_CUDA(cudaGetLastError());
    return MMX_OK;
  }
  if (dir < 0) {
    if (int rc = set_smem_col(k_mid_col<R, TILE, -1>, smem)) return rc;
    k_mid_col<R, TILE, -1><<<g, 2 * R * TILE, smem, w->stream>>>(a);
  } else {
    if (int rc = set_smem_col(k_mid_col<R, TILE, +1>, smem)) return rc;
    k_mid_col<R, TILE, +1><<<g, 2 * R * TILE, smem, w->stream>>>(a);
  }
  MMX_CUDA(cudaGetLastError());
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
