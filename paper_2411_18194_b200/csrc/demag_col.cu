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
//   k_inner_q<8>    P = 128: forward along the innermost transformed axis, multiply by the real
//                   symmetric 3x3 kernel spectrum (octant + parity), inverse, in place.  Persistent
//                   CTAs; the spectrum rows and the kernel rows of the next tile stream into shared
//                   memory (cp.async) while the current tile is transformed.
//   k_mid_pipe<16>  P = 512: the y pass of a 3-D world on large grids, same pipeline.
//   k_mid_col<R>    P = 512 / 128 / 32: the plain (one CTA per tile) y pass for everything else.
//
// The column kx = Px/2 (Nyquist) would waste a whole lane tile; it is served by separate tiles
// whose lanes run over the outer index instead (strided, but 1/257 of the data).
//
// Variants that were built, measured on c4 and removed (numbers in DESIGN.md section 8): 32-column
// inner tiles with both halves per thread (226 us), the same persistent with L2 prefetch (291 us),
// 16-column tiles with the halves in one warp but no pipeline (248 us), the cp.async pipeline with
// the kernel values in registers (207 us; 272 us with 8-column tiles); k_inner_q runs at 170 us.
// A persistent y pass with register prefetch (89 us) lost to k_mid_pipe (66 / 76 us).
#ifndef MMX_PACKED_R16
#define MMX_PACKED_R16 0   // measured on c4: y passes 68.0 / 80.8 us packed, 66.1 / 78.4 us scalar
#endif
#include "fft_reg.cuh"
#include "mmx_internal.h"

using namespace mmxreg;

namespace {

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

// cp.async with zero fill (src-size 0 when the row / column lies outside the data)
template <int BYTES>
__device__ __forceinline__ void cpa_zfill(void* smem, const void* gmem, bool valid) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
  const int n = valid ? BYTES : 0;
  if (BYTES == 16)
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(sa), "l"(gmem), "r"(n) : "memory");
  else
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(sa), "l"(gmem), "r"(n) : "memory");
}

// Fused inner pass.  16 kx columns per CTA, lane = column + 16 h, warp = j: the two halves of a line
// sit in the same warp (their inputs are one shared-memory read, their results meet by shuffle) and
// a thread carries one half of three components (48 data registers).  The spectrum rows of the
// next tile and the kernel-spectrum rows of the next tile are staged in shared memory by cp.async
// one tile ahead (one stage each, refilled as soon as every thread has read it); the 15 twiddles
// of a thread live in registers for the whole kernel.  Tile order pairs ky with Py - ky: both read
// the same kernel rows, the second read hits L2.
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
      // rows (c, pm) are equidistant in the octant when k_comp_stride = (H + 1) k_inner_stride (the
      // launcher checks it): row r = c (H + 1) + pm sits at r * k_inner_stride, no division by H + 1
      const unsigned kis = (unsigned)a.k_inner_stride;
#pragma unroll
      for (int q0 = 0; q0 < 6 * (H + 1) * (TL / 4); q0 += NT) {
        const int q = q0 + threadIdx.x;
        if (q < 6 * (H + 1) * (TL / 4)) {
          const unsigned row = q / (TL / 4), ch = q % (TL / 4);
          const unsigned sa = (unsigned)__cvta_generic_to_shared(kst + row * TL + 4 * ch);
          const float* g = a.khat + (kb + row * kis + 4 * ch);
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(g) : "memory");
        }
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
      X[0][b] = rfma(k0, mx, rfma(k3, my, rmul(k4, mz)));
      X[1][b] = rfma(k3, mx, rfma(k1, my, rmul(k5, mz)));
      X[2][b] = rfma(k4, mx, rfma(k5, my, rmul(k2, mz)));
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
  // tile-major layout of the padded side (demag_tile.cu), 0 = plain [slab][ky][xp]:
  int t_nz;                    // z rows per component (slab = c nz + z)
  unsigned t_tile, t_ks, t_nyq;  // complex elements per tile (3 nz 16), per ky (ntx tiles), offset of the Nyquist tiles
};

// position of column l (0..15) of a tile row with z index z: 16-byte chunks XOR-swizzled with (z & 7)
__device__ __forceinline__ unsigned tile_pos16(unsigned l, unsigned z) { return ((((l >> 1) ^ (z & 7u)) << 1) | (l & 1u)); }

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

// Pipelined y pass (P = 2 R^2): persistent CTAs of 8 columns x R threads per line x 2 halves
// (lane = column + 8 h + 16 (j & 1)), the rows of the next tile stream into shared memory with
// cp.async while the current tile is transformed; the halves of the inverse meet by shuffle.
// Small CTAs (16 R threads, 65-97 KB) so that three (forward) or two (inverse) of them share an SM.
// (two CTAs of 128 registers per SM beat three of 80 once the twiddles are register-resident)
template <int R, int DIR>
__global__ void __launch_bounds__(16 * R, 2) k_mid_pipe(MidColArgs a) {
  constexpr int H = R * R, P = 2 * H, TL = 8, NT = 16 * R;
  constexpr int ROWS = DIR < 0 ? H : P;   // rows of a staged tile
  constexpr int NSTG = 2;   // cp.async stages (a third forward stage was measured: 70.3 vs 69.1 us, no gain)
  constexpr int EXT = H * TL + 8;         // exchange tile of one half (+8: the halves use different banks)
  extern __shared__ __align__(16) unsigned char smraw[];
  float2* exb = reinterpret_cast<float2*>(smraw);   // [2][EXT]
  float2* stage = exb + 2 * EXT;                     // [NSTG][ROWS][TL]
  __shared__ float2 stw[P];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int kxl = lane & 7, h = (lane >> 3) & 1, j = 2 * wid + (lane >> 4);
  for (int q = threadIdx.x; q < P; q += NT) stw[q] = a.tw[q];
  const int ntm = a.ntile_main * a.nslab;
  const int nt = ntm + (a.nyq ? (a.nslab + TL - 1) / TL : 0);
  float2* ex = exb + h * EXT + kxl;
  // stage twiddles w_H^(j q) of this thread, loaded once for all tiles
  float2 tws[R];
#pragma unroll
  for (int q = 0; q < R; ++q) tws[q] = a.tw[2 * j * q];
  // forward pass: also the half twiddles w_P^(j + R u) (identity for the even half)
  float2 twp[DIR < 0 ? R : 1];
  if (DIR < 0) {
#pragma unroll
    for (int u = 0; u < R; ++u) twp[u] = h ? a.tw[j + R * u] : make_float2(1.f, 0.f);
  }

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
      unsigned xp = (unsigned)a.xp;
      unsigned so = (unsigned)slab * (unsigned)a.in_outer + (unsigned)kx0 + r0 * xp + 2 * ch;
      if (DIR > 0 && a.t_nz) {
        // rows are ky, the 64-byte half row of this tile holds its four chunks in swizzled order
        const unsigned z = (unsigned)slab % (unsigned)a.t_nz;
        const unsigned phys = ((((unsigned)kx0 >> 3) & 1u) * 4 + ch) ^ (z & 7u);
        xp = a.t_ks;
        so = ((unsigned)kx0 >> 4) * a.t_tile + (unsigned)slab * 16u + 2 * phys + r0 * xp;
      }
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
        const float2* src = a.in + (size_t)slab * a.in_outer + (size_t)row * a.xp + (a.xc - 1);
        if (DIR > 0 && a.t_nz)
          src = a.in + (a.t_nyq + ((unsigned)row >> 4) * a.t_tile + (unsigned)slab * 16u +
                        tile_pos16((unsigned)row & 15u, (unsigned)slab % (unsigned)a.t_nz));
        cpa_zfill<8>(dst + row * TL + l, src, v);
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };

  int tile = blockIdx.x;
  // prologue: NSTG - 1 tiles in flight (an empty group keeps the group count uniform past the end)
#pragma unroll
  for (int p = 0; p < NSTG - 1; ++p) {
    if (tile + p * (int)gridDim.x < nt) issue(tile + p * gridDim.x, p);
    else asm volatile("cp.async.commit_group;" ::: "memory");
  }
  int buf = 0;
  for (; tile < nt; tile += gridDim.x, buf = (buf + 1 == NSTG ? 0 : buf + 1)) {
    const int nxt = tile + (NSTG - 1) * gridDim.x;
    // (the stage refilled here was read before the block barriers of the previous iteration)
    if (nxt < nt) issue(nxt, buf == 0 ? NSTG - 1 : buf - 1);
    else asm volatile("cp.async.commit_group;" ::: "memory");
    asm volatile("cp.async.wait_group %0;" ::"n"(NSTG - 1) : "memory");
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
        v[u] = cmul(x, twp[u]);
      }
    } else {
#pragma unroll
      for (int u = 0; u < R; ++u) v[u] = xin[(2 * (j + R * u) + h) * TL];
    }
    Dft<R, DIR>::run(v);
    ex[(0 * R + j) * TL] = v[0];
#pragma unroll
    for (int q = 1; q < R; ++q) ex[(q * R + j) * TL] = ctw<DIR>(v[q], tws[q]);
    __syncthreads();
#pragma unroll
    for (int q = 0; q < R; ++q) v[q] = ex[(j * R + q) * TL];
    Dft<R, DIR>::run(v);
    const unsigned xpu = (unsigned)a.xp;
    const unsigned oo = (unsigned)slab * (unsigned)a.out_outer + (unsigned)kx;
    if (DIR < 0) {
      if (ok) {
        unsigned o0 = oo + (unsigned)(2 * j + h) * xpu, ostr = (unsigned)(2 * R) * xpu;
        if (a.t_nz) {
          const unsigned z = (unsigned)slab % (unsigned)a.t_nz, kyl = (unsigned)(2 * j + h);
          if (tile < ntm) {  // row ky = kyl + 2 R b of tile column kx
            o0 = ((unsigned)kx >> 4) * a.t_tile + (unsigned)slab * 16u + tile_pos16((unsigned)kx & 15u, z) + kyl * a.t_ks;
            ostr = (unsigned)(2 * R) * a.t_ks;
          } else {           // Nyquist column: tiles of 16 consecutive ky
            o0 = a.t_nyq + (kyl >> 4) * a.t_tile + (unsigned)slab * 16u + tile_pos16(kyl & 15u, z);
            ostr = (unsigned)(2 * R / 16) * a.t_tile;
          }
        }
#pragma unroll
        for (int b = 0; b < R; ++b) a.out[o0 + (unsigned)b * ostr] = v[b];
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
  constexpr int TL = 16;
  a.nyq = ((d.xc - 1) % TL == 0 && d.xc > 1 && L.n_outer >= TL && L.p_outer == L.n_outer) ? 1 : 0;
  if (a.nyq) { a.ntile_main = (d.xc - 1) / TL; a.xc_main = d.xc - 1; }
  else { a.ntile_main = (d.xc + TL - 1) / TL; a.xc_main = d.xc; }
  a.line_stride = L.line_stride; a.comp_stride = L.comp_stride; a.outer_stride = L.outer_stride;
  a.k_inner_stride = L.k_inner_stride; a.k_outer_stride = L.k_outer_stride; a.k_comp_stride = L.k_comp_stride;
  a.odd_inner = L.odd_inner; a.odd_outer = L.odd_outer;
  if (L.p_outer != L.n_outer) return mmx_fail(MMX_EINVAL, "inner column pass: outer extent mismatch");
  if (L.k_comp_stride != (size_t)65 * L.k_inner_stride)
    return mmx_fail(MMX_EINVAL, "inner column pass: kernel octant rows are not equidistant");
  if (3 * L.comp_stride >= (1ull << 31) || 6 * L.k_comp_stride >= (1ull << 31))
    return mmx_fail(MMX_EINVAL, "inner column pass: spectra exceed the 32-bit element offsets of this kernel");
  ProfScope ps(w, PK_INNER);
  const size_t smem = sizeof(float2) * (6 + 3) * 64 * TL + sizeof(float) * 6 * 65 * TL;
  if (int rc = set_smem_col(k_inner_q<8>, smem)) return rc;
  const int nt = a.ntile_main * L.n_outer + (a.nyq ? (L.p_outer + TL - 1) / TL : 0);
  int grid = mmx_persistent_grid(k_inner_q<8>, 256, smem, w->sm_count, 2);
  if (grid > nt) grid = nt;
  MMX_CUDA(mmx_launch(k_inner_q<8>, grid, 256, smem, w->stream, a));
  MMX_CUDA(cudaGetLastError());
  return MMX_OK;
}

bool mmx_mid_col_ok(int P, int n) { return (P == 512 || P == 128 || P == 32) && 2 * n <= P; }

// the pipelined y pass (k_mid_pipe) serves 512-point lines on grids with enough tiles to fill the GPU
bool mmx_mid_pipe_ok(const mmx_world* w, int P, int nslab) {
  const DemagPlan& d = w->dm;
  const long long ntiles = (long long)((d.xc + 15) / 16) * nslab;
  return P == 512 && ntiles >= 8LL * w->sm_count && (size_t)nslab * d.py * d.xp < (1ull << 31);
}

template <int R, int TILE>
static int mid_col_launch_t(mmx_world* w, MidColArgs& a, int dir) {
  a.nyq = ((a.xc - 1) % TILE == 0 && a.xc > 1 && a.nslab >= TILE) ? 1 : 0;
  if (a.nyq) { a.ntile_main = (a.xc - 1) / TILE; a.xc_main = a.xc - 1; }
  else { a.ntile_main = (a.xc + TILE - 1) / TILE; a.xc_main = a.xc; }
  dim3 g(a.ntile_main + a.nyq, a.nslab);
  const size_t smem = sizeof(float2) * (dir < 0 ? 2 : 3) * R * R * TILE;
  ProfScope ps(w, dir < 0 ? PK_MID_FWD : PK_MID_INV);
  const int ntiles = a.ntile_main * a.nslab + (a.nyq ? (a.nslab + TILE - 1) / TILE : 0);
  if (R == 16 && mmx_mid_pipe_ok(w, 2 * R * R, a.nslab)) {
    MidColArgs b = a;
    constexpr int TL = 8;
    b.nyq = ((a.xc - 1) % TL == 0 && a.xc > 1 && a.nslab >= TL) ? 1 : 0;
    if (b.nyq) { b.ntile_main = (a.xc - 1) / TL; b.xc_main = a.xc - 1; }
    else { b.ntile_main = (a.xc + TL - 1) / TL; b.xc_main = a.xc; }
    const int nt = b.ntile_main * a.nslab + (b.nyq ? (a.nslab + TL - 1) / TL : 0);
    const size_t sm = sizeof(float2) * (2 * (R * R * TL + 8) + 2 * (dir < 0 ? R * R : 2 * R * R) * TL);
    if (dir < 0) {
      if (int rc = set_smem_col(k_mid_pipe<16, -1>, sm)) return rc;
      int grid = mmx_persistent_grid(k_mid_pipe<16, -1>, 16 * 16, sm, w->sm_count, 2);
      MMX_CUDA(mmx_launch(k_mid_pipe<16, -1>, grid < nt ? grid : nt, 16 * 16, sm, w->stream, b));
    } else {
      if (int rc = set_smem_col(k_mid_pipe<16, +1>, sm)) return rc;
      int grid = mmx_persistent_grid(k_mid_pipe<16, +1>, 16 * 16, sm, w->sm_count, 2);
      MMX_CUDA(mmx_launch(k_mid_pipe<16, +1>, grid < nt ? grid : nt, 16 * 16, sm, w->stream, b));
    }
    MMX_CUDA(cudaGetLastError());
    return MMX_OK;
  }
  (void)ntiles;
  if (a.t_nz) return mmx_fail(MMX_EINVAL, "mid column pass: the tile-major layout needs the pipelined kernel");
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
  a.t_nz = 0; a.t_tile = a.t_ks = a.t_nyq = 0;
  if (d.tiled) {  // the padded side (spec2) is tile-major: demag_tile.cu
    a.t_nz = d.nz;
    a.t_tile = 3u * d.nz * 16u;
    a.t_ks = (unsigned)((d.xc - 1) / 16) * a.t_tile;
    a.t_nyq = (unsigned)d.py * a.t_ks;
  }
  switch (P) {
    case 512: return mid_col_launch_t<16, 16>(w, a, dir);
    case 128: return mid_col_launch_t<8, 32>(w, a, dir);
    case 32: return mid_col_launch_t<4, 32>(w, a, dir);
  }
  return mmx_fail(MMX_EINVAL, "mid column pass: unsupported length %d", P);
}
