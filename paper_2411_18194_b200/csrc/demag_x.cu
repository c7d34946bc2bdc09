// demag_x.cu -- the two passes of the demag convolution along x (the contiguous axis) for
// Px = 512, fast path of demag.cu.
//
// One warp owns one pair of real rows (a, b) packed as the complex line a + i b; lane (j, h),
// j = 0..15, h = 0..1, holds 16 points of half h of the 512-point transform in registers
// (fft_reg.cuh: P = 2 R^2, R = 16) and the only exchange between the two radix-16 stages is a
// warp-private shared-memory tile: no block barrier inside the loop.  Each warp walks over its
// row pairs and copies the rows of its next pair to shared memory with cp.async (16 B per lane,
// fully coalesced) while it transforms the current one, so its loads are always in flight.
//
//   k_x_fwd_w  M = sum_s Ms^(s) m^(s) formed while reading; Z = FFT(a + i b);
//              A[k] = (Z[k] + conj Z[P-k])/2, B[k] = (Z[k] - conj Z[P-k])/(2i), k = 0..P/2
//              -> spec1 rows (row pitch xp complex)
//   k_x_inv_w  Z[k] = A[k] + i B[k], Z[P-k] = conj A[k] + i conj B[k]; z = IFFT(Z), first Nx
//              points only; Re z -> row a, Im z -> row b of B_demag
#include "fft_reg.cuh"
#include "mmx_internal.h"

using namespace mmxreg;

namespace {

constexpr int XR = 16, XH = 256, XP = 512;
constexpr int XW = 8;                 // warps per CTA
constexpr int EXN = XH + XH / 16 + 8;  // padded exchange tile (one pad element per 16); +8: the two
                                       // halves of a line use different banks

__device__ __forceinline__ int padx(int m) { return m + (m >> 4); }

__device__ __forceinline__ void cp16(void* smem, const void* gmem) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

struct XWArgs {
  int nx, rows, xp, S, gated;
  size_t N;
  float ms[2];             // Ms of the (single) region per sublattice
  const float* yin[2];     // sel pair: state [nvec][3][N]
  const MmxCtrl* ctrl;
  const float2* tw;        // exp(-2 pi i q / 512)
  float2* spec;            // spec1 [rows][xp]
  float* bout;             // B_demag [rows][nx]
};

// per-warp shared memory of the forward pass: float in[S][2 * XH] (two rows per sublattice),
// then float2 ex[2 * EXN] (exchange tiles of the two halves; reused as Z[512])
__host__ __device__ inline size_t xfwd_warp_bytes(int S) { return (size_t)S * 2 * XH * sizeof(float) + 2 * EXN * sizeof(float2); }

// FULL: Nx = 256, an even number of rows, one sublattice (the c4 shape): sizes become constants
template <bool FULL>
__global__ void __launch_bounds__(32 * XW, 4) k_x_fwd_w(XWArgs a) {
  const int nx = FULL ? XH : a.nx, S = FULL ? 1 : a.S;
  extern __shared__ __align__(128) unsigned char smraw[];
  __shared__ float2 stw[XH];  // w_P^n for n < P/2 only (the half twiddles of the pruned input)
  // stage twiddles w_H^(j q) laid out [j][q] with a row pitch of 17: lanes (different j, same q) hit
  // different banks (stw[2 j q] has a lane stride of 4 q words: up to 8-way conflicts)
  __shared__ float2 stq[XR * (XR + 1)];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int j = lane >> 1, h = lane & 1;  // one 64-bit shared-memory wavefront = 8 j x both halves
  float* sin_ = reinterpret_cast<float*>(smraw + wid * xfwd_warp_bytes(S));
  float2* sex = reinterpret_cast<float2*>(sin_ + (size_t)S * 2 * XH);
  for (int q = threadIdx.x; q < XH; q += 32 * XW) stw[q] = a.tw[q];
  for (int q = threadIdx.x; q < XR * XR; q += 32 * XW) stq[(q / XR) * (XR + 1) + q % XR] = a.tw[2 * (q / XR) * (q % XR)];
  if (a.gated && !a.ctrl->active) return;
  const float* y = a.ctrl->sel ? a.yin[1] : a.yin[0];  // (no dynamic index into the parameter block)
  const int npair = (a.rows + 1) >> 1;
  const int nwarp = gridDim.x * XW;
  const int chunks = nx >> 1;  // 16-byte chunks of a row pair: 2 nx floats / 4

  auto prefetch = [&](int pair) {
    for (int s = 0; s < S; ++s) {
      const float* src = y + (size_t)s * 3 * a.N + (size_t)pair * 2 * nx;
      const bool full = FULL || 2 * pair + 1 < a.rows;
      for (int c = lane; c < chunks; c += 32)
        if (full || 2 * c < chunks) cp16(sin_ + s * 2 * XH + 4 * c, src + 4 * c);
    }
    cp_commit();
  };

  int pair = blockIdx.x * XW + wid;
  if (pair < npair) prefetch(pair);
  __syncthreads();  // stw
  for (; pair < npair; pair += nwarp) {
    cp_wait<0>();
    __syncwarp();
    const bool two = FULL || 2 * pair + 1 < a.rows;
    float2 v[XR];
#pragma unroll
    for (int u = 0; u < XR; ++u) {
      const int n = j + XR * u;
      float ra = 0.f, rb = 0.f;
      if (FULL || n < nx) {
        ra = a.ms[0] * sin_[n];
        rb = two ? a.ms[0] * sin_[nx + n] : 0.f;
        if (S == 2) {
          ra = fmaf(a.ms[1], sin_[2 * XH + n], ra);
          if (two) rb = fmaf(a.ms[1], sin_[2 * XH + nx + n], rb);
        }
      }
      v[u] = make_float2(ra, rb);
    }
    __syncwarp();
    if (pair + nwarp < npair) prefetch(pair + nwarp);  // overlaps the transform below
#pragma unroll
    for (int u = 0; u < XR; ++u) {
      const float2 w = h ? stw[j + XR * u] : make_float2(1.f, 0.f);  // (both halves share a warp: no branch)
      v[u] = cmul(v[u], w);
    }
    Dft<XR, -1>::run(v);
    float2* ex = sex + h * EXN;
    ex[padx(j)] = v[0];
#pragma unroll
    for (int q = 1; q < XR; ++q) ex[padx(q * XR + j)] = cmul(v[q], stq[j * (XR + 1) + q]);
    __syncwarp();
#pragma unroll
    for (int q = 0; q < XR; ++q) v[q] = ex[padx(j * XR + q)];
    Dft<XR, -1>::run(v);
    __syncwarp();
    float2* zs = sex;  // Z[k], natural order
#pragma unroll
    for (int b = 0; b < XR; ++b) zs[2 * (j + XR * b) + h] = v[b];
    __syncwarp();
    float2* o0 = a.spec + (size_t)(2 * pair) * a.xp;
    float2* o1 = o0 + a.xp;
#pragma unroll
    for (int i = 0; i <= XH / 32; ++i) {
      const int k = lane + 32 * i;
      if (k <= XH) {
        const float2 zk = zs[k], zm = zs[(XP - k) & (XP - 1)];
        o0[k] = rmul(0.5f, cadd(zk, make_float2(zm.x, -zm.y)));
        if (two) o1[k] = rmul(0.5f, cadd(make_float2(zk.y, -zk.x), make_float2(zm.y, zm.x)));
      }
    }
    __syncwarp();  // zs is rewritten by the next iteration
  }
}

struct __align__(128) XInvSmem {
  float2 in[2][XH + 16];     // [row a / b][257 kept columns]; rows and the struct are multiples of 128 bytes, so a warp's
                             // 512-byte cp.async lands on four bank rows, not five (10 % of this pass's wavefronts)
  float2 ex[2 * EXN];         // exchange tiles; reused as the two output rows [2][256] floats
};

template <bool FULL>
__global__ void __launch_bounds__(32 * XW, 3) k_x_inv_w(XWArgs a) {
  const int nx = FULL ? XH : a.nx;
  extern __shared__ __align__(128) unsigned char smraw[];
  __shared__ float2 stw[XH];  // conj(w_P^n) for the first P/2 outputs only
  // stage twiddles w_H^(j q) laid out [j][q] with a row pitch of 17: lanes (different j, same q) hit
  // different banks (stw[2 j q] has a lane stride of 4 q words: up to 8-way conflicts)
  __shared__ float2 stq[XR * (XR + 1)];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int j = lane >> 1, h = lane & 1;  // one 64-bit shared-memory wavefront = 8 j x both halves
  XInvSmem& sm = reinterpret_cast<XInvSmem*>(smraw)[wid];
  for (int q = threadIdx.x; q < XH; q += 32 * XW) stw[q] = a.tw[q];
  for (int q = threadIdx.x; q < XR * XR; q += 32 * XW) stq[(q / XR) * (XR + 1) + q % XR] = a.tw[2 * (q / XR) * (q % XR)];
  if (a.gated && !a.ctrl->active) return;
  const int npair = (a.rows + 1) >> 1;
  const int nwarp = gridDim.x * XW;
  constexpr int CH = (XH + 1 + 1) / 2;  // 16-byte chunks covering 257 complex values

  auto prefetch = [&](int pair) {
    const bool two = FULL || 2 * pair + 1 < a.rows;
    for (int r = 0; r < (two ? 2 : 1); ++r) {
      const float2* src = a.spec + (size_t)(2 * pair + r) * a.xp;
      for (int c = lane; c < CH; c += 32) cp16(&sm.in[r][2 * c], src + 2 * c);
    }
    cp_commit();
  };

  int pair = blockIdx.x * XW + wid;
  if (pair < npair) prefetch(pair);
  __syncthreads();  // stw
  for (; pair < npair; pair += nwarp) {
    cp_wait<0>();
    __syncwarp();
    const bool two = FULL || 2 * pair + 1 < a.rows;
    const float2* A = sm.in[0];
    const float2* B = sm.in[1];
    float2 v[XR];
#pragma unroll
    for (int u = 0; u < XR; ++u) {
      const int k = 2 * (j + XR * u) + h;
      const int kk = k <= XH ? k : XP - k;
      const float2 va = A[kk];
      const float2 vb = two ? B[kk] : make_float2(0.f, 0.f);
      v[u] = k <= XH ? cadd(va, make_float2(-vb.y, vb.x)) : cadd(make_float2(va.x, -va.y), make_float2(vb.y, vb.x));
    }
    __syncwarp();
    if (pair + nwarp < npair) prefetch(pair + nwarp);  // overlaps the transform below
    Dft<XR, +1>::run(v);
    float2* ex = sm.ex + h * EXN;
    ex[padx(j)] = v[0];
#pragma unroll
    for (int q = 1; q < XR; ++q) ex[padx(q * XR + j)] = cmulc(v[q], stq[j * (XR + 1) + q]);
    __syncwarp();
#pragma unroll
    for (int q = 0; q < XR; ++q) v[q] = ex[padx(j * XR + q)];
    Dft<XR, +1>::run(v);
#pragma unroll
    for (int b = 0; b < XR; ++b) {
      const float2 w = h ? stw[j + XR * b] : make_float2(1.f, 0.f);
      v[b] = cmulc(v[b], w);
    }
    __syncwarp();
    // z[n] = g0[n] + conj(w^n) g1[n]; lanes h = 0 finish n = j + 16 b for even b, lanes h = 1 for odd b
    // (bank of orow[n]: j + 16 h, all 32 lanes distinct)
    float* orow = reinterpret_cast<float*>(sm.ex);  // [2][256]
#pragma unroll
    for (int bb = 0; bb < XR / 2; ++bb) {
      const float2 mine = h ? v[2 * bb + 1] : v[2 * bb];
      const float2 send = h ? v[2 * bb] : v[2 * bb + 1];
      float2 recv;
      recv.x = __shfl_xor_sync(0xffffffffu, send.x, 1);
      recv.y = __shfl_xor_sync(0xffffffffu, send.y, 1);
      const int n = j + XR * (2 * bb + h);
      orow[n] = mine.x + recv.x;
      orow[XH + n] = mine.y + recv.y;
    }
    __syncwarp();
    float* o0 = a.bout + (size_t)(2 * pair) * nx;
    for (int c = lane; c < (nx >> 2); c += 32) {
      *reinterpret_cast<float4*>(o0 + 4 * c) = *reinterpret_cast<const float4*>(orow + 4 * c);
      if (two) *reinterpret_cast<float4*>(o0 + nx + 4 * c) = *reinterpret_cast<const float4*>(orow + XH + 4 * c);
    }
    __syncwarp();  // the output rows alias the exchange tiles of the next iteration
  }
}

}  // namespace

bool mmx_x_warp_ok(const mmx_world* w) {
  const DemagPlan& d = w->dm;
  if (d.px != XP || (d.nx & 3) || d.nx > XH || w->nreg != 1 || w->S > 2) return false;
  for (int s = 0; s < w->S; ++s)
    if (!(w->mats[(size_t)s * w->nreg].Ms > 0)) return false;
  return true;
}

int mmx_x_warp_launch(mmx_world* w, int dir, const float* const yin[2], float* bout) {
  const DemagPlan& d = w->dm;
  XWArgs a;
  a.nx = d.nx; a.rows = 3 * d.nz * d.ny; a.xp = d.xp; a.S = w->S; a.gated = 1; a.N = w->N;
  for (int s = 0; s < 2; ++s) a.ms[s] = s < w->S ? (float)w->mats[(size_t)s * w->nreg].Ms : 0.f;
  a.yin[0] = yin ? yin[0] : nullptr; a.yin[1] = yin ? yin[1] : nullptr;
  a.ctrl = w->d_ctrl; a.tw = d.tw[0]; a.spec = d.spec1; a.bout = bout;
  const int npair = (a.rows + 1) / 2;
  const bool full = d.nx == XH && (a.rows & 1) == 0 && w->S == 1;
  int blocks;
  {
    const size_t smem = dir < 0 ? xfwd_warp_bytes(a.S) * XW : sizeof(XInvSmem) * XW;
    if (dir < 0) {
      MMX_CUDA(cudaFuncSetAttribute(k_x_fwd_w<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      MMX_CUDA(cudaFuncSetAttribute(k_x_fwd_w<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      blocks = full ? mmx_persistent_grid(k_x_fwd_w<true>, 32 * XW, smem, w->sm_count, 4)
                    : mmx_persistent_grid(k_x_fwd_w<false>, 32 * XW, smem, w->sm_count, 4);
    } else {
      MMX_CUDA(cudaFuncSetAttribute(k_x_inv_w<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      MMX_CUDA(cudaFuncSetAttribute(k_x_inv_w<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      blocks = full ? mmx_persistent_grid(k_x_inv_w<true>, 32 * XW, smem, w->sm_count, 3)
                    : mmx_persistent_grid(k_x_inv_w<false>, 32 * XW, smem, w->sm_count, 3);
    }
  }
  if (blocks * XW > npair) blocks = (npair + XW - 1) / XW;
  if (dir < 0) {
    const size_t smem = xfwd_warp_bytes(a.S) * XW;
    ProfScope ps(w, PK_X_FWD);
    if (full) {
      MMX_CUDA(cudaFuncSetAttribute(k_x_fwd_w<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      MMX_CUDA(mmx_launch(k_x_fwd_w<true>, blocks, 32 * XW, smem, w->stream, a));
    } else {
      MMX_CUDA(cudaFuncSetAttribute(k_x_fwd_w<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      MMX_CUDA(mmx_launch(k_x_fwd_w<false>, blocks, 32 * XW, smem, w->stream, a));
    }
  } else {
    const size_t smem = sizeof(XInvSmem) * XW;
    ProfScope ps(w, PK_X_INV);
    if (full) {
      MMX_CUDA(cudaFuncSetAttribute(k_x_inv_w<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      MMX_CUDA(mmx_launch(k_x_inv_w<true>, blocks, 32 * XW, smem, w->stream, a));
    } else {
      MMX_CUDA(cudaFuncSetAttribute(k_x_inv_w<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      MMX_CUDA(mmx_launch(k_x_inv_w<false>, blocks, 32 * XW, smem, w->stream, a));
    }
  }
  MMX_CUDA(cudaGetLastError());
  return MMX_OK;
}
