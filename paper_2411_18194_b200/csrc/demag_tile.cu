// demag_tile.cu -- the fused innermost pass of the 3-D demag convolution on the TILE-MAJOR spectrum
// layout: forward z transform of the three components, real symmetric
// 3x3 multiply with the kernel spectrum, inverse z transform, in place.
//
// Why a second layout.  The plain layout [c][z][ky][kx] makes the 16 columns x 64 rows x 3 components
// that one tile of this pass needs 192 separate 128-byte pieces; they had to be gathered with 13
// cp.async per thread, the thread <-> column mapping was dictated by coalescing, the eight warps of a
// CTA exchanged data with each other twice per tile behind block barriers, and the two CTAs of an SM
// marched through load / transform / exchange phases in lock step: every unit of the SM (issue, fp32,
// shared memory, HBM) ended up about 50 % busy (profiles/ncu_r2_kernels.md).  Here the y pass writes
// the spectrum so that a tile IS one contiguous block per component,
//     spec2T[ky][tx][c][z][16 kx]                 tx = kx / 16, 128 bytes per (c, z) row
// (the Nyquist column kx = Px/2 is stored as tiles of 16 consecutive ky: [ky/16][c][z][16 ky]), and the
// kernel spectrum is stored at init as one ready-made shared-memory image per (ky <= Py/2, tx).  Then
//   * a tile arrives by ONE bulk-TMA copy per component (cp.async.bulk + mbarrier complete_tx; SASS
//     UBLKCP) and leaves the same way (cp.async.bulk.global.shared): no per-thread address arithmetic,
//     no cp.async, no coalescing constraint on who computes what;
//   * a warp owns two columns of the tile: lane = (column, j, half), so the radix-8 x radix-8
//     exchange is warp-private (__syncwarp) -- there is NO block barrier in the tile loop;
//   * the eight warps drift apart freely: a warp waits only on "my tile has landed" (mbarrier) and
//     the last warp to finish a tile (shared-memory ticket) writes the tile back and refills the
//     stage two tiles ahead.  Independent warps in different phases keep all units busy.
//   * tiles ky and Py - ky are consecutive in a CTA's sequence and share one kernel image (odd
//     components change sign): the kernel stage is loaded once per pair.
// The 16-byte chunks of a row are XOR-swizzled with (z & 7) -- in global memory too, so the bulk copy
// stays linear -- which makes the column-pair reads of eight different rows conflict-free; the kernel
// images are swizzled with ((kz >> 1) & 7) for the same reason.
#include "fft_reg.cuh"
#include "mbar.cuh"
#include "mmx_internal.h"

using namespace mmxreg;

namespace {

constexpr int R = 8, H = 64, P = 128, TL = 16;
constexpr int NW = 8;                              // warps per CTA, two columns each
constexpr int XS_BYTES = 3 * H * TL * 8;           // one spectrum stage: 24576
constexpr int KS_FLOATS = 6 * (H + 1) * TL;        // one kernel image: 6240 floats
constexpr int KS_BYTES = KS_FLOATS * 4;            // 24960
// Measured on c4: 2 stages + 2 regions 135.5 us; 2 + 1 (the components serialise on the one region) 140.5 us;
// 3 stages + 1 region (what fits beside the kernel image at two CTAs per SM) 139.4 us
constexpr int NXS = 2;                             // spectrum stages
constexpr int NEXR = 2;                            // exchange regions per warp
constexpr int EXR = 2 * H * 2;                     // float2 per exchange region: [half][64 rows, XOR-swizzled][2 columns]
constexpr int EX_BYTES = NW * NEXR * EXR * 8;
constexpr int SMEM_BYTES = NXS * XS_BYTES + KS_BYTES + EX_BYTES + 64;
// row (q, j) of an exchange region: q 8 + (j ^ q).  The radix-8 stage of thread j writes rows (q, j) and reads rows (j, q)
// (or the other way round): both are conflict-free, the first because the eight lanes j fill one 128-byte group, the
// second because row (j, q) sits at offset (q ^ j) of group j
__device__ __forceinline__ int exrow(int q, int j) { return (q * 8 + (j ^ q)) * 2; }

struct TileArgs {
  float2* spec;          // spec2 in tile-major layout
  const float* kimg;     // kernel images [(Py/2+1) ntx + Py/16][6][65][16], swizzled
  const float2* tw;      // exp(-2 pi i q / 128)
  const MmxCtrl* ctrl;
  int nz;                // rows per component present in memory (<= 64); the rest is zero padding
  int ntx;               // main column tiles per ky
  int py;                // transform length along y
  int ntiles;            // main tiles + Nyquist tiles
  unsigned odd_inner, odd_outer;
};

__device__ __forceinline__ unsigned s32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(s32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(s32(bar)), "r"(bytes) : "memory");
}
// wait for the phase with the given parity; after 65 536 failed polls the wait backs off and is bounded by wall time
// (mbar.cuh): a slow tile is waited for, a tile that has not landed after 10 s traps instead of hanging the GPU
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  unsigned ok = 0;
  for (int spin = 0; !ok; ++spin) {
    asm volatile(
        "{\n.reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n}\n"
        : "=r"(ok) : "r"(s32(bar)), "r"(parity) : "memory");
    if (!ok && spin > (1 << 16)) { mmx_mbar_wait_slow(s32(bar), parity); return; }
  }
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(s32(dst)), "l"(src), "r"(bytes), "r"(s32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* dst, const void* src, unsigned bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(s32(src)), "r"(bytes) : "memory");
}

// position of tile T: complex offset of its block in spec2T, kernel image index, outer wave number
struct TilePos {
  unsigned off, img;
  int ky;       // main tile: the ky of all its columns; Nyquist tile: ky of column 0
  bool nyq;
};
__device__ __forceinline__ TilePos tile_pos(const TileArgs& a, int T) {
  const int tile_elems = 3 * a.nz * TL;
  const int npair = 2 * (a.py / 2 - 1) * a.ntx;  // tiles of ky = 1 .. Py/2 - 1 and their mirrors, pairs adjacent
  TilePos p;
  p.nyq = false;
  int tx;
  if (T < npair) {
    const int q = T >> 1, kyh = 1 + q / a.ntx;
    tx = q - (kyh - 1) * a.ntx;
    p.ky = (T & 1) ? a.py - kyh : kyh;
    p.img = kyh * a.ntx + tx;
  } else if (T < npair + 2 * a.ntx) {
    const int r = T - npair;
    p.ky = r < a.ntx ? 0 : a.py / 2;
    tx = r < a.ntx ? r : r - a.ntx;
    p.img = p.ky * a.ntx + tx;
  } else {
    const int kyt = T - npair - 2 * a.ntx;
    p.nyq = true;
    p.ky = kyt * TL;
    p.img = (a.py / 2 + 1) * a.ntx + kyt;
    p.off = (unsigned)(a.py * a.ntx + kyt) * (unsigned)tile_elems;
    return p;
  }
  p.off = (unsigned)(p.ky * a.ntx + tx) * (unsigned)tile_elems;
  return p;
}

__global__ void __launch_bounds__(32 * NW, 2) k_inner_tile(TileArgs a) {
  extern __shared__ __align__(128) unsigned char smraw[];
  float2* xs0 = reinterpret_cast<float2*>(smraw);
  float* ks = reinterpret_cast<float*>(smraw + NXS * XS_BYTES);
  float2* exw = reinterpret_cast<float2*>(smraw + NXS * XS_BYTES + KS_BYTES);
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(smraw + NXS * XS_BYTES + KS_BYTES + EX_BYTES);
  unsigned long long* full = bars;       // [NXS] "spectrum stage s has landed"
  unsigned long long* kfull = bars + 3;  // "kernel image has landed"
  int* cnt = reinterpret_cast<int*>(bars + 4);  // [NXS] tickets "warps done with stage s", [3] "warps past the multiply"

  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int col = lane & 1, j = (lane >> 1) & 7, h = lane >> 4;
  if (!a.ctrl->active) return;

  // twiddles of this thread: stage w_H^(j q), half w_P^(j + R u) (identity for the even half)
  float2 tws[R], twp[R];
#pragma unroll
  for (int q = 0; q < R; ++q) {
    tws[q] = a.tw[2 * j * q];
    twp[q] = h ? a.tw[j + R * q] : make_float2(1.f, 0.f);
  }

  const int G = gridDim.x;
  const unsigned xbytes = (unsigned)a.nz * TL * 8;  // one component of a tile
  auto seqT = [&](int i) -> int { return 2 * ((int)blockIdx.x + G * (i >> 1)) + (i & 1); };
  static_assert(NXS == 2 || NXS == 3, "two or three spectrum stages");
  auto load_tile = [&](int T, int s) {
    const TilePos p = tile_pos(a, T);
    mbar_expect_tx(&full[s], 3 * xbytes);
#pragma unroll
    for (int c = 0; c < 3; ++c)
      bulk_g2s(reinterpret_cast<unsigned char*>(xs0) + s * XS_BYTES + c * (H * TL * 8), a.spec + p.off + (unsigned)c * (unsigned)(a.nz * TL),
               xbytes, &full[s]);
  };
  auto load_kimg = [&](unsigned img) {
    mbar_expect_tx(kfull, KS_BYTES);
    bulk_g2s(ks, a.kimg + (size_t)img * KS_FLOATS, KS_BYTES, kfull);
  };

  if (a.nz < H) {  // rows that are zero padding: cleared once, never written (generic proxy, fenced below)
    for (int q = threadIdx.x; q < NXS * XS_BYTES / 16; q += 32 * NW) reinterpret_cast<float4*>(smraw)[q] = make_float4(0.f, 0.f, 0.f, 0.f);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  if (threadIdx.x == 0) {
    for (int q = 0; q < NXS; ++q) mbar_init(&full[q], 1);
    mbar_init(kfull, 1);
    for (int q = 0; q < 6; ++q) cnt[q] = 0;
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (threadIdx.x == 0 && seqT(0) < a.ntiles) {
    load_tile(seqT(0), 0);
    load_kimg(tile_pos(a, seqT(0)).img);
    for (int q = 1; q < NXS; ++q)
      if (seqT(q) < a.ntiles) load_tile(seqT(q), q);
  }

  // per-thread constants of the swizzled layouts
  const int pos_lo = ((w ^ j) << 1) | col;                    // spectrum rows z with (z & 7) = j; kernel rows kz <= 64
  const int pos_hi = ((w ^ ((-j - h) & 7)) << 1) | col;       // mirrored kernel rows 128 - kz
  float2* ex0 = exw + w * NEXR * EXR + h * (H * 2) + col;      // this thread's half of region 0
  const float* kp_lo = ks + (2 * j + h) * TL + pos_lo;
  const float* kp_hi = ks + (P - 2 * j - h) * TL + pos_hi;
  const unsigned mi3 = ((a.odd_inner >> 3) & 1u) << 31, mi4 = ((a.odd_inner >> 4) & 1u) << 31, mi5 = ((a.odd_inner >> 5) & 1u) << 31;

  unsigned kuse = 0, prev_img = 0xffffffffu;
  int T = seqT(0);
  int s = 0;
  unsigned par = 0;   // parity of the current use of stage s
  for (int i = 0; T < a.ntiles; ++i) {
    const TilePos tp = tile_pos(a, T);
    const int Tn = seqT(i + 1);
    const bool more = Tn < a.ntiles;
    const unsigned next_img = more ? tile_pos(a, Tn).img : 0xffffffffu;
    float2* xs = xs0 + s * (XS_BYTES / 8) + pos_lo;
    const int ky = tp.nyq ? tp.ky + 2 * w + col : tp.ky;
    const unsigned so = 2 * ky > a.py ? 1u : 0u;

    mbar_wait(&full[s], par);
    float2 X[3][R];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
#pragma unroll
      for (int u = 0; u < R; ++u) X[c][u] = cmul(xs[(c * H + j + R * u) * TL], twp[u]);
      Dft<R, -1>::run(X[c]);
      float2* t = ex0 + (c % NEXR) * EXR;
      if (c >= NEXR) __syncwarp();  // the region is reused: its previous component has been read by every lane
      t[exrow(0, j)] = X[c][0];
#pragma unroll
      for (int q = 1; q < R; ++q) t[exrow(q, j)] = cmul(X[c][q], tws[q]);
      __syncwarp();
#pragma unroll
      for (int q = 0; q < R; ++q) X[c][q] = t[exrow(j, q)];
      Dft<R, -1>::run(X[c]);
    }
    if (tp.img != prev_img) {  // a new kernel image was requested for this tile
      mbar_wait(kfull, kuse & 1u);
      ++kuse;
      prev_img = tp.img;
    }
    // B^_i = sum_j K^_ij M^_j ; K^ real, octant + parity (sign bit flips)
    const unsigned mo3 = (so & (a.odd_outer >> 3)) << 31, mo4 = (so & (a.odd_outer >> 4)) << 31, mo5 = (so & (a.odd_outer >> 5)) << 31;
#pragma unroll
    for (int b = 0; b < R; ++b) {
      const bool mir = b > 4 || (b == 4 && (j | h) != 0);   // kz = 16 b + 2 j + h > 64
      const float* kp = b < 4 ? kp_lo + b * (2 * R * TL) : kp_hi - b * (2 * R * TL);
      const float k0 = kp[0 * (H + 1) * TL], k1 = kp[1 * (H + 1) * TL], k2 = kp[2 * (H + 1) * TL];
      const float k3 = __uint_as_float(__float_as_uint(kp[3 * (H + 1) * TL]) ^ mo3 ^ (mir ? mi3 : 0u));
      const float k4 = __uint_as_float(__float_as_uint(kp[4 * (H + 1) * TL]) ^ mo4 ^ (mir ? mi4 : 0u));
      const float k5 = __uint_as_float(__float_as_uint(kp[5 * (H + 1) * TL]) ^ mo5 ^ (mir ? mi5 : 0u));
      const float2 mx = X[0][b], my = X[1][b], mz = X[2][b];
      X[0][b] = rfma(k0, mx, rfma(k3, my, rmul(k4, mz)));
      X[1][b] = rfma(k3, mx, rfma(k1, my, rmul(k5, mz)));
      X[2][b] = rfma(k4, mx, rfma(k5, my, rmul(k2, mz)));
    }
    if (more && next_img != tp.img) {
      // the next tile needs another image: the last warp past the multiply fetches it
      __syncwarp();
      if (lane == 0) {
        __threadfence_block();
        if (atomicAdd(&cnt[NXS], 1) == NW - 1) {
          cnt[NXS] = 0;
          __threadfence_block();
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          load_kimg(next_img);
        }
      }
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      Dft<R, +1>::run(X[c]);
      float2* t = ex0 + (c % NEXR) * EXR;
      __syncwarp();  // the region's previous contents have been read by every lane
      t[exrow(j, 0)] = X[c][0];
#pragma unroll
      for (int q = 1; q < R; ++q) t[exrow(j, q)] = cmulc(X[c][q], tws[q]);
      __syncwarp();
#pragma unroll
      for (int q = 0; q < R; ++q) X[c][q] = t[exrow(q, j)];
      Dft<R, +1>::run(X[c]);
#pragma unroll
      for (int b = 0; b < R; ++b) X[c][b] = cmulc(X[c][b], twp[b]);
      // x[n] = g0[n] + conj(w_P^n) g1[n]: lanes h = 0 finish rows b < R/2, lanes h = 1 the others; the
      // result replaces the input in the stage (this warp's two columns only)
#pragma unroll
      for (int bb = 0; bb < R / 2; ++bb) {
        const float2 mine = h ? X[c][bb + R / 2] : X[c][bb];
        const float2 send = h ? X[c][bb] : X[c][bb + R / 2];
        float2 recv;
        recv.x = __shfl_xor_sync(0xffffffffu, send.x, 16);
        recv.y = __shfl_xor_sync(0xffffffffu, send.y, 16);
        const int n = j + R * (h ? bb + R / 2 : bb);
        if (n < a.nz) xs[(c * H + n) * TL] = cadd(mine, recv);
      }
    }
    // hand the finished tile to the async proxy; the last warp writes it back and refills the stage
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncwarp();
    if (lane == 0) {
      __threadfence_block();
      if (atomicAdd(&cnt[s], 1) == NW - 1) {
        cnt[s] = 0;
        __threadfence_block();
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
#pragma unroll
        for (int c = 0; c < 3; ++c)
          bulk_s2g(a.spec + tp.off + (unsigned)c * (unsigned)(a.nz * TL),
                   reinterpret_cast<unsigned char*>(xs0) + s * XS_BYTES + c * (H * TL * 8), xbytes);
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        const int T2 = seqT(i + NXS);
        if (T2 < a.ntiles) {
          asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");  // the stage has been read out
          load_tile(T2, s);
        }
      }
    }
    T = Tn;
    if (++s == NXS) { s = 0; par ^= 1u; }
  }
  if (lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");  // my write-backs are complete
}

}  // namespace

// ---- host side ---------------------------------------------------------------------------------------

// complex offset of element (slab = c nz + z, ky, kx) in the tile-major layout (also used by the y passes)
size_t mmx_tile_spec_elems(int py, int xc, int nz) {
  const int ntx = (xc - 1) / TL;
  return ((size_t)py * ntx + py / TL) * 3 * nz * TL;
}
size_t mmx_tile_kimg_floats(int py, int xc) {
  const int ntx = (xc - 1) / TL;
  return ((size_t)(py / 2 + 1) * ntx + py / TL) * KS_FLOATS;
}

bool mmx_tile_ok(const DemagPlan& d) {
  return d.nz > 1 && d.pz == P && d.nz <= H && d.py >= 32 && d.py % 32 == 0 && d.xc > 1 && (d.xc - 1) % TL == 0 &&
         mmx_tile_spec_elems(d.py, d.xc, d.nz) < (1ull << 31);
}

// kernel images from the octant spectrum khat [6][kz = 65][ky = Py/2+1][xp]: image (kyh, tx) column l is
// kx = 16 tx + l at ky = kyh; Nyquist image kyt column l is ky = 16 kyt + l (mirrored into the octant) at
// kx = xc - 1.  Float (comp, pm, l) of an image sits at (comp 65 + pm) 16 + (((l >> 1) ^ ((pm >> 1) & 7)) << 1 | (l & 1)).
void mmx_tile_kimg_build(const DemagPlan& d, const std::vector<float>& khat, std::vector<float>& out) {
  const int ntx = (d.xc - 1) / TL, kyn = d.py / 2 + 1;
  out.assign(mmx_tile_kimg_floats(d.py, d.xc), 0.f);
  auto K = [&](int comp, int pm, int kyh, int kx) -> float {
    return khat[(((size_t)comp * d.kz + pm) * d.ky + kyh) * d.xp + kx];
  };
  auto put = [&](float* img, int comp, int pm, int l, float v) {
    img[(comp * (H + 1) + pm) * TL + ((((l >> 1) ^ ((pm >> 1) & 7)) << 1) | (l & 1))] = v;
  };
#pragma omp parallel for schedule(static)
  for (int kyh = 0; kyh < kyn; ++kyh)
    for (int tx = 0; tx < ntx; ++tx) {
      float* img = out.data() + ((size_t)kyh * ntx + tx) * KS_FLOATS;
      for (int comp = 0; comp < 6; ++comp)
        for (int pm = 0; pm <= H; ++pm)
          for (int l = 0; l < TL; ++l) put(img, comp, pm, l, K(comp, pm, kyh, tx * TL + l));
    }
  for (int kyt = 0; kyt < d.py / TL; ++kyt) {
    float* img = out.data() + ((size_t)kyn * ntx + kyt) * KS_FLOATS;
    for (int comp = 0; comp < 6; ++comp)
      for (int pm = 0; pm <= H; ++pm)
        for (int l = 0; l < TL; ++l) {
          const int ky = kyt * TL + l, kom = 2 * ky > d.py ? d.py - ky : ky;
          put(img, comp, pm, l, K(comp, pm, kom, d.xc - 1));
        }
  }
}

int mmx_inner_tile_launch(mmx_world* w) {
  const DemagPlan& d = w->dm;
  TileArgs a;
  a.spec = d.spec2; a.kimg = d.kimg; a.tw = d.tw[2]; a.ctrl = w->d_ctrl;
  a.nz = d.nz; a.ntx = (d.xc - 1) / TL; a.py = d.py;
  a.ntiles = d.py * a.ntx + d.py / TL;
  a.odd_inner = (1u << 4) | (1u << 5); a.odd_outer = (1u << 3) | (1u << 5);
  ProfScope ps(w, PK_INNER);
  MMX_CUDA(cudaFuncSetAttribute(k_inner_tile, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES));
  int grid = mmx_persistent_grid(k_inner_tile, 32 * NW, SMEM_BYTES, w->sm_count, 2);
  if (2 * grid > a.ntiles) grid = a.ntiles / 2;   // (ntiles is even: every CTA starts on a pair)
  MMX_CUDA(mmx_launch(k_inner_tile, grid, 32 * NW, SMEM_BYTES, w->stream, a));
  MMX_CUDA(cudaGetLastError());
  return MMX_OK;
}
