// fft.cuh -- power-of-two complex FFT of a shared-memory tile, fp32.
//
// Used by the five demag passes (demag.cu).  A tile holds L lines of P complex points,
// laid out s[pos * LP + line] (line index fastest, LP >= L), so that the threads of a warp
// that work on the same butterfly index of neighbouring lines touch consecutive words:
// every shared-memory access of the transform is bank-conflict free without padding.
//
// Algorithm: in-place Stockham autosort, decimation in time, radix 8 with a radix-4 / radix-2
// tail (P = 8^a * {1,2,4}).  One thread owns E = min(P, 8) points of one line per stage:
//   stage (R, Ns):   for butterfly b in [0, P/R):  k = b mod Ns
//       v[r]  = x[b + r P/R] * w^(k r),  w = exp(DIR 2 pi i / (Ns R)),  r = 0..R-1
//       v     = DFT_R(v)
//       x[(b / Ns) Ns R + k + r Ns] = v[r]
// All threads load, then a block barrier, then all store, then a barrier: in place, the
// output is in natural order after the last stage.  Twiddles come from a table
// tw[q] = exp(-2 pi i q / P) built in fp64 on the host (inverse transforms conjugate it).
//
// Everything here is __host__ __device__ so the index logic can be exercised on the CPU.
#pragma once
#include <cuda_runtime.h>

#ifndef MMX_HD
#define MMX_HD __host__ __device__ __forceinline__
#endif

namespace mmxfft {

MMX_HD float2 cmul(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
MMX_HD float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
MMX_HD float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
// multiply by DIR * i  (DIR = -1: forward transform, multiply by -i)
template <int DIR>
MMX_HD float2 mul_i(float2 a) {
  return DIR < 0 ? make_float2(a.y, -a.x) : make_float2(-a.y, a.x);
}

template <int DIR>
MMX_HD void dft2(float2& a, float2& b) {
  float2 t = a;
  a = cadd(t, b);
  b = csub(t, b);
}

// 4-point DFT, natural order in and out:  X[q] = sum_r x[r] exp(DIR 2 pi i q r / 4)
template <int DIR>
MMX_HD void dft4(float2& x0, float2& x1, float2& x2, float2& x3) {
  float2 a = cadd(x0, x2), b = csub(x0, x2);
  float2 c = cadd(x1, x3), d = mul_i<DIR>(csub(x1, x3));
  x0 = cadd(a, c);
  x1 = cadd(b, d);
  x2 = csub(a, c);
  x3 = csub(b, d);
}

// 8-point DFT, natural order in and out.
template <int DIR>
MMX_HD void dft8(float2* v) {
  const float h = 0.70710678118654752440f;
  // even / odd split: E = DFT4(v0,v2,v4,v6), O = DFT4(v1,v3,v5,v7)
  float2 e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6];
  float2 o0 = v[1], o1 = v[3], o2 = v[5], o3 = v[7];
  dft4<DIR>(e0, e1, e2, e3);
  dft4<DIR>(o0, o1, o2, o3);
  // twiddles w8^q, w8 = exp(DIR 2 pi i / 8)
  // q=1: (h, DIR h); q=2: DIR i; q=3: (-h, DIR h)
  float2 t1 = DIR < 0 ? make_float2(h * (o1.x + o1.y), h * (o1.y - o1.x))
                      : make_float2(h * (o1.x - o1.y), h * (o1.y + o1.x));
  float2 t2 = mul_i<DIR>(o2);
  float2 t3 = DIR < 0 ? make_float2(h * (o3.y - o3.x), -h * (o3.x + o3.y))
                      : make_float2(-h * (o3.x + o3.y), h * (o3.x - o3.y));
  v[0] = cadd(e0, o0);
  v[4] = csub(e0, o0);
  v[1] = cadd(e1, t1);
  v[5] = csub(e1, t1);
  v[2] = cadd(e2, t2);
  v[6] = csub(e2, t2);
  v[3] = cadd(e3, t3);
  v[7] = csub(e3, t3);
}

constexpr int elems_per_thread(int P) { return P < 8 ? P : 8; }
constexpr int threads_per_line(int P) { return P / elems_per_thread(P); }
// radix of the stage that starts with stride Ns
constexpr int stage_radix(int P, int Ns) { return (P / Ns) >= 8 ? 8 : (P / Ns); }

// Load + twiddle + butterflies of one stage for thread (line, j), j in [0, P/E).
// v[u] holds point  j + u * P/E  of the line (u = q + r * E/R for butterfly q, input r).
template <int P, int DIR, int R, int NS>
MMX_HD void stage_load(const float2* __restrict__ s, int LP, int line, int j,
                       const float2* __restrict__ tw, float2* v) {
  constexpr int E = elems_per_thread(P);
  constexpr int NB = E / R;  // butterflies per thread
#pragma unroll
  for (int u = 0; u < E; ++u) v[u] = s[(j + u * (P / E)) * LP + line];
#pragma unroll
  for (int q = 0; q < NB; ++q) {
    const int b = j + q * (P / E);
    if (NS > 1) {
      const int k = b % NS;
#pragma unroll
      for (int r = 1; r < R; ++r) {
        float2 w = tw[k * r * (P / (NS * R))];
        if (DIR > 0) w.y = -w.y;
        v[q + r * NB] = cmul(v[q + r * NB], w);
      }
    }
    if (R == 8) {
      float2 t[8];
#pragma unroll
      for (int r = 0; r < 8; ++r) t[r] = v[q + r * NB];
      dft8<DIR>(t);
#pragma unroll
      for (int r = 0; r < 8; ++r) v[q + r * NB] = t[r];
    } else if (R == 4) {
      dft4<DIR>(v[q], v[q + NB], v[q + 2 * NB], v[q + 3 * NB]);
    } else if (R == 2) {
      dft2<DIR>(v[q], v[q + NB]);
    }
  }
}

template <int P, int R, int NS>
MMX_HD void stage_store(float2* __restrict__ s, int LP, int line, int j, const float2* v) {
  constexpr int E = elems_per_thread(P);
  constexpr int NB = E / R;
#pragma unroll
  for (int q = 0; q < NB; ++q) {
    const int b = j + q * (P / E);
    const int k = b % NS;
    const int j0 = (b / NS) * (NS * R) + k;
#pragma unroll
    for (int r = 0; r < R; ++r) s[(j0 + r * NS) * LP + line] = v[q + r * NB];
  }
}

#ifdef __CUDACC__
// All threads of the block must call this (it contains block barriers).  Threads with
// active == false take part in the barriers only.  The tile must be fully written and a
// barrier passed before the call; on return the result is visible to all threads.
template <int P, int DIR, int NS = 1>
struct InPlace {
  static __device__ __forceinline__ void run(float2* s, int LP, int line, int j,
                                             const float2* __restrict__ tw, bool active) {
    constexpr int R = stage_radix(P, NS);
    float2 v[elems_per_thread(P)];
    if (active) stage_load<P, DIR, R, NS>(s, LP, line, j, tw, v);
    __syncthreads();
    if (active) stage_store<P, R, NS>(s, LP, line, j, v);
    __syncthreads();
    if constexpr (NS * R < P) InPlace<P, DIR, NS * R>::run(s, LP, line, j, tw, active);
  }
};
#endif

}  // namespace mmxfft
