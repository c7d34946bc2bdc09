// fft_reg.cuh -- register-resident radix-4/8/16 DFT butterflies, fp32, for the "column" FFT
// kernels of demag.cu (one thread owns R points of a line, R threads own a line of R*R
// points, the only exchange between the two radix-R stages goes through shared memory).
//
// A transform of length P = 2 R^2 along a strided axis is split by one radix-2
// decimation-in-frequency step into its even and odd outputs,
//     X[2k]   = DFT_H( x[n] + x[n+H] )[k]
//     X[2k+1] = DFT_H( (x[n] - x[n+H]) w_P^n )[k]            H = P/2 = R^2, w_P = exp(-2 pi i/P)
// and the zero padding of the demag convolution (x[n] = 0 for n >= H on an open axis) makes
// the butterfly free: both halves start from the same H loaded points.  The inverse uses the
// mirrored decimation-in-time step and needs only the first H outputs,
//     x[n] = IDFT_H(X[2k])[n] + conj(w_P^n) IDFT_H(X[2k+1])[n].
// Each H-point transform is two radix-R stages:
//     n = j + R u, k = a + R b:   X[a + R b] = sum_j w_R^(j b) [ w_H^(j a) sum_u x[j + R u] w_R^(u a) ]
// Twiddles come from a table tw[q] = exp(-2 pi i q / P) rounded from fp64 (never products of
// fp32 twiddles), so w_H^(j a) = tw[2 j a] and w_P^n = tw[n].
#pragma once
#include <cuda_runtime.h>

namespace mmxreg {

#define MMX_DI __device__ __forceinline__

// Packed fp32 pairs (PTX add / sub / mul / fma .f32x2, sm_100: SASS FADD2 / FMUL2 / FFMA2).  On sm_100 a
// scalar FFMA / FADD / FMUL occupies the fp32 pipe of a scheduler for two cycles; the packed forms do
// two lanes' worth in the same slot, so a complex number (re, im) in one aligned register pair halves
// both the instruction count and the pipe time of the butterflies.  The SASS operands carry free
// modifiers -- swap of the halves (.LO_HI), a sign per half (.NP / .PN), scalar broadcast (.F32) --
// and ptxas folds the mov.b64 {hi, lo} packings below into them, so
//   complex multiply      a w = a (w.x, w.x) + swap(a) (-w.y, w.y)           FMUL2 + FFMA2
//   b +- i d                  = b +- (-d.y, d.x)                              one FADD2
//   real scalar k times a     = (k, k) a                                       one FMUL2 / FFMA2
// (checked with cuobjdump -sass: no MOV / PRMT is emitted for the packings).  Same IEEE operations per
// component as the scalar forms, in a different association for the multiplies.
typedef unsigned long long pk2;
MMX_DI pk2 pk(float lo, float hi) {
  pk2 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
MMX_DI pk2 pk(float2 a) { return pk(a.x, a.y); }
MMX_DI float2 up(pk2 v) {
  float2 r;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v));
  return r;
}
MMX_DI pk2 add2(pk2 a, pk2 b) { pk2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
MMX_DI pk2 sub2(pk2 a, pk2 b) { pk2 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
MMX_DI pk2 mul2(pk2 a, pk2 b) { pk2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
MMX_DI pk2 fma2(pk2 a, pk2 b, pk2 c) { pk2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }

#ifndef MMX_PACKED_F32X2
#define MMX_PACKED_F32X2 1
#endif
#ifndef MMX_PACKED_R16
#define MMX_PACKED_R16 MMX_PACKED_F32X2
#endif
MMX_DI float2 cadd_pk(float2 a, float2 b) { return up(add2(pk(a), pk(b))); }
MMX_DI float2 csub_pk(float2 a, float2 b) { return up(sub2(pk(a), pk(b))); }
MMX_DI float2 cadd_sc(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
MMX_DI float2 csub_sc(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
template <bool PK>
MMX_DI float2 caddt(float2 a, float2 b) { return PK ? cadd_pk(a, b) : cadd_sc(a, b); }
template <bool PK>
MMX_DI float2 csubt(float2 a, float2 b) { return PK ? csub_pk(a, b) : csub_sc(a, b); }
MMX_DI float2 cadd(float2 a, float2 b) { return caddt<MMX_PACKED_F32X2 != 0>(a, b); }
MMX_DI float2 csub(float2 a, float2 b) { return csubt<MMX_PACKED_F32X2 != 0>(a, b); }
#if MMX_PACKED_F32X2
MMX_DI float2 cmul(float2 a, float2 b) { return up(fma2(pk(a.y, a.x), pk(-b.y, b.y), mul2(pk(a), pk(b.x, b.x)))); }
// a * conj(b)
MMX_DI float2 cmulc(float2 a, float2 b) { return up(fma2(pk(a.y, a.x), pk(b.y, -b.y), mul2(pk(a), pk(b.x, b.x)))); }
// real scalar times complex, and its accumulate form
MMX_DI float2 rmul(float k, float2 a) { return up(mul2(pk(k, k), pk(a))); }
MMX_DI float2 rfma(float k, float2 a, float2 c) { return up(fma2(pk(k, k), pk(a), pk(c))); }
#else
MMX_DI float2 cmul(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
MMX_DI float2 cmulc(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, a.y * b.y), fmaf(a.y, b.x, -a.x * b.y));
}
MMX_DI float2 rmul(float k, float2 a) { return make_float2(k * a.x, k * a.y); }
MMX_DI float2 rfma(float k, float2 a, float2 c) { return make_float2(fmaf(k, a.x, c.x), fmaf(k, a.y, c.y)); }
#endif
// a * w (DIR < 0, forward) or a * conj(w) (DIR > 0, inverse), w a forward twiddle
template <int DIR>
MMX_DI float2 ctw(float2 a, float2 w) {
  return DIR < 0 ? cmul(a, w) : cmulc(a, w);
}
// multiply by DIR * i
template <int DIR>
MMX_DI float2 mul_i(float2 a) {
  return DIR < 0 ? make_float2(a.y, -a.x) : make_float2(-a.y, a.x);
}
// multiply by (c + i DIR s): exp(DIR i theta) with c = cos theta, s = sin theta
template <int DIR>
MMX_DI float2 rot(float2 a, float c, float s) {
  const float d = DIR < 0 ? -s : s;
#if MMX_PACKED_F32X2
  return up(fma2(pk(a.y, a.x), pk(-d, d), mul2(pk(a), pk(c, c))));
#else
  return make_float2(fmaf(a.x, c, -a.y * d), fmaf(a.x, d, a.y * c));
#endif
}

// b + (DIR i) d and b - (DIR i) d
template <int DIR, bool PK = (MMX_PACKED_F32X2 != 0)>
MMX_DI float2 cadd_i(float2 b, float2 d) {
  if (PK) return DIR < 0 ? up(add2(pk(b), pk(d.y, -d.x))) : up(add2(pk(b), pk(-d.y, d.x)));
  return DIR < 0 ? make_float2(b.x + d.y, b.y - d.x) : make_float2(b.x - d.y, b.y + d.x);
}
template <int DIR, bool PK = (MMX_PACKED_F32X2 != 0)>
MMX_DI float2 csub_i(float2 b, float2 d) {
  if (PK) return DIR < 0 ? up(sub2(pk(b), pk(d.y, -d.x))) : up(sub2(pk(b), pk(-d.y, d.x)));
  return DIR < 0 ? make_float2(b.x - d.y, b.y + d.x) : make_float2(b.x + d.y, b.y - d.x);
}

template <int DIR, bool PK = (MMX_PACKED_F32X2 != 0)>
MMX_DI void dft4(float2& x0, float2& x1, float2& x2, float2& x3) {
  const float2 a = caddt<PK>(x0, x2), b = csubt<PK>(x0, x2);
  const float2 c = caddt<PK>(x1, x3), d = csubt<PK>(x1, x3);
  x0 = caddt<PK>(a, c);
  x1 = cadd_i<DIR, PK>(b, d);
  x2 = csubt<PK>(a, c);
  x3 = csub_i<DIR, PK>(b, d);
}

// X[q] = sum_r v[r] exp(DIR 2 pi i q r / R), natural order in and out
template <int R, int DIR>
struct Dft;

template <int DIR>
struct Dft<4, DIR> {
  static MMX_DI void run(float2* v) { dft4<DIR>(v[0], v[1], v[2], v[3]); }
};

template <int DIR>
struct Dft<8, DIR> {
  static MMX_DI void run(float2* v) {
    const float h = 0.70710678118654752440f;
    float2 e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6];
    float2 o0 = v[1], o1 = v[3], o2 = v[5], o3 = v[7];
    dft4<DIR>(e0, e1, e2, e3);
    dft4<DIR>(o0, o1, o2, o3);
    const float2 t1 = rot<DIR>(o1, h, h);
    const float2 t3 = rot<DIR>(o3, -h, h);
    v[0] = cadd(e0, o0); v[4] = csub(e0, o0);
    v[1] = cadd(e1, t1); v[5] = csub(e1, t1);
    v[2] = cadd_i<DIR>(e2, o2); v[6] = csub_i<DIR>(e2, o2);
    v[3] = cadd(e3, t3); v[7] = csub(e3, t3);
  }
};

template <int DIR>
struct Dft<16, DIR> {
  // 16 = 4 x 4:  n = 4 n1 + n2,  k = k1 + 4 k2
  //   X[k1 + 4 k2] = sum_n2 w4^(n2 k2) [ w16^(n2 k1) sum_n1 v[4 n1 + n2] w4^(n1 k1) ]
  static MMX_DI void run(float2* v) {
    const float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f;
    const float h = 0.70710678118654752440f;
    float2 t[4][4];  // t[n2][k1]
#pragma unroll
    for (int n2 = 0; n2 < 4; ++n2) {
      t[n2][0] = v[n2]; t[n2][1] = v[4 + n2]; t[n2][2] = v[8 + n2]; t[n2][3] = v[12 + n2];
      dft4<DIR, MMX_PACKED_R16 != 0>(t[n2][0], t[n2][1], t[n2][2], t[n2][3]);
    }
    // w16^(n2 k1)
    t[1][1] = rot<DIR>(t[1][1], c1, s1);
    t[1][2] = rot<DIR>(t[1][2], h, h);
    t[1][3] = rot<DIR>(t[1][3], s1, c1);
    t[2][1] = rot<DIR>(t[2][1], h, h);
    t[2][2] = mul_i<DIR>(t[2][2]);
    t[2][3] = rot<DIR>(t[2][3], -h, h);
    t[3][1] = rot<DIR>(t[3][1], s1, c1);
    t[3][2] = rot<DIR>(t[3][2], -h, h);
    t[3][3] = rot<DIR>(t[3][3], -c1, -s1);  // w16^9 = -w16^1
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) {
      dft4<DIR, MMX_PACKED_R16 != 0>(t[0][k1], t[1][k1], t[2][k1], t[3][k1]);  // index k2 now lives in the first slot
      v[k1] = t[0][k1]; v[k1 + 4] = t[1][k1]; v[k1 + 8] = t[2][k1]; v[k1 + 12] = t[3][k1];
    }
  }
};

}  // namespace mmxreg
