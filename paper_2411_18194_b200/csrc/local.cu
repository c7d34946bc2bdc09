// local.cu -- fused local effective field + torque + Runge-Kutta stage combination + error /
// max-torque reduction, and the device-side step controller.
//
// Per cell c of sublattice s (partner sublattice s'):
//   B_exch  = sum_n 2 A_cn /(Ms_c h_n^2) (m_n - m_c)                  Eq.3 term 1
//   B_A12   = sum_n A12_cn /(Ms_c h_n^2) (m'_n - m'_c)                Eq.3 term 2
//   B_A0    = 4 A0 /(a^2 Ms_c) m'_c                                    Eq.3 term 3
//   B_Dhom  = (d x m2)/Ms1 on sublattice 1, (m1 x d)/Ms2 on sublattice 2      Eq.6
//   B_DMI   = sum_{n in +-x,+-y} D_cn /(Ms_c h_n) (z x e_cn) x m_n     Eq.4, interfacial subset
//           + sum_i sum_{+-} +-1/(Ms_c h_i) q_i x m_n                   Eq.4, general tensor (k_local only)
//   B_anis  = 2Ku1/Ms (u.m) u  - 2Kc1/Ms sum_i (c_i.m)[(c_j.m)^2+(c_k.m)^2] c_i
//   B_mel   = -2/Ms [B1 eps_ii m_i + B2 (eps_ij m_j + eps_ik m_k)]     Eq.9
//   B_eff   = sum of the above + B_ext + B_demag
//   tau     = -gamma/(1+alpha^2) [m x B + alpha m x (m x B)]           Eq.2
//           + Zhang-Li torque
// A neighbour takes part only if it lies in the grid (after periodic wrap) and has Ms > 0
// ("open" boundary = the pair is dropped).  A_cn, D_cn are harmonic means; A_cn, A12_cn carry
// the region-pair scale factor across grain boundaries.
// The epilogue forms the next stage state  normalise(y0 + sum_j (dt a_ij) k_j)  (Table 2,
// P:L122-131) and, on the last stage, the embedded error  max_c |sum_j (dt e_j) k_j|_2.
#include <cuda.h>
#include <cudaTypedefs.h>

#include <cstdio>

#include "mbar.cuh"
#include "mmx_internal.h"

namespace {

struct V3 {
  float x, y, z;
};
__device__ __forceinline__ V3 v3(float x, float y, float z) { V3 r = {x, y, z}; return r; }
__device__ __forceinline__ V3 operator+(V3 a, V3 b) { return v3(a.x + b.x, a.y + b.y, a.z + b.z); }
__device__ __forceinline__ V3 operator-(V3 a, V3 b) { return v3(a.x - b.x, a.y - b.y, a.z - b.z); }
__device__ __forceinline__ V3 operator*(float s, V3 a) { return v3(s * a.x, s * a.y, s * a.z); }
__device__ __forceinline__ V3 fma3(float s, V3 a, V3 b) { return v3(fmaf(s, a.x, b.x), fmaf(s, a.y, b.y), fmaf(s, a.z, b.z)); }
__device__ __forceinline__ float dot(V3 a, V3 b) { return fmaf(a.x, b.x, fmaf(a.y, b.y, a.z * b.z)); }
__device__ __forceinline__ V3 cross(V3 a, V3 b) {
  return v3(fmaf(a.y, b.z, -a.z * b.y), fmaf(a.z, b.x, -a.x * b.z), fmaf(a.x, b.y, -a.y * b.x));
}
__device__ __forceinline__ V3 ld3(const float* p, size_t N, size_t i) { return v3(p[i], p[N + i], p[2 * N + i]); }
__device__ __forceinline__ void st3(float* p, size_t N, size_t i, V3 v) { p[i] = v.x; p[N + i] = v.y; p[2 * N + i] = v.z; }
__device__ __forceinline__ float harm(float a, float b) {
  float s = a + b;
  return s != 0.f ? 2.f * a * b / s : 0.f;
}

__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// block-wide max of a non-negative float, result atomically folded into *target (bit pattern).
// NaN is mapped to +inf bits + 1 so that it survives the unsigned max and is seen by the controller.
__device__ __forceinline__ void block_max_to(float v, unsigned* target) {
  __shared__ unsigned smax[32];
  unsigned bits = (v != v) ? 0x7fc00000u : __float_as_uint(v);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) bits = max(bits, __shfl_xor_sync(0xffffffffu, bits, o));
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) smax[wid] = bits;
  __syncthreads();
  if (wid == 0) {
    const int nw = (blockDim.x + 31) >> 5;
    bits = lane < nw ? smax[lane] : 0u;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) bits = max(bits, __shfl_xor_sync(0xffffffffu, bits, o));
    if (lane == 0 && bits != 0u) atomicMax(target, bits);
  }
  __syncthreads();
}

// neighbour index of cell (ix,iy,iz) along axis by d = +-1, or -1 when outside an open axis
__device__ __forceinline__ long long nbr(const LocalArgs& a, int ix, int iy, int iz, int axis, int d) {
  int p[3] = {ix, iy, iz};
  const int n[3] = {a.nx, a.ny, a.nz};
  int q = p[axis] + d;
  if (q < 0 || q >= n[axis]) {
    if (!a.per[axis]) return -1;
    q = (q + n[axis]) % n[axis];
  }
  p[axis] = q;
  return ((long long)p[2] * a.ny + p[1]) * a.nx + p[0];
}

// Neumann boundary condition of Eq.5 as ghost cells, reading S41: normal derivatives g = d_n m of sublattice
// s and (two sublattices) of its partner o at a face with outward normal d e_axis, from
//     2 A g + A12 P_m g' = m x q_n,   2 A' g' + A12 P_m' g = m' x q'_n,   q_n = d (q_axis + interfacial part)
// solved in closed form (w = P_m m', beta = A12^2/(2A'), R = r - (A12/2A') P_m r'):
//     g.w = R.w/(2A - beta + beta |w|^2),  g = (R - beta (g.w) w)/(2A - beta),  g' = (r' - A12 P_m' g)/(2A').
__device__ __forceinline__ V3 qn_of(const LocalArgs& a, int s, int axis, float d, float Dc) {
  V3 q = v3(a.dmiq[s][axis][0], a.dmiq[s][axis][1], a.dmiq[s][axis][2]);
  if (axis == 0) q.y += Dc;        // interfacial D: q_x = D y^
  else if (axis == 1) q.x -= Dc;   //                q_y = -D x^
  return d * q;
}
__device__ __forceinline__ V3 perp(V3 v, V3 u) { return v - dot(v, u) * u; }
__device__ __forceinline__ void neumann_g(const LocalArgs& a, bool two, int s, int o, int axis, float d, V3 ms, V3 mo,
                                          const float* Ps, const float* Po, V3& gs, V3& go) {
  const float A = Ps[MP_A];
  const V3 r = cross(ms, qn_of(a, s, axis, d, Ps[MP_D]));
  gs = go = v3(0.f, 0.f, 0.f);
  if (!(A > 0.f)) return;
  if (!two || a.A12 == 0.f || !(Po[MP_A] > 0.f)) {
    gs = (0.5f / A) * r;
    if (two && Po[MP_A] > 0.f) go = (0.5f / Po[MP_A]) * cross(mo, qn_of(a, o, axis, d, Po[MP_D]));
    return;
  }
  const float iAp = 0.5f / Po[MP_A];
  const V3 rp = cross(mo, qn_of(a, o, axis, d, Po[MP_D]));
  const float beta = a.A12 * a.A12 * iAp, den = 2.f * A - beta;
  const V3 w = perp(mo, ms);
  const V3 R = r - (a.A12 * iAp) * perp(rp, ms);
  const float gw = dot(R, w) / (den + beta * dot(w, w));
  gs = (1.f / den) * (R - (beta * gw) * w);
  go = iAp * (rp - a.A12 * perp(gs, mo));
}

template <int S, bool REG>
__global__ void __launch_bounds__(256) k_local(LocalArgs a) {
  MmxCtrl* ctrl = a.ctrl;
  if (!ctrl->active) return;
  const int sel = ctrl->sel;
  const size_t N = (size_t)a.nx * a.ny * a.nz;
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const float* yin = a.yin[sel];
  float errv = 0.f, tqv = 0.f;
  bool bad = false;
  if (i < N) {
    // (32-bit index arithmetic: a world has fewer than 2^31 cells)
    const unsigned ci = (unsigned)i, rowi = ci / (unsigned)a.nx;
    const int ix = (int)(ci - rowi * (unsigned)a.nx), iz = (int)(rowi / (unsigned)a.ny), iy = (int)(rowi - (unsigned)iz * (unsigned)a.ny);
    const int rc = REG ? a.reg[i] : 0;
    long long ni[6];
    int rn[6];
#pragma unroll
    for (int q = 0; q < 6; ++q) {
      ni[q] = nbr(a, ix, iy, iz, q >> 1, (q & 1) ? -1 : +1);
      rn[q] = (REG && ni[q] >= 0) ? a.reg[ni[q]] : rc;
    }
    V3 mc[S];
#pragma unroll
    for (int s = 0; s < S; ++s) mc[s] = ld3(yin + (size_t)s * 3 * N, N, i);
    // neighbour values of every sublattice, loaded up front and unconditionally (an absent neighbour reads the centre
    // cell): the loads do not wait for the region -> material -> "is it magnetic" lookups of the neighbour, which is
    // what bounds this kernel on small, L2-resident grids (c3: 30 -> 2x us per call)
    V3 mnb[S][6];
#pragma unroll
    for (int s = 0; s < S; ++s)
#pragma unroll
      for (int q = 0; q < 6; ++q) mnb[s][q] = ld3(yin + (size_t)s * 3 * N, N, ni[q] >= 0 ? (size_t)ni[q] : i);

#pragma unroll
    for (int s = 0; s < S; ++s) {
      if (a.heff_out || a.tau_out) {
        if (s != a.heff_s) continue;
      }
      // partner sublattices o = (s + t) mod S, t = 1 .. S - 1: the inter-sublattice terms act between s and every
      // other sublattice (reading S38)
      const float* P = a.mat + ((size_t)s * a.nreg + rc) * MMX_MATW;
      const float Ms = P[MP_MS], iMs = P[MP_INVMS];
      V3 B = v3(0.f, 0.f, 0.f);
      V3 dm = v3(0.f, 0.f, 0.f);  // (u.grad) m for Zhang-Li
      V3 tau = v3(0.f, 0.f, 0.f);
      if (Ms > 0.f) {
        const float Ac = P[MP_A], Dc = P[MP_D];
        const float zlb = P[MP_ZLB];
#pragma unroll
        for (int q = 0; q < 6; ++q) {
          const int axis = q >> 1;
          const float d = (q & 1) ? -1.f : 1.f;
          V3 mn = mc[s];  // missing neighbour: centre value (only used by Zhang-Li)
          if (ni[q] >= 0) {
            const float* Pn = REG ? a.mat + ((size_t)s * a.nreg + rn[q]) * MMX_MATW : P;
            if (Pn[MP_MS] > 0.f) {
              mn = mnb[s][q];
              const bool same = rn[q] == rc;
              if (a.terms & MMX_T_EXCH) {
                // (same region: the harmonic mean of A with itself is A -- no division)
                const float wex = 2.f * (same ? Ac : harm(Ac, Pn[MP_A]) * a.scaleA11) * iMs * a.inv_h2[axis];
                B = fma3(wex, mn - mc[s], B);
              }
              if (axis < 2 && (a.terms & MMX_T_DMI)) {
                const float wd = (same ? Dc : harm(Dc, Pn[MP_D])) * iMs * a.inv_h[axis] * d;
                // (z x (d e_axis)) x m_n = d (m_z e_axis - m_axis z)
                if (axis == 0) { B.x = fmaf(wd, mn.z, B.x); B.z = fmaf(-wd, mn.x, B.z); }
                else { B.y = fmaf(wd, mn.z, B.y); B.z = fmaf(-wd, mn.y, B.z); }
              }
              if (a.has_dmiq && (a.terms & MMX_T_DMI)) {
                // general tensor of Eq.4: B_c += d /(Ms_c h_i) q_i x m_n
                const V3 qv = v3(a.dmiq[s][axis][0], a.dmiq[s][axis][1], a.dmiq[s][axis][2]);
                B = fma3(iMs * a.inv_h[axis] * d, cross(qv, mn), B);
              }
              if (S >= 2 && (a.terms & (MMX_T_A12 | MMX_T_DMI_INTER))) {
#pragma unroll
                for (int t = 1; t < S; ++t) {
                  const int o = (s + t) % S;
                  const V3 on = mnb[o][q];
                  if (a.terms & MMX_T_A12) {
                    const float w12 = a.A12 * (same ? 1.f : a.scaleA12) * iMs * a.inv_h2[axis];
                    B = fma3(w12, on - mc[o], B);
                  }
                  if (axis < 2 && (a.terms & MMX_T_DMI_INTER)) {
                    const float wd = a.Dinter * iMs * a.inv_h[axis] * d;
                    if (axis == 0) { B.x = fmaf(wd, on.z, B.x); B.z = fmaf(-wd, on.x, B.z); }
                    else { B.y = fmaf(wd, on.z, B.y); B.z = fmaf(-wd, on.y, B.z); }
                  }
                  if (a.has_dmiq12 && (a.terms & MMX_T_DMI_INTER)) {
                    // inter-sublattice tensor of Eq.4: B_c += d /(Ms_c h_i) q12_i x m'_n
                    const V3 qv = v3(a.dmiq[3][axis][0], a.dmiq[3][axis][1], a.dmiq[3][axis][2]);
                    B = fma3(iMs * a.inv_h[axis] * d, cross(qv, on), B);
                  }
                }
              }
            }
          }
          if (a.neumann && S <= 2 && !(ni[q] >= 0 && (REG ? a.mat[((size_t)s * a.nreg + rn[q]) * MMX_MATW + MP_MS] : Ms) > 0.f)) {
            // absent partner: Neumann ghost m_c + h d_n m in every pair stencil, the centre cell's own constants
            const int o = S == 2 ? 1 - s : s;
            const float* Po = a.mat + ((size_t)o * a.nreg + rc) * MMX_MATW;
            V3 gs, go;
            neumann_g(a, S == 2, s, o, axis, d, mc[s], mc[o], P, Po, gs, go);
            const float h = 1.f / a.inv_h[axis];
            const V3 mg = fma3(h, gs, mc[s]);
            if (a.terms & MMX_T_EXCH) B = fma3(2.f * Ac * iMs * a.inv_h2[axis], mg - mc[s], B);
            if (axis < 2 && (a.terms & MMX_T_DMI)) {
              const float wd = Dc * iMs * a.inv_h[axis] * d;
              if (axis == 0) { B.x = fmaf(wd, mg.z, B.x); B.z = fmaf(-wd, mg.x, B.z); }
              else { B.y = fmaf(wd, mg.z, B.y); B.z = fmaf(-wd, mg.y, B.z); }
            }
            if (a.has_dmiq && (a.terms & MMX_T_DMI)) {
              const V3 qv = v3(a.dmiq[s][axis][0], a.dmiq[s][axis][1], a.dmiq[s][axis][2]);
              B = fma3(iMs * a.inv_h[axis] * d, cross(qv, mg), B);
            }
            if (S == 2 && (a.terms & (MMX_T_A12 | MMX_T_DMI_INTER))) {
              const V3 og = fma3(h, go, mc[o]);
              if (a.terms & MMX_T_A12) B = fma3(a.A12 * iMs * a.inv_h2[axis], og - mc[o], B);
              if (axis < 2 && (a.terms & MMX_T_DMI_INTER)) {
                const float wd = a.Dinter * iMs * a.inv_h[axis] * d;
                if (axis == 0) { B.x = fmaf(wd, og.z, B.x); B.z = fmaf(-wd, og.x, B.z); }
                else { B.y = fmaf(wd, og.z, B.y); B.z = fmaf(-wd, og.y, B.z); }
              }
              if (a.has_dmiq12 && (a.terms & MMX_T_DMI_INTER)) {
                const V3 qv = v3(a.dmiq[3][axis][0], a.dmiq[3][axis][1], a.dmiq[3][axis][2]);
                B = fma3(iMs * a.inv_h[axis] * d, cross(qv, og), B);
              }
            }
          }
          if (a.has_J) {
            // central difference: (m_+ - m_-)/(2h) weighted by u_axis = zlb * J_axis
            const float wu = zlb * a.J[axis] * 0.5f * a.inv_h[axis] * d;
            dm = fma3(wu, mn, dm);
          }
        }
        if (S >= 2 && (a.terms & MMX_T_A0)) {
#pragma unroll
          for (int t = 1; t < S; ++t) B = fma3(a.a0pref * iMs, mc[(s + t) % S], B);
        }
        if (S >= 2 && (a.terms & MMX_T_DMI_HOMO)) {
          // Eq.6: eps = d . (m_a x m_b)  =>  B_a = (d x m_b)/Ms_a,  B_b = (m_a x d)/Ms_b; pairs (a, b) = (0, 1) for two
          // sublattices, the cyclic pairs (0,1), (1,2), (2,0) for three (readings S32, S38)
          const V3 dv = v3(a.dhomo[0], a.dhomo[1], a.dhomo[2]);
          if (S == 3 || s == 0) B = fma3(iMs, cross(dv, mc[(s + 1) % S]), B);
          if (S == 3 || s == 1) B = fma3(iMs, cross(mc[(s + S - 1) % S], dv), B);
        }
        if (a.terms & MMX_T_ANIS_U) {
          const V3 u = v3(P[MP_UX], P[MP_UY], P[MP_UZ]);
          B = fma3(P[MP_KU2] * dot(u, mc[s]), u, B);
        }
        if ((a.terms & MMX_T_ANIS_C) && P[MP_KC2] != 0.f) {
          const V3 c1 = v3(P[MP_C1X], P[MP_C1Y], P[MP_C1Z]);
          const V3 c2 = v3(P[MP_C2X], P[MP_C2Y], P[MP_C2Z]);
          const V3 c3 = v3(P[MP_C3X], P[MP_C3Y], P[MP_C3Z]);
          const float a1 = dot(c1, mc[s]), a2 = dot(c2, mc[s]), a3 = dot(c3, mc[s]);
          const float k = -P[MP_KC2];
          B = fma3(k * a1 * (a2 * a2 + a3 * a3), c1, B);
          B = fma3(k * a2 * (a3 * a3 + a1 * a1), c2, B);
          B = fma3(k * a3 * (a1 * a1 + a2 * a2), c3, B);
        }
        if (a.terms & MMX_T_ZEEMAN) B = B + v3(a.bext[0], a.bext[1], a.bext[2]);
        if ((a.terms & MMX_T_DEMAG) && a.bdemag) B = B + ld3(a.bdemag, N, i);
        if ((a.terms & MMX_T_MEL) && a.strain) {
          const float exx = a.strain[i], eyy = a.strain[N + i], ezz = a.strain[2 * N + i];
          const float exy = a.strain[3 * N + i], exz = a.strain[4 * N + i], eyz = a.strain[5 * N + i];
          const float p1 = -P[MP_MEL1], p2 = -P[MP_MEL2];
          const V3 m = mc[s];
          B.x += p1 * exx * m.x + p2 * (exy * m.y + exz * m.z);
          B.y += p1 * eyy * m.y + p2 * (exy * m.x + eyz * m.z);
          B.z += p1 * ezz * m.z + p2 * (exz * m.x + eyz * m.y);
        }
        // Eq.2
        const V3 m = mc[s];
        const V3 mxB = cross(m, B);
        const V3 mxmxB = cross(m, mxB);
        const float alpha = P[MP_ALPHA];
        tau = a.relax ? (-P[MP_LLG] * alpha) * mxmxB : (-P[MP_LLG]) * fma3(alpha, mxmxB, mxB);
        if (a.has_J) {
          // tau_ZL = -(1+alpha^2)^-1 [ (1 + xi alpha) m x (m x dm) + (xi - alpha) m x dm ]
          const float xi = P[MP_XI];
          const V3 mxa = cross(m, dm);
          const V3 mxmxa = cross(m, mxa);
          const float inv = -1.f / (1.f + alpha * alpha);
          tau = fma3(inv * (1.f + xi * alpha), mxmxa, tau);
          tau = fma3(inv * (xi - alpha), mxa, tau);
        }
        if (a.has_sl) {
          // Slonczewski torque (reading S37): gamma beta/(1+alpha^2) [(eps + alpha eps') m x (p x m) + (eps' - alpha eps) p x m]
          const V3 pv = v3(a.sl_mp[0], a.sl_mp[1], a.sl_mp[2]);
          const float eps = P[MP_POL] * a.sl_l2 / ((a.sl_l2 + 1.f) + (a.sl_l2 - 1.f) * dot(m, pv));
          const V3 pxm = cross(pv, m);
          const V3 mxpxm = cross(m, pxm);
          const float pref = P[MP_LLG] * a.sl_beta * iMs;
          tau = fma3(pref * (eps + alpha * a.sl_epsp), mxpxm, tau);
          tau = fma3(pref * (a.sl_epsp - alpha * eps), pxm, tau);
        }
      }
      if (a.heff_out) { st3(a.heff_out, N, i, B); continue; }
      if (a.tau_out) { st3(a.tau_out, N, i, tau); continue; }
      st3(a.kout[sel] + (size_t)s * 3 * N, N, i, tau);
      if (a.do_tq) {
        const float t2 = dot(tau, tau);
        tqv = fmaxf(tqv, sqrtf(t2));
        bad |= !(t2 == t2);
      }
      if (a.ynext[0]) {
        const float* ca = ctrl->ca[a.combine_row];
        V3 y = ld3(a.y0[sel] + (size_t)s * 3 * N, N, i);
        V3 acc = v3(0.f, 0.f, 0.f);
        for (int j = 0; j < a.n_prev; ++j) {
          const float cj = ca[j];
          if (cj != 0.f) acc = fma3(cj, ld3(a.kprev[sel][j] + (size_t)s * 3 * N, N, i), acc);
        }
        acc = fma3(ca[a.stage], tau, acc);
        y = y + acc;
        const float n2 = dot(y, y);
        if (n2 > 0.f) y = (1.f / sqrtf(n2)) * y;
        st3(a.ynext[sel] + (size_t)s * 3 * N, N, i, y);
      }
      if (a.do_err) {
        const float* ce = ctrl->ce;
        V3 e = v3(0.f, 0.f, 0.f);
        for (int j = 0; j < a.n_prev; ++j) {
          const float cj = ce[j];
          if (cj != 0.f) e = fma3(cj, ld3(a.kprev[sel][j] + (size_t)s * 3 * N, N, i), e);
        }
        e = fma3(ce[a.stage], tau, e);
        const float e2 = dot(e, e);
        errv = fmaxf(errv, sqrtf(e2));
        bad |= !(e2 == e2);
      }
    }
  }
  if (bad) errv = tqv = __int_as_float(0x7fc00000);
  if (a.do_err) block_max_to(errv, &ctrl->err_bits);
  if (a.do_tq) block_max_to(tqv, &ctrl->tq_bits);
}

// ---- fast path: one region (uniform material, Ms > 0), Nx a multiple of 4 ------------------------
// One thread owns four x-consecutive cells; every global access is a float4 (centre, y/z
// neighbours, B_demag, y0, k_j, outputs) except the two x-edge neighbours.  Same arithmetic,
// term by term, as k_local.
struct Q3 {  // four cells of a 3-vector field
  V3 c[4];
};
__device__ __forceinline__ Q3 ldq(const float* p, size_t N, size_t i) {
  const float4 x = *reinterpret_cast<const float4*>(p + i);
  const float4 y = *reinterpret_cast<const float4*>(p + N + i);
  const float4 z = *reinterpret_cast<const float4*>(p + 2 * N + i);
  Q3 q;
  q.c[0] = v3(x.x, y.x, z.x); q.c[1] = v3(x.y, y.y, z.y); q.c[2] = v3(x.z, y.z, z.z); q.c[3] = v3(x.w, y.w, z.w);
  return q;
}
__device__ __forceinline__ void stq(float* p, size_t N, size_t i, const Q3& q) {
  *reinterpret_cast<float4*>(p + i) = make_float4(q.c[0].x, q.c[1].x, q.c[2].x, q.c[3].x);
  *reinterpret_cast<float4*>(p + N + i) = make_float4(q.c[0].y, q.c[1].y, q.c[2].y, q.c[3].y);
  *reinterpret_cast<float4*>(p + 2 * N + i) = make_float4(q.c[0].z, q.c[1].z, q.c[2].z, q.c[3].z);
}

// NP = n_prev, the number of earlier k_j of the RK combination; MODE bit 0: form the next stage
// state, bit 1: form the embedded error
#define MMX_L4_BLOCK 256   // threads per CTA, two CTAs per SM (128-256 threads x 2-5 per SM measured: 93-102 us)
template <int S, int NP, int MODE>
__global__ void __launch_bounds__(MMX_L4_BLOCK, 2) k_local4(LocalArgs a) {
  // thread-private landing slots for the streamed inputs (B_demag, y0, k_j): cp.async puts them
  // in flight at the top of the kernel without holding registers; slot a of thread t is
  // lsm[a * 256 + t] (16 B per lane: conflict-free)
  extern __shared__ float4 lsm[];
  MmxCtrl* ctrl = a.ctrl;
  if (!ctrl->active) return;
  const int sel = ctrl->sel;
  const size_t N = (size_t)a.nx * a.ny * a.nz;
  const unsigned gpr = a.nx >> 2;  // groups per row
  auto stage3 = [&](int slot, const float* p, size_t idx) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const unsigned sa = (unsigned)__cvta_generic_to_shared(&lsm[(slot + c) * MMX_L4_BLOCK + threadIdx.x]);
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(p + (size_t)c * N + idx) : "memory");
    }
  };
  auto stq_stream = [&](float* p, size_t idx, const Q3& q) {
    stq(p, N, idx, q);
  };
  auto take3 = [&](int slot) -> Q3 {
    const float4 x = lsm[(slot + 0) * MMX_L4_BLOCK + threadIdx.x];
    const float4 y = lsm[(slot + 1) * MMX_L4_BLOCK + threadIdx.x];
    const float4 z = lsm[(slot + 2) * MMX_L4_BLOCK + threadIdx.x];
    Q3 q;
    q.c[0] = v3(x.x, y.x, z.x); q.c[1] = v3(x.y, y.y, z.y); q.c[2] = v3(x.z, y.z, z.z); q.c[3] = v3(x.w, y.w, z.w);
    return q;
  };
  const unsigned g = blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned rows = (unsigned)a.ny * a.nz;
  const float* yin = a.yin[sel];
  float errv = 0.f, tqv = 0.f;
  bool bad = false;
  if (g < gpr * rows) {
    const unsigned row = g / gpr;
    const int ix = (int)(g - row * gpr) << 2;
    const int iz = (int)(row / (unsigned)a.ny), iy = (int)(row - (unsigned)iz * a.ny);
    const size_t i = (size_t)row * a.nx + ix;
    // neighbour offsets (in elements) along y and z; valid flags
    long long off[6];
    bool val[6];
    {
      const bool xm = ix > 0, xp = ix + 4 < a.nx;
      val[1] = xm || a.per[0]; off[1] = xm ? -1 : (long long)a.nx - 1;
      val[0] = xp || a.per[0]; off[0] = xp ? 4 : 4 - (long long)a.nx;
      const bool ym = iy > 0, yp = iy + 1 < a.ny;
      val[3] = ym || (a.per[1] && a.ny > 1); off[3] = ym ? -(long long)a.nx : (long long)(a.ny - 1) * a.nx;
      val[2] = yp || (a.per[1] && a.ny > 1); off[2] = yp ? (long long)a.nx : -(long long)(a.ny - 1) * a.nx;
      const long long pl = (long long)a.nx * a.ny;
      const bool zm = iz > 0, zp = iz + 1 < a.nz;
      val[5] = zm || (a.per[2] && a.nz > 1); off[5] = zm ? -pl : (long long)(a.nz - 1) * pl;
      val[4] = zp || (a.per[2] && a.nz > 1); off[4] = zp ? pl : -(long long)(a.nz - 1) * pl;
    }
    Q3 mc[S];
#pragma unroll
    for (int s = 0; s < S; ++s) mc[s] = ldq(yin + (size_t)s * 3 * N, N, i);

#pragma unroll
    for (int s = 0; s < S; ++s) {
      if (a.heff_out || a.tau_out) {
        if (s != a.heff_s) continue;
      }
      const int o = S == 2 ? 1 - s : s;
      // streamed inputs of this sublattice: slot 0 B_demag, slot 3 y0, slot 6 + 3 j k_j
      constexpr bool comb = (MODE & 1) != 0, doerr = (MODE & 2) != 0;
      const bool epi = !a.heff_out && !a.tau_out;
      const float* ca = ctrl->ca[a.combine_row];
      const float* ce = ctrl->ce;
      const bool use_bd = (a.terms & MMX_T_DEMAG) && a.bdemag;
      if (use_bd) stage3(0, a.bdemag, i);
      if (MODE != 0 && epi) {
        if (comb) stage3(3, a.y0[sel] + (size_t)s * 3 * N, i);
#pragma unroll
        for (int j = 0; j < NP; ++j) {
          const float cj = comb ? ca[j] : 0.f;
          const float ej = doerr ? ce[j] : 0.f;
          if (cj != 0.f || ej != 0.f) stage3(6 + 3 * j, a.kprev[sel][j] + (size_t)s * 3 * N, i);
        }
      }
      asm volatile("cp.async.commit_group;" ::: "memory");
      const float* P = a.mat + (size_t)s * MMX_MATW;
      const float iMs = P[MP_INVMS];
      const float* ms_ = yin + (size_t)s * 3 * N;
      const float* mo_ = yin + (size_t)o * 3 * N;
      const bool use12 = S == 2 && (a.terms & (MMX_T_A12 | MMX_T_DMI_INTER));
      Q3 B, dm;
#pragma unroll
      for (int e = 0; e < 4; ++e) { B.c[e] = v3(0.f, 0.f, 0.f); dm.c[e] = v3(0.f, 0.f, 0.f); }
      const float Ac = P[MP_A], Dc = P[MP_D], zlb = P[MP_ZLB];
#pragma unroll
      for (int q = 0; q < 6; ++q) {
        const int axis = q >> 1;
        const float d = (q & 1) ? -1.f : 1.f;
        // neighbour values of the four cells along direction q (own and partner sublattice)
        Q3 mn = mc[s], on = mc[o];
        bool v[4] = {val[q], val[q], val[q], val[q]};
        if (axis == 0) {
          // interior cells take their x neighbour from the thread's own registers
          // (loads are unconditional -- an absent neighbour reads the thread's own cell -- so that
          // the compiler can issue all of them before the first use)
          const size_t ei = val[q] ? (size_t)((long long)i + off[q]) : i;
          const V3 edge = ld3(ms_, N, ei);
          V3 oedge = edge;
          if (use12) oedge = ld3(mo_, N, ei);
          if (q == 0) {
            mn.c[0] = mc[s].c[1]; mn.c[1] = mc[s].c[2]; mn.c[2] = mc[s].c[3]; mn.c[3] = edge;
            on.c[0] = mc[o].c[1]; on.c[1] = mc[o].c[2]; on.c[2] = mc[o].c[3]; on.c[3] = oedge;
            v[0] = v[1] = v[2] = true;
          } else {
            mn.c[3] = mc[s].c[2]; mn.c[2] = mc[s].c[1]; mn.c[1] = mc[s].c[0]; mn.c[0] = edge;
            on.c[3] = mc[o].c[2]; on.c[2] = mc[o].c[1]; on.c[1] = mc[o].c[0]; on.c[0] = oedge;
            v[1] = v[2] = v[3] = true;
          }
        } else {
          const size_t ni = val[q] ? (size_t)((long long)i + off[q]) : i;
          mn = ldq(ms_, N, ni);
          if (use12) on = ldq(mo_, N, ni);
        }
        const float wex = 2.f * harm(Ac, Ac) * iMs * a.inv_h2[axis];
        const float wd = harm(Dc, Dc) * iMs * a.inv_h[axis] * d;
        const float w12 = a.A12 * iMs * a.inv_h2[axis];
        const float wdi = a.Dinter * iMs * a.inv_h[axis] * d;
        const float wu = zlb * a.J[axis] * 0.5f * a.inv_h[axis] * d;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          if (v[e]) {
            if (a.terms & MMX_T_EXCH) B.c[e] = fma3(wex, mn.c[e] - mc[s].c[e], B.c[e]);
            if (axis < 2 && (a.terms & MMX_T_DMI)) {
              if (axis == 0) { B.c[e].x = fmaf(wd, mn.c[e].z, B.c[e].x); B.c[e].z = fmaf(-wd, mn.c[e].x, B.c[e].z); }
              else { B.c[e].y = fmaf(wd, mn.c[e].z, B.c[e].y); B.c[e].z = fmaf(-wd, mn.c[e].y, B.c[e].z); }
            }
            if (S == 2) {
              if (a.terms & MMX_T_A12) B.c[e] = fma3(w12, on.c[e] - mc[o].c[e], B.c[e]);
              if (axis < 2 && (a.terms & MMX_T_DMI_INTER)) {
                if (axis == 0) { B.c[e].x = fmaf(wdi, on.c[e].z, B.c[e].x); B.c[e].z = fmaf(-wdi, on.c[e].x, B.c[e].z); }
                else { B.c[e].y = fmaf(wdi, on.c[e].z, B.c[e].y); B.c[e].z = fmaf(-wdi, on.c[e].y, B.c[e].z); }
              }
            }
          }
          if (a.has_J) dm.c[e] = fma3(wu, v[e] ? mn.c[e] : mc[s].c[e], dm.c[e]);
        }
      }
      Q3 bd, tau;
      asm volatile("cp.async.wait_group 0;" ::: "memory");
      if (use_bd) bd = take3(0);
      float eps[6][4];
      const bool use_mel = (a.terms & MMX_T_MEL) && a.strain;
      if (use_mel) {
#pragma unroll
        for (int c = 0; c < 6; ++c) {
          const float4 t = *reinterpret_cast<const float4*>(a.strain + (size_t)c * N + i);
          eps[c][0] = t.x; eps[c][1] = t.y; eps[c][2] = t.z; eps[c][3] = t.w;
        }
      }
      const float alpha = P[MP_ALPHA], llg = P[MP_LLG], xi = P[MP_XI];
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const V3 m = mc[s].c[e];
        V3 Bc = B.c[e];
        if (S == 2 && (a.terms & MMX_T_A0)) Bc = fma3(a.a0pref * iMs, mc[o].c[e], Bc);
        if (S == 2 && (a.terms & MMX_T_DMI_HOMO)) {
          const V3 dv = v3(a.dhomo[0], a.dhomo[1], a.dhomo[2]);
          Bc = fma3(iMs, s == 0 ? cross(dv, mc[o].c[e]) : cross(mc[o].c[e], dv), Bc);
        }
        if (a.terms & MMX_T_ANIS_U) {
          const V3 u = v3(P[MP_UX], P[MP_UY], P[MP_UZ]);
          Bc = fma3(P[MP_KU2] * dot(u, m), u, Bc);
        }
        if ((a.terms & MMX_T_ANIS_C) && P[MP_KC2] != 0.f) {
          const V3 c1 = v3(P[MP_C1X], P[MP_C1Y], P[MP_C1Z]);
          const V3 c2 = v3(P[MP_C2X], P[MP_C2Y], P[MP_C2Z]);
          const V3 c3 = v3(P[MP_C3X], P[MP_C3Y], P[MP_C3Z]);
          const float a1 = dot(c1, m), a2 = dot(c2, m), a3 = dot(c3, m);
          const float k = -P[MP_KC2];
          Bc = fma3(k * a1 * (a2 * a2 + a3 * a3), c1, Bc);
          Bc = fma3(k * a2 * (a3 * a3 + a1 * a1), c2, Bc);
          Bc = fma3(k * a3 * (a1 * a1 + a2 * a2), c3, Bc);
        }
        if (a.terms & MMX_T_ZEEMAN) Bc = Bc + v3(a.bext[0], a.bext[1], a.bext[2]);
        if (use_bd) Bc = Bc + bd.c[e];
        if (use_mel) {
          const float p1 = -P[MP_MEL1], p2 = -P[MP_MEL2];
          Bc.x += p1 * eps[0][e] * m.x + p2 * (eps[3][e] * m.y + eps[4][e] * m.z);
          Bc.y += p1 * eps[1][e] * m.y + p2 * (eps[3][e] * m.x + eps[5][e] * m.z);
          Bc.z += p1 * eps[2][e] * m.z + p2 * (eps[4][e] * m.x + eps[5][e] * m.y);
        }
        B.c[e] = Bc;
        const V3 mxB = cross(m, Bc);
        const V3 mxmxB = cross(m, mxB);
        V3 t = a.relax ? (-llg * alpha) * mxmxB : (-llg) * fma3(alpha, mxmxB, mxB);
        if (a.has_J) {
          const V3 mxa = cross(m, dm.c[e]);
          const V3 mxmxa = cross(m, mxa);
          const float inv = -1.f / (1.f + alpha * alpha);
          t = fma3(inv * (1.f + xi * alpha), mxmxa, t);
          t = fma3(inv * (xi - alpha), mxa, t);
        }
        tau.c[e] = t;
      }
      if (a.heff_out) { stq(a.heff_out, N, i, B); continue; }
      if (a.tau_out) { stq(a.tau_out, N, i, tau); continue; }
      stq_stream(a.kout[sel] + (size_t)s * 3 * N, i, tau);
      if (a.do_tq) {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const float t2 = dot(tau.c[e], tau.c[e]);
          tqv = fmaxf(tqv, sqrtf(t2));
          bad |= !(t2 == t2);
        }
      }
      Q3 ys, er;
      if (MODE != 0 && epi) {
        if (comb) ys = take3(3);
        if (doerr) {
#pragma unroll
          for (int e = 0; e < 4; ++e) er.c[e] = v3(0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int j = 0; j < NP; ++j) {
          const float cj = comb ? ca[j] : 0.f;
          const float ej = doerr ? ce[j] : 0.f;
          if (cj != 0.f || ej != 0.f) {
            const Q3 kj = take3(6 + 3 * j);
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              if (comb) ys.c[e] = fma3(cj, kj.c[e], ys.c[e]);
              if (doerr) er.c[e] = fma3(ej, kj.c[e], er.c[e]);
            }
          }
        }
      }
      if (comb) {
        const float cs = ca[a.stage];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          V3 yy = fma3(cs, tau.c[e], ys.c[e]);
          const float n2 = dot(yy, yy);
          if (n2 > 0.f) yy = (1.f / sqrtf(n2)) * yy;
          ys.c[e] = yy;
        }
        stq(a.ynext[sel] + (size_t)s * 3 * N, N, i, ys);
      }
      if (doerr) {
        const float es = ce[a.stage];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const V3 ee = fma3(es, tau.c[e], er.c[e]);
          const float e2 = dot(ee, ee);
          errv = fmaxf(errv, sqrtf(e2));
          bad |= !(e2 == e2);
        }
      }
    }
  }
  if (bad) errv = tqv = __int_as_float(0x7fc00000);
  if (a.do_err) block_max_to(errv, &ctrl->err_bits);
  if (a.do_tq) block_max_to(tqv, &ctrl->tq_bits);
}

// ---- TMA halo-tile path: one sublattice, uniform material, open boundaries (the c4 / c1 shape) --------
// A CTA owns a tile of 64 x 4 x 2 cells.  The tile of m with its one-cell halo arrives in shared memory by
// ONE tensor-map TMA copy (cp.async.bulk.tensor.4d, box 72 x 6 x 4 x 3 floats starting at x0 - 4 so that a
// thread's four cells are a 16-byte aligned LDS.128; cells outside the grid are zero-filled by the copy
// unit and masked by the validity flags below, which is the "open" boundary of S9): the centre and all
// six neighbours are shared-memory reads, no register is held for a load in flight and there is no
// per-thread address arithmetic for the stencil.  The streamed inputs (B_demag, y0, k_j) keep their
// thread-private cp.async landing slots; outputs are float4 stores.  Same arithmetic, term by term, as
// k_local4 / k_local.  Three to five CTAs of 128 threads per SM.
constexpr int LT_TX = 64, LT_TY = 4, LT_TZ = 2, LT_BX = 72, LT_BY = LT_TY + 2, LT_BZ = LT_TZ + 2, LT_NT = 128;
constexpr int LT_HALO_BYTES = 3 * LT_BZ * LT_BY * LT_BX * 4;  // 20736

__device__ __forceinline__ unsigned lt_s32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

template <int NP, int MODE>
__global__ void __launch_bounds__(LT_NT, 3) k_local_t(LocalArgs a, const __grid_constant__ CUtensorMap tm0,
                                                      const __grid_constant__ CUtensorMap tm1) {
  extern __shared__ __align__(128) unsigned char smraw[];
  float* halo = reinterpret_cast<float*>(smraw);                             // [3][BZ][BY][BX]
  float4* lsm = reinterpret_cast<float4*>(smraw + LT_HALO_BYTES);             // landing slots [slot][NT]
  __shared__ __align__(8) unsigned long long bar;
  MmxCtrl* ctrl = a.ctrl;
  if (!ctrl->active) return;
  const int sel = ctrl->sel;
  const size_t N = (size_t)a.nx * a.ny * a.nz;
  const int x0 = blockIdx.x * LT_TX, y0 = blockIdx.y * LT_TY, z0 = blockIdx.z * LT_TZ;
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(lt_s32(&bar)) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    const CUtensorMap* tm = sel ? &tm1 : &tm0;
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(lt_s32(&bar)), "r"(LT_HALO_BYTES) : "memory");
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
        ::"r"(lt_s32(halo)), "l"(tm), "r"(x0 - 4), "r"(y0 - 1), "r"(z0 - 1), "r"(0), "r"(lt_s32(&bar)) : "memory");
  }
  const int tx = threadIdx.x & 15, ty = (threadIdx.x >> 4) & 3, tz = threadIdx.x >> 6;
  const int ix = x0 + 4 * tx, iy = y0 + ty, iz = z0 + tz;
  const bool inside = ix < a.nx && iy < a.ny && iz < a.nz;
  const size_t i = ((size_t)iz * a.ny + iy) * a.nx + ix;
  auto stage3 = [&](int slot, const float* p, size_t idx) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const unsigned sa = lt_s32(&lsm[(slot + c) * LT_NT + threadIdx.x]);
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(p + (size_t)c * N + idx) : "memory");
    }
  };
  auto take3 = [&](int slot) -> Q3 {
    const float4 x = lsm[(slot + 0) * LT_NT + threadIdx.x];
    const float4 y = lsm[(slot + 1) * LT_NT + threadIdx.x];
    const float4 z = lsm[(slot + 2) * LT_NT + threadIdx.x];
    Q3 q;
    q.c[0] = v3(x.x, y.x, z.x); q.c[1] = v3(x.y, y.y, z.y); q.c[2] = v3(x.z, y.z, z.z); q.c[3] = v3(x.w, y.w, z.w);
    return q;
  };
  constexpr bool comb = (MODE & 1) != 0, doerr = (MODE & 2) != 0;
  const bool epi = !a.heff_out && !a.tau_out;
  const float* ca = ctrl->ca[a.combine_row];
  const float* ce = ctrl->ce;
  const bool use_bd = (a.terms & MMX_T_DEMAG) && a.bdemag;
  if (inside) {
    // streamed inputs: slot 0 B_demag, slot 3 y0, slot 6 + 3 j k_j
    if (use_bd) stage3(0, a.bdemag, i);
    if (MODE != 0 && epi) {
      if (comb) stage3(3, a.y0[sel], i);
#pragma unroll
      for (int j = 0; j < NP; ++j) {
        const float cj = comb ? ca[j] : 0.f;
        const float ej = doerr ? ce[j] : 0.f;
        if (cj != 0.f || ej != 0.f) stage3(6 + 3 * j, a.kprev[sel][j], i);
      }
    }
  }
  asm volatile("cp.async.commit_group;" ::: "memory");
  {  // the halo tile has landed
    unsigned ok = 0;
    for (int spin = 0; !ok; ++spin) {
      asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\nselp.u32 %0, 1, 0, p;\n}\n"
                   : "=r"(ok) : "r"(lt_s32(&bar)) : "memory");
      if (!ok && spin > (1 << 16)) { mmx_mbar_wait_slow(lt_s32(&bar), 0); break; }   // (mbar.cuh: back-off, 10 s wall-time bound)
    }
  }
  float errv = 0.f, tqv = 0.f;
  bool bad = false;
  if (inside) {
    auto hq = [&](int dz, int dy) -> Q3 {  // the thread's four cells of row (ty + dy, tz + dz)
      const float* p = halo + ((tz + 1 + dz) * LT_BY + (ty + 1 + dy)) * LT_BX + 4 + 4 * tx;
      const float4 x = *reinterpret_cast<const float4*>(p);
      const float4 y = *reinterpret_cast<const float4*>(p + LT_BZ * LT_BY * LT_BX);
      const float4 z = *reinterpret_cast<const float4*>(p + 2 * LT_BZ * LT_BY * LT_BX);
      Q3 q;
      q.c[0] = v3(x.x, y.x, z.x); q.c[1] = v3(x.y, y.y, z.y); q.c[2] = v3(x.z, y.z, z.z); q.c[3] = v3(x.w, y.w, z.w);
      return q;
    };
    auto h1 = [&](int xo) -> V3 {  // one cell of the thread's own row at x offset xo from its first cell
      const float* p = halo + ((tz + 1) * LT_BY + (ty + 1)) * LT_BX + 4 + 4 * tx + xo;
      return v3(p[0], p[LT_BZ * LT_BY * LT_BX], p[2 * LT_BZ * LT_BY * LT_BX]);
    };
    const bool val[6] = {ix + 4 < a.nx, ix > 0, iy + 1 < a.ny, iy > 0, iz + 1 < a.nz, iz > 0};
    const Q3 mc = hq(0, 0);
    const float* P = a.mat;
    const float iMs = P[MP_INVMS];
    Q3 B, dm;
#pragma unroll
    for (int e = 0; e < 4; ++e) { B.c[e] = v3(0.f, 0.f, 0.f); dm.c[e] = v3(0.f, 0.f, 0.f); }
    const float Ac = P[MP_A], Dc = P[MP_D], zlb = P[MP_ZLB];
#pragma unroll
    for (int q = 0; q < 6; ++q) {
      const int axis = q >> 1;
      const float d = (q & 1) ? -1.f : 1.f;
      Q3 mn;
      bool v[4] = {val[q], val[q], val[q], val[q]};
      if (q == 0) {
        mn.c[0] = mc.c[1]; mn.c[1] = mc.c[2]; mn.c[2] = mc.c[3]; mn.c[3] = h1(4);
        v[0] = v[1] = v[2] = true;
      } else if (q == 1) {
        mn.c[3] = mc.c[2]; mn.c[2] = mc.c[1]; mn.c[1] = mc.c[0]; mn.c[0] = h1(-1);
        v[1] = v[2] = v[3] = true;
      } else {
        mn = hq(axis == 2 ? (q == 4 ? 1 : -1) : 0, axis == 1 ? (q == 2 ? 1 : -1) : 0);
      }
      const float wex = 2.f * harm(Ac, Ac) * iMs * a.inv_h2[axis];
      const float wd = harm(Dc, Dc) * iMs * a.inv_h[axis] * d;
      const float wu = zlb * a.J[axis] * 0.5f * a.inv_h[axis] * d;
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        if (v[e]) {
          if (a.terms & MMX_T_EXCH) B.c[e] = fma3(wex, mn.c[e] - mc.c[e], B.c[e]);
          if (axis < 2 && (a.terms & MMX_T_DMI)) {
            if (axis == 0) { B.c[e].x = fmaf(wd, mn.c[e].z, B.c[e].x); B.c[e].z = fmaf(-wd, mn.c[e].x, B.c[e].z); }
            else { B.c[e].y = fmaf(wd, mn.c[e].z, B.c[e].y); B.c[e].z = fmaf(-wd, mn.c[e].y, B.c[e].z); }
          }
        }
        if (a.has_J) dm.c[e] = fma3(wu, v[e] ? mn.c[e] : mc.c[e], dm.c[e]);
      }
    }
    Q3 bd, tau;
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    if (use_bd) bd = take3(0);
    float eps[6][4];
    const bool use_mel = (a.terms & MMX_T_MEL) && a.strain;
    if (use_mel) {
#pragma unroll
      for (int c = 0; c < 6; ++c) {
        const float4 t = *reinterpret_cast<const float4*>(a.strain + (size_t)c * N + i);
        eps[c][0] = t.x; eps[c][1] = t.y; eps[c][2] = t.z; eps[c][3] = t.w;
      }
    }
    const float alpha = P[MP_ALPHA], llg = P[MP_LLG], xi = P[MP_XI];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const V3 m = mc.c[e];
      V3 Bc = B.c[e];
      if (a.terms & MMX_T_ANIS_U) {
        const V3 u = v3(P[MP_UX], P[MP_UY], P[MP_UZ]);
        Bc = fma3(P[MP_KU2] * dot(u, m), u, Bc);
      }
      if ((a.terms & MMX_T_ANIS_C) && P[MP_KC2] != 0.f) {
        const V3 c1 = v3(P[MP_C1X], P[MP_C1Y], P[MP_C1Z]);
        const V3 c2 = v3(P[MP_C2X], P[MP_C2Y], P[MP_C2Z]);
        const V3 c3 = v3(P[MP_C3X], P[MP_C3Y], P[MP_C3Z]);
        const float a1 = dot(c1, m), a2 = dot(c2, m), a3 = dot(c3, m);
        const float k = -P[MP_KC2];
        Bc = fma3(k * a1 * (a2 * a2 + a3 * a3), c1, Bc);
        Bc = fma3(k * a2 * (a3 * a3 + a1 * a1), c2, Bc);
        Bc = fma3(k * a3 * (a1 * a1 + a2 * a2), c3, Bc);
      }
      if (a.terms & MMX_T_ZEEMAN) Bc = Bc + v3(a.bext[0], a.bext[1], a.bext[2]);
      if (use_bd) Bc = Bc + bd.c[e];
      if (use_mel) {
        const float p1 = -P[MP_MEL1], p2 = -P[MP_MEL2];
        Bc.x += p1 * eps[0][e] * m.x + p2 * (eps[3][e] * m.y + eps[4][e] * m.z);
        Bc.y += p1 * eps[1][e] * m.y + p2 * (eps[3][e] * m.x + eps[5][e] * m.z);
        Bc.z += p1 * eps[2][e] * m.z + p2 * (eps[4][e] * m.x + eps[5][e] * m.y);
      }
      B.c[e] = Bc;
      const V3 mxB = cross(m, Bc);
      const V3 mxmxB = cross(m, mxB);
      V3 t = a.relax ? (-llg * alpha) * mxmxB : (-llg) * fma3(alpha, mxmxB, mxB);
      if (a.has_J) {
        const V3 mxa = cross(m, dm.c[e]);
        const V3 mxmxa = cross(m, mxa);
        const float inv = -1.f / (1.f + alpha * alpha);
        t = fma3(inv * (1.f + xi * alpha), mxmxa, t);
        t = fma3(inv * (xi - alpha), mxa, t);
      }
      tau.c[e] = t;
    }
    if (a.heff_out) stq(a.heff_out, N, i, B);
    else if (a.tau_out) stq(a.tau_out, N, i, tau);
    else {
      stq(a.kout[sel], N, i, tau);
      if (a.do_tq) {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const float t2 = dot(tau.c[e], tau.c[e]);
          tqv = fmaxf(tqv, sqrtf(t2));
          bad |= !(t2 == t2);
        }
      }
      Q3 ys, er;
      if (MODE != 0) {
        if (comb) ys = take3(3);
        if (doerr) {
#pragma unroll
          for (int e = 0; e < 4; ++e) er.c[e] = v3(0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int j = 0; j < NP; ++j) {
          const float cj = comb ? ca[j] : 0.f;
          const float ej = doerr ? ce[j] : 0.f;
          if (cj != 0.f || ej != 0.f) {
            const Q3 kj = take3(6 + 3 * j);
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              if (comb) ys.c[e] = fma3(cj, kj.c[e], ys.c[e]);
              if (doerr) er.c[e] = fma3(ej, kj.c[e], er.c[e]);
            }
          }
        }
      }
      if (comb) {
        const float cs = ca[a.stage];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          V3 yy = fma3(cs, tau.c[e], ys.c[e]);
          const float n2 = dot(yy, yy);
          if (n2 > 0.f) yy = (1.f / sqrtf(n2)) * yy;
          ys.c[e] = yy;
        }
        stq(a.ynext[sel], N, i, ys);
      }
      if (doerr) {
        const float es = ce[a.stage];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const V3 ee = fma3(es, tau.c[e], er.c[e]);
          const float e2 = dot(ee, ee);
          errv = fmaxf(errv, sqrtf(e2));
          bad |= !(e2 == e2);
        }
      }
    }
  } else {
    asm volatile("cp.async.wait_group 0;" ::: "memory");
  }
  if (bad) errv = tqv = __int_as_float(0x7fc00000);
  if (a.do_err) block_max_to(errv, &ctrl->err_bits);
  if (a.do_tq) block_max_to(tqv, &ctrl->tq_bits);
}

// y_next = project(y0 + ca[row][0] * k1) for all vectors (m normalised, u and v not)
__global__ void __launch_bounds__(256) k_combine1(const float* y0a, const float* y0b, const float* k1a,
                                                  const float* k1b, float* yna, float* ynb, int row, int S,
                                                  int nvec, size_t N, MmxCtrl* ctrl) {
  if (!ctrl->active) return;
  const int sel = ctrl->sel;
  const float* y0 = sel ? y0b : y0a;
  const float* k1 = sel ? k1b : k1a;
  float* yn = sel ? ynb : yna;
  const float c = ctrl->ca[row][0];
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  for (int v = 0; v < nvec; ++v) {
    const size_t b = (size_t)v * 3 * N;
    V3 y = fma3(c, ld3(k1 + b, N, i), ld3(y0 + b, N, i));
    if (v < S) {
      const float n2 = dot(y, y);
      if (n2 > 0.f) y = (1.f / sqrtf(n2)) * y;
    }
    st3(yn + b, N, i, y);
  }
}

// mode 0: begin of an attempt (fill the coefficient tables from dt, clear the reductions)
// mode 1: end of an attempt (accept / reject, new dt, bookkeeping)
// mode 2: re-arm (active = 1) after a stepping call
// mode 3: first step size from max torque: dt = 0.01 / max|tau| (only when dt <= 0)
__global__ void k_controller(MmxCtrl* c, MmxTableau tab, int mode) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  if (mode == 2) { c->active = 1; return; }
  if (mode == 3) {
    if (c->dt <= 0.0) {
      const double tq = (double)__uint_as_float(c->tq_bits);
      c->dt = tq > 0.0 ? 0.01 / tq : 1e-15;
      if (c->dt_max > 0.0 && c->dt > c->dt_max) c->dt = c->dt_max;
    }
    c->max_torque = (double)__uint_as_float(c->tq_bits);
    return;
  }
  if (!c->active) return;
  if (mode == 0) {
    double dt = c->dt;
    if (!c->fixed && c->dt_max > 0.0 && dt > c->dt_max) dt = c->dt_max;
    if (c->t_end > 0.0 && c->t + dt > c->t_end) dt = c->t_end - c->t;
    c->dt = dt;
    for (int i = 0; i < MMX_MAX_STAGES; ++i) {
      for (int j = 0; j < MMX_MAX_STAGES; ++j) c->ca[i][j] = (float)(dt * tab.a[i][j]);
      c->ce[i] = (float)(dt * tab.e[i]);
      c->cc[i] = (float)tab.c[i];
    }
    c->err_bits = 0u;
    c->tq_bits = 0u;
    return;
  }
  // mode 1
  const unsigned eb = c->err_bits, tb = c->tq_bits;
  const double err = (double)__uint_as_float(eb);
  const bool bad = eb >= 0x7f800000u || tb >= 0x7f800000u;
  c->err_last = err;
  c->hist[c->hist_n % MMX_HIST] = err;
  c->hist_n++;
  c->attempts++;
  bool accept = c->fixed || !tab.embedded || err <= c->tol;
  if (bad) { c->nan_flag = 1; c->active = 0; accept = false; }
  // methods without a reusable last stage: stage 0 of this attempt measured the torque of the accepted
  // state it started from; below torque_stop the attempt is abandoned (neither accepted nor rejected)
  if (!bad && !tab.fsal && c->torque_stop > 0.0 && (double)__uint_as_float(tb) < c->torque_stop) {
    c->max_torque = (double)__uint_as_float(tb);
    c->attempts--;
    c->hist_n--;
    c->active = 0;
    return;
  }
  double dt_new = c->dt;
  if (!c->fixed && tab.embedded) {
    double fac = 2.0;
    if (err > 0.0) {
      fac = pow(c->tol / err, 1.0 / (double)c->order);
      fac = fmin(2.0, fmax(0.5, fac));
    }
    dt_new = c->dt * 0.8 * fac;
    if (c->dt_max > 0.0 && dt_new > c->dt_max) dt_new = c->dt_max;
  }
  if (accept) {
    c->t += c->dt;
    c->accepted++;
    c->sel ^= 1;
    c->max_torque = (double)__uint_as_float(tb);
    if (c->target_accepted > 0 && c->accepted >= c->target_accepted) c->active = 0;
    if (c->t_end > 0.0 && c->t >= c->t_end * (1.0 - 1e-14)) c->active = 0;
    if (tab.fsal && c->torque_stop > 0.0 && c->max_torque < c->torque_stop) c->active = 0;
  } else if (!bad) {
    c->rejected++;
  }
  c->dt = dt_new;
}

// energies: E = -c_term V sum_c Ms_c m_c . B_term,c ; fp64 accumulation
__global__ void __launch_bounds__(256) k_dot_energy(const float* m, const float* B, const uint16_t* reg,
                                                    const float* mat, int nreg, size_t N, double* acc) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  double v = 0.0;
  if (i < N) {
    const int r = reg ? reg[i] : 0;
    const double Ms = mat[(size_t)r * MMX_MATW + MP_MS];
    v = Ms * ((double)m[i] * B[i] + (double)m[N + i] * B[N + i] + (double)m[2 * N + i] * B[2 * N + i]);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __shared__ double sm[8];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) sm[wid] = v;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int k = 0; k < 8; ++k) t += sm[k];
    atomicAdd(acc, t);
  }
}

}  // namespace

// tensor map of a state buffer [3 nvec][nz][ny][nx] floats with the halo box of k_local_t, returned by value: a later
// lookup that misses on a full cache recycles slot 0, so a pointer into the cache would not survive a second call
static int tmap_for(mmx_world* w, const float* base, CUtensorMap* out) {
  for (int k = 0; k < w->n_tmaps; ++k)
    if (w->tmaps[k].base == base) { *out = *reinterpret_cast<const CUtensorMap*>(w->tmaps[k].bytes); return MMX_OK; }
  if (w->n_tmaps >= 4) w->n_tmaps = 0;
  static PFN_cuTensorMapEncodeTiled encode = nullptr;
  if (!encode) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) != cudaSuccess || !fn)
      return mmx_fail(MMX_ECUDA, "cuTensorMapEncodeTiled is not available");
    encode = reinterpret_cast<PFN_cuTensorMapEncodeTiled>(fn);
  }
  MmxTmap& t = w->tmaps[w->n_tmaps];
  const cuuint64_t dims[4] = {(cuuint64_t)w->grid[0], (cuuint64_t)w->grid[1], (cuuint64_t)w->grid[2], (cuuint64_t)(3 * w->nvec)};
  const cuuint64_t strides[3] = {(cuuint64_t)w->grid[0] * 4, (cuuint64_t)w->grid[0] * w->grid[1] * 4, (cuuint64_t)w->N * 4};
  const cuuint32_t box[4] = {LT_BX, LT_BY, LT_BZ, 3};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  const CUresult r = encode(reinterpret_cast<CUtensorMap*>(t.bytes), CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, const_cast<float*>(base), dims,
                            strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                            CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return mmx_fail(MMX_ECUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
  t.base = base;
  w->n_tmaps++;
  *out = *reinterpret_cast<const CUtensorMap*>(t.bytes);
  return MMX_OK;
}

int mmx_local_launch(mmx_world* w, const LocalArgs& a) {
  const size_t N = w->N;
  const unsigned blocks = (unsigned)((N + 255) / 256);
  const bool reg = w->nreg > 1;
  ProfScope ps(w, PK_LOCAL);
  // (the general DMI tensors, the Slonczewski torque and the Neumann boundary live in the general kernel k_local only)
  bool uniform = !reg && (w->grid[0] % 4) == 0 && !a.has_dmiq && !a.has_sl && !a.neumann;
  for (int s = 0; s < w->S && uniform; ++s) uniform = w->mats[(size_t)s * w->nreg].Ms > 0;
  if (w->S > 2) uniform = false;  // (three sublattices: general kernel)
  const bool open_all = !a.per[0] && !a.per[1] && !a.per[2];
  if (uniform && w->S == 1 && open_all) {
    // TMA halo tiles (k_local_t)
    CUtensorMap t0, t1;
    if (int rc = tmap_for(w, a.yin[0], &t0)) return rc;
    if (int rc = tmap_for(w, a.yin[1], &t1)) return rc;
    const dim3 grid((w->grid[0] + LT_TX - 1) / LT_TX, (w->grid[1] + LT_TY - 1) / LT_TY, (w->grid[2] + LT_TZ - 1) / LT_TZ);
    const int mode = (a.ynext[0] ? 1 : 0) | (a.do_err ? 2 : 0);
#define MMX_LT_GO(NP_, M_)                                                                                         \
  {                                                                                                                \
    const size_t sm_ = LT_HALO_BYTES + sizeof(float4) * LT_NT * (6 + 3 * (NP_));                                   \
    if (sm_ > 32 * 1024)                                                                                           \
      MMX_CUDA(cudaFuncSetAttribute(k_local_t<NP_, M_>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_));   \
    k_local_t<NP_, M_><<<grid, LT_NT, sm_, w->stream>>>(a, t0, t1);                                                \
  }
#define MMX_LT(NP_)                                \
  case NP_:                                        \
    if (mode == 0) MMX_LT_GO(0, 0)                 \
    else if (mode == 1) MMX_LT_GO(NP_, 1)          \
    else if (mode == 2) MMX_LT_GO(NP_, 2)          \
    else MMX_LT_GO(NP_, 3)                         \
    break;
    switch (a.n_prev) { MMX_LT(0) MMX_LT(1) MMX_LT(2) MMX_LT(3) MMX_LT(4) MMX_LT(5) MMX_LT(6) MMX_LT(7)
      default: return mmx_fail(MMX_EINVAL, "n_prev %d out of range", a.n_prev); }
  } else if (uniform) {
    const unsigned b4 = (unsigned)((N / 4 + MMX_L4_BLOCK - 1) / MMX_L4_BLOCK);
    const int mode = (a.ynext[0] ? 1 : 0) | (a.do_err ? 2 : 0);
#define MMX_L4_GO(S_, NP_, M_)                                                             \
  {                                                                                        \
    const size_t sm_ = sizeof(float4) * MMX_L4_BLOCK * (6 + 3 * (NP_));                            \
    if (sm_ > 32 * 1024)                                                                   \
      MMX_CUDA(cudaFuncSetAttribute(k_local4<S_, NP_, M_>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_)); \
    MMX_CUDA(mmx_launch(k_local4<S_, NP_, M_>, b4, MMX_L4_BLOCK, sm_, w->stream, a));                                \
  }
#define MMX_L4(S_, NP_)                                                    \
  case NP_:                                                                \
    if (mode == 0) MMX_L4_GO(S_, 0, 0)                                     \
    else if (mode == 1) MMX_L4_GO(S_, NP_, 1)                              \
    else if (mode == 2) MMX_L4_GO(S_, NP_, 2)                              \
    else MMX_L4_GO(S_, NP_, 3)                                             \
    break;
#define MMX_L4_ALL(S_) switch (a.n_prev) { MMX_L4(S_, 0) MMX_L4(S_, 1) MMX_L4(S_, 2) MMX_L4(S_, 3) MMX_L4(S_, 4) \
    MMX_L4(S_, 5) MMX_L4(S_, 6) MMX_L4(S_, 7) default: return mmx_fail(MMX_EINVAL, "n_prev %d out of range", a.n_prev); }
    if (w->S == 1) { MMX_L4_ALL(1) } else { MMX_L4_ALL(2) }
  } else if (w->S == 1) {
    if (reg) k_local<1, true><<<blocks, 256, 0, w->stream>>>(a);
    else k_local<1, false><<<blocks, 256, 0, w->stream>>>(a);
  } else if (w->S == 2) {
    if (reg) k_local<2, true><<<blocks, 256, 0, w->stream>>>(a);
    else k_local<2, false><<<blocks, 256, 0, w->stream>>>(a);
  } else {
    if (reg) k_local<3, true><<<blocks, 256, 0, w->stream>>>(a);
    else k_local<3, false><<<blocks, 256, 0, w->stream>>>(a);
  }
  w->launches++;
  MMX_CUDA(cudaGetLastError());
  return MMX_OK;
}

int mmx_combine_launch(mmx_world* w, const float* const y0[2], const float* const k1[2],
                       float* const ynext[2], int row) {
  const unsigned blocks = (unsigned)((w->N + 255) / 256);
  ProfScope ps(w, PK_COMBINE);
  MMX_CUDA(mmx_launch(k_combine1, blocks, 256, 0, w->stream, y0[0], y0[1], k1[0], k1[1], ynext[0], ynext[1], row,
                      w->S, w->nvec, w->N, w->d_ctrl));
  w->launches++;
  MMX_CUDA(cudaGetLastError());
  return MMX_OK;
}

int mmx_controller_launch(mmx_world* w, const MmxTableau& tab, int mode) {
  ProfScope ps(w, PK_CTRL);
  MMX_CUDA(mmx_launch(k_controller, 1, 32, 0, w->stream, w->d_ctrl, tab, mode));
  w->launches++;
  MMX_CUDA(cudaGetLastError());
  return MMX_OK;
}

// sum over sublattices of  Ms m . B  for the field already stored in w->scratch (per sublattice
// call): helper used by mmx_energy in api.cu
int mmx_energy_launch(mmx_world* w, unsigned s, const float* B, double* dev_acc) {
  const unsigned blocks = (unsigned)((w->N + 255) / 256);
  ProfScope ps(w, PK_ENERGY);
  k_dot_energy<<<blocks, 256, 0, w->stream>>>(w->Y[w->sel_host] + (size_t)s * 3 * w->N, B,
                                              w->nreg > 1 ? w->d_reg : nullptr,
                                              w->d_mat + (size_t)s * w->nreg * MMX_MATW, w->nreg, w->N, dev_acc);
  w->launches++;
  MMX_CUDA(cudaGetLastError());
  return MMX_OK;
}
