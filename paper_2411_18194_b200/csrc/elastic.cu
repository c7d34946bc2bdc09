// elastic.cu -- elastodynamics and magnetoelastic body force.
//
// Eq.7: rho u_tt = f_el + f_mel for cubic symmetry; strain = numeric gradient
// of u, f_el = numeric divergence of the stress; "fourth order accurate central difference
// scheme in the bulk ... lower order schemes close to and at the boundaries"; traction and
// traction-free boundary conditions impose sigma.n = t.  Eq.8: f_mel.
// In a two-sublattice magnet u, v, strain and stiffness are shared, each sublattice has its own
// B1, B2 and the body forces add.
//
// Gradient of f at index i of an axis with n cells, step h:
//   +-1, +-2 all present : (-f[+2] + 8 f[+1] - 8 f[-1] + f[-2]) / (12 h)
//   +-1 present          : (f[+1] - f[-1]) / (2 h)
//   one-sided            : (-3 f0 + 4 f[+1] - f[+2]) / (2 h)  or  (f[+1] - f0) / h  (mirrored at the far end)
//   single cell          : 0
// Divergence of sigma: the same operator, except in the first / last cell of an open axis
// where the face value s_b of sigma (from sigma.n = t, half a cell away) enters:
//   (-4 s_b + 3 s_0 + s_1) / (3 h)   resp.   (4 s_b - 3 s_{n-1} - s_{n-2}) / (3 h).
#include <cstdio>

#include "mmx_internal.h"

namespace {

struct Grid {
  int n[3];
  int per[3];
  float inv_h[3];
  size_t stride[3];
};

// d f / d x_axis at cell with coordinate p[axis] = i; f points at the cell, stride in elements
__device__ __forceinline__ float grad1(const float* f, int i, int n, bool per, size_t st, float inv_h) {
  if (n == 1) return 0.f;
  auto has = [&](int k) { return per || (i + k >= 0 && i + k < n); };
  auto at = [&](int k) {
    int q = i + k;
    if (per) q = ((q % n) + n) % n;
    return f[((long long)q - i) * (long long)st];
  };
  if (has(-2) && has(-1) && has(1) && has(2)) return (-at(2) + 8.f * at(1) - 8.f * at(-1) + at(-2)) * (inv_h / 12.f);
  if (has(-1) && has(1)) return (at(1) - at(-1)) * (0.5f * inv_h);
  if (has(1) && has(2)) return (-3.f * at(0) + 4.f * at(1) - at(2)) * (0.5f * inv_h);
  if (has(1)) return (at(1) - at(0)) * inv_h;
  if (has(-1) && has(-2)) return (3.f * at(0) - 4.f * at(-1) + at(-2)) * (0.5f * inv_h);
  if (has(-1)) return (at(0) - at(-1)) * inv_h;
  return 0.f;
}

__device__ __forceinline__ void coords(size_t i, const int n[3], int p[3]) {
  // (32-bit arithmetic: a world has fewer than 2^31 cells, mmx_world_create checks it)
  const unsigned c = (unsigned)i, row = c / (unsigned)n[0];
  p[0] = (int)(c - row * (unsigned)n[0]);
  p[2] = (int)(row / (unsigned)n[1]);
  p[1] = (int)(row - (unsigned)p[2] * (unsigned)n[1]);
}

__global__ void __launch_bounds__(256) k_strain(ElasticArgs a) {
  if (a.ctrl && !a.ctrl->active) return;
  const int sel = a.ctrl ? a.ctrl->sel : 0;
  const size_t N = (size_t)a.nx * a.ny * a.nz;
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int n[3] = {a.nx, a.ny, a.nz};
  const size_t st[3] = {1, (size_t)a.nx, (size_t)a.nx * a.ny};
  int p[3];
  coords(i, n, p);
  const float* u = a.yin[sel] + (size_t)a.S * 3 * N;  // displacement follows the S magnetisations
  float g[3][3];  // g[i][j] = d_i u_j
#pragma unroll
  for (int ax = 0; ax < 3; ++ax)
#pragma unroll
    for (int j = 0; j < 3; ++j) g[ax][j] = grad1(u + (size_t)j * N + i, p[ax], n[ax], a.per[ax], st[ax], a.inv_h[ax]);
  a.strain[i] = g[0][0];
  a.strain[N + i] = g[1][1];
  a.strain[2 * N + i] = g[2][2];
  a.strain[3 * N + i] = 0.5f * (g[0][1] + g[1][0]);
  a.strain[4 * N + i] = 0.5f * (g[0][2] + g[2][0]);
  a.strain[5 * N + i] = 0.5f * (g[1][2] + g[2][1]);
  if (a.strain_f) {
    // viscous damping: "an extra term, proportional to the strain rate, is added to the total
    // stress tensor"; stiffness-proportional Rayleigh form sigma = C : (eps(u) + beta eps(v)), so the
    // force kernel takes its stress from the strain of u + beta v.  v follows u in the state vector.
    const float* v = u + 3 * N;
    float gv[3][3];
#pragma unroll
    for (int ax = 0; ax < 3; ++ax)
#pragma unroll
      for (int j = 0; j < 3; ++j) gv[ax][j] = grad1(v + (size_t)j * N + i, p[ax], n[ax], a.per[ax], st[ax], a.inv_h[ax]);
    a.strain_f[i] = fmaf(a.beta, gv[0][0], g[0][0]);
    a.strain_f[N + i] = fmaf(a.beta, gv[1][1], g[1][1]);
    a.strain_f[2 * N + i] = fmaf(a.beta, gv[2][2], g[2][2]);
    a.strain_f[3 * N + i] = 0.5f * (fmaf(a.beta, gv[0][1] + gv[1][0], g[0][1] + g[1][0]));
    a.strain_f[4 * N + i] = 0.5f * (fmaf(a.beta, gv[0][2] + gv[2][0], g[0][2] + g[2][0]));
    a.strain_f[5 * N + i] = 0.5f * (fmaf(a.beta, gv[1][2] + gv[2][1], g[1][2] + g[2][1]));
  }
}

// sigma_ij at the cell whose strain components are e[6] = xx,yy,zz,xy,xz,yz
__device__ __forceinline__ float sigma_of(const float* eps, size_t N, long long c, int i, int j, float C11, float C12,
                                          float C44) {
  if (i == j) {
    const float exx = eps[c], eyy = eps[N + c], ezz = eps[2 * N + c];
    const float tr = exx + eyy + ezz;
    const float eii = i == 0 ? exx : (i == 1 ? eyy : ezz);
    return C11 * eii + C12 * (tr - eii);
  }
  const int k = (i + j == 1) ? 3 : ((i + j == 2) ? 4 : 5);
  return 2.f * C44 * eps[(size_t)k * N + c];
}

// d sigma_ij / d x_ax at cell i with traction face values
__device__ float div1(const ElasticArgs& a, const float* eps, size_t N, size_t cell, int ii, int jj, int pi, int n,
                      bool per, size_t st, float inv_h, float face_lo, float face_hi) {
  if (n == 1) return 0.f;
  auto S = [&](int k) {
    int q = pi + k;
    if (per) q = ((q % n) + n) % n;
    return sigma_of(eps, N, (long long)cell + ((long long)q - pi) * (long long)st, ii, jj, a.C11, a.C12, a.C44);
  };
  if (!per) {
    if (pi == 0) return (-4.f * face_lo + 3.f * S(0) + S(1)) * (inv_h / 3.f);
    if (pi == n - 1) return (4.f * face_hi - 3.f * S(0) - S(-1)) * (inv_h / 3.f);
  }
  auto has = [&](int k) { return per || (pi + k >= 0 && pi + k < n); };
  if (has(-2) && has(-1) && has(1) && has(2)) return (-S(2) + 8.f * S(1) - 8.f * S(-1) + S(-2)) * (inv_h / 12.f);
  if (has(-1) && has(1)) return (S(1) - S(-1)) * (0.5f * inv_h);
  if (has(1) && has(2)) return (-3.f * S(0) + 4.f * S(1) - S(2)) * (0.5f * inv_h);
  if (has(1)) return (S(1) - S(0)) * inv_h;
  if (has(-1) && has(-2)) return (3.f * S(0) - 4.f * S(-1) + S(-2)) * (0.5f * inv_h);
  if (has(-1)) return (S(0) - S(-1)) * inv_h;
  return 0.f;
}

__global__ void __launch_bounds__(256) k_elastic(ElasticArgs a) {
  if (a.ctrl && !a.ctrl->active) return;
  const int sel = a.ctrl ? a.ctrl->sel : 0;
  const size_t N = (size_t)a.nx * a.ny * a.nz;
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int n[3] = {a.nx, a.ny, a.nz};
  const size_t st[3] = {1, (size_t)a.nx, (size_t)a.nx * a.ny};
  int p[3];
  coords(i, n, p);
  const float* yin = a.yin[sel];
  // traction amplitude at the stage time
  float tr[3] = {0.f, 0.f, 0.f};
  // (only the cells on the traction face use it: the fp64 sine is not evaluated by the others)
  if (a.face >= 0 && p[a.face >> 1] == ((a.face & 1) ? n[a.face >> 1] - 1 : 0)) {
    double t = a.t_fixed;
    if (a.ctrl && !a.accel_out) t = a.ctrl->t + (double)a.ctrl->cc[a.stage] * a.ctrl->dt;
    const double amp = a.tamp * sin(2.0 * 3.14159265358979323846 * a.tfreq * t);
    for (int j = 0; j < 3; ++j) tr[j] = (float)(amp * a.tvec[j]);
  }
  float f[3] = {0.f, 0.f, 0.f};
  // f_el,j = sum_i d_i sigma_ij ; face value of sigma_ij on the low/high face of axis i is -+ t_j
#pragma unroll
  for (int j = 0; j < 3; ++j)
#pragma unroll
    for (int ax = 0; ax < 3; ++ax) {
      const float flo = (a.face == 2 * ax) ? -tr[j] : 0.f;
      const float fhi = (a.face == 2 * ax + 1) ? tr[j] : 0.f;
      f[j] += div1(a, a.strain_f ? a.strain_f : a.strain, N, i, ax, j, p[ax], n[ax], a.per[ax], st[ax], a.inv_h[ax], flo, fhi);
    }
  // f_mel (Eq.8), summed over sublattices
  const int rc = a.reg ? a.reg[i] : 0;
  for (int s = 0; s < a.S; ++s) {
    const float* P = a.mat + ((size_t)s * a.nreg + rc) * MMX_MATW;
    const float B1 = P[MP_B1], B2 = P[MP_B2];
    if (B1 == 0.f && B2 == 0.f) continue;
    const float* m = yin + (size_t)s * 3 * N;
    float d[3][3];  // d[i][j] = d_i m_j
    float mc[3];
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      mc[j] = m[(size_t)j * N + i];
#pragma unroll
      for (int ax = 0; ax < 3; ++ax) d[ax][j] = grad1(m + (size_t)j * N + i, p[ax], n[ax], a.per[ax], st[ax], a.inv_h[ax]);
    }
#pragma unroll
    for (int q = 0; q < 3; ++q) {
      const int b = (q + 1) % 3, c = (q + 2) % 3;
      f[q] += 2.f * B1 * mc[q] * d[q][q] + B2 * (mc[q] * (d[b][b] + d[c][c]) + mc[b] * d[b][q] + mc[c] * d[c][q]);
    }
  }
  float acc[3] = {f[0] * a.inv_rho, f[1] * a.inv_rho, f[2] * a.inv_rho};
  if (a.accel_out) {
    for (int j = 0; j < 3; ++j) a.accel_out[(size_t)j * N + i] = acc[j];
    return;
  }
  // RHS of the first-order system: du/dt = v, dv/dt = acc
  const size_t ou = (size_t)a.S * 3 * N, ov = (size_t)(a.S + 1) * 3 * N;
  float kv[2][3];
  for (int j = 0; j < 3; ++j) {
    kv[0][j] = yin[ov + (size_t)j * N + i];
    kv[1][j] = acc[j];
    a.kout[sel][ou + (size_t)j * N + i] = kv[0][j];
    a.kout[sel][ov + (size_t)j * N + i] = kv[1][j];
  }
  if (a.ynext[0]) {
    const float* ca = a.ctrl->ca[a.combine_row];
    for (int w = 0; w < 2; ++w) {
      const size_t off = w == 0 ? ou : ov;
      for (int j = 0; j < 3; ++j) {
        const size_t e = off + (size_t)j * N + i;
        float accum = 0.f;
        for (int q = 0; q < a.n_prev; ++q) {
          const float cq = ca[q];
          if (cq != 0.f) accum = fmaf(cq, a.kprev[sel][q][e], accum);
        }
        accum = fmaf(ca[a.stage], kv[w][j], accum);
        a.ynext[sel][e] = a.y0[sel][e] + accum;
      }
    }
  }
}

// (1/2) sigma : eps  and  (1/2) rho v^2, fp64 accumulation
__global__ void __launch_bounds__(256) k_elastic_energy(const float* eps, const float* v, size_t N, float C11, float C12,
                                                        float C44, double rho, double* acc) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  double es = 0.0, ek = 0.0;
  if (i < N) {
    const double exx = eps[i], eyy = eps[N + i], ezz = eps[2 * N + i];
    const double exy = eps[3 * N + i], exz = eps[4 * N + i], eyz = eps[5 * N + i];
    const double sxx = C11 * exx + C12 * (eyy + ezz), syy = C11 * eyy + C12 * (exx + ezz), szz = C11 * ezz + C12 * (exx + eyy);
    es = 0.5 * (sxx * exx + syy * eyy + szz * ezz + 2.0 * (2.0 * C44) * (exy * exy + exz * exz + eyz * eyz));
    const double vx = v[i], vy = v[N + i], vz = v[2 * N + i];
    ek = 0.5 * rho * (vx * vx + vy * vy + vz * vz);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    es += __shfl_xor_sync(0xffffffffu, es, o);
    ek += __shfl_xor_sync(0xffffffffu, ek, o);
  }
  if ((threadIdx.x & 31) == 0) {
    atomicAdd(acc, es);
    atomicAdd(acc + 1, ek);
  }
}

}  // namespace

int mmx_strain_launch(mmx_world* w, const ElasticArgs& a) {
  const unsigned blocks = (unsigned)((w->N + 255) / 256);
  ProfScope ps(w, PK_STRAIN);
  k_strain<<<blocks, 256, 0, w->stream>>>(a);
  w->launches++;
  MMX_CUDA(cudaGetLastError());
  return MMX_OK;
}

int mmx_elastic_launch(mmx_world* w, const ElasticArgs& a) {
  const unsigned blocks = (unsigned)((w->N + 255) / 256);
  ProfScope ps(w, PK_ELASTIC);
  k_elastic<<<blocks, 256, 0, w->stream>>>(a);
  w->launches++;
  MMX_CUDA(cudaGetLastError());
  return MMX_OK;
}

int mmx_elastic_energy_launch(mmx_world* w, double* es, double* ek) {
  const unsigned blocks = (unsigned)((w->N + 255) / 256);
  MMX_CUDA(cudaMemsetAsync(w->d_acc, 0, 2 * sizeof(double), w->stream));
  const float* v = w->Y[w->sel_host] + (size_t)(w->S + 1) * 3 * w->N;
  k_elastic_energy<<<blocks, 256, 0, w->stream>>>(w->strain, v, w->N, (float)w->el.C11, (float)w->el.C12,
                                                  (float)w->el.C44, w->el.rho, w->d_acc);
  w->launches++;
  double h[2];
  MMX_CUDA(cudaMemcpyAsync(h, w->d_acc, sizeof(h), cudaMemcpyDeviceToHost, w->stream));
  MMX_CUDA(cudaStreamSynchronize(w->stream));
  const double V = w->cell[0] * w->cell[1] * w->cell[2];
  *es = h[0] * V;
  *ek = h[1] * V;
  return MMX_OK;
}
