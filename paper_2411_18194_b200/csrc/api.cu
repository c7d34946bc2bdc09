// api.cu -- the C-ABI entry points of include/mmx.h: world plumbing, parameter upload, the
// per-stage launch sequence  [strain] -> [demag passes] -> local field/torque/RK combine ->
// [elastic RHS], and the explicit Runge-Kutta drivers (Table 2; classical RK4).
#include <cmath>
#include <cstdarg>
#include <cstddef>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "mmx_internal.h"

namespace {

thread_local char g_err[512] = "";

const double MU0 = 4e-7 * M_PI;
const double GAMMA0 = 1.7595e11;        // rad/(T s); the paper defers to mumax3's value
const double MU_B = 9.2740100783e-24;   // J/T
const double Q_E = 1.602176634e-19;     // C

template <typename T>
int dev_alloc(mmx_world* w, T** p, size_t count) {
  *p = nullptr;
  if (count == 0) return MMX_OK;
  cudaError_t e = cudaMalloc((void**)p, count * sizeof(T));
  if (e != cudaSuccess) {
    cudaGetLastError();
    return mmx_fail(MMX_ENOMEM, "cudaMalloc of %zu bytes failed: %s", count * sizeof(T), cudaGetErrorString(e));
  }
  w->dev_bytes += (long long)(count * sizeof(T));
  return MMX_OK;
}

template <typename T>
void dev_free(mmx_world* w, T** p, size_t count) {
  if (*p) {
    cudaFree(*p);
    w->dev_bytes -= (long long)(count * sizeof(T));
    *p = nullptr;
  }
}

void default_material(mmx_material* m) {
  memset(m, 0, sizeof(*m));
  m->gamma = GAMMA0;
  m->u[2] = 1.0;
  m->c1[0] = 1.0;
  m->c2[1] = 1.0;
}

// Largest y such that |R(i y')| <= 1 + growth for all y' in [0, y], R the stability polynomial of the tableau,
// R(z) = 1 + sum_k z^k b^T A^(k-1) 1: how far up the imaginary axis (undamped waves, u'' = -omega^2 u, y = omega dt) a step
// may reach before round-off is amplified by more than `growth` per step.  RK4: 2 sqrt 2; Bogacki-Shampine: sqrt 3;
// Dormand-Prince: 0.997; Heun, Cash-Karp and Fehlberg are not neutrally stable anywhere on the axis (|R| - 1 ~ y^4 / y^6),
// so their limit is set by the growth allowance alone.  Scanned in steps of 1e-4 up to y = 4.
double imag_axis_limit(const MmxTableau& t, double growth) {
  const int s = t.stages;
  double coef[MMX_MAX_STAGES + 1], v[MMX_MAX_STAGES], nv[MMX_MAX_STAGES];
  coef[0] = 1.0;
  for (int i = 0; i < s; ++i) v[i] = 1.0;
  for (int k = 1; k <= s; ++k) {
    double d = 0.0;
    for (int i = 0; i < s; ++i) d += t.b[i] * v[i];
    coef[k] = d;
    for (int i = 0; i < s; ++i) {
      nv[i] = 0.0;
      for (int j = 0; j < i; ++j) nv[i] += t.a[i][j] * v[j];
    }
    for (int i = 0; i < s; ++i) v[i] = nv[i];
  }
  double last = 0.0;
  for (int q = 1; q <= 40000; ++q) {
    const double y = 1e-4 * q;
    double re = 0.0, im = 0.0, p = 1.0;  // p = y^k
    for (int k = 0; k <= s; ++k) {
      switch (k & 3) { case 0: re += coef[k] * p; break; case 1: im += coef[k] * p; break;
                       case 2: re -= coef[k] * p; break; default: im -= coef[k] * p; }
      p *= y;
    }
    if (sqrt(re * re + im * im) > 1.0 + growth + 1e-13) break;
    last = y;
  }
  return last;
}

// Step bound of adaptive stepping with elastodynamics on: dt_max = 0.9 y_max / omega_max.
//   y_max      imag_axis_limit of the method with a growth allowance of 1e-6 per step
//   omega_max  largest frequency of the discrete elastic operator: the fourth-order central first derivative applied twice
//              (Eq.7) has the symbol (8 sin th - sin 2th)/(6 h) <= 1.3722 / h per axis, so
//              omega_max <= 1.3722 v_max sqrt(sum over axes with more than one cell of 1 / h_a^2); v_max the fastest wave
//              of the cubic medium, the largest of the longitudinal velocities along [100], [110], [111] and sqrt(C44/rho)
double elastic_dt_limit(const mmx_world* w, const MmxTableau& tab) {
  const double C11 = w->el.C11, C12 = w->el.C12, C44 = w->el.C44;
  double c = C11;
  if (C44 > c) c = C44;
  if (0.5 * (C11 + C12 + 2 * C44) > c) c = 0.5 * (C11 + C12 + 2 * C44);
  if ((C11 + 2 * C12 + 4 * C44) / 3.0 > c) c = (C11 + 2 * C12 + 4 * C44) / 3.0;
  double k2 = 0.0;
  for (int a = 0; a < 3; ++a)
    if (w->grid[a] > 1) k2 += 1.0 / (w->cell[a] * w->cell[a]);
  if (!(c > 0) || !(w->el.rho > 0) || !(k2 > 0)) return 0.0;
  const double omega_max = 1.3722 * sqrt(c / w->el.rho) * sqrt(k2);
  return 0.9 * imag_axis_limit(tab, 1e-6) / omega_max;
}

size_t vecN(const mmx_world* w) { return (size_t)w->nvec * 3 * w->N; }

// ---- tableaux (Table 2; classical RK4 from the textbook reference [51]) -----------
MmxTableau make_tableau(int method) {
  MmxTableau t;
  memset(&t, 0, sizeof(t));
  auto row = [&](int i, std::initializer_list<double> v) {
    int j = 0;
    for (double x : v) t.a[i][j++] = x;
  };
  auto setv = [&](double* dst, std::initializer_list<double> v) {
    int j = 0;
    for (double x : v) dst[j++] = x;
  };
  switch (method) {
    case MMX_RK4:
      t.stages = 4; t.fsal = 0; t.order = 4; t.embedded = 0;
      setv(t.c, {0, 0.5, 0.5, 1});
      row(1, {0.5}); row(2, {0, 0.5}); row(3, {0, 0, 1});
      setv(t.b, {1.0 / 6, 1.0 / 3, 1.0 / 3, 1.0 / 6});
      break;
    case MMX_HEUN12: {
      t.stages = 2; t.fsal = 0; t.order = 2; t.embedded = 1;
      setv(t.c, {0, 1});
      row(1, {1});
      setv(t.b, {0.5, 0.5});
      setv(t.e, {0.5 - 1.0, 0.5});
      break;
    }
    case MMX_BS23: {
      t.stages = 4; t.fsal = 1; t.order = 3; t.embedded = 1;
      setv(t.c, {0, 0.5, 0.75, 1});
      row(1, {0.5}); row(2, {0, 0.75}); row(3, {2.0 / 9, 1.0 / 3, 4.0 / 9});
      setv(t.b, {2.0 / 9, 1.0 / 3, 4.0 / 9, 0});
      setv(t.e, {2.0 / 9 - 7.0 / 24, 1.0 / 3 - 1.0 / 4, 4.0 / 9 - 1.0 / 3, -1.0 / 8});
      break;
    }
    case MMX_CK45: {
      t.stages = 6; t.fsal = 0; t.order = 5; t.embedded = 1;
      setv(t.c, {0, 1.0 / 5, 3.0 / 10, 3.0 / 5, 1, 7.0 / 8});
      row(1, {1.0 / 5});
      row(2, {3.0 / 40, 9.0 / 40});
      row(3, {3.0 / 10, -9.0 / 10, 6.0 / 5});
      row(4, {-11.0 / 54, 5.0 / 2, -70.0 / 27, 35.0 / 27});
      row(5, {1631.0 / 55296, 175.0 / 512, 575.0 / 13824, 44275.0 / 110592, 253.0 / 4096});
      setv(t.b, {37.0 / 378, 0, 250.0 / 621, 125.0 / 594, 0, 512.0 / 1771});
      const double b4[6] = {2825.0 / 27648, 0, 18575.0 / 48384, 13525.0 / 55296, 277.0 / 14336, 1.0 / 4};
      for (int j = 0; j < 6; ++j) t.e[j] = t.b[j] - b4[j];
      break;
    }
    case MMX_RKF45: {
      t.stages = 6; t.fsal = 0; t.order = 5; t.embedded = 1;
      setv(t.c, {0, 1.0 / 4, 3.0 / 8, 12.0 / 13, 1, 1.0 / 2});
      row(1, {1.0 / 4});
      row(2, {3.0 / 32, 9.0 / 32});
      row(3, {1932.0 / 2197, -7200.0 / 2197, 7296.0 / 2197});
      row(4, {439.0 / 216, -8, 3680.0 / 513, -845.0 / 4104});
      row(5, {-8.0 / 27, 2, -3544.0 / 2565, 1859.0 / 4104, -11.0 / 40});
      setv(t.b, {16.0 / 135, 0, 6656.0 / 12825, 28561.0 / 56430, -9.0 / 50, 2.0 / 55});
      const double b4[6] = {25.0 / 216, 0, 1408.0 / 2565, 2197.0 / 4104, -1.0 / 5, 0};
      for (int j = 0; j < 6; ++j) t.e[j] = t.b[j] - b4[j];
      break;
    }
    case MMX_DP45:
    default: {
      t.stages = 7; t.fsal = 1; t.order = 5; t.embedded = 1;
      setv(t.c, {0, 1.0 / 5, 3.0 / 10, 4.0 / 5, 8.0 / 9, 1, 1});
      row(1, {1.0 / 5});
      row(2, {3.0 / 40, 9.0 / 40});
      row(3, {44.0 / 45, -56.0 / 15, 32.0 / 9});
      row(4, {19372.0 / 6561, -25360.0 / 2187, 64448.0 / 6561, -212.0 / 729});
      row(5, {9017.0 / 3168, -355.0 / 33, 46732.0 / 5247, 49.0 / 176, -5103.0 / 18656});
      row(6, {35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84});
      setv(t.b, {35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84, 0});
      setv(t.e, {71.0 / 57600, 0, -71.0 / 16695, 71.0 / 1920, -17253.0 / 339200, 22.0 / 525, -1.0 / 40});
      break;
    }
  }
  if (!t.fsal)
    for (int j = 0; j < t.stages; ++j) t.a[t.stages][j] = t.b[j];  // final combination as an extra row
  return t;
}

int upload_params(mmx_world* w) {
  if (!w->mat_dirty) return MMX_OK;
  std::vector<float> tab((size_t)w->S * w->nreg * MMX_MATW, 0.f);
  for (int s = 0; s < w->S; ++s)
    for (int r = 0; r < w->nreg; ++r) {
      const mmx_material& m = w->mats[(size_t)s * w->nreg + r];
      float* p = tab.data() + ((size_t)s * w->nreg + r) * MMX_MATW;
      const double iMs = m.Ms > 0 ? 1.0 / m.Ms : 0.0;
      const double gamma = m.gamma > 0 ? m.gamma : GAMMA0;
      p[MP_MS] = (float)m.Ms;
      p[MP_INVMS] = (float)iMs;
      p[MP_A] = (float)m.A;
      p[MP_D] = (float)m.D;
      p[MP_ALPHA] = (float)m.alpha;
      p[MP_LLG] = (float)(gamma / (1.0 + m.alpha * m.alpha));
      p[MP_KU2] = (float)(2.0 * m.Ku1 * iMs);
      p[MP_UX] = (float)m.u[0]; p[MP_UY] = (float)m.u[1]; p[MP_UZ] = (float)m.u[2];
      p[MP_KC2] = (float)(2.0 * m.Kc1 * iMs);
      p[MP_C1X] = (float)m.c1[0]; p[MP_C1Y] = (float)m.c1[1]; p[MP_C1Z] = (float)m.c1[2];
      p[MP_C2X] = (float)m.c2[0]; p[MP_C2Y] = (float)m.c2[1]; p[MP_C2Z] = (float)m.c2[2];
      p[MP_C3X] = (float)(m.c1[1] * m.c2[2] - m.c1[2] * m.c2[1]);
      p[MP_C3Y] = (float)(m.c1[2] * m.c2[0] - m.c1[0] * m.c2[2]);
      p[MP_C3Z] = (float)(m.c1[0] * m.c2[1] - m.c1[1] * m.c2[0]);
      p[MP_MEL1] = (float)(2.0 * m.B1 * iMs);
      p[MP_MEL2] = (float)(2.0 * m.B2 * iMs);
      p[MP_B1] = (float)m.B1;
      p[MP_B2] = (float)m.B2;
      p[MP_ZLB] = (float)(MU_B * m.pol * iMs / (Q_E * (1.0 + m.xi * m.xi)));
      p[MP_XI] = (float)m.xi;
      p[MP_POL] = (float)m.pol;
    }
  MMX_CUDA(cudaMemcpyAsync(w->d_mat, tab.data(), tab.size() * sizeof(float), cudaMemcpyHostToDevice, w->stream));
  MMX_CUDA(cudaStreamSynchronize(w->stream));  // tab goes out of scope
  w->mat_dirty = false;
  return MMX_OK;
}

int alloc_state(mmx_world* w) {
  const int nvec = w->S + (w->has_elastic ? 2 : 0);
  if (w->Y[0] && nvec == w->nvec) {
    // the state keeps its shape; the viscous-damping strain buffer may still have been switched on
    if (w->has_elastic && w->el.rayleigh_beta != 0.0 && !w->strain_f)
      if (int rc = dev_alloc(w, &w->strain_f, 6 * w->N)) return rc;
    return MMX_OK;
  }
  const size_t old_cnt = vecN(w);
  const int old_nvec = w->nvec;
  float* oldY = w->Y[0] ? w->Y[w->sel_host] : nullptr;
  float* keep[2] = {w->Y[0], w->Y[1]};
  w->nvec = nvec;
  const size_t cnt = vecN(w);
  float* ny[2];
  for (int i = 0; i < 2; ++i) {
    if (int rc = dev_alloc(w, &ny[i], cnt)) return rc;
    MMX_CUDA(cudaMemsetAsync(ny[i], 0, cnt * sizeof(float), w->stream));
  }
  if (oldY) {
    const size_t ncopy = (size_t)(old_nvec < nvec ? old_nvec : nvec) * 3 * w->N;
    MMX_CUDA(cudaMemcpyAsync(ny[0], oldY, ncopy * sizeof(float), cudaMemcpyDeviceToDevice, w->stream));
    MMX_CUDA(cudaStreamSynchronize(w->stream));
  }
  for (int i = 0; i < 2; ++i) {
    dev_free(w, &keep[i], old_cnt);
    w->Y[i] = ny[i];
    dev_free(w, &w->YS[i], old_cnt);
    if (int rc = dev_alloc(w, &w->YS[i], cnt)) return rc;
  }
  for (int i = 0; i <= MMX_MAX_STAGES; ++i) {
    dev_free(w, &w->K[i], old_cnt);
    if (int rc = dev_alloc(w, &w->K[i], cnt)) return rc;
  }
  if (!w->bdemag) {
    if (int rc = dev_alloc(w, &w->bdemag, 3 * w->N)) return rc;
    if (int rc = dev_alloc(w, &w->scratch, 3 * w->N)) return rc;
  }
  if (w->has_elastic && !w->strain)
    if (int rc = dev_alloc(w, &w->strain, 6 * w->N)) return rc;
  if (w->has_elastic && w->el.rayleigh_beta != 0.0 && !w->strain_f)
    if (int rc = dev_alloc(w, &w->strain_f, 6 * w->N)) return rc;
  w->sel_host = 0;
  w->k1_valid = false;
  w->cfg_epoch++;
  w->n_tmaps = 0;  // the buffers moved
  // ctrl->sel must follow
  int zero = 0;
  MMX_CUDA(cudaMemcpyAsync(&w->d_ctrl->sel, &zero, sizeof(int), cudaMemcpyHostToDevice, w->stream));
  MMX_CUDA(cudaStreamSynchronize(w->stream));
  return MMX_OK;
}

unsigned active_terms(const mmx_world* w) {
  unsigned t = MMX_T_ALL;
  if (!(w->use_demag && w->dm.ready)) t &= ~MMX_T_DEMAG;
  if (!w->has_elastic) t &= ~MMX_T_MEL;
  if (w->S < 2) t &= ~(MMX_T_A12 | MMX_T_A0 | MMX_T_DMI_INTER | MMX_T_DMI_HOMO);
  return t;
}

void fill_local(const mmx_world* w, LocalArgs& a, unsigned terms) {
  memset(&a, 0, sizeof(a));
  a.nx = w->grid[0]; a.ny = w->grid[1]; a.nz = w->grid[2];
  a.S = w->S; a.nreg = w->nreg;
  for (int k = 0; k < 3; ++k) {
    a.per[k] = w->pbc[k] > 0;
    a.inv_h[k] = (float)(1.0 / w->cell[k]);
    a.inv_h2[k] = (float)(1.0 / (w->cell[k] * w->cell[k]));
    a.bext[k] = (float)w->bext[k];
    a.J[k] = (float)w->J[k];
  }
  a.reg = w->nreg > 1 ? w->d_reg : nullptr;
  a.mat = w->d_mat;
  a.scaleA11 = (float)w->cpl.scale_A11;
  a.scaleA12 = (float)w->cpl.scale_A12;
  a.A12 = (float)w->cpl.A12;
  a.a0pref = (float)(w->cpl.latcon > 0 ? 4.0 * w->cpl.A0 / (w->cpl.latcon * w->cpl.latcon) : 0.0);
  a.Dinter = (float)w->cpl.D_inter;
  for (int k = 0; k < 3; ++k) a.dhomo[k] = (float)w->cpl.d_homo[k];
  a.has_dmiq = w->has_dmiq ? 1 : 0;
  a.has_dmiq12 = 0;
  for (int s = 0; s < 4; ++s)
    for (int k = 0; k < 9; ++k) {
      a.dmiq[s][k / 3][k % 3] = (float)w->dmiq[s][k];
      if (s == 3 && w->dmiq[s][k] != 0.0) a.has_dmiq12 = 1;
    }
  a.has_sl = w->sl.jz != 0.0 ? 1 : 0;
  {
    const double HBAR = 1.054571817e-34;
    const double d = w->sl.thickness > 0 ? w->sl.thickness : w->grid[2] * w->cell[2];
    a.sl_beta = (float)(HBAR * w->sl.jz / (Q_E * d));
    for (int k = 0; k < 3; ++k) a.sl_mp[k] = (float)w->sl.mp[k];
    a.sl_l2 = (float)(w->sl.lambda * w->sl.lambda);
    a.sl_epsp = (float)w->sl.eps_prime;
  }
  a.terms = terms;
  a.has_J = (w->J[0] != 0.0 || w->J[1] != 0.0 || w->J[2] != 0.0) ? 1 : 0;
  a.relax = w->relax_mode ? 1 : 0;
  // Eq.5 without any DMI has the solution d_n m = d_n m' = 0: every ghost equals its cell, exchange and A12 pairs with a
  // ghost add exactly zero, and the field is that of the open boundary bit for bit.  Ghost cells are therefore formed only
  // when some DMI constant is set (the default boundary then costs nothing on the worlds without DMI).
  bool any_dmi = w->has_dmiq || w->cpl.D_inter != 0.0;
  for (size_t q = 0; q < w->mats.size() && !any_dmi; ++q) any_dmi = w->mats[q].D != 0.0;
  a.neumann = (w->boundary == MMX_BC_NEUMANN && any_dmi) ? 1 : 0;
  a.bdemag = (terms & MMX_T_DEMAG) ? w->bdemag : nullptr;
  a.strain = (terms & MMX_T_MEL) ? w->strain : nullptr;
  a.ctrl = w->d_ctrl;
  a.vec_stride = 3 * w->N;
}

void fill_elastic(const mmx_world* w, ElasticArgs& a) {
  memset(&a, 0, sizeof(a));
  a.nx = w->grid[0]; a.ny = w->grid[1]; a.nz = w->grid[2];
  a.S = w->S; a.nreg = w->nreg;
  for (int k = 0; k < 3; ++k) {
    a.per[k] = w->pbc[k] > 0;
    a.inv_h[k] = (float)(1.0 / w->cell[k]);
    a.tvec[k] = (float)w->el.traction_vec[k];
  }
  a.reg = w->nreg > 1 ? w->d_reg : nullptr;
  a.mat = w->d_mat;
  a.C11 = (float)w->el.C11; a.C12 = (float)w->el.C12; a.C44 = (float)w->el.C44;
  a.inv_rho = (float)(1.0 / w->el.rho);
  a.face = w->el.traction_face;
  a.tamp = w->el.traction_amp; a.tfreq = w->el.traction_freq;
  a.strain = w->strain;
  a.beta = (float)w->el.rayleigh_beta;
  a.strain_f = w->el.rayleigh_beta != 0.0 ? w->strain_f : nullptr;
  a.vec_stride = 3 * w->N;
}

struct CtrlHost {  // leading part of MmxCtrl, up to (not including) ca
  MmxCtrl c;
};

// The leading part of the controller block (everything before the coefficient tables) travels between host and
// device without the copy engines: a write is a one-thread kernel that takes the words as its parameter, a read is a
// one-warp kernel that stores them into mapped pinned host memory.  A stepping call therefore never queues behind a
// caller's bulk cudaMemcpyAsync on another stream (the end-to-end leg of bench.py overlaps 50 MB copies with the step).
constexpr int CTRL_HEAD_WORDS = (int)(offsetof(MmxCtrl, ca) / sizeof(unsigned));
struct CtrlHead {
  unsigned w[CTRL_HEAD_WORDS];
};
__global__ void k_ctrl_put(MmxCtrl* c, CtrlHead h) {
  unsigned* dst = reinterpret_cast<unsigned*>(c);
  for (int i = threadIdx.x; i < CTRL_HEAD_WORDS; i += blockDim.x) dst[i] = h.w[i];
}
__global__ void k_ctrl_get(const MmxCtrl* c, unsigned* host_mapped) {
  const unsigned* src = reinterpret_cast<const unsigned*>(c);
  for (int i = threadIdx.x; i < CTRL_HEAD_WORDS; i += blockDim.x) host_mapped[i] = src[i];
  __threadfence_system();
}

int read_ctrl(mmx_world* w, MmxCtrl* h) {
  if (!w->h_ctrl) {
    MMX_CUDA(cudaMemcpyAsync(h, w->d_ctrl, offsetof(MmxCtrl, ca), cudaMemcpyDeviceToHost, w->stream));
    MMX_CUDA(cudaStreamSynchronize(w->stream));
    return MMX_OK;
  }
  k_ctrl_get<<<1, 32, 0, w->stream>>>(w->d_ctrl, w->h_ctrl);
  MMX_CUDA(cudaGetLastError());
  MMX_CUDA(cudaStreamSynchronize(w->stream));
  memcpy(h, w->h_ctrl, offsetof(MmxCtrl, ca));
  return MMX_OK;
}

int write_ctrl(mmx_world* w, const MmxCtrl* h) {
  CtrlHead hd;
  memcpy(hd.w, h, offsetof(MmxCtrl, ca));
  k_ctrl_put<<<1, 32, 0, w->stream>>>(w->d_ctrl, hd);
  MMX_CUDA(cudaGetLastError());
  return MMX_OK;
}

// buffers of one RK step, as "sel pairs" (index with ctrl->sel)
struct StepBufs {
  const float* kj[2][MMX_MAX_STAGES];
};

int prepare(mmx_world* w) {
  if (int rc = alloc_state(w)) return rc;
  return upload_params(w);
}

// One evaluation of the right-hand side at the stage state `yin`, output k into `kout`,
// with the optional RK epilogue described by la (already filled except for pointers here).
int eval_stage(mmx_world* w, LocalArgs& la, ElasticArgs* ea) {
  if (w->has_elastic && ea) {
    if (int rc = mmx_strain_launch(w, *ea)) return rc;
  }
  if (la.terms & MMX_T_DEMAG) {
    if (int rc = mmx_demag_launch(w, la.yin, w->bdemag)) return rc;
  }
  if (int rc = mmx_local_launch(w, la)) return rc;
  if (w->has_elastic && ea) {
    if (int rc = mmx_elastic_launch(w, *ea)) return rc;
  }
  return MMX_OK;
}

int run_steps(mmx_world* w, const mmx_rk_opts* o, mmx_rk_stats* stats) {
  if (int rc = prepare(w)) return rc;
  const MmxTableau tab = make_tableau(o->method);
  if (!tab.embedded && !o->fixed_dt) return mmx_fail(MMX_EINVAL, "method %d has no error estimate: fixed_dt required", o->method);
  if (o->fixed_dt && !(o->dt0 > 0)) return mmx_fail(MMX_EINVAL, "fixed_dt needs dt0 > 0");
  if (o->fixed_dt && o->nsteps <= 0 && o->t_end <= 0) return mmx_fail(MMX_EINVAL, "fixed_dt needs nsteps or t_end");
  const int s = tab.stages;
  const long long launches0 = w->launches;
  const unsigned terms = active_terms(w);

  MmxCtrl h;
  if (int rc = read_ctrl(w, &h)) return rc;
  if (o->t_end > 0 && h.t >= o->t_end) {  // already there: no zero or backward step
    if (stats) {
      stats->accepted = stats->rejected = 0;
      stats->t = h.t; stats->dt = o->dt0 > 0 ? o->dt0 : h.dt; stats->last_err = 0.0; stats->max_torque = h.max_torque;
      stats->launches = 0;
    }
    return MMX_OK;
  }
  h.dt = o->dt0 > 0 ? o->dt0 : 0.0;
  h.dt_max = o->dt_max > 0 ? o->dt_max : 0.0;
  if (w->has_elastic && !o->fixed_dt && !(h.dt_max > 0)) {
    // the error estimate covers the magnetic variables only: keep dt inside the elastic limit of this method
    h.dt_max = elastic_dt_limit(w, tab);
  }
  h.tol = o->tol > 0 ? o->tol : 1e-5;
  h.t_end = o->t_end > 0 ? o->t_end : 0.0;
  h.torque_stop = o->torque_stop > 0 ? o->torque_stop : 0.0;
  h.accepted = h.rejected = h.attempts = 0;
  h.target_accepted = o->nsteps > 0 ? o->nsteps : 0;
  h.active = 1;
  h.fixed = o->fixed_dt ? 1 : 0;
  h.nan_flag = 0;
  h.order = tab.order;
  h.hist_n = 0;
  h.err_bits = h.tq_bits = 0;
  h.err_last = 0;
  if (int rc = write_ctrl(w, &h)) return rc;

  // sel pairs
  float* Ycur[2] = {w->Y[0], w->Y[1]};
  float* Ynew[2] = {w->Y[1], w->Y[0]};
  float* Kfirst[2] = {w->K[0], w->K[MMX_MAX_STAGES]};
  float* Klast[2] = {w->K[MMX_MAX_STAGES], w->K[0]};
  auto kbuf = [&](int j, int which) -> float* {
    if (j == 0) return Kfirst[which];
    if (tab.fsal && j == s - 1) return Klast[which];
    return w->K[j];
  };
  auto ybuf = [&](int i, int which) -> float* {  // stage state Y_i
    if (i == 0) return Ycur[which];
    if (tab.fsal && i == s - 1) return Ynew[which];
    return w->YS[i & 1];
  };

  auto stage_eval = [&](int i, bool epilogue) -> int {
    LocalArgs la;
    fill_local(w, la, terms);
    ElasticArgs ea;
    if (w->has_elastic) fill_elastic(w, ea);
    for (int q = 0; q < 2; ++q) {
      la.yin[q] = ybuf(i, q);
      la.kout[q] = kbuf(i, q);
      la.y0[q] = Ycur[q];
      for (int j = 0; j < i; ++j) la.kprev[q][j] = kbuf(j, q);
    }
    la.stage = i;
    la.n_prev = i;
    if (epilogue) {
      if (i < s - 1) {
        for (int q = 0; q < 2; ++q) la.ynext[q] = ybuf(i + 1, q);
        la.combine_row = i + 1;
      } else if (!tab.fsal) {
        for (int q = 0; q < 2; ++q) la.ynext[q] = Ynew[q];
        la.combine_row = s;
      }
      la.do_err = (tab.embedded && i == s - 1) ? 1 : 0;
    }
    la.do_tq = tab.fsal ? (i == s - 1 || !epilogue) : (i == 0);
    if (w->has_elastic) {
      ea.ctrl = w->d_ctrl;
      ea.stage = i; ea.n_prev = la.n_prev; ea.combine_row = la.combine_row;
      for (int q = 0; q < 2; ++q) {
        ea.yin[q] = la.yin[q]; ea.kout[q] = la.kout[q]; ea.y0[q] = la.y0[q]; ea.ynext[q] = la.ynext[q];
        for (int j = 0; j < i; ++j) ea.kprev[q][j] = la.kprev[q][j];
      }
    }
    return eval_stage(w, la, w->has_elastic ? &ea : nullptr);
  };

  // k1 at the current state (FSAL methods keep it across steps; also gives the first dt)
  const bool need_first_dt = !(o->dt0 > 0);
  if ((tab.fsal && !(w->k1_valid && w->k1_method == o->method)) || need_first_dt) {
    if (int rc = mmx_controller_launch(w, tab, 0)) return rc;  // clears reductions, fills cc
    if (int rc = stage_eval(0, false)) return rc;
    if (int rc = mmx_controller_launch(w, tab, 3)) return rc;
    w->k1_valid = tab.fsal;
    w->k1_method = o->method;
  }

  auto attempt = [&]() -> int {
    if (int rc = mmx_controller_launch(w, tab, 0)) return rc;
    if (tab.fsal) {
      const float* y0[2] = {Ycur[0], Ycur[1]};
      const float* k1[2] = {Kfirst[0], Kfirst[1]};
      float* yn[2] = {ybuf(1, 0), ybuf(1, 1)};
      if (int rc = mmx_combine_launch(w, y0, k1, yn, 1)) return rc;
    } else {
      if (int rc = stage_eval(0, true)) return rc;
    }
    for (int i = 1; i < s; ++i)
      if (int rc = stage_eval(i, true)) return rc;
    return mmx_controller_launch(w, tab, 1);
  };

  // One attempt = one CUDA graph launch.  Captured on first use per (method, configuration epoch);
  // any failure to capture falls back to plain launches.  Off while the per-kernel profiler runs.
  auto attempt_fast = [&]() -> int {
    if (!w->use_graphs || w->prof) return attempt();
    if (!(w->step_graph && w->graph_method == o->method && w->graph_epoch == w->cfg_epoch)) {
      if (w->step_graph) { cudaGraphExecDestroy(w->step_graph); w->step_graph = nullptr; }
      const long long l0 = w->launches;
      cudaGraph_t graph = nullptr;
      if (cudaStreamBeginCapture(w->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
        cudaGetLastError();
        w->use_graphs = false;
        return attempt();
      }
      const int rc = attempt();
      const cudaError_t ce = cudaStreamEndCapture(w->stream, &graph);
      w->graph_launches = w->launches - l0;
      w->launches = l0;
      if (rc != MMX_OK || ce != cudaSuccess || graph == nullptr ||
          cudaGraphInstantiate(&w->step_graph, graph, 0) != cudaSuccess) {
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        w->step_graph = nullptr;
        w->use_graphs = false;
        return rc != MMX_OK ? rc : attempt();
      }
      cudaGraphDestroy(graph);
      w->graph_method = o->method;
      w->graph_epoch = w->cfg_epoch;
    }
    MMX_CUDA(cudaGraphLaunch(w->step_graph, w->stream));
    w->launches += w->graph_launches;
    return MMX_OK;
  };

  const long long max_attempts = o->max_attempts > 0 ? o->max_attempts : 1000000;
  long long done = 0;
  while (done < max_attempts) {
    long long chunk;
    if (o->fixed_dt && o->nsteps > 0) chunk = o->nsteps - done;
    else chunk = 8;
    if (chunk > max_attempts - done) chunk = max_attempts - done;
    if (chunk > 4096) chunk = 4096;
    if (chunk <= 0) break;
    for (long long q = 0; q < chunk; ++q)
      if (int rc = attempt_fast()) return rc;
    done += chunk;
    if (int rc = read_ctrl(w, &h)) return rc;
    if (!h.active) break;
    if (o->fixed_dt && o->nsteps > 0 && done >= o->nsteps) break;
  }
  if (int rc = mmx_controller_launch(w, tab, 2)) return rc;
  if (int rc = read_ctrl(w, &h)) return rc;
  w->sel_host = h.sel;
  if (!tab.fsal) w->k1_valid = false;
  if (stats) {
    stats->accepted = h.accepted; stats->rejected = h.rejected;
    stats->t = h.t; stats->dt = h.dt; stats->last_err = h.err_last; stats->max_torque = h.max_torque;
    stats->launches = w->launches - launches0;
  }
  if (h.nan_flag) return mmx_fail(MMX_ENAN, "NaN/Inf in the error or torque reduction at t = %g", h.t);
  return MMX_OK;
}

int copy_out(mmx_world* w, const float* dev, float* out, int mem, size_t count) {
  MMX_CUDA(cudaMemcpyAsync(out, dev, count * sizeof(float),
                           mem == MMX_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, w->stream));
  if (mem == MMX_HOST) MMX_CUDA(cudaStreamSynchronize(w->stream));
  return MMX_OK;
}

// field pieces needed by an evaluation at the current state
int eval_prereq(mmx_world* w, unsigned terms) {
  const float* yin[2] = {w->Y[w->sel_host], w->Y[w->sel_host]};
  if (terms & MMX_T_MEL) {
    ElasticArgs ea;
    fill_elastic(w, ea);
    ea.yin[0] = ea.yin[1] = yin[0];
    if (int rc = mmx_strain_launch(w, ea)) return rc;
  }
  if (terms & MMX_T_DEMAG) {
    if (int rc = mmx_demag_launch(w, yin, w->bdemag)) return rc;
  }
  return MMX_OK;
}

}  // namespace

int mmx_fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}

extern "C" {

const char* mmx_last_error(void) { return g_err; }
const char* mmx_version(void) { return "mmx 0.3 (sm_100a)"; }
int mmx_abi_version(void) { return MMX_ABI_VERSION; }

int mmx_rk_imag_stability_limit(int method, double growth, double* y_max) {
  if (!y_max) return mmx_fail(MMX_EINVAL, "NULL argument");
  if (method < MMX_RK4 || method > MMX_RKF45) return mmx_fail(MMX_EINVAL, "unknown method %d", method);
  if (!(growth >= 0)) return mmx_fail(MMX_EINVAL, "growth must be >= 0");
  *y_max = imag_axis_limit(make_tableau(method), growth);
  return MMX_OK;
}

int mmx_world_create(const int grid[3], const double cellsize[3], const int pbc[3], int n_sublattices,
                     void* cuda_stream, mmx_world** out) {
  if (!grid || !cellsize || !pbc || !out) return mmx_fail(MMX_EINVAL, "NULL argument");
  *out = nullptr;
  if (n_sublattices < 1 || n_sublattices > 3) return mmx_fail(MMX_EINVAL, "n_sublattices must be 1, 2 or 3");
  for (int a = 0; a < 3; ++a) {
    if (grid[a] < 1) return mmx_fail(MMX_EINVAL, "grid[%d] = %d", a, grid[a]);
    if (!(cellsize[a] > 0)) return mmx_fail(MMX_EINVAL, "cellsize[%d] must be > 0", a);
    if (pbc[a] < 0) return mmx_fail(MMX_EINVAL, "pbc[%d] < 0", a);
  }
  if ((double)grid[0] * grid[1] * grid[2] > 2.0e9) return mmx_fail(MMX_EINVAL, "grid too large");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return mmx_fail(MMX_ECUDA, "no CUDA device: libmmx has no CPU fallback");
  }
  mmx_world* w = new (std::nothrow) mmx_world();
  if (!w) return mmx_fail(MMX_ENOMEM, "host allocation failed");
  for (int a = 0; a < 3; ++a) { w->grid[a] = grid[a]; w->cell[a] = cellsize[a]; w->pbc[a] = pbc[a]; }
  w->S = n_sublattices;
  w->nvec = w->S;
  w->N = (size_t)grid[0] * grid[1] * grid[2];
  w->stream = (cudaStream_t)cuda_stream;
  w->own_stream = false;
  if (!w->stream) {
    // The legacy default stream cannot be captured into a CUDA graph.  A world created on it runs on
    // its own *blocking* stream instead, which the runtime orders against the legacy default stream
    // in both directions, so callers that enqueue on stream 0 see the same ordering as before.
    if (cudaStreamCreate(&w->stream) == cudaSuccess) w->own_stream = true;
    else { cudaGetLastError(); w->stream = nullptr; }
  }
  w->has_dmiq = false;
  for (int s = 0; s < 4; ++s)
    for (int k = 0; k < 9; ++k) w->dmiq[s][k] = 0.0;
  memset(&w->sl, 0, sizeof(w->sl));
  w->relax_mode = false;
  // P:L161 "The Neumann boundary conditions as given in Eq. (5) are the default in mumax+"; Eq.5 is written for a
  // sublattice and its partner, so a three-sublattice world starts open (mmx_set_boundary refuses Neumann there)
  w->boundary = n_sublattices <= 2 ? MMX_BC_NEUMANN : MMX_BC_OPEN;
  w->n_tmaps = 0;
  w->step_graph = nullptr; w->graph_method = -1; w->graph_epoch = -1; w->cfg_epoch = 0; w->graph_launches = 0;
  w->use_graphs = getenv("MMX_NO_GRAPH") == nullptr;
  {
    int dev = 0;
    cudaGetDevice(&dev);
    w->sm_count = 148;
    cudaDeviceGetAttribute(&w->sm_count, cudaDevAttrMultiProcessorCount, dev);
    if (w->sm_count <= 0) w->sm_count = 148;
  }
  w->nreg = 1;
  w->d_reg = nullptr;
  w->mats.resize(w->S);
  for (auto& m : w->mats) default_material(&m);
  w->d_mat = nullptr;
  w->mat_dirty = true;
  memset(&w->cpl, 0, sizeof(w->cpl));
  w->cpl.scale_A11 = w->cpl.scale_A12 = 1.0;
  w->cpl.latcon = 0.35e-9;
  for (int a = 0; a < 3; ++a) w->bext[a] = w->J[a] = 0.0;
  w->has_elastic = false;
  memset(&w->el, 0, sizeof(w->el));
  w->el.traction_face = -1;
  w->use_demag = true;
  memset(&w->dm, 0, sizeof(w->dm));
  w->Y[0] = w->Y[1] = w->YS[0] = w->YS[1] = nullptr;
  for (int i = 0; i <= MMX_MAX_STAGES; ++i) w->K[i] = nullptr;
  w->bdemag = w->strain = w->strain_f = w->scratch = nullptr;
  w->d_ctrl = nullptr; w->d_acc = nullptr; w->h_ctrl = nullptr;
  w->sel_host = 0; w->k1_valid = false; w->k1_method = -1;
  w->dev_bytes = 0; w->launches = 0;
  w->prof = false;
  int rc = dev_alloc(w, &w->d_mat, (size_t)w->S * MMX_MATW);
  if (!rc) rc = dev_alloc(w, &w->d_ctrl, 1);
  if (!rc) rc = dev_alloc(w, &w->d_acc, 64);
  if (!rc) {
    MmxCtrl* hc = new (std::nothrow) MmxCtrl();
    if (!hc) rc = mmx_fail(MMX_ENOMEM, "host allocation failed");
    else {
      memset(hc, 0, sizeof(*hc));
      hc->active = 1;
      cudaError_t e = cudaMemcpy(w->d_ctrl, hc, sizeof(*hc), cudaMemcpyHostToDevice);
      delete hc;
      if (e != cudaSuccess) rc = mmx_fail(MMX_ECUDA, "ctrl upload failed: %s", cudaGetErrorString(e));
    }
  }
  if (!rc && cudaHostAlloc(reinterpret_cast<void**>(&w->h_ctrl), offsetof(MmxCtrl, ca), cudaHostAllocMapped) != cudaSuccess) {
    cudaGetLastError();
    w->h_ctrl = nullptr;  // (read_ctrl falls back to a plain copy)
  }
  if (rc) { mmx_world_destroy(w); return rc; }
  *out = w;
  return MMX_OK;
}

int mmx_world_destroy(mmx_world* w) {
  if (!w) return MMX_OK;
  cudaStreamSynchronize(w->stream);
  cudaFree(w->d_reg); cudaFree(w->d_mat); cudaFree(w->d_ctrl); cudaFree(w->d_acc);
  if (w->h_ctrl) cudaFreeHost(w->h_ctrl);
  for (int i = 0; i < 2; ++i) { cudaFree(w->Y[i]); cudaFree(w->YS[i]); }
  for (int i = 0; i <= MMX_MAX_STAGES; ++i) cudaFree(w->K[i]);
  cudaFree(w->bdemag); cudaFree(w->strain); cudaFree(w->strain_f); cudaFree(w->scratch);
  for (int a = 0; a < 3; ++a) cudaFree(w->dm.tw[a]);
  cudaFree(w->dm.spec1); cudaFree(w->dm.spec2); cudaFree(w->dm.khat); cudaFree(w->dm.kimg);
  if (w->step_graph) cudaGraphExecDestroy(w->step_graph);
  if (w->own_stream) cudaStreamDestroy(w->stream);
  cudaGetLastError();
  delete w;
  return MMX_OK;
}

int mmx_set_regions(mmx_world* w, const uint16_t* region_of_cell, int mem, int n_regions) {
  if (!w) return mmx_fail(MMX_EINVAL, "NULL world");
  if (n_regions < 1 || n_regions > 65536) return mmx_fail(MMX_EINVAL, "n_regions = %d", n_regions);
  if (!region_of_cell) n_regions = 1;
  if (region_of_cell && mem == MMX_HOST) {
    for (size_t i = 0; i < w->N; ++i)
      if (region_of_cell[i] >= n_regions) return mmx_fail(MMX_EINVAL, "region index %d >= n_regions at cell %zu", region_of_cell[i], i);
  }
  cudaStreamSynchronize(w->stream);
  if (n_regions != w->nreg) {
    dev_free(w, &w->d_mat, (size_t)w->S * w->nreg * MMX_MATW);
    w->nreg = n_regions;
    if (int rc = dev_alloc(w, &w->d_mat, (size_t)w->S * w->nreg * MMX_MATW)) return rc;
    w->mats.assign((size_t)w->S * w->nreg, mmx_material());
    for (auto& m : w->mats) default_material(&m);
  }
  w->mat_dirty = true;
  if (region_of_cell) {
    if (!w->d_reg)
      if (int rc = dev_alloc(w, &w->d_reg, w->N)) return rc;
    MMX_CUDA(cudaMemcpyAsync(w->d_reg, region_of_cell, w->N * sizeof(uint16_t),
                             mem == MMX_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, w->stream));
    MMX_CUDA(cudaStreamSynchronize(w->stream));
  }
  w->k1_valid = false;
  w->cfg_epoch++;  // kernel arguments change: the captured step graph is stale
  return MMX_OK;
}

int mmx_set_material(mmx_world* w, int sublattice, int region, const mmx_material* mat) {
  if (!w || !mat) return mmx_fail(MMX_EINVAL, "NULL argument");
  if (sublattice < 0 || sublattice >= w->S) return mmx_fail(MMX_EINVAL, "sublattice %d out of range", sublattice);
  if (region < 0 || region >= w->nreg) return mmx_fail(MMX_EINVAL, "region %d out of range (n_regions = %d)", region, w->nreg);
  if (mat->Ms < 0 || mat->alpha < 0) return mmx_fail(MMX_EINVAL, "Ms and alpha must be >= 0");
  w->mats[(size_t)sublattice * w->nreg + region] = *mat;
  w->mat_dirty = true;
  w->k1_valid = false;
  w->cfg_epoch++;  // kernel arguments change: the captured step graph is stale
  return MMX_OK;
}

int mmx_set_coupling(mmx_world* w, const mmx_coupling* c) {
  if (!w || !c) return mmx_fail(MMX_EINVAL, "NULL argument");
  if (c->A0 != 0.0 && !(c->latcon > 0)) return mmx_fail(MMX_EINVAL, "A0 != 0 needs latcon > 0");
  w->cpl = *c;
  w->k1_valid = false;
  w->cfg_epoch++;  // kernel arguments change: the captured step graph is stale
  return MMX_OK;
}

int mmx_set_bext(mmx_world* w, const double B[3]) {
  if (!w || !B) return mmx_fail(MMX_EINVAL, "NULL argument");
  for (int a = 0; a < 3; ++a) w->bext[a] = B[a];
  w->k1_valid = false;
  w->cfg_epoch++;  // kernel arguments change: the captured step graph is stale
  return MMX_OK;
}

int mmx_set_current(mmx_world* w, const double J[3]) {
  if (!w || !J) return mmx_fail(MMX_EINVAL, "NULL argument");
  for (int a = 0; a < 3; ++a) w->J[a] = J[a];
  w->k1_valid = false;
  w->cfg_epoch++;  // kernel arguments change: the captured step graph is stale
  return MMX_OK;
}

int mmx_set_dmi_tensor(mmx_world* w, int sublattice, const double q[9]) {
  if (!w) return mmx_fail(MMX_EINVAL, "NULL world");
  if (sublattice == MMX_DMI_INTER) {
    if (w->S < 2) return mmx_fail(MMX_EINVAL, "the inter-sublattice DMI tensor needs two or three sublattices");
    sublattice = 3;
  } else if (sublattice < 0 || sublattice >= w->S) {
    return mmx_fail(MMX_EINVAL, "sublattice %d out of range", sublattice);
  }
  for (int k = 0; k < 9; ++k) w->dmiq[sublattice][k] = q ? q[k] : 0.0;
  w->has_dmiq = false;
  for (int s = 0; s < 4; ++s)
    for (int k = 0; k < 9; ++k) w->has_dmiq = w->has_dmiq || w->dmiq[s][k] != 0.0;
  w->k1_valid = false;
  w->cfg_epoch++;  // kernel arguments change: the captured step graph is stale
  return MMX_OK;
}

int mmx_set_boundary(mmx_world* w, int kind) {
  if (!w) return mmx_fail(MMX_EINVAL, "NULL world");
  if (kind != MMX_BC_OPEN && kind != MMX_BC_NEUMANN) return mmx_fail(MMX_EINVAL, "unknown boundary kind %d", kind);
  if (kind == MMX_BC_NEUMANN && w->S > 2)
    return mmx_fail(MMX_EINVAL, "the Neumann boundary condition of Eq.5 is written for one sublattice and its partner");
  w->boundary = kind;
  w->k1_valid = false;
  w->cfg_epoch++;  // kernel arguments change: the captured step graph is stale
  return MMX_OK;
}

int mmx_set_slonczewski(mmx_world* w, const mmx_slonczewski* sl) {
  if (!w) return mmx_fail(MMX_EINVAL, "NULL world");
  if (!sl) {
    memset(&w->sl, 0, sizeof(w->sl));
  } else {
    const double n = sqrt(sl->mp[0] * sl->mp[0] + sl->mp[1] * sl->mp[1] + sl->mp[2] * sl->mp[2]);
    if (sl->jz != 0.0 && !(n > 0)) return mmx_fail(MMX_EINVAL, "Slonczewski torque needs a fixed-layer direction mp");
    if (sl->jz != 0.0 && !(sl->lambda >= 1.0)) return mmx_fail(MMX_EINVAL, "Slonczewski Lambda must be >= 1");
    w->sl = *sl;
    for (int k = 0; k < 3; ++k) w->sl.mp[k] = n > 0 ? sl->mp[k] / n : 0.0;
  }
  w->k1_valid = false;
  w->cfg_epoch++;  // kernel arguments change: the captured step graph is stale
  return MMX_OK;
}

int mmx_set_elastic(mmx_world* w, const mmx_elastic* e) {
  if (!w) return mmx_fail(MMX_EINVAL, "NULL world");
  if (e) {
    if (!(e->rho > 0)) return mmx_fail(MMX_EINVAL, "rho must be > 0");
    if (e->traction_face < -1 || e->traction_face > 5) return mmx_fail(MMX_EINVAL, "traction_face out of range");
    if (!(e->rayleigh_beta >= 0)) return mmx_fail(MMX_EINVAL, "rayleigh_beta must be >= 0");
    w->el = *e;
    w->has_elastic = true;
  } else {
    w->has_elastic = false;
  }
  w->k1_valid = false;
  w->cfg_epoch++;  // kernel arguments change: the captured step graph is stale
  if (w->Y[0]) return alloc_state(w);
  return MMX_OK;
}

int mmx_enable_demag(mmx_world* w, int on) {
  if (!w) return mmx_fail(MMX_EINVAL, "NULL world");
  w->use_demag = on != 0;
  w->k1_valid = false;
  w->cfg_epoch++;  // kernel arguments change: the captured step graph is stale
  return MMX_OK;
}

static int field_vec(mmx_world* w, int field, int* vec) {
  switch (field) {
    case MMX_F_M0: *vec = 0; return MMX_OK;
    case MMX_F_M1:
      if (w->S < 2) return mmx_fail(MMX_EINVAL, "world has one sublattice");
      *vec = 1; return MMX_OK;
    case MMX_F_M2:
      if (w->S < 3) return mmx_fail(MMX_EINVAL, "world has fewer than three sublattices");
      *vec = 2; return MMX_OK;
    case MMX_F_U:
    case MMX_F_V:
      if (!w->has_elastic) return mmx_fail(MMX_ESTATE, "elastic fields need mmx_set_elastic first");
      *vec = w->S + (field == MMX_F_V ? 1 : 0); return MMX_OK;
    default: return mmx_fail(MMX_EINVAL, "unknown field %d", field);
  }
}

int mmx_set_state(mmx_world* w, int field, const float* buf, int mem) {
  if (!w || !buf) return mmx_fail(MMX_EINVAL, "NULL argument");
  int vec;
  if (int rc = field_vec(w, field, &vec)) return rc;
  if (int rc = alloc_state(w)) return rc;
  MMX_CUDA(cudaMemcpyAsync(w->Y[w->sel_host] + (size_t)vec * 3 * w->N, buf, 3 * w->N * sizeof(float),
                           mem == MMX_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, w->stream));
  if (mem == MMX_HOST) MMX_CUDA(cudaStreamSynchronize(w->stream));
  w->k1_valid = false;
  return MMX_OK;
}

int mmx_get_state(mmx_world* w, int field, float* buf, int mem) {
  if (!w || !buf) return mmx_fail(MMX_EINVAL, "NULL argument");
  int vec;
  if (int rc = field_vec(w, field, &vec)) return rc;
  if (int rc = alloc_state(w)) return rc;
  return copy_out(w, w->Y[w->sel_host] + (size_t)vec * 3 * w->N, buf, mem, 3 * w->N);
}

int mmx_set_time(mmx_world* w, double t) {
  if (!w) return mmx_fail(MMX_EINVAL, "NULL world");
  MMX_CUDA(cudaMemcpyAsync(&w->d_ctrl->t, &t, sizeof(double), cudaMemcpyHostToDevice, w->stream));
  MMX_CUDA(cudaStreamSynchronize(w->stream));
  w->k1_valid = false;
  return MMX_OK;
}

int mmx_get_time(mmx_world* w, double* t) {
  if (!w || !t) return mmx_fail(MMX_EINVAL, "NULL argument");
  MMX_CUDA(cudaMemcpyAsync(t, &w->d_ctrl->t, sizeof(double), cudaMemcpyDeviceToHost, w->stream));
  MMX_CUDA(cudaStreamSynchronize(w->stream));
  return MMX_OK;
}

int mmx_newell_tensor_host(const int grid[3], const double cellsize[3], const int pbc[3],
                           double analytic_cutoff_cells, double* out, long long out_len) {
  if (!grid || !cellsize || !pbc || !out) return mmx_fail(MMX_EINVAL, "NULL argument");
  std::vector<double> oct;
  int n[3];
  if (int rc = mmx_newell_octant(grid, cellsize, pbc, analytic_cutoff_cells, oct, n)) return rc;
  if ((long long)oct.size() != out_len) return mmx_fail(MMX_EINVAL, "out_len %lld, expected %zu", out_len, oct.size());
  memcpy(out, oct.data(), oct.size() * sizeof(double));
  return MMX_OK;
}

int mmx_kernel_spectrum_host(const int grid[3], const double cellsize[3], const int pbc[3],
                             double analytic_cutoff_cells, float* out, long long out_len, long long dims_out[5]) {
  if (!grid || !cellsize || !pbc || !dims_out) return mmx_fail(MMX_EINVAL, "NULL argument");
  mmx_world tmp;
  for (int a = 0; a < 3; ++a) { tmp.grid[a] = grid[a]; tmp.pbc[a] = pbc[a]; tmp.cell[a] = cellsize[a]; }
  if (int rc = mmx_demag_plan_sizes(&tmp)) return rc;
  const DemagPlan& d = tmp.dm;
  dims_out[0] = d.px; dims_out[1] = d.py; dims_out[2] = d.pz; dims_out[3] = d.xp;
  dims_out[4] = 6LL * d.kz * d.ky * d.xp;
  if (!out) return MMX_OK;
  if (out_len != dims_out[4]) return mmx_fail(MMX_EINVAL, "out_len %lld, expected %lld", out_len, dims_out[4]);
  std::vector<double> oct;
  int n[3];
  if (int rc = mmx_newell_octant(grid, cellsize, pbc, analytic_cutoff_cells, oct, n)) return rc;
  const int P[3] = {d.px, d.py, d.pz};
  std::vector<float> khat;
  const double scale = -MU0 / ((double)d.px * d.py * d.pz);
  if (int rc = mmx_kernel_spectrum(grid, pbc, P, d.xp, oct, n, scale, khat)) return rc;
  memcpy(out, khat.data(), khat.size() * sizeof(float));
  return MMX_OK;
}

int mmx_demag_kernel_init(mmx_world* w, double analytic_cutoff_cells) {
  if (!w) return mmx_fail(MMX_EINVAL, "NULL world");
  DemagPlan& d = w->dm;
  if (int rc = mmx_demag_plan_sizes(w)) return rc;
  std::vector<double> oct;
  int n[3];
  if (int rc = mmx_newell_octant(w->grid, w->cell, w->pbc, analytic_cutoff_cells, oct, n)) return rc;
  const int P[3] = {d.px, d.py, d.pz};
  std::vector<float> khat;
  const double scale = -MU0 / ((double)d.px * d.py * d.pz);
  if (int rc = mmx_kernel_spectrum(w->grid, w->pbc, P, d.xp, oct, n, scale, khat)) return rc;
  cudaStreamSynchronize(w->stream);
  // 3-D worlds with 128-point z lines on grids large enough for the pipelined y pass keep the padded
  // spectrum tile-major and the kernel spectrum as per-tile images (demag_tile.cu)
  d.tiled = mmx_tile_ok(d) && mmx_mid_col_ok(d.py, d.ny) && mmx_mid_pipe_ok(w, d.py, 3 * d.nz);
  std::vector<float> kimg;
  if (d.tiled) mmx_tile_kimg_build(d, khat, kimg);
  if (!d.spec1) {
    if (d.tiled) {
      if (int rc = dev_alloc(w, &d.kimg, kimg.size())) return rc;
    } else {
      if (int rc = dev_alloc(w, &d.khat, khat.size())) return rc;
    }
    if (int rc = dev_alloc(w, &d.spec1, (size_t)3 * d.nz * d.ny * d.xp)) return rc;
    if (d.nz > 1 && d.py > 1)
      if (int rc = dev_alloc(w, &d.spec2, d.tiled ? mmx_tile_spec_elems(d.py, d.xc, d.nz) : (size_t)3 * d.nz * d.py * d.xp)) return rc;
    for (int a = 0; a < 3; ++a) {
      std::vector<float2> tw(P[a]);
      for (int q = 0; q < P[a]; ++q) {
        const double ang = -2.0 * M_PI * q / P[a];
        tw[q] = make_float2((float)cos(ang), (float)sin(ang));
      }
      if (int rc = dev_alloc(w, &d.tw[a], (size_t)P[a])) return rc;
      MMX_CUDA(cudaMemcpy(d.tw[a], tw.data(), tw.size() * sizeof(float2), cudaMemcpyHostToDevice));
    }
  }
  if (d.tiled) MMX_CUDA(cudaMemcpy(d.kimg, kimg.data(), kimg.size() * sizeof(float), cudaMemcpyHostToDevice));
  else MMX_CUDA(cudaMemcpy(d.khat, khat.data(), khat.size() * sizeof(float), cudaMemcpyHostToDevice));
  d.ready = true;
  w->k1_valid = false;
  w->cfg_epoch++;  // kernel arguments change: the captured step graph is stale
  return MMX_OK;
}

int mmx_eval_heff(mmx_world* w, int sublattice, unsigned term_mask, float* out, int mem) {
  if (!w || !out) return mmx_fail(MMX_EINVAL, "NULL argument");
  if (sublattice < 0 || sublattice >= w->S) return mmx_fail(MMX_EINVAL, "sublattice %d out of range", sublattice);
  if ((term_mask & MMX_T_DEMAG) && !w->dm.ready) return mmx_fail(MMX_ESTATE, "demag term requested before mmx_demag_kernel_init");
  if (int rc = prepare(w)) return rc;
  unsigned terms = term_mask;
  if (!w->has_elastic) terms &= ~MMX_T_MEL;
  if (w->S < 2) terms &= ~(MMX_T_A12 | MMX_T_A0 | MMX_T_DMI_INTER | MMX_T_DMI_HOMO);
  if (int rc = eval_prereq(w, terms)) return rc;
  LocalArgs la;
  fill_local(w, la, terms);
  la.yin[0] = la.yin[1] = w->Y[w->sel_host];
  float* dst = mem == MMX_DEVICE ? out : w->scratch;
  la.heff_out = dst;
  la.heff_s = sublattice;
  if (int rc = mmx_local_launch(w, la)) return rc;
  if (mem == MMX_HOST) return copy_out(w, w->scratch, out, mem, 3 * w->N);
  return MMX_OK;
}

int mmx_eval_torque(mmx_world* w, int sublattice, float* out, int mem) {
  if (!w || !out) return mmx_fail(MMX_EINVAL, "NULL argument");
  if (sublattice < 0 || sublattice >= w->S) return mmx_fail(MMX_EINVAL, "sublattice %d out of range", sublattice);
  if (int rc = prepare(w)) return rc;
  const unsigned terms = active_terms(w);
  if (int rc = eval_prereq(w, terms)) return rc;
  LocalArgs la;
  fill_local(w, la, terms);
  la.yin[0] = la.yin[1] = w->Y[w->sel_host];
  float* dst = mem == MMX_DEVICE ? out : w->scratch;
  la.tau_out = dst;
  la.heff_s = sublattice;
  if (int rc = mmx_local_launch(w, la)) return rc;
  if (mem == MMX_HOST) return copy_out(w, w->scratch, out, mem, 3 * w->N);
  return MMX_OK;
}

int mmx_eval_accel(mmx_world* w, float* out, int mem) {
  if (!w || !out) return mmx_fail(MMX_EINVAL, "NULL argument");
  if (!w->has_elastic) return mmx_fail(MMX_ESTATE, "mmx_set_elastic has not been called");
  if (int rc = prepare(w)) return rc;
  double t = 0;
  if (int rc = mmx_get_time(w, &t)) return rc;
  ElasticArgs ea;
  fill_elastic(w, ea);
  ea.yin[0] = ea.yin[1] = w->Y[w->sel_host];
  ea.t_fixed = t;
  if (int rc = mmx_strain_launch(w, ea)) return rc;
  float* dst = mem == MMX_DEVICE ? out : w->scratch;
  ea.accel_out = dst;
  if (int rc = mmx_elastic_launch(w, ea)) return rc;
  if (mem == MMX_HOST) return copy_out(w, w->scratch, out, mem, 3 * w->N);
  return MMX_OK;
}

int mmx_energy(mmx_world* w, unsigned term_mask, double* joule_out) {
  if (!w || !joule_out) return mmx_fail(MMX_EINVAL, "NULL argument");
  if (int rc = prepare(w)) return rc;
  unsigned terms = term_mask & active_terms(w);
  if (int rc = eval_prereq(w, terms)) return rc;
  MMX_CUDA(cudaMemsetAsync(w->d_acc, 0, 64 * sizeof(double), w->stream));
  int slot = 0;
  double coef[64];
  for (int s = 0; s < w->S; ++s)
    for (int b = 0; b < 11; ++b) {  // one pass per term bit of MMX_T_ALL
      const unsigned bit = 1u << b;
      if (!(terms & bit)) continue;
      LocalArgs la;
      fill_local(w, la, bit);
      la.yin[0] = la.yin[1] = w->Y[w->sel_host];
      la.heff_out = w->scratch;
      la.heff_s = s;
      if (int rc = mmx_local_launch(w, la)) return rc;
      if (int rc = mmx_energy_launch(w, (unsigned)s, w->scratch, w->d_acc + slot)) return rc;
      coef[slot] = bit == MMX_T_ZEEMAN ? 1.0 : (bit == MMX_T_ANIS_C ? 0.25 : 0.5);
      ++slot;
    }
  double h[64];
  MMX_CUDA(cudaMemcpyAsync(h, w->d_acc, 64 * sizeof(double), cudaMemcpyDeviceToHost, w->stream));
  MMX_CUDA(cudaStreamSynchronize(w->stream));
  const double V = w->cell[0] * w->cell[1] * w->cell[2];
  double E = 0;
  for (int q = 0; q < slot; ++q) E += -coef[q] * V * h[q];
  *joule_out = E;
  return MMX_OK;
}

int mmx_elastic_energy(mmx_world* w, double* strain_energy, double* kinetic_energy) {
  if (!w || !strain_energy || !kinetic_energy) return mmx_fail(MMX_EINVAL, "NULL argument");
  if (!w->has_elastic) return mmx_fail(MMX_ESTATE, "mmx_set_elastic has not been called");
  if (int rc = prepare(w)) return rc;
  if (int rc = eval_prereq(w, MMX_T_MEL)) return rc;
  return mmx_elastic_energy_launch(w, strain_energy, kinetic_energy);
}

int mmx_max_torque(mmx_world* w, double* out) {
  if (!w || !out) return mmx_fail(MMX_EINVAL, "NULL argument");
  if (int rc = prepare(w)) return rc;
  const unsigned terms = active_terms(w);
  if (int rc = eval_prereq(w, terms)) return rc;
  unsigned zero = 0;
  MMX_CUDA(cudaMemcpyAsync(&w->d_ctrl->tq_bits, &zero, sizeof(zero), cudaMemcpyHostToDevice, w->stream));
  LocalArgs la;
  fill_local(w, la, terms);
  la.yin[0] = la.yin[1] = w->Y[w->sel_host];
  la.kout[0] = la.kout[1] = w->K[1];
  la.do_tq = 1;
  if (int rc = mmx_local_launch(w, la)) return rc;
  unsigned bits = 0;
  MMX_CUDA(cudaMemcpyAsync(&bits, &w->d_ctrl->tq_bits, sizeof(bits), cudaMemcpyDeviceToHost, w->stream));
  MMX_CUDA(cudaStreamSynchronize(w->stream));
  float f;
  memcpy(&f, &bits, sizeof(f));
  *out = (double)f;
  if (bits >= 0x7f800000u) return mmx_fail(MMX_ENAN, "NaN/Inf torque");
  return MMX_OK;
}

int mmx_stray_field(mmx_world* w, double height, float* out, int mem) {
  if (!w || !out) return mmx_fail(MMX_EINVAL, "NULL argument");
  if (w->pbc[0] || w->pbc[1] || w->pbc[2]) return mmx_fail(MMX_EINVAL, "mmx_stray_field needs open boundaries");
  if (!(height > -0.5 * w->cell[2])) return mmx_fail(MMX_EINVAL, "the probe layer must lie above the centre of the top layer");
  if (int rc = prepare(w)) return rc;
  const size_t cnt = (size_t)3 * w->grid[0] * w->grid[1];
  float* dst = out;
  float* tmp = nullptr;
  if (mem == MMX_HOST) {
    MMX_CUDA(cudaMalloc(&tmp, cnt * sizeof(float)));
    dst = tmp;
  }
  int rc = mmx_stray_launch(w, height, 0.0, dst);
  if (!rc && mem == MMX_HOST) rc = copy_out(w, tmp, out, MMX_HOST, cnt);
  cudaFree(tmp);
  return rc;
}

int mmx_step_rk4(mmx_world* w, double dt, long long nsteps) {
  if (!w) return mmx_fail(MMX_EINVAL, "NULL world");
  if (!(dt > 0) || nsteps < 0) return mmx_fail(MMX_EINVAL, "dt must be > 0 and nsteps >= 0");
  if (nsteps == 0) return MMX_OK;
  mmx_rk_opts o;
  memset(&o, 0, sizeof(o));
  o.method = MMX_RK4; o.fixed_dt = 1; o.dt0 = dt; o.nsteps = nsteps;
  return run_steps(w, &o, nullptr);
}

int mmx_step_rk45(mmx_world* w, const mmx_rk_opts* opts, mmx_rk_stats* stats) {
  if (!w || !opts) return mmx_fail(MMX_EINVAL, "NULL argument");
  if (opts->method < MMX_RK4 || opts->method > MMX_RKF45) return mmx_fail(MMX_EINVAL, "unknown method %d", opts->method);
  if (opts->nsteps <= 0 && opts->t_end <= 0 && opts->torque_stop <= 0 && opts->max_attempts <= 0)
    return mmx_fail(MMX_EINVAL, "no stopping criterion");
  return run_steps(w, opts, stats);
}

int mmx_relax(mmx_world* w, double torque_stop, double tol, long long max_attempts, mmx_rk_stats* stats) {
  if (!w) return mmx_fail(MMX_EINVAL, "NULL world");
  if (!(torque_stop > 0)) return mmx_fail(MMX_EINVAL, "mmx_relax needs torque_stop > 0");
  double t0 = 0;
  if (int rc = mmx_get_time(w, &t0)) return rc;
  mmx_rk_opts o;
  memset(&o, 0, sizeof(o));
  o.method = MMX_DP45; o.tol = tol; o.torque_stop = torque_stop; o.max_attempts = max_attempts;
  w->relax_mode = true;
  w->k1_valid = false;
  w->cfg_epoch++;  // the local kernels' arguments change: the captured step graph is stale
  int rc = run_steps(w, &o, stats);
  w->relax_mode = false;
  w->k1_valid = false;
  w->cfg_epoch++;
  const int rc2 = mmx_set_time(w, t0);
  if (stats) stats->t = t0;
  return rc ? rc : rc2;
}

int mmx_get_err_history(mmx_world* w, double* host_out, int n, int* n_out) {
  if (!w || !host_out || !n_out || n < 0) return mmx_fail(MMX_EINVAL, "bad argument");
  MmxCtrl h;
  if (int rc = read_ctrl(w, &h)) return rc;
  int have = h.hist_n < MMX_HIST ? h.hist_n : MMX_HIST;
  if (have > n) have = n;
  std::vector<double> hist(MMX_HIST);
  MMX_CUDA(cudaMemcpyAsync(hist.data(), w->d_ctrl->hist, sizeof(double) * MMX_HIST, cudaMemcpyDeviceToHost, w->stream));
  MMX_CUDA(cudaStreamSynchronize(w->stream));
  for (int q = 0; q < have; ++q) host_out[q] = hist[(size_t)(h.hist_n - have + q) % MMX_HIST];
  *n_out = have;
  return MMX_OK;
}

int mmx_profile_enable(mmx_world* w, int on) {
  if (!w) return mmx_fail(MMX_EINVAL, "NULL world");
  cudaStreamSynchronize(w->stream);
  for (auto& r : w->prof_recs) { cudaEventDestroy(r.e0); cudaEventDestroy(r.e1); }
  w->prof_recs.clear();
  w->prof = on != 0;
  return MMX_OK;
}

int mmx_profile_read(mmx_world* w, double* ms_out, long long* count_out, int n) {
  if (!w || !ms_out || !count_out || n < PK_COUNT) return mmx_fail(MMX_EINVAL, "need room for %d categories", PK_COUNT);
  MMX_CUDA(cudaStreamSynchronize(w->stream));
  for (int i = 0; i < n; ++i) { ms_out[i] = 0.0; count_out[i] = 0; }
  for (auto& r : w->prof_recs) {
    float ms = 0.f;
    MMX_CUDA(cudaEventElapsedTime(&ms, r.e0, r.e1));
    ms_out[r.cat] += ms;
    count_out[r.cat] += 1;
    cudaEventDestroy(r.e0);
    cudaEventDestroy(r.e1);
  }
  w->prof_recs.clear();
  return MMX_OK;
}

int mmx_device_bytes(mmx_world* w, long long* bytes) {
  if (!w || !bytes) return mmx_fail(MMX_EINVAL, "NULL argument");
  *bytes = w->dev_bytes;
  return MMX_OK;
}

int mmx_graph_enable(mmx_world* w, int on) {
  if (!w) return mmx_fail(MMX_EINVAL, "NULL world");
  w->use_graphs = on != 0;
  return MMX_OK;
}

int mmx_graph_info(mmx_world* w, long long* kernels_per_replay) {
  if (!w || !kernels_per_replay) return mmx_fail(MMX_EINVAL, "NULL argument");
  *kernels_per_replay = (w->step_graph && w->graph_epoch == w->cfg_epoch) ? w->graph_launches : 0;
  return MMX_OK;
}

}  // extern "C"
