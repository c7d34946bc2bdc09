// newell.cpp -- host-side (one-time) construction of the magnetostatic kernel.
//
// P:L142-144 (section 3.1.2): the demagnetising tensor is evaluated "using the analytical
// result [58] below a certain cutoff radius and the asymptotic result [59] above that
// radius"; periodic boundary conditions "also affect the calculation of the magnetostatic
// fields".
//
//  * near field: Newell's closed-form cell-cell interaction, N_xx = D[f]/(4 pi V),
//    N_xy = D[g]/(4 pi V), D = 27-point second difference; evaluated in 80-bit long double
//    because the difference cancels ~ (R/cell)^5 digits.
//  * far field: the cell-cell average of the point-dipole tensor
//        N_ij(r) = -(V/4pi) < d_i d_j 1/|r + t| >,   t = s - s',  s, s' uniform in a cell,
//    evaluated with a 3-point Gauss rule per axis for the triangular density of t_k
//    (nodes 0, +-sqrt(2/5) D_k, weights 7/12, 5/24, 5/24: exact through 5th order in D/R).
//  * periodic axes: K(d) = sum_{i=-R..R} N(d + i L) for 0 <= d <= N/2, the d = N/2 tie
//    averaged over its two images (odd components vanish there).
//  * spectrum: the octant is even/odd-extended on the padded box per axis and transformed
//    with a plain fp64 radix-2 FFT; the result is real; it is scaled (the caller folds
//    -mu0/(Px Py Pz) in) and rounded to fp32.
//
// Sign convention: B = -mu0 sum_r' N(r - r') M(r'), trace N(0) = 1.
#include <cmath>
#include <complex>
#include <cstdio>
#include <vector>

#include "mmx_internal.h"

typedef long double ld;

namespace {

const int PARITY[6][3] = {{1, 1, 1}, {1, 1, 1}, {1, 1, 1}, {-1, -1, 1}, {-1, 1, -1}, {1, -1, -1}};

inline ld sdiv(ld a, ld b) { return b != 0 ? a / b : (ld)0; }

ld newell_f(ld x, ld y, ld z) {
  ld x2 = x * x, y2 = y * y, z2 = z * z;
  ld R = sqrtl(x2 + y2 + z2);
  ld r = 0;
  r += 0.5L * y * (z2 - x2) * asinhl(sdiv(y, sqrtl(x2 + z2)));
  r += 0.5L * z * (y2 - x2) * asinhl(sdiv(z, sqrtl(x2 + y2)));
  r -= x * y * z * atanl(sdiv(y * z, x * R));
  r += (2 * x2 - y2 - z2) * R / 6;
  return r;
}

ld newell_g(ld x, ld y, ld z) {
  ld x2 = x * x, y2 = y * y, z2 = z * z;
  ld R = sqrtl(x2 + y2 + z2);
  ld r = 0;
  r += x * y * z * asinhl(sdiv(z, sqrtl(x2 + y2)));
  r += y / 6 * (3 * z2 - y2) * asinhl(sdiv(x, sqrtl(y2 + z2)));
  r += x / 6 * (3 * z2 - x2) * asinhl(sdiv(y, sqrtl(x2 + z2)));
  r -= z * z2 / 6 * atanl(sdiv(x * y, z * R));
  r -= z * y2 / 2 * atanl(sdiv(x * z, y * R));
  r -= z * x2 / 2 * atanl(sdiv(y * z, x * R));
  r -= x * y * R / 3;
  return r;
}

// primitive F_comp at a lattice point (X, Y, Z)
ld primitive(int comp, ld X, ld Y, ld Z) {
  switch (comp) {
    case 0: return newell_f(X, Y, Z);
    case 1: return newell_f(Y, X, Z);
    case 2: return newell_f(Z, Y, X);
    case 3: return newell_g(X, Y, Z);
    case 4: return newell_g(X, Z, Y);
    default: return newell_g(Y, Z, X);
  }
}

// far field: 27-node quadrature of F_ij = 3 r_i r_j / R^5 - delta_ij / R^3
double far_field(int comp, double x, double y, double z, const double cell[3]) {
  static const int IA[6] = {0, 1, 2, 0, 0, 1}, IB[6] = {0, 1, 2, 1, 2, 2};
  const double node = std::sqrt(0.4);
  const double wn[3] = {5.0 / 24.0, 7.0 / 12.0, 5.0 / 24.0};
  double acc = 0;
  for (int a = -1; a <= 1; ++a)
    for (int b = -1; b <= 1; ++b)
      for (int c = -1; c <= 1; ++c) {
        double r[3] = {x + a * node * cell[0], y + b * node * cell[1], z + c * node * cell[2]};
        double R2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
        double R = std::sqrt(R2);
        double F = 3.0 * r[IA[comp]] * r[IB[comp]] / (R2 * R2 * R) - (IA[comp] == IB[comp] ? 1.0 / (R2 * R) : 0.0);
        acc += wn[a + 1] * wn[b + 1] * wn[c + 1] * F;
      }
  double V = cell[0] * cell[1] * cell[2];
  return -(V / (4.0 * M_PI)) * acc;
}

// N_comp on offsets (i dx + sx, j dy + sy, k dz + sz), 0 <= i < n0 ..., accumulated into acc
void add_octant(int comp, const int n[3], const double cell[3], double cutoff_cells, const double shift[3],
                double* acc) {
  const double cmax = std::fmax(cell[0], std::fmax(cell[1], cell[2]));
  const double rcut2 = cutoff_cells * cmax * cutoff_cells * cmax;
  const ld V = (ld)cell[0] * (ld)cell[1] * (ld)cell[2];
  const ld pref = 1.0L / (4.0L * 3.14159265358979323846264338327950288L * V);
  // near region: points with R^2 < rcut2.  Build the primitive on the bounding box (+1 halo) lazily.
  int lo[3], hi[3];
  bool any_near = false;
  for (int a = 0; a < 3; ++a) { lo[a] = n[a]; hi[a] = -1; }
#pragma omp parallel for collapse(2) schedule(static)
  for (int k = 0; k < n[2]; ++k)
    for (int j = 0; j < n[1]; ++j) {
      for (int i = 0; i < n[0]; ++i) {
        double X = i * cell[0] + shift[0], Y = j * cell[1] + shift[1], Z = k * cell[2] + shift[2];
        double R2 = X * X + Y * Y + Z * Z;
        size_t idx = ((size_t)k * n[1] + j) * n[0] + i;
        if (R2 >= rcut2) acc[idx] += far_field(comp, X, Y, Z, cell);
      }
    }
  for (int k = 0; k < n[2]; ++k)
    for (int j = 0; j < n[1]; ++j)
      for (int i = 0; i < n[0]; ++i) {
        double X = i * cell[0] + shift[0], Y = j * cell[1] + shift[1], Z = k * cell[2] + shift[2];
        if (X * X + Y * Y + Z * Z < rcut2) {
          any_near = true;
          int p[3] = {i, j, k};
          for (int a = 0; a < 3; ++a) {
            if (p[a] < lo[a]) lo[a] = p[a];
            if (p[a] > hi[a]) hi[a] = p[a];
          }
        }
      }
  if (!any_near) return;
  const int e0 = hi[0] - lo[0] + 3, e1 = hi[1] - lo[1] + 3, e2 = hi[2] - lo[2] + 3;
  std::vector<ld> F((size_t)e0 * e1 * e2);
#pragma omp parallel for collapse(2) schedule(static)
  for (int k = 0; k < e2; ++k)
    for (int j = 0; j < e1; ++j)
      for (int i = 0; i < e0; ++i) {
        ld X = (ld)(lo[0] + i - 1) * (ld)cell[0] + (ld)shift[0];
        ld Y = (ld)(lo[1] + j - 1) * (ld)cell[1] + (ld)shift[1];
        ld Z = (ld)(lo[2] + k - 1) * (ld)cell[2] + (ld)shift[2];
        F[((size_t)k * e1 + j) * e0 + i] = primitive(comp, X, Y, Z);
      }
  const ld w[3] = {1, -2, 1};
  for (int k = lo[2]; k <= hi[2]; ++k)
    for (int j = lo[1]; j <= hi[1]; ++j)
      for (int i = lo[0]; i <= hi[0]; ++i) {
        double X = i * cell[0] + shift[0], Y = j * cell[1] + shift[1], Z = k * cell[2] + shift[2];
        if (X * X + Y * Y + Z * Z >= rcut2) continue;
        ld s = 0;
        for (int c = 0; c < 3; ++c)
          for (int b = 0; b < 3; ++b)
            for (int a = 0; a < 3; ++a)
              s -= w[a] * w[b] * w[c] *
                   F[((size_t)(k - lo[2] + c) * e1 + (j - lo[1] + b)) * e0 + (i - lo[0] + a)];
        acc[((size_t)k * n[1] + j) * n[0] + i] += (double)(s * pref);
      }
}

void fft_inplace(std::complex<double>* x, int n) {
  // iterative radix-2 decimation in time, forward (exp(-i ...))
  for (int i = 1, j = 0; i < n; ++i) {
    int bit = n >> 1;
    for (; j & bit; bit >>= 1) j ^= bit;
    j ^= bit;
    if (i < j) std::swap(x[i], x[j]);
  }
  for (int len = 2; len <= n; len <<= 1) {
    for (int i = 0; i < n; i += len)
      for (int k = 0; k < len / 2; ++k) {
        double ang = -2.0 * M_PI * k / len;
        std::complex<double> wk(std::cos(ang), std::sin(ang));
        std::complex<double> u = x[i + k], v = x[i + k + len / 2] * wk;
        x[i + k] = u + v;
        x[i + k + len / 2] = u - v;
      }
  }
}

}  // namespace

int mmx_newell_octant(const int grid[3], const double cell[3], const int pbc[3], double cutoff_cells,
                      std::vector<double>& out, int n[3]) {
  if (cutoff_cells <= 0) cutoff_cells = 32.0;
  for (int a = 0; a < 3; ++a) n[a] = pbc[a] > 0 ? grid[a] / 2 + 1 : grid[a];
  const size_t cnt = (size_t)n[0] * n[1] * n[2];
  out.assign(6 * cnt, 0.0);
  const double L[3] = {grid[0] * cell[0], grid[1] * cell[1], grid[2] * cell[2]};
  for (int comp = 0; comp < 6; ++comp) {
    double* acc = out.data() + comp * cnt;
    for (int iz = -pbc[2]; iz <= pbc[2]; ++iz)
      for (int iy = -pbc[1]; iy <= pbc[1]; ++iy)
        for (int ix = -pbc[0]; ix <= pbc[0]; ++ix) {
          double shift[3] = {ix * L[0], iy * L[1], iz * L[2]};
          add_octant(comp, n, cell, cutoff_cells, shift, acc);
        }
    // tie at d = N/2 on an even periodic axis: mean of the images at +N/2 and -N/2
    for (int a = 0; a < 3; ++a) {
      if (pbc[a] > 0 && grid[a] % 2 == 0 && grid[a] > 1) {
        const double f = 0.5 * (1 + PARITY[comp][a]);
        for (int k = 0; k < n[2]; ++k)
          for (int j = 0; j < n[1]; ++j)
            for (int i = 0; i < n[0]; ++i) {
              int p[3] = {i, j, k};
              if (p[a] == grid[a] / 2) acc[((size_t)k * n[1] + j) * n[0] + i] *= f;
            }
      }
    }
  }
  return MMX_OK;
}

// Transform the octant to the real spectrum octant [6][kz][ky][xp] (x: 0..Px/2).
int mmx_kernel_spectrum(const int grid[3], const int pbc[3], const int P[3], int xp,
                        const std::vector<double>& octant, const int n[3], double scale,
                        std::vector<float>& khat) {
  const int kx = P[0] / 2 + 1;
  const int ky = P[1] > 1 ? P[1] / 2 + 1 : 1;
  const int kz = P[2] > 1 ? P[2] / 2 + 1 : 1;
  khat.assign((size_t)6 * kz * ky * xp, 0.f);
  const size_t cnt = (size_t)n[0] * n[1] * n[2];
  for (int comp = 0; comp < 6; ++comp) {
    // work array: current extents e[a] per axis, starts as the octant
    int e[3] = {n[0], n[1], n[2]};
    std::vector<double> cur(octant.begin() + comp * cnt, octant.begin() + (comp + 1) * cnt);
    int nodd = 0;
    for (int a = 0; a < 3; ++a) {
      const int Pa = P[a];
      const int outn = a == 0 ? kx : (a == 1 ? ky : kz);
      const int par = PARITY[comp][a];
      int ne[3] = {e[0], e[1], e[2]};
      ne[a] = outn;
      std::vector<double> nxt((size_t)ne[0] * ne[1] * ne[2], 0.0);
      if (Pa == 1) {
        // untransformed single-cell axis: K(0); odd components vanish
        for (int k = 0; k < ne[2]; ++k)
          for (int j = 0; j < ne[1]; ++j)
            for (int i = 0; i < ne[0]; ++i)
              nxt[((size_t)k * ne[1] + j) * ne[0] + i] = par > 0 ? cur[((size_t)k * e[1] + j) * e[0] + i] : 0.0;
        if (par < 0) ++nodd;
      } else {
        if (par < 0) ++nodd;
        const int o1 = (a + 1) % 3, o2 = (a + 2) % 3;
        const long long lines = (long long)e[o1] * e[o2];
#pragma omp parallel
        {
          std::vector<std::complex<double>> buf(Pa);
#pragma omp for schedule(static)
          for (long long ln = 0; ln < lines; ++ln) {
            int p[3];
            p[o1] = (int)(ln % e[o1]);
            p[o2] = (int)(ln / e[o1]);
            for (int q = 0; q < Pa; ++q) buf[q] = 0.0;
            for (int d = 0; d < e[a]; ++d) {
              p[a] = d;
              double v = cur[((size_t)p[2] * e[1] + p[1]) * e[0] + p[0]];
              // offsets d and -d (index Pa - d); on an open axis |d| < N <= Pa/2, on a periodic
              // axis d <= N/2 and the tie d = N/2 maps onto itself (already averaged).
              if (d == 0) buf[0] = v;
              else if (2 * d == Pa) buf[d] = par > 0 ? v : 0.0;
              else { buf[d] = v; buf[Pa - d] = par > 0 ? v : -v; }
            }
            fft_inplace(buf.data(), Pa);
            for (int q = 0; q < outn; ++q) {
              p[a] = q;
              // even: real part; odd: FFT = -i S with S real  ->  keep S = -imag
              double v = par > 0 ? buf[q].real() : -buf[q].imag();
              nxt[((size_t)p[2] * ne[1] + p[1]) * ne[0] + p[0]] = v;
            }
          }
        }
      }
      cur.swap(nxt);
      e[0] = ne[0]; e[1] = ne[1]; e[2] = ne[2];
    }
    // each odd axis contributes a factor (-i); two of them give -1 (components have 0 or 2)
    const double sgn = (nodd == 2) ? -1.0 : 1.0;
    float* dst = khat.data() + (size_t)comp * kz * ky * xp;
    for (int k = 0; k < kz; ++k)
      for (int j = 0; j < ky; ++j)
        for (int i = 0; i < kx; ++i)
          dst[((size_t)k * ky + j) * xp + i] = (float)(sgn * scale * cur[((size_t)k * e[1] + j) * e[0] + i]);
  }
  (void)grid; (void)pbc;
  return MMX_OK;
}

// N_comp(i dx, j dy, dz) on the non-negative quadrant of in-plane offsets at a fixed z offset dz (any real number, not
// a multiple of the cell height): the cell-to-cell tensor between a source layer and a probe layer above the magnet
// (mmx_stray_field).  out: [6][ny][nx].
int mmx_newell_quadrant_at(int nx, int ny, const double cell[3], double dz, double cutoff_cells, std::vector<double>& out) {
  if (cutoff_cells <= 0) cutoff_cells = 32.0;
  const int n[3] = {nx, ny, 1};
  const size_t cnt = (size_t)nx * ny;
  out.assign(6 * cnt, 0.0);
  const double shift[3] = {0.0, 0.0, dz};
  for (int comp = 0; comp < 6; ++comp) add_octant(comp, n, cell, cutoff_cells, shift, out.data() + comp * cnt);
  return MMX_OK;
}
