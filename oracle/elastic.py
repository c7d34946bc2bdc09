"""ORACLE (test infrastructure): elastodynamics and magnetoelastic body force.

P:L169-177 (Eq.7): rho u_tt = f_tot for cubic symmetry; "f_el is computed as the
numeric divergence of the stress, while the strain is calculated with the
numeric gradient of the displacement ... traction and traction-free boundary
conditions impose sigma.n = t ... Both spatial derivative calculations utilize
a fourth order accurate central difference scheme in the bulk material.  Lower
order schemes are used close to and at the boundaries."  Eq.8 P:L181-184.

Readings S23/S24:
  gradient at a cell: 4th-order central where the four neighbours +-1,+-2 exist,
  else 2nd-order central, else one-sided (-3f0+4f1-f2)/(2h) or (f1-f0)/h,
  else 0 (single-cell axis).
  divergence of sigma: the same operator, except in a boundary cell of an open
  axis, where the face value sigma_b (from sigma.n = t, at distance h/2) enters:
  d sigma|_0 = +-(-4 sigma_b + 3 sigma_0 + sigma_1)/(3h).
  The elastic medium fills the whole grid (no holes).
"""
from __future__ import annotations

import numpy as np

EPS_KEYS = ("xx", "yy", "zz", "xy", "xz", "yz")


def _take(f, axis, i):
    sl = [slice(None)] * f.ndim
    sl[f.ndim - 1 - axis] = i
    return f[tuple(sl)]


def gradient(f, axis, h, periodic):
    """d f / d x_axis for a scalar array f [Nz,Ny,Nx] with the order-fallback rule."""
    ax = f.ndim - 1 - axis
    n = f.shape[ax]
    out = np.zeros_like(f)
    if n == 1:
        return out

    def plane(i):
        sl = [slice(None)] * f.ndim
        sl[ax] = i
        return tuple(sl)

    todo = range(n)
    if n >= 5 and not periodic:
        # bulk cells 2..n-3 all have +-1, +-2: same 4th-order formula as below, in one slice op
        def sh(k):
            sl = [slice(None)] * f.ndim
            sl[ax] = slice(2 + k, n - 2 + k)
            return f[tuple(sl)]
        out[plane(slice(2, n - 2))] = (-sh(2) + 8 * sh(1) - 8 * sh(-1) + sh(-2)) / (12 * h)
        todo = (0, 1, n - 2, n - 1)
    for i in todo:
        def has(k):
            return periodic or (0 <= i + k < n)

        def at(k):
            return f[plane((i + k) % n)]
        if has(-2) and has(-1) and has(1) and has(2):
            val = (-at(2) + 8 * at(1) - 8 * at(-1) + at(-2)) / (12 * h)
        elif has(-1) and has(1):
            val = (at(1) - at(-1)) / (2 * h)
        elif has(1) and has(2):
            val = (-3 * at(0) + 4 * at(1) - at(2)) / (2 * h)
        elif has(1):
            val = (at(1) - at(0)) / h
        elif has(-1) and has(-2):
            val = (3 * at(0) - 4 * at(-1) + at(-2)) / (2 * h)
        elif has(-1):
            val = (at(0) - at(-1)) / h
        else:
            val = 0.0
        out[plane(i)] = val
    return out


def strain(u, cell, pbc):
    """Tensor strain eps_ij = (d_i u_j + d_j u_i)/2 from displacement u [3,Nz,Ny,Nx]."""
    g = [[gradient(u[j], i, cell[i], pbc[i] > 0) for j in range(3)] for i in range(3)]  # g[i][j] = d_i u_j
    return dict(xx=g[0][0], yy=g[1][1], zz=g[2][2],
                xy=0.5 * (g[0][1] + g[1][0]), xz=0.5 * (g[0][2] + g[2][0]), yz=0.5 * (g[1][2] + g[2][1]))


def stress(eps, C11, C12, C44):
    """sigma_ii = C11 eps_ii + C12 (eps_jj + eps_kk); sigma_ij = 2 C44 eps_ij (cubic symmetry)."""
    return dict(xx=C11 * eps["xx"] + C12 * (eps["yy"] + eps["zz"]),
                yy=C11 * eps["yy"] + C12 * (eps["xx"] + eps["zz"]),
                zz=C11 * eps["zz"] + C12 * (eps["xx"] + eps["yy"]),
                xy=2 * C44 * eps["xy"], xz=2 * C44 * eps["xz"], yz=2 * C44 * eps["yz"])


def viscous_stress(v, beta, C11, C12, C44, cell, pbc):
    """"viscous damping, where an extra term, proportional to the strain rate, is added to
    the total stress tensor"; Table 1 names its coefficient "stiffness coefficient of the
    Rayleigh damping", a time (0.1 ps).  Reading S31: stiffness-proportional Rayleigh
    damping, sigma_visc = beta C : eps_dot with eps_dot = sym grad v (same gradient operator)."""
    return {k: beta * val for k, val in stress(strain(v, cell, pbc), C11, C12, C44).items()}


def div_axis(s, axis, h, periodic, face_lo, face_hi):
    """d s / d x_axis with the face values of s on the two open faces of that axis."""
    n = s.shape[s.ndim - 1 - axis]
    out = gradient(s, axis, h, periodic)
    if periodic or n == 1:
        return out
    lo = [slice(None)] * s.ndim
    hi = [slice(None)] * s.ndim
    lo[s.ndim - 1 - axis], hi[s.ndim - 1 - axis] = 0, n - 1
    out[tuple(lo)] = (-4 * face_lo + 3 * _take(s, axis, 0) + _take(s, axis, 1)) / (3 * h)
    out[tuple(hi)] = (4 * face_hi - 3 * _take(s, axis, n - 1) - _take(s, axis, n - 2)) / (3 * h)
    return out


_SIG = {(0, 0): "xx", (1, 1): "yy", (2, 2): "zz", (0, 1): "xy", (1, 0): "xy",
        (0, 2): "xz", (2, 0): "xz", (1, 2): "yz", (2, 1): "yz"}
_FACES = {"x-": (0, -1), "x+": (0, +1), "y-": (1, -1), "y+": (1, +1), "z-": (2, -1), "z+": (2, +1)}


def elastic_force(sig, cell, pbc, tractions=None):
    """f_el,j = sum_i d_i sigma_ij.  `tractions`: dict face -> 3-vector t (Pa) with
    sigma.n = t on that face (n the outward normal); faces not listed are traction free."""
    tractions = tractions or {}
    # face value of sigma_ij on the low/high face of axis i:  n = -+e_i  =>  sigma_ij = -+ t_j
    face = {(i, sgn): np.zeros(3) for i in range(3) for sgn in (-1, 1)}
    for name, t in tractions.items():
        i, sgn = _FACES[name]
        face[(i, sgn)] = sgn * np.asarray(t, float)
    f = np.zeros((3,) + sig["xx"].shape)
    for j in range(3):
        for i in range(3):
            f[j] += div_axis(sig[_SIG[(i, j)]], i, cell[i], pbc[i] > 0,
                             face[(i, -1)][j], face[(i, +1)][j])
    return f


def magnetoelastic_force(m, B1, B2, cell, pbc):
    """Eq.8 with d m by the gradient operator above (S24)."""
    d = [[gradient(m[j], i, cell[i], pbc[i] > 0) for j in range(3)] for i in range(3)]  # d[i][j] = d_i m_j
    f = np.empty_like(m)
    for a in range(3):
        b, c = (a + 1) % 3, (a + 2) % 3
        f[a] = (2 * B1 * m[a] * d[a][a]
                + B2 * (m[a] * (d[b][b] + d[c][c]) + m[b] * d[b][a] + m[c] * d[c][a]))
    return f
