"""ORACLE (test infrastructure): demagnetising tensor of uniformly magnetised cuboid cells.

P:L142-144 (section 3.1.2): "using the analytical result [58] below a certain
cutoff radius and the asymptotic result [59] above that radius".

* analytic branch: Newell's closed forms f (diagonal) and g (off-diagonal),
  combined with the 27-point second-difference operator,
  evaluated in extended precision (np.longdouble) to tame the cancellation.
* asymptotic branch (reading S12): Taylor expansion of the cell-cell averaged
  dipole kernel  N_ij = -(V/4pi) < d_i d_j (1/|r+t|) >,  t = s-s' the difference
  of two points uniformly distributed in a cell (<t_k^2> = D_k^2/6,
  <t_k^4> = D_k^4/15), kept through 4th order in the cell size.
* periodic axes (reading S13): K(d) = sum_{i=-R..R} N(d + i L), |d| <= N/2,
  the d = +-N/2 tie averaged.

Sign convention: B = -mu0 * sum_r' N(r-r') M(r'), so N_xx + N_yy + N_zz = 1 at r = 0.
"""
from __future__ import annotations

import numpy as np

LD = np.longdouble

COMPS = ("xx", "yy", "zz", "xy", "xz", "yz")
# parity of N_ij under reflection of each axis (x, y, z): -1 if the axis appears once in ij
PARITY = {"xx": (1, 1, 1), "yy": (1, 1, 1), "zz": (1, 1, 1),
          "xy": (-1, -1, 1), "xz": (-1, 1, -1), "yz": (1, -1, -1)}


# ----------------------------------------------------------------------
# analytic branch
# ----------------------------------------------------------------------
def _safe_div(a, b):
    out = np.zeros_like(a)
    np.divide(a, b, out=out, where=(b != 0))
    return out


def newell_f(x, y, z):
    """Newell f(x,y,z); N_xx = D[f]/(4 pi V).  Terms whose argument is 0/0 are dropped."""
    x, y, z = np.broadcast_arrays(LD(1) * x, LD(1) * y, LD(1) * z)
    x2, y2, z2 = x * x, y * y, z * z
    R = np.sqrt(x2 + y2 + z2)
    t1 = 0.5 * y * (z2 - x2) * np.arcsinh(_safe_div(y, np.sqrt(x2 + z2)))
    t2 = 0.5 * z * (y2 - x2) * np.arcsinh(_safe_div(z, np.sqrt(x2 + y2)))
    t3 = -x * y * z * np.arctan(_safe_div(y * z, x * R))
    t4 = (2 * x2 - y2 - z2) * R / 6
    return t1 + t2 + t3 + t4


def newell_g(x, y, z):
    """Newell g(x,y,z); N_xy = D[g]/(4 pi V)."""
    x, y, z = np.broadcast_arrays(LD(1) * x, LD(1) * y, LD(1) * z)
    x2, y2, z2 = x * x, y * y, z * z
    R = np.sqrt(x2 + y2 + z2)
    t1 = x * y * z * np.arcsinh(_safe_div(z, np.sqrt(x2 + y2)))
    t2 = y / 6 * (3 * z2 - y2) * np.arcsinh(_safe_div(x, np.sqrt(y2 + z2)))
    t3 = x / 6 * (3 * z2 - x2) * np.arcsinh(_safe_div(y, np.sqrt(x2 + z2)))
    t4 = -z * z2 / 6 * np.arctan(_safe_div(x * y, z * R))
    t5 = -z * y2 / 2 * np.arctan(_safe_div(x * z, y * R))
    t6 = -z * x2 / 2 * np.arctan(_safe_div(y * z, x * R))
    t7 = -x * y * R / 3
    return t1 + t2 + t3 + t4 + t5 + t6 + t7


def _second_difference(F):
    """27-point operator  -sum_{a,b,c in {-1,0,1}} w_a w_b w_c F,  w = (1,-2,1),
    applied to F sampled on lattice points -1..n along each axis (shape n+2)."""
    w = (1.0, -2.0, 1.0)
    nz, ny, nx = (s - 2 for s in F.shape)
    out = np.zeros((nz, ny, nx), dtype=F.dtype)
    for a in range(3):
        for b in range(3):
            for c in range(3):
                out -= w[a] * w[b] * w[c] * F[c:c + nz, b:b + ny, a:a + nx]
    return out


def _analytic_block(comp, ix, iy, iz, cell, shift):
    """N_comp at offsets (ix[i]*dx + shift_x, ...) on the outer-product lattice, analytic."""
    dx, dy, dz = (LD(c) for c in cell)
    # lattice points -1..n around every requested offset: offsets are contiguous integer ranges
    def ext(i, d, s):
        i = np.asarray(i)
        e = np.concatenate(([i[0] - 1], i, [i[-1] + 1])).astype(LD)
        return e * d + LD(s)
    X = ext(ix, dx, shift[0])[None, None, :]
    Y = ext(iy, dy, shift[1])[None, :, None]
    Z = ext(iz, dz, shift[2])[:, None, None]
    if comp == "xx":
        F = newell_f(X, Y, Z)
    elif comp == "yy":
        F = newell_f(Y, X, Z)
    elif comp == "zz":
        F = newell_f(Z, Y, X)
    elif comp == "xy":
        F = newell_g(X, Y, Z)
    elif comp == "xz":
        F = newell_g(X, Z, Y)
    elif comp == "yz":
        F = newell_g(Y, Z, X)
    else:
        raise ValueError(comp)
    V = dx * dy * dz
    return _second_difference(F) / (4 * LD(np.pi) * V)


# ----------------------------------------------------------------------
# asymptotic branch: derivatives of 1/R as polynomial / R^(2n+1)
# ----------------------------------------------------------------------
def _poly_add(p, q, s=1.0):
    out = dict(p)
    for k, v in q.items():
        out[k] = out.get(k, 0.0) + s * v
    return out


def _poly_mul_mono(p, mono, coef=1.0):
    return {(k[0] + mono[0], k[1] + mono[1], k[2] + mono[2]): coef * v for k, v in p.items()}


def _poly_dpartial(p, axis):
    out = {}
    for k, v in p.items():
        if k[axis] > 0:
            kk = list(k)
            kk[axis] -= 1
            out[tuple(kk)] = out.get(tuple(kk), 0.0) + v * k[axis]
    return out


def _deriv(p, n, axis):
    """d/dx_axis [ p / R^(2n+1) ] = [ (dp) R^2 - (2n+1) x p ] / R^(2n+3)."""
    dp = _poly_dpartial(p, axis)
    out = {}
    for mono in ((2, 0, 0), (0, 2, 0), (0, 0, 2)):
        out = _poly_add(out, _poly_mul_mono(dp, mono))
    xm = [0, 0, 0]
    xm[axis] = 1
    out = _poly_add(out, _poly_mul_mono(p, tuple(xm), -(2 * n + 1)))
    return out, n + 1


def _deriv_multi(axes):
    p, n = {(0, 0, 0): 1.0}, 0
    for a in axes:
        p, n = _deriv(p, n, a)
    return p, n


def _poly_eval(p, x, y, z):
    out = np.zeros(np.broadcast(x, y, z).shape)
    for (a, b, c), v in p.items():
        if v != 0.0:
            out = out + v * x ** a * y ** b * z ** c
    return out


_AX = {"x": 0, "y": 1, "z": 2}


def asymptotic(comp, x, y, z, cell):
    """Far-field N_comp(x,y,z) through 4th order in the cell size (reading S12)."""
    i, j = _AX[comp[0]], _AX[comp[1]]
    d = [float(c) for c in cell]
    p2, _ = _deriv_multi((i, j))
    p4, p6 = {}, {}
    for k in range(3):
        q, _ = _deriv_multi((i, j, k, k))
        p4 = _poly_add(p4, q, d[k] ** 2 / 12.0)
        q, _ = _deriv_multi((i, j, k, k, k, k))
        p6 = _poly_add(p6, q, d[k] ** 4 / 360.0)
        for l in range(k + 1, 3):
            q, _ = _deriv_multi((i, j, k, k, l, l))
            p6 = _poly_add(p6, q, d[k] ** 2 * d[l] ** 2 / 144.0)
    x, y, z = np.broadcast_arrays(np.asarray(x, float), np.asarray(y, float), np.asarray(z, float))
    R2 = x * x + y * y + z * z
    R = np.sqrt(R2)
    V = d[0] * d[1] * d[2]
    with np.errstate(divide="ignore", invalid="ignore"):
        val = (_poly_eval(p2, x, y, z) / R ** 5 + _poly_eval(p4, x, y, z) / R ** 9
               + _poly_eval(p6, x, y, z) / R ** 13)
    return -(V / (4 * np.pi)) * val


# ----------------------------------------------------------------------
# tensor on the non-negative octant of offsets
# ----------------------------------------------------------------------
def newell_octant(comp, n, cell, cutoff_cells=32.0, shift=(0.0, 0.0, 0.0)):
    """N_comp at offsets (i dx + shift_x, j dy + shift_y, k dz + shift_z),
    0 <= i < n[0] etc.  Returns float64 [n2, n1, n0] (z, y, x order).

    Analytic inside |r| < cutoff_cells * max(cell), asymptotic outside (S11)."""
    nx, ny, nz = n
    ix, iy, iz = np.arange(nx), np.arange(ny), np.arange(nz)
    X = ix[None, None, :] * cell[0] + shift[0]
    Y = iy[None, :, None] * cell[1] + shift[1]
    Z = iz[:, None, None] * cell[2] + shift[2]
    R2 = X * X + Y * Y + Z * Z
    rcut = cutoff_cells * max(cell)
    near = R2 < rcut * rcut
    out = np.empty((nz, ny, nx))
    far = ~near
    if far.any():
        Xb, Yb, Zb = np.broadcast_arrays(X, Y, Z)
        out[far] = asymptotic(comp, Xb[far], Yb[far], Zb[far], cell)
    if near.any():
        # bounding index box of the near region (contiguous ranges along each axis)
        kz, ky, kx = np.nonzero(near)
        bx = np.arange(kx.min(), kx.max() + 1)
        by = np.arange(ky.min(), ky.max() + 1)
        bz = np.arange(kz.min(), kz.max() + 1)
        blk = _analytic_block(comp, bx, by, bz, cell, shift).astype(np.float64)
        sub = near[np.ix_(bz, by, bx)]
        view = out[np.ix_(bz, by, bx)]
        view[sub] = blk[sub]
        out[np.ix_(bz, by, bx)] = view
    return out


def self_term(cell):
    """(N_xx, N_yy, N_zz) at zero offset for one cell of edge lengths `cell`."""
    return tuple(float(newell_octant(c, (1, 1, 1), cell)[0, 0, 0]) for c in ("xx", "yy", "zz"))


def kernel_octant(grid, cell, pbc=(0, 0, 0), cutoff_cells=32.0):
    """Demag kernel K_comp(d) for 0 <= d_a <= M_a, where M_a = N_a - 1 on an open
    axis and floor(N_a/2) on a periodic one (images summed, tie averaged).
    Returns dict comp -> float64 [Mz+1, My+1, Mx+1]."""
    n = [(g // 2 + 1) if p > 0 else g for g, p in zip(grid, pbc)]
    L = [g * c for g, c in zip(grid, cell)]
    rng = [range(-p, p + 1) if p > 0 else (0,) for p in pbc]
    out = {}
    for comp in COMPS:
        acc = np.zeros((n[2], n[1], n[0]))
        for iz in rng[2]:
            for iy in rng[1]:
                for ix in rng[0]:
                    acc += newell_octant(comp, n, cell, cutoff_cells,
                                         shift=(ix * L[0], iy * L[1], iz * L[2]))
        # tie at d = N/2 on an even periodic axis: average of d=+N/2 and d=-N/2
        par = PARITY[comp]
        for a, (g, p) in enumerate(zip(grid, pbc)):
            if p > 0 and g % 2 == 0 and g > 1:
                sl = [slice(None)] * 3
                sl[2 - a] = g // 2
                acc[tuple(sl)] *= 0.5 * (1 + par[a])
        out[comp] = acc
    return out


def kernel_lookup(octant, comp, d, grid, pbc):
    """K_comp at signed integer offsets d = (dx, dy, dz) (arrays), using the parity
    of N_ij and, on periodic axes, wrapping d into [-N/2, N/2]."""
    sign = 1.0
    idx = []
    for a in range(3):
        da = np.asarray(d[a])
        if pbc[a] > 0:
            g = grid[a]
            da = (da + g // 2) % g - g // 2  # [-g/2, g/2)
        sign = sign * np.where(da < 0, PARITY[comp][a], 1.0)
        idx.append(np.abs(da))
    return sign * octant[comp][idx[2], idx[1], idx[0]]
