"""ORACLE (test infrastructure): local effective-field terms and torques.

All arrays are float64, vector fields are [3, Nz, Ny, Nx] (component first),
per-cell scalars [Nz, Ny, Nx].  Axis numbering: 0 = x, 1 = y, 2 = z.

Citations: exchange Eq.3; DMI Eq.4; anisotropy / Zeeman
P:L116-118 ("implemented in the same way as in mumax3" -- readings S3, S16);
magnetoelastic field Eq.9; LLG torque Eq.2; Zhang-Li
torque P:L110 (reading S17).  Boundary reading S9 (OPEN = a stencil pair whose
partner does not exist contributes nothing).
"""
from __future__ import annotations

import numpy as np

from .constants import HBAR, MU_B, Q_E


# ----------------------------------------------------------------------
# neighbour access
# ----------------------------------------------------------------------
def neighbour(a, axis, d, periodic):
    """Value of `a` at cell c + d*e_axis, and whether that cell is inside the grid
    (after wrapping on a periodic axis).  Outside cells read as 0."""
    ax = a.ndim - 1 - axis
    n = a.shape[ax]
    if periodic:
        return np.roll(a, -d, axis=ax), np.ones(a.shape[-3:], dtype=bool)
    out = np.zeros_like(a)
    ex = np.zeros(a.shape[-3:], dtype=bool)
    if abs(d) < n:
        src = [slice(None)] * a.ndim
        dst = [slice(None)] * a.ndim
        if d > 0:
            dst[ax], src[ax] = slice(0, n - d), slice(d, n)
        else:
            dst[ax], src[ax] = slice(-d, n), slice(0, n + d)
        out[tuple(dst)] = a[tuple(src)]
        exd = [slice(None)] * 3
        exd[2 - axis] = dst[ax]
        ex[tuple(exd)] = True
    return out, ex


def _harmonic(a, b):
    s = a + b
    out = np.zeros_like(s)
    np.divide(2 * a * b, s, out=out, where=(s != 0))
    return out


def _inv(ms):
    out = np.zeros_like(ms)
    np.divide(1.0, ms, out=out, where=(ms > 0))
    return out


# ----------------------------------------------------------------------
# Eq.3: exchange-like pair terms
# ----------------------------------------------------------------------
def pair_laplacian(mq, Ms, Apar, reg, scale, cell, pbc, factor, ghost=None):
    """sum over the 6 neighbours n of  factor * A_cn / Ms_c * (mq_n - mq_c) / h_n^2,
    A_cn = harmonic mean of Apar at c and n, times `scale` when c and n lie in
    different regions (S3, S4).  factor=2, mq=m^(s), Apar=A11: first term of Eq.3;
    factor=1, mq=m^(s'), Apar=A12: second term (S5).
    ghost: None = open boundary (S9: a pair whose partner is absent adds nothing); else a dict
    (axis, d) -> ghost values of mq behind an absent partner (Neumann boundary of Eq.5, reading S41), which
    then enter the pair with the centre cell's own Apar."""
    B = np.zeros_like(mq)
    iMs = _inv(Ms)
    for axis in range(3):
        h = cell[axis]
        for d in (+1, -1):
            mn, ex = neighbour(mq, axis, d, pbc[axis] > 0)
            Msn, _ = neighbour(Ms, axis, d, pbc[axis] > 0)
            An, _ = neighbour(Apar, axis, d, pbc[axis] > 0)
            rn, _ = neighbour(reg, axis, d, pbc[axis] > 0)
            ok = ex & (Msn > 0) & (Ms > 0)
            Acn = _harmonic(Apar, An) * np.where(rn == reg, 1.0, scale)
            B += np.where(ok, factor * Acn * iMs / (h * h), 0.0)[None] * (mn - mq)
            if ghost is not None:
                absent = ~ok & (Ms > 0)
                B += np.where(absent, factor * Apar * iMs / (h * h), 0.0)[None] * (ghost[(axis, d)] - mq)
    return B


def homogeneous_exchange(m_other, Ms, A0, latcon):
    """Third term of Eq.3: 4 A0 / (Ms a^2) m^(s')."""
    return (4.0 * A0 / (latcon * latcon)) * _inv(Ms)[None] * m_other


# ----------------------------------------------------------------------
# Eq.4, interfacial subset (S7): D_xzx = D_yzy = +D, D_xxz = D_yyz = -D
# ----------------------------------------------------------------------
def dmi_homogeneous(m_other, Ms, d, s):
    """Eq.6: energy density eps = d . (m^(s) x m^(s')) between the two sublattices of a
    cell, d the DMI vector in J/m^3.  Reading S32: (s, s') = (first, second) sublattice.  Then
    eps = m1 . (m2 x d) = m2 . (d x m1), so B^(1) = -(m2 x d)/Ms1 = (d x m2)/Ms1 and
    B^(2) = -(d x m1)/Ms2 = (m1 x d)/Ms2.  `m_other` is the partner sublattice, `s` this one."""
    dv = np.asarray(d, float).reshape(3, 1, 1, 1) * np.ones_like(m_other)
    B = cross(dv, m_other) if s == 0 else cross(m_other, dv)
    return B * _inv(Ms)[None]


def dmi_tensor(mq, Ms, q, cell, pbc, ghost=None):
    """General DMI of Eq.4 for s = s': eps = sum_ijk D_ijk m_j d_i m_k with
    D_ijk = -D_ikj, "9 independent components".  For each axis i the antisymmetric 3x3 block is a
    vector q_i, D_ijk = sum_l eps_jkl q_il, so eps = sum_i q_i . (m x d_i m) and
    B = -(1/Ms) delta E/delta m = (2/Ms) sum_i q_i x d_i m.  Discretised pair by pair like the
    interfacial term (central difference; a pair whose partner is absent or has Ms = 0 adds
    nothing, reading S9):  B_c = sum_i sum_{d=+-1} d / (Ms_c h_i) q_i x m_(c + d e_i).
    q: [3 axes][3] in J/m^2, uniform (reading S33).  Interfacial D is q_x = D y^, q_y = -D x^;
    bulk (Bloch) DMI eps = D m.(curl m) is q_i = -D e_i
    (m.(curl m) = -sum_i e_i.(m x d_i m))."""
    B = np.zeros_like(mq)
    iMs = _inv(Ms)
    q = np.asarray(q, float)
    for axis in range(3):
        if not np.any(q[axis]):
            continue
        h = cell[axis]
        qv = q[axis].reshape(3, 1, 1, 1) * np.ones_like(mq)
        for d in (+1, -1):
            mn, ex = neighbour(mq, axis, d, pbc[axis] > 0)
            Msn, _ = neighbour(Ms, axis, d, pbc[axis] > 0)
            ok = ex & (Msn > 0) & (Ms > 0)
            w = np.where(ok, iMs / h, 0.0) * d
            B += w[None] * cross(qv, mn)
            if ghost is not None:   # Neumann boundary (reading S41): the absent partner is the ghost value
                wg = np.where(~ok & (Ms > 0), iMs / h, 0.0) * d
                B += wg[None] * cross(qv, ghost[(axis, d)])
    return B


def dmi_interfacial(mq, Ms, D, cell, pbc, ghost=None):
    """B = sum_{n in +-x, +-y} D_cn / (Ms_c h_n) (z^ x e_cn) x mq_n ;
    continuum limit (2D/Ms)(dx m_z, dy m_z, -dx m_x - dy m_y)."""
    B = np.zeros_like(mq)
    iMs = _inv(Ms)
    for axis in (0, 1):
        h = cell[axis]
        for d in (+1, -1):
            mn, ex = neighbour(mq, axis, d, pbc[axis] > 0)
            Msn, _ = neighbour(Ms, axis, d, pbc[axis] > 0)
            Dn, _ = neighbour(D, axis, d, pbc[axis] > 0)
            ok = ex & (Msn > 0) & (Ms > 0)
            w = np.where(ok, _harmonic(D, Dn) * iMs / h, 0.0) * d
            # (z^ x (d x^)) x m = d ( m_z, 0, -m_x);  (z^ x (d y^)) x m = d (0, m_z, -m_y)
            B[axis] += w * mn[2]
            B[2] -= w * mn[axis]
            if ghost is not None:   # Neumann boundary (reading S41): ghost value, the centre cell's own D
                wg = np.where(~ok & (Ms > 0), D * iMs / h, 0.0) * d
                B[axis] += wg * ghost[(axis, d)][2]
                B[2] -= wg * ghost[(axis, d)][axis]
    return B


# ----------------------------------------------------------------------
# anisotropy, Zeeman (S16)
# ----------------------------------------------------------------------
def uniaxial(m, Ms, Ku1, u):
    """B = (2 Ku1 / Ms) (u.m) u ; u [3,Nz,Ny,Nx] unit axis per cell."""
    return (2.0 * Ku1 * _inv(Ms) * (u * m).sum(axis=0))[None] * u


def cubic(m, Ms, Kc1, c1, c2):
    """B = -(2 Kc1/Ms) sum_i (c_i.m) [ (c_j.m)^2 + (c_k.m)^2 ] c_i, c3 = c1 x c2."""
    c3 = np.cross(c1, c2, axis=0)
    a = [(c * m).sum(axis=0) for c in (c1, c2, c3)]
    pref = -2.0 * Kc1 * _inv(Ms)
    B = np.zeros_like(m)
    for i, c in enumerate((c1, c2, c3)):
        j, k = (i + 1) % 3, (i + 2) % 3
        B += (pref * a[i] * (a[j] ** 2 + a[k] ** 2))[None] * c
    return B


def zeeman(m, Ms, bext):
    return np.asarray(bext, float)[:, None, None, None] * (Ms > 0)[None] * np.ones_like(m)


# ----------------------------------------------------------------------
# Eq.9: magnetoelastic (Villari) field; eps = dict xx,yy,zz,xy,xz,yz of tensor strain
# ----------------------------------------------------------------------
def magnetoelastic_field(m, Ms, B1, B2, eps):
    pref = -2.0 * _inv(Ms)
    out = np.empty_like(m)
    out[0] = pref * (B1 * eps["xx"] * m[0] + B2 * (eps["xy"] * m[1] + eps["xz"] * m[2]))
    out[1] = pref * (B1 * eps["yy"] * m[1] + B2 * (eps["xy"] * m[0] + eps["yz"] * m[2]))
    out[2] = pref * (B1 * eps["zz"] * m[2] + B2 * (eps["xz"] * m[0] + eps["yz"] * m[1]))
    return out


# ----------------------------------------------------------------------
# torques
# ----------------------------------------------------------------------
def cross(a, b):
    return np.stack([a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0]])


def llg_torque(m, B, alpha, gamma, precession=True):
    """Eq.2: tau = -gamma/(1+alpha^2) [ m x B + alpha m x (m x B) ]   (1/s).
    precession=False drops the m x B term: the damping-only torque that a relaxation follows ("after
    letting a non-collinear antiferromagnet relax from a random state"; the paper does not say how -- reading
    S39: as mumax3's relax(), the precession term is switched off and the damping term is integrated with the
    adaptive scheme until the torque falls below a threshold)."""
    mxB = cross(m, B)
    if not precession:
        return (-gamma / (1.0 + alpha * alpha))[None] * (alpha[None] * cross(m, mxB))
    return (-gamma / (1.0 + alpha * alpha))[None] * (mxB + alpha[None] * cross(m, mxB))


def directional_derivative(m, uvec, Ms, cell, pbc):
    """(u.grad) m by 2-point central differences; a missing neighbour takes the
    centre value (S17).  uvec [3,Nz,Ny,Nx] in m/s."""
    out = np.zeros_like(m)
    for axis in range(3):
        h = cell[axis]
        per = pbc[axis] > 0
        mp, exp_ = neighbour(m, axis, +1, per)
        mm, exm = neighbour(m, axis, -1, per)
        Mp, _ = neighbour(Ms, axis, +1, per)
        Mm, _ = neighbour(Ms, axis, -1, per)
        mp = np.where((exp_ & (Mp > 0))[None], mp, m)
        mm = np.where((exm & (Mm > 0))[None], mm, m)
        out += uvec[axis][None] * (mp - mm) / (2.0 * h)
    return out


def zhang_li_torque(m, Ms, alpha, pol, xi, J, cell, pbc):
    """tau_ZL = -(1+alpha^2)^-1 [ (1+xi alpha) m x (m x (u.grad)m) + (xi-alpha) m x (u.grad)m ],
    u = mu_B P J / (e Ms (1+xi^2))  [m/s]   (S17; per sublattice with its own Ms, S18)."""
    Jv = np.asarray(J, float)
    uvec = (MU_B * pol * _inv(Ms) / (Q_E * (1.0 + xi * xi)))[None] * Jv[:, None, None, None]
    a = directional_derivative(m, uvec, Ms, cell, pbc)
    mxa = cross(m, a)
    mxmxa = cross(m, mxa)
    return (-1.0 / (1.0 + alpha * alpha))[None] * ((1.0 + xi * alpha)[None] * mxmxa
                                                   + (xi - alpha)[None] * mxa)


def slonczewski_torque(m, Ms, alpha, gamma, pol, jz, mp, lam, eps_prime, thickness):
    """Slonczewski spin-transfer torque ("as formulated by ... Slonczewski [29], implemented in
    the same way as in mumax3"; the paper prints no formula -- reading S37).  In Gilbert form a current
    density jz through a free layer of thickness d, polarised along the fixed-layer direction m_p, adds
        T = gamma beta [ eps m x (m_p x m) - eps' m x m_p ],     beta = hbar jz / (e Ms d)   [T]
        eps = P Lambda^2 / ((Lambda^2 + 1) + (Lambda^2 - 1) (m . m_p))
    to  dm/dt = -gamma m x B + alpha m x dm/dt + T.  Solving for dm/dt (as for Eq.2) gives the explicit torque
        tau_SL = gamma beta / (1 + alpha^2) [ (eps + alpha eps') m x (m_p x m) - (eps' - alpha eps) m x m_p ].
    m_p [3]: direction of the fixed layer (normalised here); returns 1/s."""
    mp = np.asarray(mp, float)
    mpv = (mp / np.sqrt((mp * mp).sum())).reshape(3, 1, 1, 1) * np.ones_like(m)   # m_p is a direction
    beta = HBAR * jz / (Q_E * thickness) * _inv(Ms)
    l2 = lam * lam
    eps = pol * l2 / ((l2 + 1.0) + (l2 - 1.0) * (m * mpv).sum(axis=0))
    pxm = cross(mpv, m)
    mxpxm = cross(m, pxm)
    pref = gamma * beta / (1.0 + alpha * alpha)
    return (pref * (eps + alpha * eps_prime))[None] * mxpxm + (pref * (eps_prime - alpha * eps))[None] * pxm


# ----------------------------------------------------------------------
# Eq.5: Neumann boundary condition as ghost cells -- reading S41
# ----------------------------------------------------------------------
def neumann_ghosts(m, A11, qn_of, A12, cell):
    """Ghost values behind the six faces of every cell, for one or two sublattices.

    Eq.5:  2 A11^(s) d_n m^(s) = A12 (d_n m^(s') x m^(s)) x m^(s) + D^(s).(n (x) m^(s)),  n the outward normal.
    Readings (S41): (i) the contraction is the one the variation of Eq.4 fixes, D.(n (x) m) = m x q_n with
    q_n = sum_i n_i q_i (interfacial D: q_x = D y^, q_y = -D x^), so that Eq.5 is the natural boundary condition
    of the energy of Eq.3 + Eq.4; (ii) (a x m) x m = -(a - (a.m) m) = -P_m a, so for two sublattices the normal
    derivatives g = d_n m, g' = d_n m' solve the linear system
        2 A  g  + A12 P_m  g' = m  x q_n  = r
        2 A' g' + A12 P_m' g  = m' x q'_n = r'
    whose closed-form solution is, with w = P_m m', beta = A12^2/(2A'), R = r - (A12/2A') P_m r':
        g.w = R.w / (2A - beta + beta |w|^2),   g = (R - beta (g.w) w)/(2A - beta),   g' = (r' - A12 P_m' g)/(2A');
    one sublattice: g = r/(2A).  (iii) the ghost behind the face (axis i, side d) is m_c + h_i g (first order in h,
    as mumax3 does for its DMI boundary), and enters every pair stencil in place of the absent partner.

    m: list of S arrays [3,Nz,Ny,Nx]; A11: list of S per-cell arrays; qn_of(s, axis, d) -> [3,Nz,Ny,Nx] the vector
    q_n = d q_axis of sublattice s per cell; A12 scalar.  Returns list over s of dict (axis, d) -> ghost array."""
    S = len(m)
    assert S <= 2, "Eq.5 is written for a sublattice s and its partner s'"
    proj = lambda a, u: a - (a * u).sum(axis=0)[None] * u
    out = [dict() for _ in range(S)]
    for axis in range(3):
        for d in (+1, -1):
            r = [cross(m[s], qn_of(s, axis, d)) for s in range(S)]
            iA = [np.where(A11[s] > 0, 1.0 / np.where(A11[s] > 0, 2.0 * A11[s], 1.0), 0.0) for s in range(S)]
            if S == 1 or A12 == 0.0:
                g = [iA[s][None] * r[s] for s in range(S)]
            else:
                g = [None, None]
                a2, a2p = 2.0 * A11[0], 2.0 * A11[1]
                beta = A12 * A12 * iA[1]
                w = proj(m[1], m[0])
                R = r[0] - (A12 * iA[1])[None] * proj(r[1], m[0])
                den = a2 - beta
                gw = (R * w).sum(axis=0) / (den + beta * (w * w).sum(axis=0))
                g[0] = (R - (beta * gw)[None] * w) / den[None]
                g[1] = iA[1][None] * (r[1] - A12 * proj(g[0], m[1]))
                del a2p
            for s in range(S):
                out[s][(axis, d)] = m[s] + cell[axis] * g[s]
    return out
