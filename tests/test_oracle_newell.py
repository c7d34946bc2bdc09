"""Pins for oracle/newell.py and oracle/demag.py (P1-P5, P19 of DESIGN.md)."""
import os

import numpy as np
import pytest

from oracle import demag as dm
from oracle import newell as nw
from oracle.constants import MU0

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def test_P1_selfterm_golden():
    """N_xx+N_yy+N_zz = 1; cube = 1/3; values printed in SURVEY 8c (golden file)."""
    for line in open(os.path.join(GOLDEN, "newell_selfterm.txt")):
        if line.startswith("#") or not line.strip():
            continue
        v = [float(x) for x in line.split()]
        got = nw.self_term(tuple(v[:3]))
        assert abs(sum(got) - 1.0) < 1e-13
        np.testing.assert_allclose(got, v[3:], atol=2e-10)


def test_P2_trace_and_parity():
    cell = (2e-9, 3e-9, 1.5e-9)
    o = {c: nw.newell_octant(c, (6, 5, 4), cell) for c in nw.COMPS}
    tr = o["xx"] + o["yy"] + o["zz"]
    tr[0, 0, 0] -= 1.0
    assert np.abs(tr).max() < 1e-13
    # off-diagonals vanish on their symmetry planes (odd parity)
    assert np.abs(o["xy"][:, 0, :]).max() < 1e-15 and np.abs(o["xy"][:, :, 0]).max() < 1e-15
    assert np.abs(o["xz"][0, :, :]).max() < 1e-15 and np.abs(o["yz"][:, 0, :]).max() < 1e-15
    # explicit odd parity through a shifted evaluation: N_xy(-x) = -N_xy(x)
    a = nw.newell_octant("xy", (1, 1, 1), cell, shift=(2 * cell[0], cell[1], cell[2]))
    b = nw.newell_octant("xy", (1, 1, 1), cell, shift=(-2 * cell[0], cell[1], cell[2]))
    assert a[0, 0, 0] != 0 and abs(a[0, 0, 0] + b[0, 0, 0]) < 1e-15


def _gauss_pair_average(fun, r, cell, n=6):
    """< fun(r + s - s') > over s, s' uniform in the cell, by Gauss-Legendre quadrature."""
    x, w = np.polynomial.legendre.leggauss(n)
    x, w = 0.5 * x, 0.5 * w
    acc = 0.0
    pts = [(xi, wi) for xi, wi in zip(x, w)]
    t = {}
    for a in range(3):  # distribution of s_a - s'_a on the tensor grid
        T = (x[:, None] - x[None, :]) * cell[a]
        W = w[:, None] * w[None, :]
        t[a] = (T.ravel(), W.ravel())
    TX, TY, TZ = np.meshgrid(t[0][0], t[1][0], t[2][0], indexing="ij")
    WX, WY, WZ = np.meshgrid(t[0][1], t[1][1], t[2][1], indexing="ij")
    return float((fun(r[0] + TX, r[1] + TY, r[2] + TZ) * WX * WY * WZ).sum())


def test_brute_force_pair_integral():
    """N_ij(r) = -(V/4pi) < d_i d_j 1/|r+s-s'| >: 6-D Gauss quadrature of the point-dipole
    kernel between two separated cells, independent of Newell's closed forms."""
    cell = (1.0, 1.4, 0.6)
    V = cell[0] * cell[1] * cell[2]
    r_idx = (2, 1, 1)
    r = tuple(i * c for i, c in zip(r_idx, cell))

    def F(i, j):
        def f(x, y, z):
            R2 = x * x + y * y + z * z
            c = (x, y, z)
            return 3 * c[i] * c[j] / R2 ** 2.5 - (1.0 if i == j else 0.0) / R2 ** 1.5
        return f
    ax = {"x": 0, "y": 1, "z": 2}
    for comp in nw.COMPS:
        want = -(V / (4 * np.pi)) * _gauss_pair_average(F(ax[comp[0]], ax[comp[1]]), r, cell, n=7)
        got = nw.newell_octant(comp, (3, 2, 2), cell, cutoff_cells=1e9)[r_idx[2], r_idx[1], r_idx[0]]
        assert abs(got - want) < 2e-7 * abs(want) + 1e-12, (comp, got, want)


def test_P3_dipole_limit_and_branch_agreement():
    cell = (4e-9, 4e-9, 4e-9)
    V = 64e-27
    i = (20, 25, 30)
    x, y, z = (k * 4e-9 for k in i)
    R = np.sqrt(x * x + y * y + z * z)
    an = {c: nw.newell_octant(c, (21, 26, 31), cell, cutoff_cells=1e9)[30, 25, 20] for c in nw.COMPS}
    asy = {c: nw.newell_octant(c, (21, 26, 31), cell, cutoff_cells=0.1)[30, 25, 20] for c in nw.COMPS}
    dip = dict(xx=V / (4 * np.pi) * (1 / R ** 3 - 3 * x * x / R ** 5), xy=V / (4 * np.pi) * (-3 * x * y / R ** 5),
               yz=V / (4 * np.pi) * (-3 * y * z / R ** 5), zz=V / (4 * np.pi) * (1 / R ** 3 - 3 * z * z / R ** 5))
    for c, d in dip.items():
        assert abs(an[c] - d) < 2e-3 * abs(d)          # point dipole: O((cell/R)^2) corrections
    for c in nw.COMPS:
        assert abs(an[c] - asy[c]) < 1e-7 * abs(an[c])  # two independent branches agree far away
    # ... and still agree at the default switch radius with an elongated cell
    cell = (7.8125e-9, 7.8125e-9, 3e-9)
    a = nw.newell_octant("xx", (34, 3, 2), cell, cutoff_cells=1e9)[1, 2, 33]
    b = nw.newell_octant("xx", (34, 3, 2), cell, cutoff_cells=0.1)[1, 2, 33]
    assert abs(a - b) < 1e-7 * abs(a)


@pytest.mark.parametrize("n,cell", [((4, 2, 3), (1.0, 1.5, 0.7)), ((3, 3, 3), (2.0, 2.0, 2.0))])
def test_P4_uniform_box_equals_big_cell(n, cell):
    """Average demag factor of a uniformly magnetised block of n cells = self term of one
    cell with the block's edge lengths (exact identity); cube block -> 1/3."""
    oct_ = nw.kernel_octant(n, cell)
    big = nw.self_term(tuple(k * c for k, c in zip(n, cell)))
    for a, comp in enumerate(("xx", "yy", "zz")):
        M = np.zeros((3, n[2], n[1], n[0]))
        M[a] = 1.0
        B = dm.demag_direct(M, oct_, n, (0, 0, 0))
        assert abs(-B[a].mean() / MU0 - big[a]) < 1e-12
        for b in range(3):
            if b != a:
                assert abs(B[b].mean()) < 1e-18  # off-diagonals average to zero
    if n == (3, 3, 3):
        np.testing.assert_allclose(big, (1 / 3,) * 3, atol=1e-13)


def test_P19_thin_film():
    """64x64x1 flat cells: N_z of the film close to 1 and equal to the big-cell value."""
    n, cell = (64, 64, 1), (4e-9, 4e-9, 1e-9)
    oct_ = nw.kernel_octant(n, cell)
    M = np.zeros((3, 1, 64, 64))
    M[2] = 1.0
    spec = dm.kernel_spectrum(oct_, n, (0, 0, 0))
    B = dm.demag_fft(M, spec, n, (0, 0, 0))
    nz_film = -B[2].mean() / MU0
    big = nw.self_term((256e-9, 256e-9, 1e-9))
    assert abs(nz_film - big[2]) < 1e-10
    assert 0.98 < nz_film < 1.0


@pytest.mark.parametrize("grid,pbc", [((8, 8, 4), (0, 0, 0)), ((5, 3, 2), (0, 0, 0)),
                                      ((8, 8, 1), (2, 2, 0)), ((8, 4, 2), (3, 0, 0))])
def test_P5_direct_vs_fft(grid, pbc):
    rng = np.random.default_rng(5)
    cell = (2e-9, 3e-9, 1e-9)
    oct_ = nw.kernel_octant(grid, cell, pbc)
    M = rng.standard_normal((3, grid[2], grid[1], grid[0])) * 1e5
    Bd = dm.demag_direct(M, oct_, grid, pbc)
    Bf = dm.demag_fft(M, dm.kernel_spectrum(oct_, grid, pbc), grid, pbc)
    assert np.abs(Bd - Bf).max() < 1e-12 * np.abs(Bd).max()


def test_pbc_kernel_against_explicit_images():
    """Periodic kernel (S13) vs an explicit open-boundary sum over replicated copies of the
    magnet: equal up to the truncation of the outermost image shell."""
    grid, cell, R = (4, 4, 1), (2e-9, 2e-9, 1e-9), 6
    rng = np.random.default_rng(7)
    M = rng.standard_normal((3, 1, 4, 4))
    oct_p = nw.kernel_octant(grid, cell, (R, R, 0))
    Bp = dm.demag_direct(M, oct_p, grid, (R, R, 0))
    rep = 2 * R + 1
    big = (grid[0] * rep, grid[1] * rep, 1)
    Mbig = np.tile(M, (1, 1, rep, rep))
    oct_o = nw.kernel_octant(big, cell)
    c0 = R * 4
    tg = [(c0 + i, c0 + j, 0) for j in range(4) for i in range(4)]
    Bo = dm.demag_direct(Mbig, oct_o, big, (0, 0, 0), targets=tg).reshape(3, 1, 4, 4)
    # difference = edge images that one window has and the other has not: O((cell/(R L))^3) each
    assert np.abs(Bp - Bo).max() < 2e-2 * np.abs(Bo).max()
    assert np.abs(Bp - Bo).max() > 0  # the windows do differ (definition, not identity)


def test_P26_stray_field_above_the_magnet():
    """P26 (pins oracle/demag.py::stray_field_at_height, reading S40).
    (a) closed form: on the axis of a uniformly z-magnetised square slab (side a, thickness t) the surface-charge
        picture gives B_z(z) = (mu0 Ms / 4 pi) [Omega(z - t/2) - Omega(z + t/2)], Omega(d) = 4 atan(a^2/(4 d sqrt(d^2 + a^2/2)))
        the solid angle of the square seen from distance d; probe cells small against the height, so the cell average
        equals the point value to O((cell/height)^2).
    (b) far field: one magnetised cell seen from 40 cells above is a point dipole.
    (c) tie to the validated in-magnet kernel (P4, P5): in a two-layer magnet the field that layer 0 alone creates in
        layer 1 is the stray field of layer 0 at height dz/2 above its surface."""
    from oracle import demag as dm
    from oracle.constants import MU0
    # (a)
    n, h, t, Ms = 21, 2e-9, 3e-9, 8e5
    M = np.zeros((3, 1, n, n)); M[2] = Ms
    a = n * h
    for height in (20e-9, 60e-9):
        B = dm.stray_field_at_height(M, (n, n, 1), (h, h, t), height)
        zc = t / 2 + height                                   # probe centre above the slab centre
        om = lambda d: 4 * np.arctan(a * a / (4 * d * np.sqrt(d * d + a * a / 2)))
        want = MU0 * Ms / (4 * np.pi) * (om(zc - t / 2) - om(zc + t / 2))
        assert abs(B[2, n // 2, n // 2] - want) < 2e-3 * abs(want), (height, B[2, n // 2, n // 2], want)
        assert abs(B[0, n // 2, n // 2]) < 1e-9 * abs(want) and abs(B[1, n // 2, n // 2]) < 1e-9 * abs(want)
    # (b)
    n, h = 9, 1e-9
    M = np.zeros((3, 1, n, n)); mom = np.array([0.3, -0.5, 0.8]) * 1e6
    M[:, 0, 4, 4] = mom
    height = 40e-9
    B = dm.stray_field_at_height(M, (n, n, 1), (h, h, h), height, cutoff_cells=8.0)
    for (ty, tx) in ((4, 4), (0, 8), (7, 2)):
        r = np.array([(tx - 4) * h, (ty - 4) * h, h / 2 + height])
        rn = np.linalg.norm(r)
        want = MU0 / (4 * np.pi) * h ** 3 * (3 * r * (mom @ r) / rn ** 5 - mom / rn ** 3)
        np.testing.assert_allclose(B[:, ty, tx], want, rtol=2e-3, atol=1e-6 * np.abs(want).max())
    # (c)
    rng = np.random.default_rng(8)
    grid, cell = (6, 5, 2), (2e-9, 3e-9, 1.5e-9)
    M = rng.standard_normal((3, 2, 5, 6)) * 5e5
    M0 = M.copy(); M0[:, 1] = 0.0
    octant = nw.kernel_octant(grid, cell)
    ref = dm.demag_direct(M0, octant, grid, (0, 0, 0))[:, 1]
    got = dm.stray_field_at_height(M0[:, :1], (6, 5, 1), cell, cell[2] / 2)
    np.testing.assert_allclose(got, ref, rtol=1e-10, atol=1e-12 * np.abs(ref).max())
