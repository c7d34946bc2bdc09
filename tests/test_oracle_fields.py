"""Pins for oracle/fields.py and the energy bookkeeping of oracle/world.py (P6, P10, P11)."""
import numpy as np
import pytest

import workloads as wl
from oracle import fields as fl
from oracle.constants import (T_A0, T_A12, T_ANIS_C, T_ANIS_U, T_DEMAG, T_DMI, T_DMI_HOMO, T_DMI_INTER,
                              T_EXCH, T_MEL, T_ZEEMAN)
from oracle.world import World


def test_P6_exchange_spin_wave():
    """m = (cos kx, sin kx, 0), periodic: B_exch = -(2A/Ms)(2/h^2)(1 - cos kh) m."""
    nx, h, A, Ms = 32, 2e-9, 1.3e-11, 8e5
    k = 2 * np.pi * 3 / (nx * h)
    x = (np.arange(nx) + 0.5) * h
    m = np.zeros((3, 1, 1, nx))
    m[0, 0, 0], m[1, 0, 0] = np.cos(k * x), np.sin(k * x)
    one = np.ones((1, 1, nx))
    B = fl.pair_laplacian(m, Ms * one, A * one, np.zeros((1, 1, nx), int), 1.0, (h, h, h), (1, 0, 0), 2.0)
    want = -(2 * A / Ms) * (2 / h ** 2) * (1 - np.cos(k * h)) * m
    np.testing.assert_allclose(B, want, rtol=0, atol=1e-12 * np.abs(want).max())


def test_P6b_inter_sublattice_exchange_spin_waves():
    """Eq.3 second term, through World.field_terms so the sublattice wiring is pinned
    too: two periodic sublattices carrying spin waves of DIFFERENT wave numbers k1, k2 (and
    different Ms).  B_A12 on sublattice s must be (A12/Ms_s) lap m^(s') -- the OTHER sublattice's
    wave, factor 1 (not the 2 of the first term), divided by its OWN Ms:
        B_A12^(1) = -(A12/Ms1)(2/h^2)(1 - cos k2 h) m2,   B_A12^(2) = -(A12/Ms2)(2/h^2)(1 - cos k1 h) m1.
    The same world also pins the first term on each sublattice with its own A11, Ms (P6)."""
    nx, ny, h = 48, 4, 2e-9
    A12, Ms, A11 = -1.0e-12, (4.0e5, 2.5e5), (1.0e-11, 0.7e-11)
    ks = [2 * np.pi * q / (nx * h) for q in (3, 5)]
    x = (np.arange(nx) + 0.5) * h
    ms = []
    for k in ks:
        m = np.zeros((3, 1, ny, nx))
        m[0], m[1] = np.cos(k * x)[None, None, :], np.sin(k * x)[None, None, :]
        ms.append(m)
    spec = wl.WorldSpec(name="sw2", grid=(nx, ny, 1), cell=(h, h, h), pbc=(1, 1, 0), S=2, demag=False,
                        mat=wl.make_mat(2, Ms=np.array(Ms)[:, None], A=np.array(A11)[:, None]),
                        coupling=wl.default_coupling(A12=A12), m=[m.astype(np.float32) for m in ms])
    w = World(spec)
    w.m = [m.copy() for m in ms]
    for s in range(2):
        o = 1 - s
        got = w.field_terms(s, terms=T_A12)[T_A12]
        want = -(A12 / Ms[s]) * (2 / h ** 2) * (1 - np.cos(ks[o] * h)) * ms[o]
        np.testing.assert_allclose(got, want, rtol=0, atol=1e-12 * np.abs(want).max())
        got = w.field_terms(s, terms=T_EXCH)[T_EXCH]
        want = -(2 * A11[s] / Ms[s]) * (2 / h ** 2) * (1 - np.cos(ks[s] * h)) * ms[s]
        np.testing.assert_allclose(got, want, rtol=0, atol=1e-12 * np.abs(want).max())


def test_P11_dmi_cycloid_and_continuum():
    """m = (sin kx, 0, cos kx): B_DMI = -(2D/Ms)(sin kh / h) m; 2-D continuum limit
    (2D/Ms)(dx mz, dy mz, -dx mx - dy my) for a smooth texture."""
    nx, h, D, Ms = 40, 2e-9, 3e-3, 5.8e5
    k = 2 * np.pi * 2 / (nx * h)
    x = (np.arange(nx) + 0.5) * h
    m = np.zeros((3, 1, 1, nx))
    m[0, 0, 0], m[2, 0, 0] = np.sin(k * x), np.cos(k * x)
    one = np.ones((1, 1, nx))
    B = fl.dmi_interfacial(m, Ms * one, D * one, (h, h, h), (1, 0, 0))
    want = -(2 * D / Ms) * (np.sin(k * h) / h) * m
    np.testing.assert_allclose(B, want, rtol=0, atol=1e-12 * np.abs(want).max())
    # 2-D smooth texture, periodic, checks the y-direction signs
    n = 64
    X, Y = np.meshgrid((np.arange(n) + 0.5) * h, (np.arange(n) + 0.5) * h, indexing="xy")
    L = n * h
    th = 0.3 * np.sin(2 * np.pi * X / L) + 0.2 * np.cos(2 * np.pi * Y / L) + 1.0
    ph = 0.4 * np.sin(2 * np.pi * Y / L) + 0.1 * np.sin(2 * np.pi * X / L)
    m = np.stack([np.sin(th) * np.cos(ph), np.sin(th) * np.sin(ph), np.cos(th)])[:, None]
    one = np.ones((1, n, n))
    B = fl.dmi_interfacial(m, Ms * one, D * one, (h, h, h), (1, 1, 0))

    def d(f, ax):  # spectral derivative of a periodic array
        kk = 2j * np.pi * np.fft.fftfreq(n, h)
        shape = [1, 1, 1]
        shape[ax] = n
        return np.real(np.fft.ifft(np.fft.fft(f, axis=ax) * kk.reshape(shape), axis=ax))
    want = (2 * D / Ms) * np.stack([d(m[2], 2), d(m[2], 1), -d(m[0], 2) - d(m[1], 1)])
    assert np.abs(B - want).max() < 5e-3 * np.abs(want).max()  # O((kh)^2) stencil error


def _toy_world(pbc, seed=3, elastic=False):
    rng = np.random.default_rng(seed)
    grid = (5, 4, 3)
    S, R = 2, 3
    mat = wl.make_mat(S, R,
                      Ms=np.array([[4e5, 5e5, 3e5], [4.5e5, 3.5e5, 5.5e5]]),
                      A=np.array([[1e-11, 0.7e-11, 1.3e-11], [0.9e-11, 1.1e-11, 0.8e-11]]),
                      alpha=0.1, Ku1=np.array([[6e4, 3e4, 8e4], [5e4, 7e4, 2e4]]),
                      Kc1=np.array([[1e4, -2e4, 3e4], [2e4, 1e4, -1e4]]),
                      D=np.array([[1e-3, 2e-3, 0.5e-3], [1.5e-3, 1e-3, 2e-3]]),
                      B1=-1e7, B2=-0.7e7)
    ax = rng.standard_normal((S, R, 3))
    mat["u"] = ax / np.linalg.norm(ax, axis=-1, keepdims=True)
    c1 = rng.standard_normal((S, R, 3))
    c1 /= np.linalg.norm(c1, axis=-1, keepdims=True)
    c2 = np.cross(c1, rng.standard_normal((S, R, 3)))
    c2 /= np.linalg.norm(c2, axis=-1, keepdims=True)
    mat["c1"], mat["c2"] = c1, c2
    spec = wl.WorldSpec(
        name="toy", grid=grid, cell=(2e-9, 2.5e-9, 1.5e-9), pbc=pbc, S=S,
        regions=rng.integers(0, R, (grid[2], grid[1], grid[0])).astype(np.uint16), mat=mat,
        coupling=wl.default_coupling(A0=-4e-13, A12=-1e-12, D_inter=0.8e-3, scale_A11=0.25, scale_A12=0.5,
                                     d_homo=(3e4, -2e4, 5e4), bc="open"),   # open: the BC of the discrete pair energy (P10)
        bext=(0.05, -0.02, 0.1),
        elastic=dict(C11=2.5e11, C12=1.5e11, C44=1.0e11, rho=6800.0) if elastic else None,
        m=[wl.random_unit(rng, grid), wl.random_unit(rng, grid)],
        u=(rng.standard_normal((3, grid[2], grid[1], grid[0])) * 1e-12).astype(np.float32) if elastic else None,
        v=np.zeros((3, grid[2], grid[1], grid[0]), np.float32) if elastic else None)
    return World(spec, demag_mode="direct")


@pytest.mark.parametrize("pbc", [(0, 0, 0), (1, 1, 0)])
@pytest.mark.parametrize("term", [T_EXCH, T_DMI, T_ANIS_U, T_ANIS_C, T_ZEEMAN, T_DEMAG, T_A12, T_A0,
                                  T_DMI_INTER, T_MEL, T_DMI_HOMO])
def test_P10_field_is_energy_gradient(pbc, term):
    """B_term = -(1/(Ms V)) dE_term/dm (unconstrained derivative of the oracle's energy),
    including OPEN boundary pairs, region-pair scaling and two sublattices."""
    w = _toy_world(pbc, elastic=True)
    B = [w.heff(s, terms=term) for s in range(2)]
    rng = np.random.default_rng(11)
    scale = max(np.abs(B[0]).max(), np.abs(B[1]).max())
    assert scale > 0
    for _ in range(6):
        s = int(rng.integers(0, 2))
        c = int(rng.integers(0, 3))
        iz, iy, ix = (int(rng.integers(0, n)) for n in (3, 4, 5))
        m0 = w.m[s][c, iz, iy, ix]
        hstep = 1e-4
        E = []
        for sgn in (+1, -1):
            w.m[s][c, iz, iy, ix] = m0 + sgn * hstep
            E.append(w.energy(term))
        w.m[s][c, iz, iy, ix] = m0
        dE = (E[0] - E[1]) / (2 * hstep)
        want = -dE / (w.p[s]["Ms"][iz, iy, ix] * w.V)
        assert abs(B[s][c, iz, iy, ix] - want) < 1e-6 * scale, (term, s, c)


def test_open_boundary_pairs_contribute_nothing():
    """S9: a uniform state has zero exchange field in every cell, also at open edges,
    and the DMI field of a uniform state is an edge-only term."""
    grid = (6, 5, 2)
    one = np.ones((2, 5, 6))
    m = np.zeros((3, 2, 5, 6))
    m[0] = 0.6
    m[2] = 0.8
    B = fl.pair_laplacian(m, 8e5 * one, 1e-11 * one, np.zeros((2, 5, 6), int), 1.0, (1e-9,) * 3, (0, 0, 0), 2.0)
    assert np.abs(B).max() == 0.0
    Bd = fl.dmi_interfacial(m, 8e5 * one, 1e-3 * one, (1e-9,) * 3, (0, 0, 0))
    assert np.abs(Bd[:, :, 1:-1, 1:-1]).max() < 1e-18
    assert np.abs(Bd[:, :, :, 0]).max() > 0


def test_anisotropy_special_cases():
    one = np.ones((1, 1, 1))
    m = np.array([0.6, 0.0, 0.8]).reshape(3, 1, 1, 1)
    z = np.array([0.0, 0.0, 1.0]).reshape(3, 1, 1, 1)
    x = np.array([1.0, 0.0, 0.0]).reshape(3, 1, 1, 1)
    y = np.array([0.0, 1.0, 0.0]).reshape(3, 1, 1, 1)
    Bu = fl.uniaxial(m, 8e5 * one, 5e5 * one, z)
    np.testing.assert_allclose(Bu.ravel(), [0, 0, 2 * 5e5 / 8e5 * 0.8])
    # cubic: B_x = -(2Kc1/Ms) m_x (m_y^2 + m_z^2)
    Bc = fl.cubic(m, 8e5 * one, 1e4 * one, x, y)
    np.testing.assert_allclose(Bc.ravel(), [-(2e4 / 8e5) * 0.6 * 0.64, 0, -(2e4 / 8e5) * 0.8 * 0.36], atol=1e-18)


def test_P21_homogeneous_dmi_is_the_gradient_of_eq6():
    """Eq.6 defines the term by its energy density eps = d . (m1 x m2).  The oracle
    implements the FIELD; here the paper's energy is written out and differentiated numerically:
    B^(s) = -(1/(Ms V)) d/dm^(s) [ V sum_cells d . (m1 x m2) ].  Pins the form and both signs."""
    w = _toy_world((0, 0, 0))
    d = np.asarray(w.cpl["d_homo"], float)

    def eq6_energy():
        c = np.cross(np.moveaxis(w.m[0], 0, -1), np.moveaxis(w.m[1], 0, -1))
        return w.V * float((c @ d).sum())

    B = [w.field_terms(s, terms=T_DMI_HOMO)[T_DMI_HOMO] for s in range(2)]
    scale = max(np.abs(B[0]).max(), np.abs(B[1]).max())
    rng = np.random.default_rng(5)
    for _ in range(12):
        s, c = int(rng.integers(0, 2)), int(rng.integers(0, 3))
        iz, iy, ix = (int(rng.integers(0, n)) for n in (3, 4, 5))
        m0 = w.m[s][c, iz, iy, ix]
        E = []
        for sgn in (+1, -1):
            w.m[s][c, iz, iy, ix] = m0 + sgn * 1e-4
            E.append(eq6_energy())
        w.m[s][c, iz, iy, ix] = m0
        want = -(E[0] - E[1]) / 2e-4 / (w.p[s]["Ms"][iz, iy, ix] * w.V)
        assert abs(B[s][c, iz, iy, ix] - want) < 1e-8 * scale, (s, c)
    assert abs(w.energy(T_DMI_HOMO) - eq6_energy()) < 1e-10 * abs(eq6_energy())


def _dijk_from_q(q):
    """D_ijk = sum_l eps_jkl q_il (antisymmetric in j, k): the paper's rank-3 tensor from the three
    per-axis vectors."""
    eps = np.zeros((3, 3, 3))
    eps[0, 1, 2] = eps[1, 2, 0] = eps[2, 0, 1] = 1.0
    eps[0, 2, 1] = eps[2, 1, 0] = eps[1, 0, 2] = -1.0
    return np.einsum("jkl,il->ijk", eps, np.asarray(q, float))


def test_P22_general_dmi_tensor_is_the_gradient_of_eq4():
    """Eq.4 for s = s': eps = sum_ijk D_ijk m_j d_i m_k, D_ijk = -D_ikj, 9 independent
    components.  The paper's energy is written out on a periodic grid with central differences and
    differentiated numerically; the oracle's field must be its gradient.  Pins form, signs, the
    factor 2 and the mapping D_ijk <-> q_i (reading S33)."""
    rng = np.random.default_rng(21)
    n = (6, 5, 4)                                   # (nx, ny, nz)
    cell = (2e-9, 2.5e-9, 1.5e-9)
    q = 1e-3 * rng.standard_normal((3, 3))
    D = _dijk_from_q(q)
    assert np.allclose(D, -np.swapaxes(D, 1, 2))
    m = rng.standard_normal((3, n[2], n[1], n[0]))
    Ms = 5e5 * np.ones(m.shape[1:])
    V = float(np.prod(cell))

    def eq4_energy(mm):
        E = 0.0
        for i in range(3):
            ax = 3 - i                               # array axis of spatial axis i in [3, z, y, x]
            dm = (np.roll(mm, -1, axis=ax) - np.roll(mm, 1, axis=ax)) / (2 * cell[i])
            E += np.einsum("jk,jzyx,kzyx->", D[i], mm, dm)
        return V * E

    B = fl.dmi_tensor(m, Ms, q, cell, (1, 1, 1))
    scale = np.abs(B).max()
    for _ in range(15):
        c = int(rng.integers(0, 3))
        iz, iy, ix = (int(rng.integers(0, k)) for k in (n[2], n[1], n[0]))
        m0 = m[c, iz, iy, ix]
        E = []
        for sgn in (+1, -1):
            m[c, iz, iy, ix] = m0 + sgn * 1e-4
            E.append(eq4_energy(m))
        m[c, iz, iy, ix] = m0
        want = -(E[0] - E[1]) / 2e-4 / (Ms[iz, iy, ix] * V)
        assert abs(B[c, iz, iy, ix] - want) < 1e-7 * scale, c


def test_P22_bulk_dmi_helix_closed_form_and_interfacial_special_case():
    """Bulk (Bloch) DMI eps = D m.(curl m): since m.(curl m) = -sum_i e_i.(m x d_i m) this is
    q_i = -D e_i.  For the helix m = (0, cos kx, sin kx), curl m = -k m, so
    B = -(2D/Ms) curl m -> (2D/Ms)(sin kh / h) m on the grid.  And with q_x = D y^,
    q_y = -D x^ the general term must reproduce the interfacial one cell by cell (open edges too)."""
    nx, h, D, Ms = 32, 2e-9, 1.2e-3, 6e5
    k = 2 * np.pi * 3 / (nx * h)
    x = (np.arange(nx) + 0.5) * h
    m = np.zeros((3, 1, 1, nx))
    m[1, 0, 0], m[2, 0, 0] = np.cos(k * x), np.sin(k * x)
    one = Ms * np.ones((1, 1, nx))
    B = fl.dmi_tensor(m, one, -D * np.eye(3), (h, h, h), (1, 0, 0))
    np.testing.assert_allclose(B, (2 * D / Ms) * np.sin(k * h) / h * m, atol=1e-12 * np.abs(B).max())
    rng = np.random.default_rng(4)
    mm = rng.standard_normal((3, 3, 5, 6))
    Msr = 5e5 * np.ones(mm.shape[1:])
    Msr[1, 2, 3] = 0.0                              # a hole: its pairs drop out in both forms
    qi = np.array([[0, D, 0], [-D, 0, 0], [0, 0, 0]], float)
    for pbc in [(0, 0, 0), (1, 1, 0)]:
        a = fl.dmi_tensor(mm, Msr, qi, (2e-9, 3e-9, 1e-9), pbc)
        b = fl.dmi_interfacial(mm, Msr, D * np.ones_like(Msr), (2e-9, 3e-9, 1e-9), pbc)
        np.testing.assert_allclose(a, b, atol=1e-12 * np.abs(b).max())


def test_P22b_inter_sublattice_dmi_tensor_is_the_gradient_of_eq4():
    """Eq.4 for s != s': the double sum over (s, s') with D^(1,2) = D^(2,1) is written out on a
    periodic grid, eps = sum_ijk D_ijk (m1_j d_i m2_k + m2_j d_i m1_k), and differentiated numerically with respect
    to either sublattice; the oracle's inter-sublattice field, taken through World.field_terms (so the partner
    wiring and the per-sublattice Ms are pinned too), must be its gradient."""
    rng = np.random.default_rng(33)
    grid, cell = (6, 5, 4), (2e-9, 2.5e-9, 1.5e-9)
    spec = wl.make("c3", grid)
    spec.cell, spec.pbc, spec.regions, spec.demag = cell, (1, 1, 1), None, False
    spec.mat = wl.make_mat(2, Ms=np.array([[4e5], [7e5]]), A=1e-11, alpha=0.1)
    q12 = 1e-3 * rng.standard_normal((3, 3))
    spec.coupling = wl.default_coupling(latcon=0.35e-9)
    spec.coupling["dmi_q12"] = q12
    spec.m = [rng.standard_normal((3, grid[2], grid[1], grid[0])).astype(np.float32) for _ in range(2)]
    w = World(spec)
    D = _dijk_from_q(q12)
    V = float(np.prod(cell))

    def eq4_energy(m1, m2):
        E = 0.0
        for i in range(3):
            ax = 3 - i
            d1 = (np.roll(m1, -1, axis=ax) - np.roll(m1, 1, axis=ax)) / (2 * cell[i])
            d2 = (np.roll(m2, -1, axis=ax) - np.roll(m2, 1, axis=ax)) / (2 * cell[i])
            E += np.einsum("jk,jzyx,kzyx->", D[i], m1, d2) + np.einsum("jk,jzyx,kzyx->", D[i], m2, d1)
        return V * E

    B = [w.field_terms(s, terms=T_DMI_INTER)[T_DMI_INTER] for s in range(2)]
    scale = max(np.abs(b).max() for b in B)
    for _ in range(16):
        s = int(rng.integers(0, 2))
        c = int(rng.integers(0, 3))
        iz, iy, ix = (int(rng.integers(0, k)) for k in (grid[2], grid[1], grid[0]))
        m0 = w.m[s][c, iz, iy, ix]
        E = []
        for sgn in (+1, -1):
            w.m[s][c, iz, iy, ix] = m0 + sgn * 1e-4
            E.append(eq4_energy(w.m[0], w.m[1]))
        w.m[s][c, iz, iy, ix] = m0
        want = -(E[0] - E[1]) / 2e-4 / (w.p[s]["Ms"][iz, iy, ix] * V)
        assert abs(B[s][c, iz, iy, ix] - want) < 1e-7 * scale, (s, c)
    # and the interfacial special case: q12_x = D y^, q12_y = -D x^ equals coupling D_inter = D
    Dv = 1.3e-3
    spec2 = spec.copy()
    spec2.pbc = (0, 1, 0)
    spec2.coupling["dmi_q12"] = np.array([[0, Dv, 0], [-Dv, 0, 0], [0, 0, 0]], float)
    spec3 = spec2.copy()
    spec3.coupling["dmi_q12"] = None
    spec3.coupling["D_inter"] = Dv
    for s in range(2):
        a = World(spec2).field_terms(s, terms=T_DMI_INTER)[T_DMI_INTER]
        b = World(spec3).field_terms(s, terms=T_DMI_INTER)[T_DMI_INTER]
        np.testing.assert_allclose(a, b, atol=1e-12 * np.abs(b).max())


def _three_sublattice_spec(grid, pbc, seed):
    rng = np.random.default_rng(seed)
    spec = wl.make("c3", grid)
    spec.S, spec.pbc, spec.regions, spec.demag, spec.J = 3, pbc, None, False, (0.0, 0.0, 0.0)
    spec.cell = (2e-9, 2.5e-9, 1.5e-9)
    spec.mat = wl.make_mat(3, Ms=np.array([[4e5], [7e5], [5e5]]), A=1e-11, alpha=0.1)
    spec.coupling = wl.default_coupling(A0=-2.5e-11, A12=-1.5e-11, latcon=0.35e-9, D_inter=0.0,
                                        d_homo=(2e5, -1e5, 1e6))
    spec.m = [wl.random_unit(rng, grid) for _ in range(3)]
    return spec


def test_P25_three_sublattices_fields_are_the_gradient_of_the_pair_energies():
    """P:L120 ("adding a third sublattice with the same interaction terms as the first two"; reading S38).  The
    inter-sublattice energies are written out pair by pair, independently of the oracle's field code,
        E = V sum_cells [ -(4 A0/a^2) sum_{s<s'} m_s.m_s'  -  A12 sum_{s<s'} m_s . lap m_s'  +  d . sum_cyc m_s x m_{s+1} ]
    (periodic grid, 7-point Laplacian) and differentiated numerically; World.field_terms for each of the three
    sublattices must be the gradient.  Pins the sums over both partners, the factor of each term and the cyclic
    order of Eq.6 for three sublattices."""
    grid = (5, 4, 3)
    spec = _three_sublattice_spec(grid, (1, 1, 1), 44)
    w = World(spec)
    c = w.cpl
    V = w.V

    def lap(a):
        out = np.zeros_like(a)
        for ax, h in ((3, spec.cell[0]), (2, spec.cell[1]), (1, spec.cell[2])):
            out += (np.roll(a, 1, axis=ax) + np.roll(a, -1, axis=ax) - 2 * a) / h ** 2
        return out

    def energy(m):
        E = 0.0
        for s in range(3):
            for t in range(s + 1, 3):
                E += -(4 * c["A0"] / c["latcon"] ** 2) * (m[s] * m[t]).sum() - c["A12"] * (m[s] * lap(m[t])).sum()
            E += (np.asarray(c["d_homo"]).reshape(3, 1, 1, 1) * np.cross(m[s], m[(s + 1) % 3], axis=0)).sum()
        return V * E

    bits = T_A0 | T_A12 | T_DMI_HOMO
    B = [w.heff(s, terms=bits) for s in range(3)]
    scale = max(np.abs(b).max() for b in B)
    rng = np.random.default_rng(5)
    for _ in range(18):
        s, comp = int(rng.integers(0, 3)), int(rng.integers(0, 3))
        iz, iy, ix = (int(rng.integers(0, k)) for k in (grid[2], grid[1], grid[0]))
        m0 = w.m[s][comp, iz, iy, ix]
        E = []
        for sgn in (+1, -1):
            w.m[s][comp, iz, iy, ix] = m0 + sgn * 1e-4
            E.append(energy(w.m))
        w.m[s][comp, iz, iy, ix] = m0
        want = -(E[0] - E[1]) / 2e-4 / (w.p[s]["Ms"][iz, iy, ix] * V)
        assert abs(B[s][comp, iz, iy, ix] - want) < 1e-7 * scale, (s, comp)
    assert abs(w.energy(bits) - energy(w.m)) < 1e-9 * abs(energy(w.m))


def test_P25_the_120_degree_state_closed_forms():
    """Three sublattices at 120 degrees in the plane, uniform: with the homogeneous exchange A0 < 0 alone every
    sublattice feels B = -(4 A0/(Ms a^2)) m_s -- parallel to m_s, so the torque vanishes exactly -- and the energy is
    (3/2)(4 A0/a^2) V per cell; a DMI vector d z^ adds +-(3 sqrt(3)/2) d V per cell, the sign being the chirality
    (the sense in which sublattices 0 -> 1 -> 2 go round), which pins the cyclic order of Eq.6 for S = 3."""
    grid = (4, 3, 1)
    n = grid[0] * grid[1] * grid[2]
    spec = _three_sublattice_spec(grid, (0, 0, 0), 1)
    spec.coupling.update(A12=0.0, d_homo=(0.0, 0.0, 0.0))
    spec.mat["A"][:] = 0.0
    ang = lambda k, chi: np.array([np.cos(chi * 2 * np.pi * k / 3 + 0.3), np.sin(chi * 2 * np.pi * k / 3 + 0.3), 0.0])
    for chi in (+1, -1):
        s2 = spec.copy()
        s2.m = [np.tile(ang(k, chi).reshape(3, 1, 1, 1), (1, grid[2], grid[1], grid[0])).astype(np.float32) for k in range(3)]
        w = World(s2)
        w.m = [np.tile(ang(k, chi).reshape(3, 1, 1, 1), (1, grid[2], grid[1], grid[0])) for k in range(3)]
        pref = 4 * w.cpl["A0"] / w.cpl["latcon"] ** 2
        for s in range(3):
            B = w.heff(s, terms=T_A0)
            np.testing.assert_allclose(B, -(pref / w.p[s]["Ms"])[None] * w.m[s], rtol=1e-12)
            assert np.abs(w.torque(s, terms=T_A0)).max() < 1e-6 * GAMMA_ * abs(pref) / 4e5
        np.testing.assert_allclose(w.energy(T_A0), 1.5 * pref * w.V * n, rtol=1e-12)
        w.cpl["d_homo"] = (0.0, 0.0, 1.0e6)
        np.testing.assert_allclose(w.energy(T_DMI_HOMO), chi * 1.5 * np.sqrt(3.0) * 1.0e6 * w.V * n, rtol=1e-12)


GAMMA_ = 1.7595e11


def _neumann_spec(grid, S, seed, pbc=(0, 0, 0)):
    rng = np.random.default_rng(seed)
    spec = wl.make("c3" if S == 2 else "c1", grid)
    spec.pbc, spec.regions, spec.demag, spec.J = pbc, None, False, (0.0, 0.0, 0.0)
    spec.cell = (2e-9, 2.5e-9, 1.5e-9)
    spec.mat = wl.make_mat(S, Ms=np.array([[4e5], [7e5]])[:S], A=np.array([[1.0e-11], [0.8e-11]])[:S], alpha=0.1,
                           D=np.array([[1.2e-3], [0.7e-3]])[:S])
    spec.coupling = wl.default_coupling(A12=-3e-12 if S == 2 else 0.0, latcon=0.35e-9)
    spec.coupling["dmi_q"] = 0.6e-3 * rng.standard_normal((S, 3, 3))
    spec.coupling["bc"] = "neumann"
    spec.m = [wl.random_unit(rng, grid) for _ in range(S)]
    return spec


def test_P27_neumann_ghosts_satisfy_eq5_as_printed():
    """Eq.5 with the ghost derivatives g = d_n m, g' = d_n m' that oracle/fields.py::neumann_ghosts builds
    its ghost cells from (reading S41):   2 A11 g = A12 (g' x m) x m + m x q_n   for both sublattices, every face,
    the left side and the paper's double cross product written out here independently of the closed-form solve.
    Special cases: one sublattice g = m x q_n/(2A); a collinear antiferromagnet (m' = -m, equal A and D) has g' = -g and
    g = m x q_n/(2 A11 - A12)."""
    from oracle import fields as fl
    spec = _neumann_spec((5, 4, 3), 2, 9)
    w = World(spec)
    gh = w.ghosts(w.m)
    q = np.asarray(spec.coupling["dmi_q"])
    A12 = spec.coupling["A12"]
    for axis in range(3):
        for d in (+1, -1):
            g = [(gh[s][(axis, d)] - w.m[s]) / spec.cell[axis] for s in range(2)]
            for s in range(2):
                o = 1 - s
                qn = np.zeros((3,) + w.m[s].shape[1:])
                if axis == 0:
                    qn[1] = w.p[s]["D"]
                elif axis == 1:
                    qn[0] = -w.p[s]["D"]
                qn = d * (qn + q[s][axis].reshape(3, 1, 1, 1))
                lhs = 2 * w.p[s]["A"][None] * g[s]
                rhs = A12 * fl.cross(fl.cross(g[o], w.m[s]), w.m[s]) + fl.cross(w.m[s], qn)
                np.testing.assert_allclose(lhs, rhs, atol=1e-6 * np.abs(rhs).max())   # (|m| = 1 to fp32 rounding)
                assert np.abs((g[s] * w.m[s]).sum(axis=0)).max() < 1e-6 * np.abs(g[s]).max()   # d_n m is tangent to the sphere
    # collinear antiferromagnet
    s2 = spec.copy()
    s2.mat["A"][:], s2.mat["D"][:] = 1e-11, 1e-3
    s2.coupling["dmi_q"] = None
    s2.m = [spec.m[0], (-spec.m[0]).astype(np.float32)]
    w = World(s2)
    gh = w.ghosts(w.m)
    qx = np.zeros_like(w.m[0]); qx[1] = 1e-3
    g0 = (gh[0][(0, +1)] - w.m[0]) / s2.cell[0]
    g1 = (gh[1][(0, +1)] - w.m[1]) / s2.cell[0]
    np.testing.assert_allclose(g0, fl.cross(w.m[0], qx) / (2e-11 - A12), atol=1e-9 * np.abs(g0).max())
    np.testing.assert_allclose(g1, -g0, atol=1e-9 * np.abs(g0).max())


@pytest.mark.parametrize("hscale", [1.0, 0.25])
def test_P27_neumann_minus_open_is_the_local_boundary_term(hscale):
    """One sublattice: putting the ghost m_c + h d_n m behind an absent neighbour into the exchange AND the DMI pair
    stencils, their O(1/h) parts cancel exactly (only then is the boundary condition the natural one of the energy of
    Eq.3 + Eq.4 -- a ghost derivative wrong by any factor leaves a term that grows like 1/h) and what remains is
        B_neumann - B_open = sum over absent neighbours (1/(2 A Ms)) q_i x (m_c x q_i),
    independent of the cell size, = minus the gradient of the surface energy -(V/4A) |m x q_i|^2.  Checked on a random
    3-D state at two cell sizes, q_i = interfacial + general tensor."""
    from oracle import fields as fl
    spec = _neumann_spec((5, 4, 3), 1, 19)
    spec.cell = tuple(hscale * c for c in spec.cell)
    so = spec.copy()
    so.coupling["bc"] = "open"
    wn, wo = World(spec), World(so)
    diff = wn.heff(0, terms=T_EXCH | T_DMI) - wo.heff(0, terms=T_EXCH | T_DMI)
    m, A, Ms, D = wn.m[0], 1.0e-11, 4e5, 1.2e-3
    q = np.asarray(spec.coupling["dmi_q"])[0].copy()
    q[0] += [0, D, 0]
    q[1] += [-D, 0, 0]
    want = np.zeros_like(m)
    nx, ny, nz = spec.grid
    for axis, n in ((0, nx), (1, ny), (2, nz)):
        qv = q[axis].reshape(3, 1, 1, 1) * np.ones_like(m)
        term = fl.cross(qv, fl.cross(m, qv)) / (2 * A * Ms)
        for edge in (0, n - 1):
            sl = [slice(None)] * 4
            sl[3 - axis] = edge
            want[tuple(sl)] += term[tuple(sl)]
    np.testing.assert_allclose(diff, want, atol=1e-9 * np.abs(want).max())
    assert np.abs(want).max() > 1e-3   # tesla: the term is not negligible at nm cell sizes


@pytest.mark.parametrize("S", [1, 2])
def test_the_default_boundary_is_eq5_and_reduces_to_open_without_dmi(S):
    """P:L161 "The Neumann boundary conditions as given in Eq. (5) are the default in mumax+": a world that names no
    boundary kind uses the ghost cells of Eq.5, which matters as soon as there is DMI.  Without any DMI Eq.5 reads
    2 A11 d_n m = A12 (d_n m' x m) x m, whose solution is d_n m = d_n m' = 0: the default then IS the open boundary."""
    spec = _neumann_spec((6, 5, 2), S, 23)
    named, default, opened = spec.copy(), spec.copy(), spec.copy()
    del default.coupling["bc"]
    opened.coupling["bc"] = "open"
    for s in range(S):
        Bn, Bd, Bo = (World(x).heff(s, terms=T_EXCH | T_DMI | T_A12) for x in (named, default, opened))
        assert np.array_equal(Bd, Bn)
        assert np.abs(Bd - Bo).max() > 1e-3 * np.abs(Bo).max()
    for x in (default, opened):
        x.mat["D"][:] = 0.0
        x.coupling["dmi_q"] = None
    for s in range(S):
        Bd, Bo = (World(x).heff(s, terms=T_EXCH | T_DMI | T_A12) for x in (default, opened))
        assert np.abs(Bd - Bo).max() <= 1e-13 * np.abs(Bo).max()
