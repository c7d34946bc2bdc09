"""GPU parity of the SURVEY 8(f) "NEXT" rows against the fp64 oracle (through the C-ABI): Slonczewski torque
(reading S37), inter-sublattice general DMI tensor (Eq.4, s != s').  Same bars as everywhere: per-cell relative field /
torque error 1e-5, max |delta m| 1e-4 after a fixed-step trajectory."""
import numpy as np
import pytest

import paper_2411_18194_b200 as mmx
import workloads as wl
from oracle import constants as oc
from gpu_util import FIELD_TOL, TRAJ_TOL, field_err, max_dm, pair
from test_gpu_fields import _rich_spec

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name,grid", [("c1", (64, 16, 1)), ("c4", (20, 12, 6)), ("c3", (48, 24, 1))])
def test_slonczewski_torque_and_trajectory(name, grid):
    """P:L39, L110; reading S37.  Torque of every sublattice with the spin-transfer term switched on (uniform
    worlds, a world with 1669-grain-style regions, 3-D), against the oracle; the term must matter; 30 DP45 steps."""
    spec = _rich_spec(name, grid, seed=5)
    spec.mat["pol"][:] = 0.56
    sl = dict(jz=-4.0e11, mp=(0.3, -0.2, 0.93), eps_prime=0.02, thickness=3e-9)
    sl["lambda"] = 1.4
    spec.coupling["slonczewski"] = sl
    g, o = pair(spec)
    plain = spec.copy()
    plain.coupling["slonczewski"] = None
    from gpu_util import pair_oracle
    o0 = pair_oracle(plain)
    for s in range(spec.S):
        ref = o.torque(s)
        assert field_err(o0.torque(s), ref) > 1e-3            # the spin-transfer torque is a visible part of tau
        assert field_err(g.eval_torque(s), ref) < FIELD_TOL, (name, s)
    dt = spec.integrator["dt"]
    g.step_rk45(method=mmx.DP45, fixed_dt=True, dt0=dt, nsteps=30)
    o.step_dp45_fixed(dt, 30)
    for s in range(spec.S):
        assert max_dm(g.get_state(mmx.F_M[s]), o.m[s]) <= TRAJ_TOL
    # clearing it restores the plain torque
    g.set_slonczewski(jz=0.0)
    g.set_state(mmx.F_M0, np.ascontiguousarray(spec.m[0], dtype=np.float32))
    if spec.S == 2:
        g.set_state(mmx.F_M1, np.ascontiguousarray(spec.m[1], dtype=np.float32))
    assert field_err(g.eval_torque(0), o0.torque(0)) < FIELD_TOL
    g.destroy()


def test_slonczewski_switching_closed_form_on_the_cuda_path():
    """P23 end to end on the GPU: macrospin, fixed layer along z, Lambda = 1:
    m_z(t) = tanh(gamma (alpha (B + beta eps') + beta eps) t /(1 + alpha^2) + atanh m_z(0))."""
    HBAR, QE, GAMMA = 1.054571817e-34, 1.602176634e-19, 1.7595e11
    Ms, alpha, P, d, B, epsp, jz = 8.0e5, 0.02, 0.4, 2e-9, 0.2, 0.05, -6.0e11
    spec = wl.make("c1", (4, 1, 1))
    spec.demag = False
    spec.mat["alpha"][:] = alpha
    spec.mat["pol"][:] = P
    spec.mat["A"][:] = 0.0
    spec.bext = (0.0, 0.0, B)
    m0 = np.array([np.sin(0.6), 0.0, np.cos(0.6)])
    spec.m = [np.tile(m0.reshape(3, 1, 1, 1), (1, 1, 1, 4)).astype(np.float32)]
    sl = dict(jz=jz, mp=(0.0, 0.0, 1.0), eps_prime=epsp, thickness=d)
    sl["lambda"] = 1.0
    spec.coupling["slonczewski"] = sl
    g = mmx.World.from_spec(spec)
    dt, n = 2e-14, 2000
    g.step_rk4(dt, n)
    beta = HBAR * jz / (QE * Ms * d)
    rate = GAMMA * (alpha * (B + beta * epsp) + beta * P / 2) / (1 + alpha ** 2)
    mz = np.tanh(rate * n * dt + np.arctanh(float(spec.m[0][2, 0, 0, 0])))
    assert rate < 0                                             # beyond the switching current: m_z falls
    got = g.get_state(mmx.F_M0)[2, 0, 0, :]
    assert np.abs(got - mz).max() < 2e-5, (got, mz)
    g.destroy()


@pytest.mark.parametrize("grid,pbc", [((48, 24, 1), (0, 0, 0)), ((32, 16, 1), (2, 2, 0)), ((20, 12, 4), (0, 0, 0))])
def test_inter_sublattice_dmi_tensor(grid, pbc):
    """Eq.4, the third tensor "used to describe the intersublattice interaction": per-sublattice field under
    MMX_T_DMI_INTER (added to the interfacial D_inter), total field, torque, energy and a 20-step trajectory on a
    two-sublattice world with regions (c3 recipe), open / periodic / 3-D."""
    spec = _rich_spec("c3", grid, seed=29)
    spec.pbc = pbc
    rng = np.random.default_rng(37)
    spec.coupling["dmi_q12"] = 1e-3 * rng.standard_normal((3, 3))
    spec.coupling["dmi_q"] = 0.5e-3 * rng.standard_normal((2, 3, 3))
    g, o = pair(spec)
    plain = spec.copy()
    plain.coupling["dmi_q12"] = None
    from gpu_util import pair_oracle
    o0 = pair_oracle(plain)
    for s in range(2):
        ref = o.field_terms(s, terms=oc.T_DMI_INTER)[oc.T_DMI_INTER]
        assert field_err(o0.field_terms(s, terms=oc.T_DMI_INTER)[oc.T_DMI_INTER], ref) > 1e-2   # the tensor part matters
        assert field_err(g.eval_heff(s, mmx.T_DMI_INTER), ref) < FIELD_TOL, s
        assert field_err(g.eval_heff(s, mmx.T_ALL), o.heff(s)) < FIELD_TOL, s
        assert field_err(g.eval_torque(s), o.torque(s)) < FIELD_TOL, s
    Eg, Eo = g.energy(mmx.T_DMI_INTER), o.energy(oc.T_DMI_INTER)
    assert abs(Eg - Eo) < 1e-5 * abs(Eo)
    dt = spec.integrator["dt"]
    g.step_rk45(method=mmx.DP45, fixed_dt=True, dt0=dt, nsteps=20)
    o.step_dp45_fixed(dt, 20)
    for s in range(2):
        assert max_dm(g.get_state(mmx.F_M[s]), o.m[s]) <= TRAJ_TOL
    g.destroy()


def test_argument_errors_of_the_new_setters():
    spec = wl.make("c1", (8, 4, 1))
    g = mmx.World.from_spec(spec, demag=False)
    with pytest.raises(mmx.MmxError):
        g.set_dmi_tensor(mmx.DMI_INTER, np.ones((3, 3)))       # one sublattice: no inter-sublattice tensor
    with pytest.raises(mmx.MmxError):
        g.set_slonczewski(jz=1e11, mp=(0, 0, 0))               # no fixed-layer direction
    kw = {"lambda": 0.5}
    with pytest.raises(mmx.MmxError):
        g.set_slonczewski(jz=1e11, mp=(0, 0, 1), **kw)          # Lambda < 1
    g.destroy()


def test_relax_driver_matches_the_oracle_and_leaves_time_alone():
    """mmx_relax (reading S39): damping-only torque, adaptive DP45 to a torque threshold.  Macrospin closed form on the
    CUDA path (azimuth frozen, m_z = tanh), then a c2 film: the library and the oracle start from the same seeded state,
    both stop below the threshold, the relaxed states agree (same minimum: |dm| small), the energy went down, the
    simulation time did not move and ordinary stepping afterwards has its precession back."""
    GAMMA = 1.7595e11
    spec = wl.make("c1", (4, 1, 1))
    spec.demag = False
    spec.mat["alpha"][:] = 0.3
    spec.mat["A"][:] = 0.0
    spec.bext = (0.0, 0.0, 0.7)
    m0 = np.array([0.48, 0.36, 0.8])
    spec.m = [np.tile(m0.reshape(3, 1, 1, 1), (1, 1, 1, 4)).astype(np.float32)]
    g = mmx.World.from_spec(spec)
    st = g.relax(torque_stop=1e-4 * GAMMA, tol=1e-7)
    m = g.get_state(mmx.F_M0)[:, 0, 0, 0].astype(np.float64)
    assert st["accepted"] > 0 and g.get_time() == 0.0
    assert abs(np.arctan2(m[1], m[0]) - np.arctan2(0.36, 0.48)) < 2e-6      # no precession
    assert 1 - m[2] < 1e-6                                                  # relaxed along the field
    g.destroy()

    spec = wl.make("c2", (32, 32, 1))
    g, o = pair(spec)
    E0 = g.energy(mmx.T_ALL)
    stop = 2e-3 * GAMMA
    sg = g.relax(torque_stop=stop)
    so = o.relax(stop)
    assert sg["max_torque"] < stop and sg["rejected"] >= 0 and g.get_time() == 0.0
    assert abs(sg["accepted"] - so["accepted"]) <= 2
    assert max_dm(g.get_state(mmx.F_M0), o.m[0]) < 5e-4                      # same relaxed state (S21/S39: unpinned path)
    assert g.energy(mmx.T_ALL) < E0
    assert abs(g.energy(mmx.T_ALL) - o.energy(oc.T_ALL)) < 1e-4 * abs(o.energy(oc.T_ALL))
    # precession is back: one fixed DP45 step equals the oracle's ordinary step from the relaxed state
    o.m = [g.get_state(mmx.F_M0).astype(np.float64)]
    o._k1 = None
    g.step_rk45(method=mmx.DP45, fixed_dt=True, dt0=2e-14, nsteps=5)
    o.step_dp45_fixed(2e-14, 5)
    assert max_dm(g.get_state(mmx.F_M0), o.m[0]) < 1e-5
    g.destroy()


def _three_sublattice_spec(grid, pbc, seed, regions=True):
    rng = np.random.default_rng(seed)
    spec = _rich_spec("c3", grid, seed=seed)          # grains, anisotropy axes, current: the c3 recipe ...
    R = spec.n_regions
    spec.S, spec.pbc = 3, pbc
    for k, tab in list(spec.mat.items()):              # ... with a third sublattice appended to every material table
        spec.mat[k] = np.concatenate([tab, tab[:1]], axis=0)
    spec.mat["Ms"][2] = 5.0e5
    spec.mat["D"][2] = 0.7e-3
    spec.mat["Ku1"][2] = 8e4
    if not regions:
        spec.regions = None
        for k, tab in list(spec.mat.items()):
            spec.mat[k] = tab[:, :1].copy()
    spec.coupling.update(A0=-2.5e-11, A12=-1.5e-12, D_inter=0.4e-3, d_homo=(2e5, -1e5, 1e6))
    spec.m = [wl.random_unit(rng, grid) for _ in range(3)]
    return spec


@pytest.mark.parametrize("grid,pbc,regions", [((48, 24, 1), (0, 0, 0), True), ((32, 16, 1), (2, 2, 0), False),
                                              ((20, 12, 4), (0, 0, 0), True)])
def test_three_sublattices(grid, pbc, regions):
    """P:L120, reading S38: a non-collinear antiferromagnet with three exchange-coupled sublattices (Fig.3's kind of
    world: grains, reduced inter-grain exchange, interfacial + homogeneous DMI).  Every inter-sublattice term, the demag
    field of M = sum_s Ms m_s, the total field, torque and energy of each sublattice, and a 20-step trajectory."""
    spec = _three_sublattice_spec(grid, pbc, 61, regions)
    spec.coupling["dmi_q12"] = 1e-3 * np.random.default_rng(2).standard_normal((3, 3))
    g, o = pair(spec)
    for s in range(3):
        ref = o.field_terms(s)
        for bit in (mmx.T_A12, mmx.T_A0, mmx.T_DMI_INTER, mmx.T_DMI_HOMO, mmx.T_DEMAG, mmx.T_EXCH, mmx.T_DMI):
            assert field_err(g.eval_heff(s, bit), ref[bit]) < FIELD_TOL, (s, bit)
        assert field_err(g.eval_heff(s, mmx.T_ALL), o.heff(s)) < FIELD_TOL, s
        assert field_err(g.eval_torque(s), o.torque(s)) < FIELD_TOL, s
    for bit in (mmx.T_A0, mmx.T_A12, mmx.T_DMI_HOMO, mmx.T_ALL):
        Eg, Eo = g.energy(bit), o.energy(bit)
        assert abs(Eg - Eo) < 2e-5 * abs(Eo), bit
    dt = 2e-15
    g.step_rk45(method=mmx.DP45, fixed_dt=True, dt0=dt, nsteps=20)
    o.step_dp45_fixed(dt, 20)
    for s in range(3):
        assert max_dm(g.get_state(mmx.F_M[s]), o.m[s]) <= TRAJ_TOL
    g.destroy()


def test_the_120_degree_state_is_an_equilibrium_of_the_cuda_path():
    """P25's closed form end to end: three sublattices at 120 degrees under the homogeneous exchange alone: zero torque
    (to fp32 rounding of a 300 T exchange field), B_s = -(4 A0/(Ms a^2)) m_s."""
    grid = (8, 4, 1)
    spec = _three_sublattice_spec(grid, (0, 0, 0), 3, regions=False)
    spec.demag, spec.J = False, (0.0, 0.0, 0.0)
    spec.coupling.update(A12=0.0, D_inter=0.0, d_homo=(0.0, 0.0, 0.0))
    for k in ("A", "D", "Ku1", "Kc1"):
        spec.mat[k][:] = 0.0
    spec.bext = (0.0, 0.0, 0.0)
    spec.m = [np.tile(np.array([np.cos(2 * np.pi * k / 3 + 0.3), np.sin(2 * np.pi * k / 3 + 0.3), 0.0]).reshape(3, 1, 1, 1),
                      (1, 1, grid[1], grid[0])).astype(np.float32) for k in range(3)]
    g = mmx.World.from_spec(spec)
    pref = 4 * spec.coupling["A0"] / spec.coupling["latcon"] ** 2
    for s in range(3):
        B = g.eval_heff(s, mmx.T_ALL & ~mmx.T_DEMAG).astype(np.float64)
        want = -(pref / spec.mat["Ms"][s, 0]) * spec.m[s].astype(np.float64)
        assert np.abs(B - want).max() < 1e-6 * np.abs(want).max()
        tau = g.eval_torque(s).astype(np.float64)
        assert np.abs(tau).max() < 1e-6 * 1.7595e11 * np.abs(want).max()
    g.destroy()


@pytest.mark.parametrize("name,grid,height", [("c1", (40, 24, 1), 60e-9), ("c4", (20, 18, 3), 7e-9), ("three", (36, 20, 1), 60e-9)])
def test_stray_field_above_the_magnet(name, grid, height):
    """P:L84, Fig.3; reading S40: the field in a probe layer above the magnet against the oracle's term-by-term sum with the
    z-shifted Newell tensor: one layer, several layers (each with its own z offset), and the Fig.3 kind of world (three
    sublattices with different Ms and grains, M = sum_s Ms m_s; cell 1 x 1 x 30 nm, probe 60 nm above the surface)."""
    if name == "three":
        spec = _three_sublattice_spec(grid, (0, 0, 0), 71)
        spec.cell = (1e-9, 1e-9, 30e-9)
    else:
        spec = _rich_spec(name, grid, seed=13)
    g, o = pair(spec)
    got, ref = g.stray_field(height), o.stray_field(height)
    assert field_err(got[:, None], ref[:, None]) < FIELD_TOL, name
    assert np.abs(got[2] - ref[2]).max() < FIELD_TOL * np.abs(ref[2]).max()          # the imaged component, B_z
    g.destroy()


def test_stray_field_argument_errors_and_the_on_axis_closed_form():
    """Periodic worlds are refused; the on-axis closed form of a uniformly magnetised square slab (P26a) on the CUDA path."""
    spec = wl.make("c2", (16, 16, 1))
    g = mmx.World.from_spec(spec, demag=False)
    with pytest.raises(mmx.MmxError):
        g.stray_field(10e-9)
    g.destroy()
    n, h, t, Ms, height = 21, 2e-9, 3e-9, 8e5, 60e-9
    spec = wl.make("c1", (n, n, 1))
    spec.cell, spec.demag = (h, h, t), False
    spec.mat["Ms"][:] = Ms
    m = np.zeros((3, 1, n, n), np.float32); m[2] = 1.0
    spec.m = [m]
    g = mmx.World.from_spec(spec)
    B = g.stray_field(height)
    a, zc = n * h, t / 2 + height
    om = lambda d: 4 * np.arctan(a * a / (4 * d * np.sqrt(d * d + a * a / 2)))
    want = 4e-7 * np.pi * Ms / (4 * np.pi) * (om(zc - t / 2) - om(zc + t / 2))
    assert abs(B[2, n // 2, n // 2] - want) < 2e-3 * abs(want)
    g.destroy()


@pytest.mark.parametrize("name,grid,pbc", [("c1", (24, 12, 1), (0, 0, 0)), ("c4", (12, 10, 5), (0, 0, 0)), ("c3", (32, 16, 1), (0, 0, 0)),
                                           ("c3", (24, 16, 2), (0, 2, 0))])
def test_neumann_boundary_condition(name, grid, pbc):
    """Eq.5, the paper's default boundary condition, reading S41: ghost cells in the exchange, A12 and DMI
    pairs (interfacial + general tensors), one and two sublattices, grains and holes (a cell next to an empty cell is a
    boundary cell), mixed periodic / Neumann axes: each term, the total field, torque, energy and a short trajectory
    against the oracle; the boundary condition must matter."""
    spec = _rich_spec(name, grid, seed=43)
    spec.pbc = pbc
    rng = np.random.default_rng(47)
    spec.coupling["dmi_q"] = 0.8e-3 * rng.standard_normal((spec.S, 3, 3))
    if spec.S == 2:
        spec.coupling["dmi_q12"] = 0.5e-3 * rng.standard_normal((3, 3))
        spec.mat["Ms"][:, 3] = 0.0                      # one grain is empty: its neighbours see a boundary
    spec.coupling["bc"] = "neumann"
    g, o = pair(spec)
    so = spec.copy()
    so.coupling["bc"] = "open"
    from gpu_util import pair_oracle
    o_open = pair_oracle(so)
    bits = [mmx.T_EXCH, mmx.T_DMI] + ([mmx.T_A12, mmx.T_DMI_INTER] if spec.S == 2 else [])
    for s in range(spec.S):
        mag = (o.p[s]["Ms"] > 0)[None]
        ref = o.field_terms(s)
        assert field_err(o_open.heff(s) * mag, o.heff(s) * mag) > 1e-3
        for bit in bits:
            assert field_err(g.eval_heff(s, bit), ref[bit] * mag) < FIELD_TOL, (name, s, bit)
        B = o.heff(s) * mag
        if spec.demag:
            B = B - ref[oc.T_DEMAG] * (~mag)               # (library convention S35: B_eff = 0 in empty cells)
        assert field_err(g.eval_heff(s, mmx.T_ALL), o.heff(s) * mag) < FIELD_TOL, (name, s)
        assert field_err(g.eval_torque(s), o.torque(s)) < FIELD_TOL, (name, s)
    Eg, Eo = g.energy(mmx.T_EXCH | mmx.T_DMI), o.energy(oc.T_EXCH | oc.T_DMI)
    assert abs(Eg - Eo) < 1e-5 * abs(Eo)
    dt = spec.integrator["dt"]
    g.step_rk45(method=mmx.DP45, fixed_dt=True, dt0=dt, nsteps=20)
    o.step_dp45_fixed(dt, 20)
    for s in range(spec.S):
        assert max_dm(g.get_state(mmx.F_M[s]), o.m[s]) <= TRAJ_TOL
    g.set_boundary("open")
    for s in range(spec.S):
        g.set_state(mmx.F_M[s], np.ascontiguousarray(spec.m[s], dtype=np.float32))
    mag = (o.p[0]["Ms"] > 0)[None]
    assert field_err(g.eval_heff(0, mmx.T_EXCH | mmx.T_DMI), o_open.heff(0, terms=oc.T_EXCH | oc.T_DMI) * mag) < FIELD_TOL
    g.destroy()


@pytest.mark.parametrize("name,grid", [("c1", (24, 12, 1)), ("c3", (32, 16, 1))])
def test_default_boundary_is_neumann(name, grid):
    """Eq.5 is the default.  A world on which mmx_set_boundary is never called (one or two sublattices, DMI
    present) gives the oracle's default, which is the Neumann field and not the open one; with every DMI constant zero
    the default is the open boundary bit for bit (and stays on the kernels of the open case)."""
    spec = _rich_spec(name, grid, seed=61)
    spec.coupling.pop("bc", None)
    g, o = pair(spec)
    so = spec.copy()
    so.coupling["bc"] = "open"
    from gpu_util import pair_oracle
    o_open = pair_oracle(so)
    for s in range(spec.S):
        mag = (o.p[s]["Ms"] > 0)[None]
        assert field_err(o_open.heff(s) * mag, o.heff(s) * mag) > 1e-3
        assert field_err(g.eval_heff(s, mmx.T_ALL), o.heff(s) * mag) < FIELD_TOL, (name, s)
    g.destroy()
    for sp in (spec, so):
        sp.mat["D"][:] = 0.0
        sp.coupling["D_inter"] = 0.0
        sp.coupling["dmi_q"] = None
        sp.coupling.pop("dmi_q12", None)
    gd, go = mmx.World.from_spec(spec), mmx.World.from_spec(so)
    for s in range(spec.S):
        assert np.array_equal(gd.eval_heff(s, mmx.T_ALL), go.eval_heff(s, mmx.T_ALL))
    gd.destroy(); go.destroy()
