"""GPU parity, dynamics: fixed-step trajectories of every config (reduced sizes here; the full-size c4 field check is in
test_gpu_fields.py) against the fp64 oracle: max |delta m| <= 1e-4
(north_star), DP45 error estimates, the adaptive controller, |m| = 1."""
import numpy as np
import pytest

import paper_2411_18194_b200 as mmx
import workloads as wl
from gpu_util import assert_estimates, TRAJ_TOL, gpu_m, max_dm, pair, pair_oracle

pytestmark = pytest.mark.gpu


def _compare_state(g, o, spec, tol=TRAJ_TOL):
    for s in range(spec.S):
        m = g.get_state(mmx.F_M[s])
        assert max_dm(m, o.m[s]) <= tol, (s, max_dm(m, o.m[s]))
        np.testing.assert_allclose((m.astype(np.float64) ** 2).sum(axis=0), 1.0, atol=1e-6)


def test_c1_rk4_full_protocol():
    """BASELINE config 1 exactly: 64x16x1, RK4, dt = 1e-13, 2000 steps."""
    spec = wl.c1()
    g, o = pair(spec)
    g.step_rk4(1e-13, 2000)
    o.step_rk4(1e-13, 2000)
    _compare_state(g, o, spec)
    assert abs(g.get_time() - 2000e-13) < 1e-20
    g.destroy()


@pytest.mark.parametrize("name,grid,nsteps", [("c2", (64, 64, 1), 200), ("c3", (128, 32, 1), 200),
                                              ("c4", (32, 32, 8), 100), ("c4", (20, 12, 3), 50),
                                              ("c4", (136, 40, 36), 30),  # register-resident fast paths
                                              ("c5", (64, 32, 1), 200)])
def test_dp45_fixed_step_trajectory(name, grid, nsteps):
    spec = wl.make(name, grid)
    dt = spec.integrator["dt"]
    g, o = pair(spec)
    bmax = max(float(np.sqrt((o.heff(s) ** 2).sum(axis=0)).max()) for s in range(spec.S))
    st = g.step_rk45(method=mmx.DP45, fixed_dt=True, dt0=dt, nsteps=nsteps)
    errs = o.step_dp45_fixed(dt, nsteps)
    assert st["accepted"] == nsteps and st["rejected"] == 0
    _compare_state(g, o, spec)
    hist = g.get_err_history(nsteps)
    assert len(hist) == nsteps
    # fp32 floor of the estimate dt |sum_j e_j k_j|: the torque m x B is formed in fp32 from a field
    # that is nearly parallel to m (33 T of inter-sublattice exchange in c5), so each k_j carries an
    # absolute rounding error of about gamma max|B_eff| 2^-24 per operation, ~16 operations deep, and
    # the combination weights it with sum_j |e_j| = 0.16 (Dormand-Prince, Table 2):
    #   atol = 16 * 2^-24 * 0.16 * dt * gamma * max|B_eff|
    atol = 16 * 2.0 ** -24 * 0.16 * dt * 1.7595e11 * bmax
    assert_estimates(hist, errs, max(atol, 1e-9))
    if spec.elastic is not None:
        u, v = g.get_state(mmx.F_U), g.get_state(mmx.F_V)
        assert np.abs(u - o.u).max() <= 1e-4 * max(np.abs(o.u).max(), 1e-30)
        assert np.abs(v - o.v).max() <= 1e-4 * max(np.abs(o.v).max(), 1e-30)
    g.destroy()


def test_rk4_two_sublattice_with_current():
    spec = wl.make("c3", (128, 32, 1))
    g, o = pair(spec)
    g.step_rk4(5e-15, 200)
    o.step_rk4(5e-15, 200)
    _compare_state(g, o, spec)
    g.destroy()


def test_split_calls_equal_one_call():
    """FSAL bookkeeping across calls: 2 x 25 steps == 50 steps, bit for bit."""
    spec = wl.make("c4", (16, 16, 4))
    a = mmx.World.from_spec(spec)
    b = mmx.World.from_spec(spec)
    a.step_rk45(fixed_dt=True, dt0=1e-13, nsteps=50)
    b.step_rk45(fixed_dt=True, dt0=1e-13, nsteps=25)
    b.step_rk45(fixed_dt=True, dt0=1e-13, nsteps=25)
    assert np.array_equal(a.get_state(mmx.F_M0), b.get_state(mmx.F_M0))
    a.destroy(); b.destroy()


def test_adaptive_controller_matches_oracle():
    """Adaptive DP45 (controller reading S21) from a first step 60x the one the controller settles on:
    both sides reject several times, shrink and recover; every attempt must take the same accept /
    reject decision with the same step size and estimate (per-attempt calls, max_attempts = 1, the
    proposed dt handed back in), then a free-running stretch must end at the same time and state."""
    spec = wl.make("c2", (32, 32, 1))
    g, o = pair(spec)
    tol = 1e-5
    settle = o.run_dp45(tol=tol, nsteps=12)["dt"]
    o = pair_oracle(spec)
    log = []
    o.run_dp45(tol=tol, dt0=60 * settle, max_attempts=16, log=log)
    nrej = sum(1 for _, _, ok in log if not ok)
    assert nrej >= 3 and len(log) - nrej >= 3, log
    dt = 60 * settle
    for k, (dt_ref, err_ref, ok_ref) in enumerate(log):
        st = g.step_rk45(method=mmx.DP45, tol=tol, dt0=dt, max_attempts=1)
        assert (st["accepted"] == 1) == ok_ref and st["accepted"] + st["rejected"] == 1, (k, st, log[k])
        assert abs(dt - dt_ref) <= 1e-3 * dt_ref, (k, dt, dt_ref)
        assert abs(st["last_err"] - err_ref) <= 2e-2 * err_ref + 1e-9, (k, st["last_err"], err_ref)
        dt = st["dt"]
    _compare_state(g, o, spec)
    n = 20
    st = g.step_rk45(method=mmx.DP45, tol=tol, dt0=dt, nsteps=n)
    ref = o.run_dp45(tol=tol, dt0=dt, nsteps=n)
    assert st["accepted"] == n == ref["accepted"] and st["rejected"] == ref["rejected"]
    assert abs(st["t"] - ref["t"]) <= 1e-4 * ref["t"]
    # the two sides now stand at slightly different times (their step sizes follow estimates that agree
    # to ~1e-3): the states may differ by that time offset times the largest |dm/dt|, on top of TRAJ_TOL
    _compare_state(g, o, spec, tol=TRAJ_TOL + o.max_torque() * abs(st["t"] - ref["t"]))
    g.destroy()


def test_nan_in_the_state_is_reported_and_leaves_the_accepted_state_alone():
    """MMX_ENAN ("NaN guard"): one NaN cell written through mmx_set_state must
    surface as status MMX_ENAN from the stepping call, with no step accepted, the time and the
    state buffer of the accepted side untouched, and max_torque reporting it too."""
    spec = wl.make("c4", (16, 16, 8))
    g = mmx.World.from_spec(spec)
    g.step_rk45(method=mmx.DP45, fixed_dt=True, dt0=1e-13, nsteps=3)
    t0 = g.get_time()
    m = g.get_state(mmx.F_M0).copy()
    m[1, 3, 5, 7] = np.nan
    g.set_state(mmx.F_M0, m)
    for kw in (dict(fixed_dt=True, dt0=1e-13, nsteps=5), dict(tol=1e-5, nsteps=5), dict(method=mmx.CK45, tol=1e-5, nsteps=5)):
        with pytest.raises(mmx.MmxError) as ei:
            g.step_rk45(**kw)
        assert ei.value.code == -5, ei.value          # MMX_ENAN
        assert g.get_time() == t0
        back = g.get_state(mmx.F_M0)
        assert np.array_equal(back, m, equal_nan=True)
    with pytest.raises(mmx.MmxError) as ei:
        g.max_torque()
    assert ei.value.code == -5
    # the world is usable again once the state is repaired
    m[1, 3, 5, 7] = 0.0
    m /= np.sqrt((m.astype(np.float64) ** 2).sum(axis=0, keepdims=True)).astype(np.float32)
    g.set_state(mmx.F_M0, m)
    st = g.step_rk45(method=mmx.DP45, fixed_dt=True, dt0=1e-13, nsteps=2)
    assert st["accepted"] == 2
    g.destroy()


def test_t_end_already_reached_and_elastic_step_clamp():
    """(a) a stepping call whose t_end is not ahead of the current time does nothing
    (no zero or backward step, dt untouched); (b) with elastodynamics on, adaptive stepping keeps
    dt at or below the elastic bound of the method (mmx.h, mmx_step_rk45) although the magnetic error is ~ 0."""
    spec = wl.make("c1", (32, 16, 1))
    g = mmx.World.from_spec(spec)
    st = g.step_rk45(method=mmx.DP45, tol=1e-5, t_end=1e-12)
    assert abs(st["t"] - 1e-12) < 1e-24
    m = g.get_state(mmx.F_M0)
    st2 = g.step_rk45(method=mmx.DP45, tol=1e-5, t_end=1e-12)
    assert st2["accepted"] == 0 and st2["rejected"] == 0 and st2["t"] == st["t"]
    st3 = g.step_rk45(method=mmx.DP45, tol=1e-5, t_end=0.5e-12)
    assert st3["accepted"] == 0 and st3["t"] == st["t"]
    assert np.array_equal(g.get_state(mmx.F_M0), m)
    st4 = g.step_rk45(method=mmx.DP45, tol=1e-5, t_end=1.5e-12)
    assert st4["accepted"] > 0 and abs(st4["t"] - 1.5e-12) < 1e-24
    g.destroy()
    spec = wl.make("c5", (64, 32, 1))
    spec.demag = False
    g = mmx.World.from_spec(spec)
    vmax = np.sqrt((2.5e11 + 2 * 1.5e11 + 4 * 1.0e11) / 3 / 6800.0)                    # [111] longitudinal: the fastest
    lim = 0.9 * mmx.rk_imag_stability_limit(mmx.DP45, 1e-6) / (1.3722 * vmax * np.sqrt(2) / 2e-9)
    assert lim < 0.5 * 2e-9 / np.sqrt(2.5e11 / 6800.0)                                 # (below the round-1 bound)
    st = g.step_rk45(method=mmx.DP45, tol=1e-3, dt0=1e-15, nsteps=60)
    assert st["accepted"] == 60 and st["dt"] <= lim * (1 + 1e-12), (st, lim)
    u = g.get_state(mmx.F_U)
    assert np.all(np.isfinite(u)) and np.abs(u).max() < 1e-9      # stable: no CFL blow-up
    st = g.step_rk45(method=mmx.DP45, tol=1e-3, dt0=1e-15, nsteps=40, dt_max=2e-14)
    assert st["dt"] <= 2e-14 * (1 + 1e-12)
    g.destroy()


def test_adaptive_t_end_and_reject_path():
    spec = wl.make("c1", (32, 16, 1))
    g, o = pair(spec)
    # a far too large first step must be rejected and leave the state untouched
    m0 = g.get_state(mmx.F_M0)
    st = g.step_rk45(method=mmx.DP45, tol=1e-7, dt0=5e-11, max_attempts=1)
    assert st["accepted"] == 0 and st["rejected"] == 1
    assert np.array_equal(g.get_state(mmx.F_M0), m0)
    st = g.step_rk45(method=mmx.DP45, tol=1e-5, t_end=2e-12)
    assert abs(st["t"] - 2e-12) < 1e-20
    o.run_dp45(tol=1e-5, t_end=2e-12)
    g.destroy()


def test_c1_relaxation_reaches_torque_threshold():
    """BASELINE config 1: RK45 relaxation until max torque < 1e-4 (T, i.e. |tau|/gamma; S26)."""
    spec = wl.c1()
    g = mmx.World.from_spec(spec)
    gamma = 1.7595e11
    e0 = g.energy()
    st = g.step_rk45(method=mmx.DP45, tol=1e-5, torque_stop=1e-4 * gamma, max_attempts=200000)
    assert st["max_torque"] < 1e-4 * gamma
    assert g.max_torque() < 1.5e-4 * gamma
    assert g.energy() < e0
    g.destroy()


@pytest.mark.parametrize("method,order", [(mmx.RK4, 4), (mmx.DP45, 5), (mmx.HEUN12, 2), (mmx.BS23, 3),
                                          (mmx.CK45, 5), (mmx.RKF45, 5)])
def test_macrospin_closed_form_every_tableau(method, order):
    """Table 2 methods on the damped macrospin: m_z(t) = tanh(alpha gamma B t/(1+alpha^2) + atanh m_z0)."""
    spec = wl.make("c1", (4, 2, 1))
    spec.demag = False
    spec.mat["A"][:] = 0.0
    spec.mat["alpha"][:] = 0.1
    spec.bext = (0.0, 0.0, 1.0)
    m = np.zeros_like(spec.m[0])
    m[0], m[2] = np.sqrt(1 - 0.25), 0.5
    spec.m = [m]
    g = mmx.World.from_spec(spec)
    gamma, alpha, B = 1.7595e11, 0.1, 1.0
    T = 2e-11
    n = {2: 4000, 3: 800, 4: 200, 5: 100}[order]
    g.step_rk45(method=method, fixed_dt=True, dt0=T / n, nsteps=n)
    mz = g.get_state(mmx.F_M0)[2]
    ref = np.tanh(alpha * gamma * B * T / (1 + alpha ** 2) + np.arctanh(0.5))
    assert np.abs(mz - ref).max() < 2e-5
    g.destroy()


def test_graph_replay_equals_plain_launches_and_follows_parameter_changes():
    """A step is replayed as a CUDA graph; the result must be bit-identical to plain launches, and a
    parameter change between two stepping calls must rebuild the graph (kernel arguments are baked in)."""
    spec = wl.make("c2", (32, 32, 1))
    dt = spec.integrator["dt"]
    a = mmx.World.from_spec(spec)
    b = mmx.World.from_spec(spec)
    b.graph_enable(False)
    for w in (a, b):
        w.step_rk45(method=mmx.DP45, fixed_dt=True, dt0=dt, nsteps=7)
    assert a.graph_info() > 0 and b.graph_info() == 0
    assert np.array_equal(a.get_state(mmx.F_M0), b.get_state(mmx.F_M0))
    for w in (a, b):
        w.set_bext((0.05, -0.3, 0.2))
    assert a.graph_info() == 0          # stale: rebuilt on the next stepping call
    for w in (a, b):
        w.step_rk45(method=mmx.DP45, fixed_dt=True, dt0=dt, nsteps=7)
        w.step_rk4(dt, 3)
    assert a.graph_info() > 0
    assert np.array_equal(a.get_state(mmx.F_M0), b.get_state(mmx.F_M0))
    a.destroy(); b.destroy()


def test_weak_ferromagnet_canting_is_an_equilibrium_of_the_cuda_path():
    """Eq.6 closed form, end to end on the GPU: with antiferromagnetic homogeneous exchange
    J = -4 A0/a^2 and d along z the state canted by atan(d/J) has no torque; the state canted the
    other way has (reading S32 fixes which one is which)."""
    Ms, A0, a, dz = 4.0e5, -4.0e-13, 0.35e-9, 2.0e5
    J = -4 * A0 / (a * a)
    delta0 = np.arctan(dz / J)
    scale = 1.7595e11 * J / Ms
    tq = {}
    for name, delta in (("right", delta0), ("wrong", -delta0)):
        spec = wl.make("c3", (8, 4, 1))
        spec.regions = None
        for k, v in spec.mat.items():
            spec.mat[k] = v[:, :1].copy()
        spec.mat["Ms"][:] = Ms
        spec.mat["Ku1"][:] = 0.0
        spec.mat["D"][:] = 0.0
        spec.J = (0.0, 0.0, 0.0)
        spec.demag = False
        spec.coupling.update(A0=A0, A12=0.0, D_inter=0.0, latcon=a, d_homo=(0.0, 0.0, dz))
        phi1 = 0.3
        for s, phi in ((0, phi1), (1, phi1 + np.pi + delta)):
            spec.m[s][:] = 0
            spec.m[s][0], spec.m[s][1] = np.cos(phi), np.sin(phi)
        g = mmx.World.from_spec(spec)
        tq[name] = g.max_torque()
        g.destroy()
    assert tq["right"] < 1e-5 * scale, tq      # fp32: cancellation of two ~33 T fields
    assert tq["wrong"] > 1e-3 * scale, tq


def test_c4_full_size_invariants_of_the_trajectory():
    """BASELINE config 4 at full size (256x256x64, the launch configuration bench.py times).  The
    oracle cannot follow a trajectory at this size, so properties that hold at any size are checked
    (P8, P9): |m| = 1 after every call, the total energy falls monotonically (alpha = 0.1 > 0), and the
    energy lost equals the dissipated power  P = (alpha Ms V / gamma) sum_c |tau_c|^2  integrated by
    the trapezoid rule over short stretches (dE/dt = -alpha gamma/(1+alpha^2) sum Ms V |m x B|^2)."""
    spec = wl.make("c4")
    assert tuple(spec.grid) == (256, 256, 64)
    g = mmx.World.from_spec(spec)
    Ms, alpha, gamma = float(spec.mat["Ms"][0, 0]), float(spec.mat["alpha"][0, 0]), 1.7595e11
    V = float(np.prod(spec.cell))

    def power():
        tau = g.eval_torque(0).astype(np.float64)
        return alpha * Ms * V / gamma * float((tau ** 2).sum())

    dt, n = 2e-14, 4
    E = [g.energy()]
    P = [power()]
    for _ in range(3):
        st = g.step_rk45(method=mmx.DP45, fixed_dt=True, dt0=dt, nsteps=n)
        assert st["accepted"] == n
        m = g.get_state(mmx.F_M0).astype(np.float64)
        np.testing.assert_allclose((m ** 2).sum(axis=0), 1.0, atol=2e-6)
        E.append(g.energy())
        P.append(power())
        assert E[-1] < E[-2]
        lost = E[-2] - E[-1]
        trapezoid = 0.5 * (P[-2] + P[-1]) * n * dt
        assert abs(lost - trapezoid) < 0.02 * lost, (lost, trapezoid)
    g.destroy()


def test_every_setter_invalidates_the_step_graph():
    """Kernel arguments are baked into the captured graph: each configuration call must make the next
    stepping call rebuild it (and a cleared DMI tensor must give the plain result again)."""
    spec = wl.make("c2", (32, 32, 1))
    dt = spec.integrator["dt"]
    g = mmx.World.from_spec(spec)
    ref = mmx.World.from_spec(spec)
    ref.graph_enable(False)

    def step_both():
        for w in (g, ref):
            w.step_rk45(method=mmx.DP45, fixed_dt=True, dt0=dt, nsteps=3)
        assert g.graph_info() > 0
        assert np.array_equal(g.get_state(mmx.F_M0), ref.get_state(mmx.F_M0))

    step_both()
    q = 1e-3 * np.arange(9, dtype=np.float64).reshape(3, 3)
    changes = [lambda w: w.set_bext((0.0, 0.2, -0.1)),
               lambda w: w.set_current((1e11, 0.0, 0.0)),
               lambda w: w.set_dmi_tensor(0, q),
               lambda w: w.set_dmi_tensor(0, None),
               lambda w: w.enable_demag(False),
               lambda w: w.enable_demag(True)]
    for change in changes:
        for w in (g, ref):
            change(w)
        assert g.graph_info() == 0
        step_both()
    g.destroy(); ref.destroy()


@pytest.mark.parametrize("method", [mmx.DP45, mmx.BS23, mmx.CK45])
def test_long_undamped_3d_elastic_run_at_the_step_bound(method):
    """adaptive stepping of an undamped 3-D elastic medium with a magnet that never limits the step.  dt
    sits on the automatic bound for 1e4 steps; every elastic mode lies inside the method's imaginary-axis stability
    interval, so the elastic energy of a rough (all wave numbers) initial displacement must not grow.  With the round-1
    bound 0.5 h / sqrt(C11/rho) imposed by hand the top modes of Dormand-Prince are outside (omega dt ~ 1.3 > 0.997) and the
    same run gains energy: the test has teeth.  The medium is periodic: there the discrete operator of Eq.7 is symmetric and
    the bound is sharp.  (With free surfaces the one-sided boundary stencils make the operator non-normal; the oracle's
    matrix on 8 x 6 x 4 cells has eigenvalues off the real axis and an undamped run grows at ~3e10 / s whatever dt is --
    DESIGN.md section 11; the paper's demonstration runs with Rayleigh damping.)"""
    spec = wl.make("c5", (16, 8, 8))
    spec.pbc = (1, 1, 1)
    spec.demag = False
    spec.mat["B1"][:] = 0.0
    spec.mat["B2"][:] = 0.0
    spec.elastic = dict(spec.elastic, traction=None)
    mx = np.zeros((3, 8, 8, 16), np.float32)
    mx[0] = 1.0
    spec.m = [mx, -mx]                                   # both sublattices on a cubic easy axis: no torque, ever
    rng = np.random.default_rng(5)
    u0 = (1e-13 * rng.standard_normal((3, 8, 8, 16))).astype(np.float32)
    vmax = np.sqrt((2.5e11 + 2 * 1.5e11 + 4 * 1.0e11) / 3 / 6800.0)
    lim = 0.9 * mmx.rk_imag_stability_limit(method, 1e-6) / (1.3722 * vmax * np.sqrt(sum(1.0 / c ** 2 for c in spec.cell)))

    def run(dt_max, nsteps):
        g = mmx.World.from_spec(spec)
        g.set_state(mmx.F_U, u0)
        g.set_state(mmx.F_V, np.zeros_like(u0))
        E0 = sum(g.elastic_energy())
        st = g.step_rk45(method=method, tol=1e-2, dt0=1e-16, nsteps=nsteps, dt_max=dt_max)
        E1 = sum(g.elastic_energy())
        ok = np.all(np.isfinite(g.get_state(mmx.F_U)))
        g.destroy()
        return st, E0, E1, ok

    st, E0, E1, ok = run(0.0, 10000)
    h = min(spec.cell)
    assert st["accepted"] == 10000 and ok
    assert abs(st["dt"] - lim) < 1e-9 * lim, (st, lim)          # the magnet is quiet: dt sits on the bound of mmx.h
    assert 0 < E1 <= E0 * (1 + 1e-2), (E0, E1)
    if method == mmx.DP45:
        st, E0, E1, ok = run(0.5 * h / np.sqrt(2.5e11 / 6800.0), 10000)
        assert (not ok) or E1 > 2 * E0, (E0, E1)
