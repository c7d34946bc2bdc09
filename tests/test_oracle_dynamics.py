"""Pins for the torque and the integrators of the oracle (P7, P8, P9, P12, P13, P14)."""
from fractions import Fraction as Fr

import numpy as np

import workloads as wl
from oracle import fields as fl
from oracle import rk
from oracle.constants import GAMMA, MU_B, Q_E, T_ALL
from oracle.world import World


def _macrospin(alpha, B=1.0, m0=(0.6, 0.0, 0.8)):
    m = np.array(m0, np.float64).reshape(3, 1, 1, 1)
    spec = wl.WorldSpec(name="macro", grid=(1, 1, 1), cell=(1e-9,) * 3, demag=False,
                        mat=wl.make_mat(1, Ms=8e5, alpha=alpha), coupling=wl.default_coupling(),
                        bext=(0, 0, B), m=[m.astype(np.float32)])
    w = World(spec)
    w.m = [m.copy()]  # exact double start
    return w


def _macrospin_exact(alpha, B, m0, t):
    mz = np.tanh(alpha * GAMMA * B * t / (1 + alpha ** 2) + np.arctanh(m0[2]))
    phi = np.arctan2(m0[1], m0[0]) + GAMMA * B * t / (1 + alpha ** 2)
    s = np.sqrt(1 - mz * mz)
    return np.array([s * np.cos(phi), s * np.sin(phi), mz])


def test_P7_macrospin_precession_and_damping():
    for alpha in (0.0, 0.02, 0.5):
        w = _macrospin(alpha)
        w.step_rk4(1e-13, 500)
        want = _macrospin_exact(alpha, 1.0, (0.6, 0.0, 0.8), 500e-13)
        np.testing.assert_allclose(w.m[0].ravel(), want, atol=2e-9)
        assert abs(np.linalg.norm(w.m[0].ravel()) - 1) < 1e-15  # P8


def _order_conditions(a, c, order):
    """Rooted-tree order conditions of an explicit Runge-Kutta method up to `order` <= 5 (Butcher):
    list of (elementary-weight vector Phi, 1/gamma); weights b reach the order iff b.Phi = 1/gamma."""
    one = np.ones_like(c)
    Ac = a @ c
    trees = {1: [(one, 1.0)],
             2: [(c, 1 / 2)],
             3: [(c ** 2, 1 / 3), (Ac, 1 / 6)],
             4: [(c ** 3, 1 / 4), (c * Ac, 1 / 8), (a @ c ** 2, 1 / 12), (a @ Ac, 1 / 24)],
             5: [(c ** 4, 1 / 5), (c ** 2 * Ac, 1 / 10), (c * (a @ c ** 2), 1 / 15), (c * (a @ Ac), 1 / 30),
                 (Ac * Ac, 1 / 20), (a @ c ** 3, 1 / 20), (a @ (c * Ac), 1 / 40), (a @ (a @ c ** 2), 1 / 60),
                 (a @ (a @ Ac), 1 / 120)]}
    return [t for p in range(1, order + 1) for t in trees[p]]


def _residual(tab_a, c, wts, order):
    return max(abs(float(wts @ phi) - g) for phi, g in _order_conditions(tab_a, c, order))


def test_P14_tableau_identities():
    """Every pair of Table 2 + RK4: row sums, sum b = sum b* = 1, and the rooted-tree
    order conditions: the propagated weights b satisfy all conditions up to the convergence order
    the table prints and NOT the next order; the embedded weights b* = b - e those up to the
    error-estimate order it prints, and not the next.  A wrong sign, a swapped entry or a dropped
    term in any a_ij, b_j or e_j fails one of these."""
    cases = [(rk.RK4, 4, None), (rk.HEUN12, 2, 1), (rk.BS23, 3, 2), (rk.CK45, 5, 4), (rk.RKF45, 5, 4), (rk.DP45, 5, 4)]
    for tab, p, pe in cases:
        s = tab.stages
        a = np.zeros((s, s))
        for i, row in enumerate(tab.a):
            a[i, :len(row)] = row
        c = np.array(tab.c)
        b = np.array(tab.b)
        assert tab.order == p
        assert abs(b.sum() - 1) < 1e-15
        np.testing.assert_allclose(a.sum(axis=1), c, atol=1e-15)
        assert np.all(np.triu(a) == 0)                      # explicit
        assert _residual(a, c, b, p) < 1e-14, tab
        if p < 5:
            assert _residual(a, c, b, p + 1) > 1e-3, tab    # and not more
        if pe is None:
            assert tab.e is None
            continue
        bs = b - np.array(tab.e)
        assert abs(bs.sum() - 1) < 1e-15
        assert _residual(a, c, bs, pe) < 1e-14, tab
        assert _residual(a, c, bs, pe + 1) > 1e-4, tab
        if tab.fsal:                                         # last row of a equals b
            np.testing.assert_allclose(a[s - 1, :s - 1], b[:s - 1], atol=0)
            assert b[s - 1] == 0
    # e = b - b*, b* the embedded 4th-order weights of the Dormand-Prince pair (ref [55])
    bstar = [Fr(5179, 57600), 0, Fr(7571, 16695), Fr(393, 640), Fr(-92097, 339200), Fr(187, 2100), Fr(1, 40)]
    for bj, bs_, ej in zip(rk.DP45.b, bstar, rk.DP45.e):
        assert abs((bj - float(bs_)) - ej) < 1e-16
    assert rk.EMBEDDED["ck45"][0] is rk.CK45 and rk.EMBEDDED["ck45"][1] == 4


TABLEAUX = {"rk4": rk.RK4, "heun12": rk.HEUN12, "bs23": rk.BS23, "ck45": rk.CK45, "rkf45": rk.RKF45, "dp45": rk.DP45}


def _final_error(method, dt, T=2e-11, alpha=0.3):
    w = _macrospin(alpha, B=2.0)
    n = int(round(T / dt))
    if method == "rk4":
        w.step_rk4(dt, n)
    else:
        w.step_embedded_fixed(dt, n, TABLEAUX[method])
    return np.abs(w.m[0].ravel() - _macrospin_exact(alpha, 2.0, (0.6, 0.0, 0.8), n * dt)).max()


def test_P14_observed_orders():
    """Table 2: observed global convergence order of every method against the closed-form
    macrospin, and the dt-scaling of the embedded error estimate: a pair whose embedded solution has
    order q gives an estimate ~ dt^(q+1)."""
    for method, p, q, dts in (("rk4", 4, None, (1e-12, 0.5e-12)), ("heun12", 2, 1, (2e-13, 1e-13)),
                              ("bs23", 3, 2, (4e-13, 2e-13)), ("ck45", 5, 4, (1e-12, 0.5e-12)),
                              ("rkf45", 5, 4, (1e-12, 0.5e-12)), ("dp45", 5, 4, (1e-12, 0.5e-12))):
        e1, e2 = _final_error(method, dts[0]), _final_error(method, dts[1])
        assert p - 0.4 < np.log2(e1 / e2) < p + 0.5, (method, np.log2(e1 / e2))
        if q is None:
            continue
        est = []
        for dt in dts:
            w = _macrospin(0.3, B=2.0)
            est.append(w.step_embedded_fixed(dt, 1, TABLEAUX[method])[0])
        assert q + 0.6 < np.log2(est[0] / est[1]) < q + 1.4, (method, np.log2(est[0] / est[1]))


def test_P14_adaptive_run_meets_its_tolerance():
    """Controller reading S21 on the closed-form macrospin with every embedded pair: the adaptive run
    lands on t_end exactly, rejects at least once from a far too large first step, and its global
    error stays within a small multiple of tol (a wrong sign in an e row makes the estimate useless:
    either no step is ever rejected or the error is orders of magnitude above tol)."""
    for name in ("heun12", "bs23", "ck45", "rkf45", "dp45"):
        w = _macrospin(0.3, B=2.0)
        tol = 1e-6
        log = []
        st = w.run_adaptive(TABLEAUX[name], tol=tol, dt0=2e-11, t_end=2e-11, log=log)
        assert abs(st["t"] - 2e-11) < 1e-24 and st["rejected"] >= 1, (name, st)
        err = np.abs(w.m[0].ravel() - _macrospin_exact(0.3, 2.0, (0.6, 0.0, 0.8), 2e-11)).max()
        assert err < 30 * tol * max(1, st["accepted"] / 10), (name, err, st)
        assert all(e <= tol for _, e, ok in log if ok) and all(e > tol for _, e, ok in log if not ok)


def _small_world(alpha, seed=21, S=1, J=(0, 0, 0)):
    rng = np.random.default_rng(seed)
    grid = (6, 4, 2)
    spec = wl.WorldSpec(
        name="small", grid=grid, cell=(3e-9, 3e-9, 2e-9), S=S,
        mat=wl.make_mat(S, Ms=8e5, A=1.3e-11, alpha=alpha, Ku1=5e4, D=1e-3, Kc1=2e4),
        coupling=wl.default_coupling(A0=-4e-15, A12=-1e-12, D_inter=3e-4, bc="open"), bext=(0.0, 0.01, 0.05), J=J,   # open: the BC of the pair energy
        m=[wl.smoothed_random_unit(rng, grid, 2.0) for _ in range(S)])
    return World(spec, demag_mode="direct")


def test_P9_energy_conservation_and_dissipation():
    """alpha = 0: total energy constant to integrator order.  alpha > 0:
    dE/dt = -alpha gamma/(1+alpha^2) sum Ms V |m x B|^2."""
    drift = []
    for dt in (4e-14, 2e-14):
        w = _small_world(0.0, S=2)
        E0 = w.energy()
        w.step_rk4(dt, int(round(8e-13 / dt)))
        drift.append(abs(w.energy() - E0) / abs(E0))
    assert drift[0] < 1e-6 and drift[1] < drift[0] / 8
    alpha = 0.2
    w = _small_world(alpha, S=2)
    rate = 0.0
    for s in range(2):
        mxB = fl.cross(w.m[s], w.heff(s))
        rate += -alpha * GAMMA / (1 + alpha ** 2) * float((w.p[s]["Ms"][None] * mxB ** 2).sum()) * w.V
    E0 = w.energy()
    dt = 1e-15
    w.step_rk4(dt, 1)
    E1 = w.energy()
    w.step_rk4(dt, 1)
    E2 = w.energy()
    num = (-3 * E0 + 4 * E1 - E2) / (2 * dt)
    assert rate < 0 and abs(num - rate) < 1e-4 * abs(rate)


def test_P12_antiferromagnetic_resonance():
    """Two antiparallel macrospins, small tilt: omega = gamma sqrt(B_A (2 B_E + B_A)),
    B_E = -4 A0/(Ms a^2), B_A = 2 Ku/Ms  -> 128.3 GHz for the c3 numbers."""
    Ms, A0, a, Ku = 4.0e5, -4.0e-13, 0.35e-9, 6.4e4
    BE, BA = -4 * A0 / (Ms * a * a), 2 * Ku / Ms
    f_want = GAMMA * np.sqrt(BA * (2 * BE + BA)) / (2 * np.pi)
    assert abs(f_want - 128.3e9) < 0.1e9
    m1 = np.array([1e-4, 0, 1.0]).reshape(3, 1, 1, 1)
    m2 = np.array([0, 0, -1.0]).reshape(3, 1, 1, 1)
    spec = wl.WorldSpec(name="afmr", grid=(1, 1, 1), cell=(2e-9,) * 3, S=2, demag=False,
                        mat=wl.make_mat(2, Ms=Ms, Ku1=Ku, alpha=0.0),
                        coupling=wl.default_coupling(A0=A0, latcon=a),
                        m=[m1.astype(np.float32), m2.astype(np.float32)])
    w = World(spec)
    w.m = [m1 / np.linalg.norm(m1), m2.copy()]
    dt, n = 1e-14, 2400
    xs = []
    for _ in range(n):
        w.step_dp45_fixed(dt, 1)
        xs.append(w.m[0][0, 0, 0, 0] - w.m[1][0, 0, 0, 0] * 0)  # m1_x
    xs = np.array(xs)
    t = dt * np.arange(1, n + 1)
    zc = np.nonzero(np.sign(xs[1:]) != np.sign(xs[:-1]))[0]
    tz = t[zc] - xs[zc] * dt / (xs[zc + 1] - xs[zc])
    # m1_x(t) = sum of the two degenerate circular modes: pure cos(omega t) -> half periods
    f_got = 0.5 / np.mean(np.diff(tz))
    assert abs(f_got - f_want) < 2e-3 * f_want


def test_P21_weak_ferromagnet_canting_angle():
    """Two macrospins with antiferromagnetic homogeneous exchange eps = J m1.m2 (J = -4 A0/a^2 > 0) and
    the homogeneous DMI of Eq.6 with d along z, eps_D = d z.(m1 x m2): for in-plane spins with
    Delta = phi2 - phi1 the energy is J cos(Delta) + d sin(Delta), stationary where tan(Delta) = d/J
    and minimal at Delta = pi + atan(d/J) (weak-ferromagnetic canting).  The oracle's torque must
    vanish exactly there, its energy must be a minimum there, and the state canted the other way
    must feel a torque.  (A relaxation run is not used: without anisotropy the out-of-plane mode of
    this pair relaxes on a nanosecond scale.)"""
    Ms, A0, a, dz = 4.0e5, -4.0e-13, 0.35e-9, 2.0e5
    J = -4 * A0 / (a * a)
    delta0 = np.arctan(dz / J)

    def world(delta, phi1=0.3):
        m1 = np.array([np.cos(phi1), np.sin(phi1), 0.0]).reshape(3, 1, 1, 1)
        m2 = np.array([np.cos(phi1 + np.pi + delta), np.sin(phi1 + np.pi + delta), 0.0]).reshape(3, 1, 1, 1)
        spec = wl.WorldSpec(name="wfm", grid=(1, 1, 1), cell=(2e-9,) * 3, S=2, demag=False,
                            mat=wl.make_mat(2, Ms=Ms, alpha=0.5),
                            coupling=wl.default_coupling(A0=A0, latcon=a, d_homo=(0.0, 0.0, dz)),
                            m=[m1.astype(np.float32), m2.astype(np.float32)])
        w = World(spec)
        w.m = [m1, m2]
        return w

    scale = GAMMA * J / Ms                      # torque scale of the exchange field, 1/s
    assert world(delta0).max_torque() < 1e-12 * scale
    assert world(-delta0).max_torque() > 1e-3 * scale          # wrong chirality is not an equilibrium
    assert world(0.0).max_torque() > 1e-3 * scale              # neither is the collinear state
    e0 = world(delta0).energy()
    for eps in (1e-3, -1e-3):
        assert world(delta0 + eps).energy() > e0
    V = (2e-9) ** 3
    assert abs(e0 - V * (J * np.cos(np.pi + delta0) + dz * np.sin(np.pi + delta0))) < 1e-9 * abs(e0)


def test_P13_zhang_li():
    """alpha = xi: the Zhang-Li torque reduces to the transverse part of (u.grad)m, with
    u = mu_B P j/(e Ms (1+xi^2)) (71.6 m/s for the c3 numbers); a wall translates rigidly at -u."""
    Ms, P, xi, j = 4.0e5, 0.5, 0.1, 1e12
    u = MU_B * P * j / (Q_E * Ms * (1 + xi * xi))
    assert abs(u - 71.6) < 0.1
    nx, h = 160, 2e-9
    A, Ku = 1.0e-11, 6.4e4
    spec = wl.WorldSpec(name="zl", grid=(nx, 1, 1), cell=(h, h, h), demag=False,
                        mat=wl.make_mat(1, Ms=Ms, A=A, Ku1=Ku, alpha=xi, pol=P, xi=xi),
                        coupling=wl.default_coupling(), J=(j, 0, 0),
                        m=[wl.neel_wall((nx, 1, 1), (h, h, h), 0.5 * nx * h, np.sqrt(A / Ku))])
    w = World(spec)
    p = w.p[0]
    tzl = fl.zhang_li_torque(w.m[0], p["Ms"], p["alpha"], p["pol"], p["xi"], w.J, w.cell, w.pbc)
    a = fl.directional_derivative(w.m[0], np.array([u, 0, 0]).reshape(3, 1, 1, 1) * np.ones_like(w.m[0]),
                                  p["Ms"], w.cell, w.pbc)
    a_perp = a - (a * w.m[0]).sum(axis=0)[None] * w.m[0]
    np.testing.assert_allclose(tzl, a_perp, atol=1e-9 * np.abs(a).max())
    # dynamic: wall centre q from integral of m_z (m_z = tanh((x-q)/D)  =>  sum m_z h = L - 2q)
    w.spec.J, w.J = (0, 0, 0), (0, 0, 0)
    w.step_rk4(5e-14, 400)  # settle the analytic profile on the lattice (alpha = 0.1: partly)
    w.J = (j, 0, 0)
    q0 = 0.5 * (nx * h - w.m[0][2].sum() * h)
    T = 4e-11
    w.step_rk4(5e-14, int(round(T / 5e-14)))
    q1 = 0.5 * (nx * h - w.m[0][2].sum() * h)
    assert abs((q1 - q0) / T + u) < 0.02 * u


def test_P23_slonczewski_macrospin_closed_form():
    """P23 (pins reading S37: prefactor hbar/(e Ms d), eps(Lambda = 1) = P/2, the alpha mixing and the role of eps').
    Macrospin in B z^ with the fixed layer along z^ and Lambda = 1: from the Gilbert form
    dm/dt = -gamma m x B + alpha m x dm/dt + gamma beta [eps m x (z x m) - eps' m x z] one gets, exactly,
        m_z(t) = tanh( gamma (alpha (B + beta eps') + beta eps) t / (1 + alpha^2) + atanh m_z(0) )
        dphi/dt = gamma ((B + beta eps') - alpha beta eps) / (1 + alpha^2)
    so the damping-like torque cancels the Gilbert damping at beta eps = -alpha (B + beta eps') (switching current)."""
    from oracle.constants import HBAR, Q_E
    Ms, alpha, P, d, B, epsp = 8.0e5, 0.02, 0.4, 2e-9, 0.2, 0.05
    spec = wl.make("c1", (1, 1, 1))
    spec.demag = False
    spec.mat["alpha"][:] = alpha
    spec.mat["pol"][:] = P
    spec.mat["A"][:] = 0.0
    spec.bext = (0.0, 0.0, B)
    m0 = np.array([np.sin(0.6), 0.0, np.cos(0.6)])
    for jz in (-3.0e11, +2.0e11, 0.0):
        s2 = spec.copy()
        s2.m = [m0.reshape(3, 1, 1, 1).astype(np.float32)]
        s2.coupling["slonczewski"] = dict(jz=jz, mp=(0.0, 0.0, 1.0), **{"lambda": 1.0}, eps_prime=epsp, thickness=d)
        o = World(s2)
        beta = HBAR * jz / (Q_E * Ms * d)
        eps = P / 2.0
        rate = GAMMA * (alpha * (B + beta * epsp) + beta * eps) / (1 + alpha ** 2)
        omega = GAMMA * ((B + beta * epsp) - alpha * beta * eps) / (1 + alpha ** 2)
        dt, n = 2e-14, 2000
        o.step_rk4(dt, n)
        t = n * dt
        mz = np.tanh(rate * t + np.arctanh(float(o.spec.m[0][2, 0, 0, 0])))
        phi = np.arctan2(o.m[0][1, 0, 0, 0], o.m[0][0, 0, 0, 0])
        assert abs(o.m[0][2, 0, 0, 0] - mz) < 1e-7, (jz, o.m[0][2, 0, 0, 0], mz)
        assert abs(np.angle(np.exp(1j * (phi - omega * t)))) < 1e-6, (jz, phi, omega * t)
    # the damping-like torque exactly compensates the Gilbert damping at the switching current
    jc = -alpha * B * Q_E * Ms * d / (HBAR * (P / 2.0 + alpha * epsp))
    s2 = spec.copy()
    s2.m = [m0.reshape(3, 1, 1, 1).astype(np.float32)]
    s2.coupling["slonczewski"] = dict(jz=jc, mp=(0.0, 0.0, 1.0), **{"lambda": 1.0}, eps_prime=epsp, thickness=d)
    o = World(s2)
    assert abs(o.torque(0)[2, 0, 0, 0]) < 1e-6 * GAMMA * B


def test_slonczewski_angular_dependence():
    """eps(m . m_p) of reading S37 at its three closed-form points: P/2 (parallel), P Lambda^2/2 (antiparallel),
    P Lambda^2/(Lambda^2 + 1) (perpendicular) -- read off the torque on a spin perpendicular to m_p, and the
    vanishing torque at m = +-m_p."""
    from oracle import fields as fl
    from oracle.constants import HBAR, Q_E
    Ms, P, lam, d, jz = 5.0e5, 0.6, 1.7, 3e-9, 1e11
    one = lambda v: np.asarray(v, float).reshape(3, 1, 1, 1)
    arr = lambda x: np.full((1, 1, 1), float(x))
    beta = HBAR * jz / (Q_E * Ms * d)
    tau = fl.slonczewski_torque(one((1, 0, 0)), arr(Ms), arr(0.0), arr(GAMMA), arr(P), jz, (0, 0, 1), lam, 0.0, d)
    # m = x^, m_p = z^, alpha = 0: tau = gamma beta eps (z - 0) = gamma beta eps z^, eps = P L^2/(L^2+1)
    np.testing.assert_allclose(tau[:, 0, 0, 0], [0, 0, GAMMA * beta * P * lam ** 2 / (lam ** 2 + 1)], rtol=1e-12, atol=1e-3)
    for sgn in (+1, -1):
        tau = fl.slonczewski_torque(one((0, 0, sgn)), arr(Ms), arr(0.1), arr(GAMMA), arr(P), jz, (0, 0, 1), lam, 0.3, d)
        assert np.abs(tau).max() == 0.0
    th = 1e-6   # nearly (anti)parallel: |tau| / sin(theta) -> gamma beta eps(+-1)
    for sgn, eps in ((+1, P / 2), (-1, P * lam ** 2 / 2)):
        m = one((np.sin(th), 0, sgn * np.cos(th)))
        tau = fl.slonczewski_torque(m, arr(Ms), arr(0.0), arr(GAMMA), arr(P), jz, (0, 0, 1), lam, 0.0, d)
        np.testing.assert_allclose(np.sqrt((tau ** 2).sum()) / np.sin(th), GAMMA * abs(beta) * eps, rtol=1e-5)


def test_P24_relaxation_closed_form_and_energy_descent():
    """P24 (pins reading S39).  Damping-only torque of a macrospin in B z^: the azimuth stays put and
    m_z(t) = tanh(alpha gamma B t/(1 + alpha^2) + atanh m_z(0)) -- the damping part of P7 with the precession gone.
    On an exchange + anisotropy + demag film the relaxation lowers the energy monotonically and ends in a state
    whose FULL LLG torque is below the same threshold times sqrt(1 + alpha^2)/alpha (|m x B| is common to both)."""
    alpha, B = 0.3, 0.7
    w = _macrospin(alpha, B, (0.48, 0.36, 0.8))
    w.precession = False
    dt, n = 1e-13, 300
    w.step_rk4(dt, n)
    mz = np.tanh(alpha * GAMMA * B * n * dt / (1 + alpha ** 2) + np.arctanh(0.8))
    got = w.m[0][:, 0, 0, 0]
    assert abs(got[2] - mz) < 1e-9
    assert abs(np.arctan2(got[1], got[0]) - np.arctan2(0.36, 0.48)) < 1e-12
    spec = wl.make("c2", (16, 16, 1))
    o = World(spec)
    E = [o.energy(T_ALL)]
    o.precession = False
    for _ in range(40):
        o.run_adaptive(rk.DP45, 1e-5, nsteps=3)
        E.append(o.energy(T_ALL))
    assert all(b <= a + 1e-9 * abs(a) for a, b in zip(E, E[1:]))
    o.precession = True
    o2 = World(spec)
    a = float(spec.mat["alpha"][0, 0])
    stop = 1e-3 * GAMMA   # 1 mT in torque units
    st = o2.relax(stop)
    assert st["accepted"] > 0 and o2.t == 0.0 and o2.precession
    assert o2.max_torque() < stop * np.sqrt(1 + a * a) / a * 1.0001
    assert o2.energy(T_ALL) < E[0]


def _cubic_macrospin(m, Kc1, Ms, c1, c2, alpha=0.0):
    mat = wl.make_mat(1, Ms=Ms, Kc1=Kc1, alpha=alpha)
    mat["c1"][:] = c1
    mat["c2"][:] = c2
    spec = wl.WorldSpec(name="cubic", grid=(1, 1, 1), cell=(2e-9, 3e-9, 4e-9), S=1, demag=False, mat=mat,
                        coupling=wl.default_coupling(), m=[np.asarray(m, np.float32).reshape(3, 1, 1, 1)])
    w = World(spec)
    w.m = [np.asarray(m, float).reshape(3, 1, 1, 1) / np.linalg.norm(m)]
    return w


def test_P28_cubic_anisotropy_energy_closed_forms():
    """P:L116 (cubic anisotropy "implemented in the same way as in mumax3"): the first-order cubic energy density is
    K_c1 (a1^2 a2^2 + a2^2 a3^2 + a3^2 a1^2), a_i the direction cosines on the cubic axes.  Its textbook values --
    0 along <100>, K_c1/4 along <110>, K_c1/3 along <111> -- are typed in here as numbers; the oracle's energy is
    -1/4 sum Ms V m.B_cubic, so these fix the product (energy factor 1/4) x (field factor 2 K_c1/Ms), and P10 (field =
    energy gradient, which fixes their ratio) then fixes each.  The axes are a rotated frame, so a slip in c3 = c1 x c2 or
    in the index pattern (a_i times the OTHER two squares) shows as well."""
    from oracle.world import T_ANIS_C
    Kc1, Ms = 1.0e4, 4.0e5
    V = 2e-9 * 3e-9 * 4e-9
    c1 = np.array([2.0, 1.0, 2.0]) / 3.0
    c2 = np.array([1.0, 2.0, -2.0]) / 3.0
    c3 = np.cross(c1, c2)
    for m, want in ((c1, 0.0), (c3, 0.0), (c1 + c2, Kc1 * V / 4), (c2 - c3, Kc1 * V / 4), (c1 + c2 + c3, Kc1 * V / 3),
                    (c1 - c2 + c3, Kc1 * V / 3)):
        E = _cubic_macrospin(m, Kc1, Ms, c1, c2).energy(T_ANIS_C)
        assert abs(E - want) < 1e-12 * Kc1 * V, (m, E, want)
    # one generic direction: cosines (0.6, 0, 0.8) -> K (0.36 * 0.64) = 0.2304 K
    E = _cubic_macrospin(0.6 * c1 + 0.8 * c3, Kc1, Ms, c1, c2).energy(T_ANIS_C)
    assert abs(E - 0.2304 * Kc1 * V) < 1e-12 * Kc1 * V


def test_P28_cubic_anisotropy_precession_frequency():
    """The dynamic pin of the field's prefactor (like P12 for the uniaxial term): for K_c1 > 0 the cubic axes are easy, and a
    spin tilted by a small angle from c1 precesses about it in the anisotropy field B_A = 2 K_c1 / Ms at omega = gamma B_A
    (alpha = 0) -- the curvature of K_c1 a1^2 (a2^2 + a3^2) at the axis.  A factor 2 or 1/2 in fields.cubic moves the
    frequency by that factor; the energy-based pins above cannot see a slip made in both the field and the 1/4."""
    Kc1, Ms = 6.0e4, 4.0e5
    c1 = np.array([2.0, 1.0, 2.0]) / 3.0
    c2 = np.array([1.0, 2.0, -2.0]) / 3.0
    f_want = GAMMA * (2 * Kc1 / Ms) / (2 * np.pi)          # 8.40 GHz
    assert abs(f_want - 8.4012e9) < 1e6
    w = _cubic_macrospin(c1 + 1e-3 * c2, Kc1, Ms, c1, c2)
    dt, n = 2e-13, 1500                                     # 2.5 periods
    xs = []
    for _ in range(n):
        w.step_dp45_fixed(dt, 1)
        xs.append(float((w.m[0][:, 0, 0, 0] * c2).sum()))  # component along c2: cos(omega t)
    xs = np.array(xs)
    t = dt * np.arange(1, n + 1)
    zc = np.nonzero(np.sign(xs[1:]) != np.sign(xs[:-1]))[0]
    tz = t[zc] - xs[zc] * dt / (xs[zc + 1] - xs[zc])
    assert len(tz) >= 4
    f_got = 0.5 / np.mean(np.diff(tz))
    assert abs(f_got - f_want) < 2e-3 * f_want, (f_got, f_want)
