"""GPU parity of every embedded pair of Table 2 against the oracle's tableaux (oracle/rk.py,
pinned by P14): fixed-step trajectories with the embedded error history -- the only thing that reads the
`e` rows of the library's tableaux -- the adaptive accept / reject sequence, and the torque stop."""
import numpy as np
import pytest

import paper_2411_18194_b200 as mmx
import workloads as wl
from oracle import rk as ork
from gpu_util import assert_estimates, TRAJ_TOL, max_dm, pair, pair_oracle
from test_gpu_configs import _estimate_floor

pytestmark = pytest.mark.gpu

PAIRS = [(mmx.HEUN12, ork.HEUN12), (mmx.BS23, ork.BS23), (mmx.CK45, ork.CK45), (mmx.RKF45, ork.RKF45),
         (mmx.DP45, ork.DP45)]
IDS = ["heun12", "bs23", "ck45", "rkf45", "dp45"]


@pytest.mark.parametrize("name,grid", [("c4", (16, 16, 8)), ("c2", (32, 32, 1))])
@pytest.mark.parametrize("method,tab", PAIRS, ids=IDS)
def test_fixed_step_trajectory_and_error_history(method, tab, name, grid):
    spec = wl.make(name, grid)
    dt, n = spec.integrator["dt"], 50
    g, o = pair(spec)
    floor = _estimate_floor(o, spec, dt, tab)
    st = g.step_rk45(method=method, fixed_dt=True, dt0=dt, nsteps=n)
    errs = o.step_embedded_fixed(dt, n, tab)
    assert st["accepted"] == n and st["rejected"] == 0
    d = max_dm(g.get_state(mmx.F_M0), o.m[0])
    assert d <= TRAJ_TOL, d
    hist = g.get_err_history(n)
    assert len(hist) == n
    assert_estimates(hist, errs, floor)
    assert min(errs) > 20 * floor or tab.order == 5     # the comparison is not vacuous for the low orders
    g.destroy()


@pytest.mark.parametrize("method,tab", PAIRS, ids=IDS)
def test_adaptive_sequence_per_method(method, tab):
    """From a first step 60x too large both sides must reject, shrink and recover identically: the
    accept / reject decision of every attempt, and the step size and the estimate of every attempt
    (dt follows err^(1/order): a relative error d of the fp32 estimate moves dt by d / order)."""
    spec = wl.make("c2", (32, 32, 1))
    g, o = pair(spec)
    tol, nat = 1e-5, 14
    first = o.run_adaptive(tab, tol=tol, nsteps=12)     # finds the step size the controller settles on
    o = pair_oracle(spec)
    dt0 = 60 * first["dt"]
    log = []
    o.run_adaptive(tab, tol=tol, dt0=dt0, max_attempts=nat, log=log)
    assert sum(1 for _, _, ok in log if not ok) >= 3 and sum(1 for _, _, ok in log if ok) >= 3, log
    dt = dt0
    for k, (dt_ref, err_ref, ok_ref) in enumerate(log):
        st = g.step_rk45(method=method, tol=tol, dt0=dt, max_attempts=1)
        ok = st["accepted"] == 1
        assert ok == ok_ref and st["accepted"] + st["rejected"] == 1, (k, st, log[k])
        assert abs(dt - dt_ref) <= 1e-3 * dt_ref, (k, dt, dt_ref)
        assert abs(st["last_err"] - err_ref) <= 2e-2 * err_ref + 1e-9, (k, st["last_err"], err_ref)
        dt = st["dt"]
    assert abs(g.get_time() - o.t) <= 1e-3 * o.t
    assert max_dm(g.get_state(mmx.F_M0), o.m[0]) <= TRAJ_TOL + o.max_torque() * abs(g.get_time() - o.t)
    g.destroy()


@pytest.mark.parametrize("method", [mmx.HEUN12, mmx.BS23, mmx.CK45, mmx.RKF45, mmx.DP45], ids=IDS)
def test_torque_stop_every_method(method):
    """A relaxation call whose only stopping criterion is torque_stop must end for every method -- also
    those without a reusable last stage, which test the first stage of the next attempt -- well before
    max_attempts, with the reported torque below the threshold and equal to the torque of the
    returned state."""
    spec = wl.make("c1", (32, 16, 1))
    g = mmx.World.from_spec(spec)
    gamma = 1.7595e11
    stop = 2e-2 * gamma
    st = g.step_rk45(method=method, tol=1e-4, torque_stop=stop, max_attempts=200000)
    assert st["accepted"] + st["rejected"] < 150000, st
    assert 0 < st["max_torque"] < stop, st
    tq = g.max_torque()
    assert abs(tq - st["max_torque"]) <= 1e-4 * tq, (tq, st)
    g.destroy()
