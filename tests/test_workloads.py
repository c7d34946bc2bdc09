"""The seeded input generators: shapes, determinism, unit norm, structure of each config."""
import numpy as np
import pytest

import workloads as wl
from oracle.world import World

SMALL = {"c1": (64, 16, 1), "c2": (32, 32, 1), "c3": (64, 32, 1), "c4": (16, 16, 8), "c5": (64, 16, 1)}


@pytest.mark.parametrize("name", list(SMALL))
def test_generators(name):
    a, b = wl.make(name, SMALL[name]), wl.make(name, SMALL[name])
    nx, ny, nz = SMALL[name]
    assert len(a.m) == a.S
    for ma, mb in zip(a.m, b.m):
        assert ma.dtype == np.float32 and ma.shape == (3, nz, ny, nx)
        assert np.array_equal(ma, mb)
        np.testing.assert_allclose((ma.astype(np.float64) ** 2).sum(axis=0), 1.0, atol=3e-7)
    if a.regions is not None:
        assert a.regions.dtype == np.uint16 and a.regions.max() < a.n_regions
        np.testing.assert_allclose(np.linalg.norm(a.mat["u"], axis=-1), 1.0, atol=1e-12)
        assert (a.mat["u"][..., 2] >= np.cos(np.deg2rad(10.0)) - 1e-12).all()
    if name == "c3":
        assert np.array_equal(a.m[1], -a.m[0]) and a.J[0] == 1e12
    if name == "c5":
        assert a.u is not None and a.elastic["traction"]["freq"] == 5e9


def test_full_size_shapes_match_baseline_json():
    assert wl.c1().grid == (64, 16, 1) and wl.c1().cell == (7.8125e-9, 7.8125e-9, 3e-9)
    s = wl.c3()
    assert s.grid == (1024, 128, 1) and s.n_regions == 1669 and s.S == 2


@pytest.mark.parametrize("name", list(SMALL))
def test_oracle_runs_every_config(name):
    w = World(wl.make(name, SMALL[name]))
    if name == "c1":
        w.step_rk4(1e-13, 3)
    else:
        errs = w.step_dp45_fixed(w.spec.integrator["dt"], 2)
        assert all(np.isfinite(errs)) and errs[0] > 0
    for m in w.m:
        np.testing.assert_allclose((m ** 2).sum(axis=0), 1.0, atol=1e-14)  # P8


def test_oracle_adaptive_controller():
    w = World(wl.make("c2", (16, 16, 1)))
    st = w.run_dp45(tol=1e-5, nsteps=8)
    assert st["accepted"] == 8 and st["dt"] > 0 and st["last_err"] <= 1e-5
    # a far too large first step must be rejected and shrunk
    w = World(wl.make("c2", (16, 16, 1)))
    st = w.run_dp45(tol=1e-5, dt0=1e-11, nsteps=2)
    assert st["rejected"] >= 1
