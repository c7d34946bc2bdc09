#!/usr/bin/env python
"""Writes the stored expected values of the full-size fixed-step parity protocol (reading
S29) -- calls ONLY `oracle/` and the seeded generators in `workloads/`, never the CUDA path.

    python tests/golden/make_trajectory_goldens.py c2 c3_rk4 c3_dp45 c5 c4      (any subset)

For every BASELINE.json config at its stated size the fp64 oracle integrates the protocol as written
(c2 DP45 dt = 2e-14 x 500; c3 RK4 and DP45 dt = 5e-15 x 400; c5 DP45 dt = 5e-15 x 400; c4 DP45
dt = 1e-13 x 100) and the final state is stored as float32 (rounding 6e-8, against the 1e-4
tolerance of the comparison) in tests/golden/traj_<case>.npz together with the per-step DP45 error
estimates (float64).  c2 / c3 / c5 store the whole grid; c4 (4.2 M cells, 50 MB per field) stores a sample of the
oracle's whole-grid result: the regular sub-lattice ix % 4 == 1, iy % 4 == 2, iz % 2 == 1 (1/32 of
the grid), the complete planes iz = 0 and iz = 63, and the complete rows iy in {0, 255} of plane
iz = 31 (flat cell indices stored beside the values).
The oracle needs about 0.35 s (c2), 2.7 s (c3), 1.3 s (c5) and 20 s (c4) per DP45 step on 8 cores,
which is why these runs are stored and not repeated inside the GPU tests; the GPU tests compare
the CUDA path against these files (tests/test_gpu_configs.py).
"""
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402
from oracle.world import World  # noqa: E402

CASES = {  # case -> (config, method, dt, nsteps)   SURVEY 8d "Fixed-step parity protocol"
    "c2": ("c2", "dp45", 2e-14, 500),
    "c3_rk4": ("c3", "rk4", 5e-15, 400),
    "c3_dp45": ("c3", "dp45", 5e-15, 400),
    "c5": ("c5", "dp45", 5e-15, 400),
    "c4": ("c4", "dp45", 1e-13, 100),
}


def c4_sample_mask(grid):
    nx, ny, nz = grid
    iz, iy, ix = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    mask = (ix % 4 == 1) & (iy % 4 == 2) & (iz % 2 == 1)
    mask |= (iz == 0) | (iz == nz - 1)
    mask |= (iz == nz // 2 - 1) & ((iy == 0) | (iy == ny - 1))
    return mask


def run(case):
    name, method, dt, nsteps = CASES[case]
    spec = wl.make(name)
    o = World(spec)
    t0 = time.time()
    errs = []
    chunk = 10
    for k in range(0, nsteps, chunk):
        n = min(chunk, nsteps - k)
        if method == "rk4":
            o.step_rk4(dt, n)
        else:
            errs += o.step_dp45_fixed(dt, n)
        print("%s: %d / %d steps, %.0f s" % (case, k + n, nsteps, time.time() - t0), flush=True)
    out = {"dt": np.float64(dt), "nsteps": np.int64(nsteps), "errs": np.asarray(errs, np.float64),
           "grid": np.asarray(spec.grid, np.int64)}
    if name == "c4":
        mask = c4_sample_mask(spec.grid)
        out["mask_index"] = np.flatnonzero(mask.ravel()).astype(np.int32)
        out["m0"] = o.m[0].reshape(3, -1)[:, out["mask_index"]].astype(np.float32)
    else:
        for s in range(spec.S):
            out["m%d" % s] = o.m[s].astype(np.float32)
        if spec.elastic is not None:
            out["u"] = o.u.astype(np.float64)   # tiny magnitudes (1e-13 m): keep fp64
            out["v"] = o.v.astype(np.float64)
    np.savez_compressed(os.path.join(HERE, "traj_%s.npz" % case), **out)
    print("%s: written, %.0f s" % (case, time.time() - t0), flush=True)


if __name__ == "__main__":
    for c in (sys.argv[1:] or list(CASES)):
        run(c)
