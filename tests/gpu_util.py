"""Helpers of the GPU parity tests: build the CUDA world and the oracle world from the same
seeded WorldSpec, and the error measures of BASELINE.json's north_star (readings S27)."""
import numpy as np

import paper_2411_18194_b200 as mmx
from oracle.world import World as OracleWorld

FIELD_TOL = 1e-5   # per-cell relative field error (north_star)
TRAJ_TOL = 1e-4    # max |delta m| after a fixed-step trajectory (north_star)


def field_err(got, ref):
    """max_c |dB_c|_2 / max(|B_c|_2, 0.1 RMS|B|)   (reading S27)."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    d = np.sqrt(((got - ref) ** 2).sum(axis=0))
    n = np.sqrt((ref ** 2).sum(axis=0))
    rms = np.sqrt((n ** 2).mean())
    if rms == 0.0:
        return float(d.max())
    return float((d / np.maximum(n, 0.1 * rms)).max())


def torque_err_conditioned(got, ref, B, alpha, gamma):
    """Torque parity for states near equilibrium.  There tau = -gamma' [m x B +
    alpha m x (m x B)] is a small remainder of a large field nearly parallel to m (33 T of
    inter-sublattice exchange in c3 / c5), so an admissible field error of FIELD_TOL |B| already moves
    the torque by gamma' (1 + alpha) FIELD_TOL |B| -- far more than FIELD_TOL |tau|.  The criterion is
    the north_star field tolerance propagated through Eq.2:
        max_c |d tau_c| / (gamma' (1 + alpha) max(|B_c|, 0.1 RMS|B|)),   gamma' = gamma / (1 + alpha^2)."""
    d = np.sqrt(((np.asarray(got, np.float64) - ref) ** 2).sum(axis=0))
    n = np.sqrt((np.asarray(B, np.float64) ** 2).sum(axis=0))
    rms = np.sqrt((n ** 2).mean())
    scale = gamma / (1 + alpha ** 2) * (1 + alpha) * np.maximum(n, 0.1 * rms)
    return float((d / scale).max())


EST_RTOL = 1e-3   # embedded error estimate of a fixed-step run, relative (SURVEY 8d "rel. 1e-3")


def assert_estimates(got, ref, floor):
    """Error-estimate history of a fixed-step run against the oracle's: |got - ref| <= EST_RTOL ref + floor, floor the
    absolute fp32 rounding floor of the estimate derived in DESIGN.md section 10 (passed in by the test).  Wherever the
    estimate is >= 100 floor this is a relative comparison at 1e-3 (+ at most 1e-2 from the floor); floor-limited entries
    are held by the floor alone.  On failure the message carries the measured ratio."""
    got, ref = np.asarray(got, np.float64), np.asarray(ref, np.float64)
    assert got.shape == ref.shape
    d = np.abs(got - ref)
    worst = float(((d - floor) / np.maximum(ref, 1e-300)).max())
    assert (d <= EST_RTOL * ref + floor).all(), "estimate history: max (|d| - floor) / est = %.3g, bar %.1g" % (worst, EST_RTOL)


def max_dm(a, b):
    return float(np.abs(np.asarray(a, np.float64) - np.asarray(b, np.float64)).max())


def pair(spec, demag_mode="fft", demag=None):
    """(cuda world, oracle world) for one spec."""
    if demag is not None:
        spec = spec.copy()
        spec.demag = demag
    g = mmx.World.from_spec(spec)
    o = OracleWorld(spec, demag_mode=demag_mode)
    return g, o


def pair_oracle(spec, demag_mode="fft"):
    """A fresh oracle world alone (no CUDA world)."""
    return OracleWorld(spec, demag_mode=demag_mode)


def gpu_m(g, S):
    return [g.get_state(mmx.F_M[s]) for s in range(S)]
