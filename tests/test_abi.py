"""Host-side checks that need no GPU: the C-ABI library loads and exports every symbol that
include/mmx.h declares; the host-only entry points (Newell tensor, kernel spectrum) agree with
the oracle; argument errors are reported, and world creation fails loudly without a device."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_2411_18194_b200 as mmx
from paper_2411_18194_b200 import binding, build
from oracle import demag as odm
from oracle import newell as onw
from oracle.constants import MU0

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return mmx.load()


def test_every_declared_symbol_is_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "mmx.h")).read()
    declared = set(re.findall(r"^(?:int|const char\*)\s+(mmx_[a-z0-9_]+)\s*\(", hdr, flags=re.M))
    assert len(declared) >= 25
    raw = ctypes.CDLL(binding.LIB_PATH)
    for name in declared:
        assert hasattr(raw, name), name
    assert declared == set(binding.PROTOTYPES), declared ^ set(binding.PROTOTYPES)


def test_struct_layouts_match_header():
    assert ctypes.sizeof(binding.Material) == 20 * 8
    assert ctypes.sizeof(binding.Coupling) == 9 * 8
    assert ctypes.sizeof(binding.RkOpts) == 64 and ctypes.sizeof(binding.RkStats) == 56
    assert ctypes.sizeof(binding.Elastic) == 88


def test_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(mmx.MmxError) as e:
        mmx.World((4, 4, 1), (1e-9, 1e-9, 1e-9))
    assert e.value.code == -3 and "no CPU fallback" in str(e.value)


def test_argument_errors(lib):
    dims = (ctypes.c_longlong * 5)()
    I3, D3 = ctypes.c_int * 3, ctypes.c_double * 3
    rc = lib.mmx_kernel_spectrum_host(I3(6, 4, 1), D3(1e-9, 1e-9, 1e-9), I3(1, 0, 0), 32.0, None, 0, dims)
    assert rc == -1 and b"power of two" in lib.mmx_last_error()
    rc = lib.mmx_kernel_spectrum_host(I3(4096, 4, 1), D3(1e-9, 1e-9, 1e-9), I3(0, 0, 0), 32.0, None, 0, dims)
    assert rc == -1
    assert lib.mmx_world_destroy(None) == 0
    assert lib.mmx_step_rk4(None, 1e-13, 1) == -1
    # entry points added after the first path: NULL world is an argument error, never a crash
    q9 = (ctypes.c_double * 9)()
    n = ctypes.c_longlong()
    assert lib.mmx_set_dmi_tensor(None, 0, q9) == -1
    assert lib.mmx_graph_enable(None, 1) == -1
    assert lib.mmx_graph_info(None, ctypes.byref(n)) == -1
    assert lib.mmx_set_elastic(None, None) == -1 and lib.mmx_set_coupling(None, None) == -1


@pytest.mark.parametrize("grid,cell,pbc", [((8, 8, 4), (4e-9, 4e-9, 4e-9), (0, 0, 0)),
                                           ((70, 9, 2), (7.8125e-9, 7.8125e-9, 3e-9), (0, 0, 0)),
                                           ((16, 16, 1), (2e-9, 2e-9, 1e-9), (4, 4, 0))])
def test_library_newell_tensor_equals_oracle(lib, grid, cell, pbc):
    """Two independent evaluations (library: long double + Gauss quadrature of the dipole tensor;
    oracle: long double + Taylor moments) agree to 1e-12 of the self term."""
    mine = mmx.newell_tensor_host(grid, cell, pbc)
    ref = onw.kernel_octant(grid, cell, pbc)
    for i, c in enumerate(onw.COMPS):
        assert np.abs(mine[i] - ref[c]).max() < 1e-12, c


@pytest.mark.parametrize("grid,cell,pbc", [((8, 8, 4), (4e-9, 4e-9, 4e-9), (0, 0, 0)),
                                           ((8, 16, 1), (2e-9, 2e-9, 1e-9), (2, 2, 0)),
                                           ((8, 4, 2), (2e-9, 3e-9, 1e-9), (1, 0, 0))])
def test_library_kernel_spectrum_equals_oracle(lib, grid, cell, pbc):
    kh, P = mmx.kernel_spectrum_host(grid, cell, pbc)
    assert tuple(P) == tuple(odm.padded_size(grid, pbc))
    sp = odm.kernel_spectrum(onw.kernel_octant(grid, cell, pbc), grid, pbc)
    scale = -MU0 / (P[0] * P[1] * P[2])
    for i, c in enumerate(onw.COMPS):
        ref = sp[c][:kh.shape[1], :kh.shape[2], :]
        assert np.abs(ref.imag).max() < 1e-12          # the spectrum is real
        got = kh[i][:, :, :ref.shape[2]] / scale
        assert np.abs(got - ref.real).max() < 3e-7 * max(np.abs(ref.real).max(), 1.0)


def test_padding_rule():
    _, P = mmx.kernel_spectrum_host((20, 12, 3), (1e-9,) * 3)
    assert P == (64, 32, 8)
    _, P = mmx.kernel_spectrum_host((1, 1, 1), (1e-9,) * 3)
    assert P == (2, 1, 1)


def test_imaginary_axis_stability_limits_of_the_tableaux(lib):
    """mmx_rk_imag_stability_limit (the elastic step bound of mmx_step_rk45): closed forms where they exist -- RK4
    |R(iy)|^2 = 1 - y^6/72 + y^8/576 <= 1 up to 2 sqrt 2, Bogacki-Shampine 1 - y^4/12 + y^6/36 <= 1 up to sqrt 3, Heun
    |R|^2 = 1 + y^4/4 -- and for every method the stability polynomial of the oracle's exact-fraction tableau (Table 2,
    P:L122-131) evaluated independently on both sides of the returned limit."""
    from oracle import rk
    assert abs(mmx.rk_imag_stability_limit(mmx.RK4) - 2 * np.sqrt(2)) < 1.5e-4
    assert abs(mmx.rk_imag_stability_limit(mmx.BS23) - np.sqrt(3)) < 1.5e-4
    g = 1e-6
    assert abs(mmx.rk_imag_stability_limit(mmx.HEUN12, g) - (4 * ((1 + g) ** 2 - 1)) ** 0.25) < 1.5e-4
    tabs = {mmx.RK4: rk.RK4, mmx.DP45: rk.DP45, mmx.HEUN12: rk.HEUN12, mmx.BS23: rk.BS23, mmx.CK45: rk.CK45, mmx.RKF45: rk.RKF45}
    for method, tab in tabs.items():
        s = tab.stages
        A = np.zeros((s, s))
        for i, row in enumerate(tab.a):
            A[i, :len(row)] = [float(x) for x in row]
        b = np.array([float(x) for x in tab.b])
        R = lambda y: abs(1 + 1j * y * (b @ np.linalg.solve(np.eye(s) - 1j * y * A, np.ones(s))))
        for growth in (0.0, 1e-6):
            y = mmx.rk_imag_stability_limit(method, growth)
            assert 0 <= y < 3.0
            if y > 0:
                assert max(R(t) for t in np.linspace(0, y, 400)) <= 1 + growth + 1e-12, (method, growth)
            assert R(y + 2e-4) > 1 + growth, (method, growth)
    assert mmx.rk_imag_stability_limit(mmx.DP45) < 1.0 < mmx.rk_imag_stability_limit(mmx.BS23)
    with pytest.raises(mmx.MmxError):
        mmx.rk_imag_stability_limit(17)
