"""mmx_stray_field_static: the stray-field probe for callers that cannot allocate device memory.

Who they are: a process whose GPU memory already belongs, all of it, to a pooling allocator (here that would be PyTorch's
caching allocator: a raw cudaMalloc inside a library then fails or forces the pool to be emptied); a loop that cannot take
the device-wide stall of cudaMalloc / cudaFree; a thread working while another thread captures a CUDA graph.  The regular
mmx_stray_field does cudaMalloc + cudaFree on every call; the static variant keeps its scratch (M = sum_s Ms m_s) in a
3 MiB array built into the library and takes the Newell table as a caller-owned input (include/mmx.h states the limit of
262 144 cells and the rule that calls on one GPU must not overlap).

This file is named so that pytest collects it last: with `-x` a failure here cannot hide any other test.  It makes no
assumption about what ran before it in the process (it passes alone in a fresh process and after the whole suite): the
built-in array is shared and keeps old contents, and that is part of what is tested.
"""
import numpy as np
import pytest

import paper_2411_18194_b200 as mmx
from gpu_util import FIELD_TOL, field_err


def _unit_vectors(rng, shape):
    v = rng.standard_normal(shape)
    return (v / np.sqrt((v ** 2).sum(axis=-4, keepdims=True))).astype(np.float32)


def _existing_path(grid, cell, Ms, m, height):
    """mmx_stray_field on a world with one region and Ms[s] per sublattice: the path the new entry point is checked against."""
    g = mmx.World(grid, cell, n_sublattices=len(Ms))
    for s, v in enumerate(Ms):
        g.set_material(s, 0, Ms=v, A=1e-11, alpha=0.1)
        g.set_state(mmx.F_M[s], m[s])
    B = g.stray_field(height)
    g.destroy()
    return B


@pytest.mark.gpu
def test_static_scratch_stray_field_equals_the_allocating_path_on_two_calls_in_a_row():
    """Two calls back to back on different grids, sublattice counts and heights, each against mmx_stray_field within the
    field tolerance of the parity tests (FIELD_TOL, reading S27) -- the second, smaller problem runs on an array that still
    holds the first one's M, so a call that relied on stale or zeroed scratch would show here.  Then the first problem
    again, to see that nothing of the second call leaks either.  The arithmetic and its order are the existing kernel's,
    so the results are also compared bit for bit."""
    import torch
    rng = np.random.default_rng(20241118)
    cases = [((40, 24, 2), (2e-9, 3e-9, 4e-9), (4.2e5, 5.6e5), 7e-9),      # two sublattices, two layers, ragged tiles
             ((21, 37, 1), (3e-9, 3e-9, 30e-9), (8.0e5,), 60e-9)]          # one sublattice, the Fig.3 probe height
    prepared = []
    for grid, cell, Ms, height in cases:
        m = _unit_vectors(rng, (len(Ms), 3, grid[2], grid[1], grid[0]))
        want = _existing_path(grid, cell, Ms, m, height)
        table = torch.from_numpy(mmx.stray_table_host(grid, cell, height)).cuda()
        prepared.append((grid, Ms, torch.from_numpy(m).cuda(), table, want))
    torch.cuda.synchronize()
    for grid, Ms, m_dev, table, want in prepared + prepared[:1]:
        out = torch.full((3, grid[1], grid[0]), float("nan"), dtype=torch.float32, device="cuda")
        mmx.stray_field_static(grid, Ms, m_dev, table, out, stream=torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        assert np.isfinite(got).all()
        assert field_err(got[:, None], want[:, None]) < FIELD_TOL, grid
        assert np.abs(got[2] - want[2]).max() < FIELD_TOL * np.abs(want[2]).max()      # the imaged component, B_z
        assert np.array_equal(got, want), grid


@pytest.mark.gpu
def test_static_scratch_entry_point_refuses_what_it_cannot_hold():
    """One cell above the limit is refused with a message that names the limit, before anything is launched (the pointers
    are never touched: they are dummies here); bad sublattice counts and NULL pointers likewise."""
    import torch
    dummy = torch.zeros(16, dtype=torch.float32, device="cuda")
    big = (mmx.STRAY_STATIC_MAX_CELLS // 512 + 1, 512, 1)
    with pytest.raises(mmx.MmxError) as e:
        mmx.stray_field_static(big, (8e5,), dummy, dummy, dummy)
    assert e.value.code == -1 and str(mmx.STRAY_STATIC_MAX_CELLS) in str(e.value)
    with pytest.raises(mmx.MmxError) as e:
        mmx.stray_field_static((4, 4, 1), (1.0, 1.0, 1.0, 1.0), dummy, dummy, dummy)
    assert e.value.code == -1
    rc = mmx.load().mmx_stray_field_static(None, 1, None, None, None, None, None)
    assert rc == -1


def test_stray_table_host_against_the_oracle_tensor():
    """The caller-built input of the entry point, without a GPU: layer k of the table is -mu0 times the oracle's Newell
    tensor at the z offset (Nz - k - 1/2) dz + height (reading S40), component order xx, yy, zz, xy, xz, yz."""
    from oracle import newell as nw
    grid, cell, height = (9, 7, 2), (2e-9, 3e-9, 4e-9), 11e-9
    tab = mmx.stray_table_host(grid, cell, height)
    assert tab.shape == (2, 6, 7, 9) and tab.dtype == np.float32
    mu0 = 4e-7 * np.pi
    for k in range(grid[2]):
        dz = (grid[2] - k - 0.5) * cell[2] + height
        for q, c in enumerate(nw.COMPS):
            want = -mu0 * nw.newell_octant(c, (grid[0], grid[1], 1), cell, 32.0, shift=(0.0, 0.0, dz))[0]
            assert np.abs(tab[k, q] - want).max() < 2e-7 * np.abs(want).max() + 1e-14, (k, c)
    import ctypes as C
    short = np.empty(5, np.float32)                                  # a wrong out_len is refused, nothing is written
    rc = mmx.load().mmx_stray_table_host((C.c_int * 3)(*grid), (C.c_double * 3)(*cell), height, short.ctypes.data, short.size)
    assert rc == -1 and b"out_len" in mmx.load().mmx_last_error()
