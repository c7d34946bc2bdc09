"""ORACLE (test infrastructure): magnetostatic field.

P:L144: "In the case of antiferromagnets, the vector sum of the spins within a
simulation cell is computed prior to evaluating the resulting field."

Definition:  B_i(r) = -mu0 sum_{r'} sum_j K_ij(r - r') M_j(r'),
M = sum_s Ms^(s) m^(s).  `demag_direct` IS that definition (O(N^2));
`demag_fft` is the same convolution through zero-padded FFTs (scipy.fft as a
library step) and is validated against the direct sum in
tests/test_oracle_newell.py (P5).
"""
from __future__ import annotations

import numpy as np
import scipy.fft as sfft

from . import newell as nw
from .constants import MU0

_PAIR = {(0, 0): "xx", (1, 1): "yy", (2, 2): "zz", (0, 1): "xy", (1, 0): "xy",
         (0, 2): "xz", (2, 0): "xz", (1, 2): "yz", (2, 1): "yz"}


def demag_direct(M, octant, grid, pbc, targets=None):
    """Direct sum.  M float64 [3,Nz,Ny,Nx] (A/m).  `targets`: optional list of
    (ix,iy,iz) cells to evaluate (sampled parity at full size); default all cells.
    Returns B [3, ...] in tesla: full grid, or [3, len(targets)]."""
    nx, ny, nz = grid
    iz, iy, ix = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    all_cells = targets is None
    if all_cells:
        targets = list(zip(ix.ravel(), iy.ravel(), iz.ravel()))
    B = np.zeros((3, len(targets)))
    for t, (tx, ty, tz) in enumerate(targets):
        d = (tx - ix, ty - iy, tz - iz)
        K = {c: nw.kernel_lookup(octant, c, d, grid, pbc) for c in nw.COMPS}
        for i in range(3):
            acc = 0.0
            for j in range(3):
                acc += np.sum(K[_PAIR[(i, j)]] * M[j])
            B[i, t] = -MU0 * acc
    return B.reshape(3, nz, ny, nx) if all_cells else B


def padded_size(grid, pbc):
    """FFT length per axis: N on a periodic or single-cell axis, 2N on an open one."""
    return tuple(g if (p > 0 or g == 1) else 2 * g for g, p in zip(grid, pbc))


def kernel_spectrum(octant, grid, pbc):
    """rfftn of the kernel laid out with wrap-around on the padded box.
    Returns dict comp -> complex128 [Pz, Py, Px/2+1]."""
    P = padded_size(grid, pbc)
    out = {}
    for comp in nw.COMPS:
        d = []
        for a in range(3):
            j = np.arange(P[a])
            if pbc[a] > 0 or grid[a] == 1:
                da = np.where(j <= P[a] // 2, j, j - P[a])
            else:
                da = np.where(j < grid[a], j, j - P[a])  # j == N: offset -N, unused
            d.append(da)
        DZ, DY, DX = np.meshgrid(d[2], d[1], d[0], indexing="ij")
        valid = np.ones_like(DX, dtype=bool)
        for a, D in enumerate((DX, DY, DZ)):
            if not (pbc[a] > 0 or grid[a] == 1):
                valid &= np.abs(D) < grid[a]
        Dc = [np.where(valid, D, 0) for D in (DX, DY, DZ)]
        K = np.where(valid, nw.kernel_lookup(octant, comp, Dc, grid, pbc), 0.0)
        out[comp] = sfft.rfftn(K, axes=(0, 1, 2), workers=-1)
    return out


def demag_fft(M, spectrum, grid, pbc):
    """Zero-padded FFT convolution; M float64 [3,Nz,Ny,Nx] -> B [3,Nz,Ny,Nx] tesla."""
    nx, ny, nz = grid
    P = padded_size(grid, pbc)
    Mh = [sfft.rfftn(M[j], s=(P[2], P[1], P[0]), axes=(0, 1, 2), workers=-1) for j in range(3)]
    B = np.empty_like(M)
    for i in range(3):
        acc = 0
        for j in range(3):
            acc = acc + spectrum[_PAIR[(i, j)]] * Mh[j]
        b = sfft.irfftn(acc, s=(P[2], P[1], P[0]), axes=(0, 1, 2), workers=-1)
        B[i] = -MU0 * b[:nz, :ny, :nx]
    return B


def stray_field_at_height(M, grid, cell, height, cutoff_cells=32.0):
    """Field of the magnet in a probe layer above it ("we calculate the out-of-plane component of the magnet's
    stray field 60 nm above the film's surface"; reading S40: the probe layer has the magnet's in-plane grid and cell
    size, its cells are centred `height` above the top surface, and the value is the average over a probe cell, like
    every field of the method).  The definition, term by term:
        B_i(x, y) = -mu0 sum_{x', y', k} sum_j N_ij(x - x', y - y', Dz_k) M_j(x', y', k),
        Dz_k = (Nz - k - 1/2) dz + height           (centre of source layer k to centre of the probe layer),
    N the cell-to-cell Newell tensor of oracle/newell.py at a z offset that is not a multiple of dz.  Open boundaries.
    M float64 [3, Nz, Ny, Nx] in A/m; returns B [3, Ny, Nx] in tesla."""
    nx, ny, nz = grid
    iy, ix = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    B = np.zeros((3, ny, nx))
    for k in range(nz):
        dzk = (nz - k - 0.5) * cell[2] + height
        quad = {c: nw.newell_octant(c, (nx, ny, 1), cell, cutoff_cells, shift=(0.0, 0.0, dzk))[0] for c in nw.COMPS}
        for ty in range(ny):
            for tx in range(nx):
                dx, dy = tx - ix, ty - iy
                for c in nw.COMPS:
                    par = nw.PARITY[c]
                    Kc = np.where(dx < 0, par[0], 1.0) * np.where(dy < 0, par[1], 1.0) * quad[c][np.abs(dy), np.abs(dx)]
                    for (i, j), name in _PAIR.items():
                        if name == c:
                            B[i, ty, tx] += -MU0 * np.sum(Kc * M[j, k])
    return B
