"""Seeded synthetic input generators shared by the oracle and the CUDA path.

This module holds NONE of the method's arithmetic (no field, torque, FFT or
Runge-Kutta code): it only describes worlds (grid, cell size, boundary kind,
material tables, region maps) and draws initial states.  Both `oracle/` and
`paper_2411_18194_b200/` consume the `WorldSpec` objects it returns; neither of
those two imports the other.

The five configurations follow /root/repo/BASELINE.json `configs[0..4]`
("c1".."c5"); the recipes (distributions, seeds, wall profiles, grain
generator) are the ones stated in SURVEY.md section 8(d) and DESIGN.md.  They
are synthetic stand-ins shaped like the paper's demonstrations (PAPER.md L41,
L47, L84) -- the paper's own data sets are not available.

Everything is generated with numpy.random.default_rng(seed) (PCG64) on the host
and stored as float32, so both sides read bit-identical inputs.
"""
from __future__ import annotations

import copy
from dataclasses import dataclass, field

import numpy as np

# Names of the per-(sublattice, region) scalar material parameters.
MAT_SCALARS = ("Ms", "A", "alpha", "Ku1", "Kc1", "D", "B1", "B2", "pol", "xi", "gamma")
# Names of the per-(sublattice, region) 3-vector material parameters.
MAT_VECTORS = ("u", "c1", "c2")

GAMMA_DEFAULT = 1.7595e11  # rad/(T s); SURVEY S1 (the paper defers to mumax3's value)


@dataclass
class WorldSpec:
    """Plain description of one simulation world."""
    name: str
    grid: tuple            # (Nx, Ny, Nz)
    cell: tuple            # (dx, dy, dz) in metres
    pbc: tuple = (0, 0, 0)  # periodic image repetitions per axis, 0 = open
    S: int = 1              # number of sublattices (1, 2 or 3)
    regions: np.ndarray | None = None   # uint16 [Nz,Ny,Nx]; None = one region
    mat: dict = field(default_factory=dict)       # name -> float64 [S,R] or [S,R,3]
    coupling: dict = field(default_factory=dict)  # A0, A12, latcon, D_inter, scale_A11, scale_A12
    bext: tuple = (0.0, 0.0, 0.0)   # tesla
    J: tuple = (0.0, 0.0, 0.0)      # A/m^2
    elastic: dict | None = None     # C11, C12, C44, rho, traction{face, vec, amp, freq}
    demag: bool = True
    cutoff_cells: float = 32.0      # analytic/asymptotic switch radius
    m: list = field(default_factory=list)  # S arrays float32 [3,Nz,Ny,Nx]
    u: np.ndarray | None = None     # displacement float32 [3,Nz,Ny,Nx]
    v: np.ndarray | None = None     # velocity float32 [3,Nz,Ny,Nx]
    integrator: dict = field(default_factory=dict)  # suggested fixed-step parity protocol

    @property
    def n_regions(self) -> int:
        return int(self.mat["Ms"].shape[1])

    @property
    def ncells(self) -> int:
        return int(self.grid[0] * self.grid[1] * self.grid[2])

    def copy(self) -> "WorldSpec":
        return copy.deepcopy(self)


def make_mat(S: int, R: int = 1, **kw) -> dict:
    """Material table with every parameter present; unspecified ones are zero
    (gamma: default; axes u,c1,c2: z,x,y)."""
    mat = {k: np.zeros((S, R)) for k in MAT_SCALARS}
    mat["gamma"][:] = GAMMA_DEFAULT
    mat["u"] = np.tile(np.array([0.0, 0.0, 1.0]), (S, R, 1))
    mat["c1"] = np.tile(np.array([1.0, 0.0, 0.0]), (S, R, 1))
    mat["c2"] = np.tile(np.array([0.0, 1.0, 0.0]), (S, R, 1))
    for k, val in kw.items():
        arr = np.asarray(val, dtype=np.float64)
        mat[k][...] = arr
    return mat


def default_coupling(**kw) -> dict:
    c = dict(A0=0.0, A12=0.0, latcon=0.35e-9, D_inter=0.0, scale_A11=1.0, scale_A12=1.0,
             d_homo=(0.0, 0.0, 0.0), dmi_q=None)   # dmi_q: [S][3][3] per-axis DMI vectors of Eq.4, J/m^2
    # bc: "open" | "neumann"; absent = the paper's default (Eq.5 for one or two sublattices).  BASELINE.json's
    # configurations 1, 3 and 4 say "open boundaries" in words, so their specs carry bc="open".
    c.update(kw)
    return c


# --------------------------------------------------------------------------
# state generators
# --------------------------------------------------------------------------
def random_unit(rng, grid) -> np.ndarray:
    """3 iid normals per cell, normalised: uniform on the sphere."""
    nx, ny, nz = grid
    m = rng.standard_normal((3, nz, ny, nx))
    m /= np.sqrt((m * m).sum(axis=0, keepdims=True))
    return m.astype(np.float32)


def _renorm32(m) -> np.ndarray:
    m = np.asarray(m, dtype=np.float64)
    m = m / np.sqrt((m * m).sum(axis=0, keepdims=True))
    return m.astype(np.float32)


def smoothed_random_unit(rng, grid, sigma_cells=3.0) -> np.ndarray:
    """Random field blurred by a periodic Gaussian of `sigma_cells`, renormalised
    (input generation only: a separable circular blur with an explicit kernel)."""
    nx, ny, nz = grid
    m = rng.standard_normal((3, nz, ny, nx))
    for axis, n in ((-1, nx), (-2, ny)):
        if n == 1:
            continue
        d = np.arange(n)
        d = np.minimum(d, n - d)
        w = np.exp(-0.5 * (d / sigma_cells) ** 2)
        w /= w.sum()
        out = np.zeros_like(m)
        for j in np.nonzero(w > 1e-12)[0]:
            out += w[j] * np.roll(m, j, axis=axis)
        m = out
    return _renorm32(m)


def neel_wall(grid, cell, x0, width, sign=1.0) -> np.ndarray:
    """m=(sech xi, 0, tanh xi), xi=(x-x0)/width, x = cell centres."""
    nx, ny, nz = grid
    x = (np.arange(nx) + 0.5) * cell[0]
    xi = (x - x0) / width
    m = np.zeros((3, nz, ny, nx))
    m[0] = (1.0 / np.cosh(xi))[None, None, :]
    m[2] = np.tanh(xi)[None, None, :]
    return _renorm32(sign * m)


def multi_wall(grid, cell, n_walls, delta) -> np.ndarray:
    """theta(x)=sum_k (-1)^(k+1) 2 atan exp((x-x_k)/delta), x_k=k L/(n_walls+1);
    m=(cos theta, 0, sin theta)."""
    nx, ny, nz = grid
    x = (np.arange(nx) + 0.5) * cell[0]
    L = nx * cell[0]
    theta = np.zeros(nx)
    for k in range(1, n_walls + 1):
        xk = k * L / (n_walls + 1)
        theta += (-1.0) ** (k + 1) * 2.0 * np.arctan(np.exp((x - xk) / delta))
    m = np.zeros((3, nz, ny, nx))
    m[0] = np.cos(theta)[None, None, :]
    m[2] = np.sin(theta)[None, None, :]
    return _renorm32(m)


def voronoi_regions(rng, grid, cell, n_seeds) -> np.ndarray:
    """Nearest-seed (Voronoi) region index per cell, seeds uniform in the xy box."""
    from scipy.spatial import cKDTree
    nx, ny, nz = grid
    seeds = np.stack([rng.uniform(0, nx * cell[0], n_seeds),
                      rng.uniform(0, ny * cell[1], n_seeds)], axis=1)
    x = (np.arange(nx) + 0.5) * cell[0]
    y = (np.arange(ny) + 0.5) * cell[1]
    X, Y = np.meshgrid(x, y, indexing="xy")  # [ny,nx]
    _, idx = cKDTree(seeds).query(np.stack([X.ravel(), Y.ravel()], axis=1))
    reg2d = idx.reshape(ny, nx).astype(np.uint16)
    return np.ascontiguousarray(np.broadcast_to(reg2d[None], (nz, ny, nx)))


def cone_axes(rng, n, half_angle_deg) -> np.ndarray:
    """n unit vectors within `half_angle_deg` of +z: cos(theta)~U[cos(a),1], phi~U[0,2pi)."""
    ct = rng.uniform(np.cos(np.deg2rad(half_angle_deg)), 1.0, n)
    ph = rng.uniform(0.0, 2 * np.pi, n)
    st = np.sqrt(1 - ct * ct)
    return np.stack([st * np.cos(ph), st * np.sin(ph), ct], axis=1)


# --------------------------------------------------------------------------
# the five BASELINE.json configurations
# --------------------------------------------------------------------------
def c1(grid=(64, 16, 1), seed=1001) -> WorldSpec:
    """BASELINE.json configs[0]: ferromagnetic thin strip, demag + exchange, RK4 dt=1e-13 x2000."""
    rng = np.random.default_rng(seed)
    return WorldSpec(
        name="c1", grid=tuple(grid), cell=(7.8125e-9, 7.8125e-9, 3e-9),
        mat=make_mat(1, Ms=8.0e5, A=1.3e-11, alpha=0.5), coupling=default_coupling(bc="open"),   # "open boundaries"
        m=[random_unit(rng, grid)],
        integrator=dict(method="rk4", dt=1e-13, nsteps=2000))


def c2(grid=(256, 256, 1), seed=1002) -> WorldSpec:
    """configs[1]: periodic film with DMI, uniaxial anisotropy, Zeeman; DP45 tol 1e-5."""
    rng = np.random.default_rng(seed)
    return WorldSpec(
        name="c2", grid=tuple(grid), cell=(2e-9, 2e-9, 1e-9), pbc=(4, 4, 0),
        mat=make_mat(1, Ms=5.8e5, A=1.5e-11, D=3.0e-3, Ku1=8.0e5, alpha=0.3),
        # "periodic in-plane"; the one-cell z axis has no stencil partner and interfacial DMI no z term, so the
        # boundary kind is immaterial there: stated as open, which keeps the periodic fast kernels in the tests
        coupling=default_coupling(bc="open"), bext=(0.0, 0.0, 0.1),
        m=[smoothed_random_unit(rng, grid, 3.0)],
        integrator=dict(method="dp45", dt=2e-14, nsteps=500, tol=1e-5))


def c3(grid=(1024, 128, 1), seed=1003, grain_diameter=20e-9) -> WorldSpec:
    """configs[2]: two-sublattice polycrystalline AFM strip, Zhang-Li torque, Neel wall."""
    rng = np.random.default_rng(seed)
    cell = (2e-9, 2e-9, 2e-9)
    nx, ny, nz = grid
    area = nx * cell[0] * ny * cell[1]
    n_grains = max(1, int(round(area / (np.pi * (grain_diameter / 2) ** 2))))
    regions = voronoi_regions(rng, grid, cell, n_grains)
    axes = cone_axes(rng, n_grains, 10.0)
    mat = make_mat(2, n_grains, Ms=4.0e5, A=1.0e-11, alpha=0.01, Ku1=6.4e4, D=1.0e-3,
                   pol=0.5, xi=0.1)
    mat["u"][:] = axes[None]
    x0 = 0.5 * nx * cell[0]           # 1024 nm on the full grid
    width = np.sqrt(1.0e-11 / 6.4e4)  # 12.5 nm
    m1 = neel_wall(grid, cell, x0, width)
    return WorldSpec(
        name="c3", grid=tuple(grid), cell=cell, S=2, regions=regions, mat=mat,
        coupling=default_coupling(A0=-4.0e-13, A12=-1.0e-12, latcon=0.35e-9, D_inter=0.0, bc="open"),   # "open boundaries"
        J=(1e12, 0.0, 0.0), m=[m1, (-m1).astype(np.float32)],
        integrator=dict(method="dp45", dt=5e-15, nsteps=400))


def c4(grid=(256, 256, 64), seed=1004) -> WorldSpec:
    """configs[3]: bulk ferromagnetic box, demag-dominated; the roofline headline config."""
    rng = np.random.default_rng(seed)
    return WorldSpec(
        name="c4", grid=tuple(grid), cell=(4e-9, 4e-9, 4e-9),
        mat=make_mat(1, Ms=1.0e6, A=1.0e-11, alpha=0.1), coupling=default_coupling(bc="open"),   # "open boundaries"
        m=[random_unit(rng, grid)],
        integrator=dict(method="dp45", dt=1e-13, nsteps=100))


def c5(grid=(512, 128, 1), seed=1005) -> WorldSpec:
    """configs[4]: magnetoelastic AFM racetrack; m1, m2, u, v co-integrated."""
    cell = (2e-9, 2e-9, 2e-9)
    delta = np.sqrt(1.0e-11 / 1.0e4)  # 31.6 nm
    m1 = multi_wall(grid, cell, 4, delta)
    nx, ny, nz = grid
    zeros = np.zeros((3, nz, ny, nx), dtype=np.float32)
    return WorldSpec(
        name="c5", grid=tuple(grid), cell=cell, S=2,
        mat=make_mat(2, Ms=4.0e5, A=1.0e-11, alpha=0.005, Kc1=1.0e4, B1=-1.0e7, B2=-1.0e7),
        coupling=default_coupling(A0=-4.0e-13, latcon=0.35e-9),
        elastic=dict(C11=2.5e11, C12=1.5e11, C44=1.0e11, rho=6800.0,
                     traction=dict(face="x-", vec=(0.0, 0.0, 1.0), amp=1e8, freq=5e9)),
        m=[m1, (-m1).astype(np.float32)], u=zeros.copy(), v=zeros.copy(),
        integrator=dict(method="dp45", dt=5e-15, nsteps=400))


CONFIGS = {"c1": c1, "c2": c2, "c3": c3, "c4": c4, "c5": c5}


def make(name: str, grid=None, **kw) -> WorldSpec:
    """Build configuration `name`; `grid` overrides the size (reduced parity cases)."""
    if grid is not None:
        kw["grid"] = tuple(grid)
    return CONFIGS[name](**kw)
