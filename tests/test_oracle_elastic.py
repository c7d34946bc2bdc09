"""Pins for oracle/elastic.py and the magnetoelastic terms (P15, P16, P17)."""
import os

import numpy as np

import workloads as wl
from oracle import elastic as el
from oracle import fields as fl
from oracle.world import World

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _paper_numbers():
    out = {}
    for line in open(os.path.join(GOLDEN, "paper_elastic_numbers.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, v, tol = line.split()
        out[k] = (float(v), float(tol))
    return out


def test_gradient_operator_orders():
    h = 0.1
    x = (np.arange(40) + 0.5) * h
    f = np.sin(x).reshape(1, 1, -1)
    g = el.gradient(f, 0, h, False)
    err = np.abs(g - np.cos(x))[0, 0]
    assert err[2:-2].max() < 4e-6          # 4th order in the bulk: h^4/30
    assert err[1] < 3e-3 and err[0] < 5e-3  # 2nd order next to / at the boundary
    # polynomial exactness: cubic is exact in the bulk, quadratic at the boundary
    np.testing.assert_allclose(el.gradient((x ** 2).reshape(1, 1, -1), 0, h, False)[0, 0], 2 * x, atol=1e-12)
    # periodic: 4th order everywhere, symbol k_eff = (8 sin kh - sin 2kh)/(6h)
    n = 32
    xp = np.arange(n) * h
    k = 2 * np.pi * 3 / (n * h)
    gp = el.gradient(np.sin(k * xp).reshape(1, 1, -1), 0, h, True)[0, 0]
    keff = (8 * np.sin(k * h) - np.sin(2 * k * h)) / (6 * h)
    np.testing.assert_allclose(gp, keff * np.cos(k * xp), atol=1e-12)
    # single-cell axis: derivative is zero
    assert np.all(el.gradient(np.ones((1, 3, 4)), 2, h, False) == 0)


def test_P16_patch_test():
    """Linear displacement field -> uniform stress; with t = sigma.n applied on every face the
    body force vanishes in every cell, including boundary cells."""
    grid, cell = (7, 6, 5), (2e-9, 3e-9, 2.5e-9)
    C11, C12, C44 = 3.3e11, 0.6e11, 1.1e11
    G = np.array([[1e-3, 2e-3, -1e-3], [0.5e-3, -2e-3, 1.5e-3], [3e-3, 1e-3, 0.7e-3]])  # G[i][j] = d_i u_j
    z, y, x = np.meshgrid(*[(np.arange(n) + 0.5) * c for n, c in zip(grid[::-1], cell[::-1])], indexing="ij")
    u = np.stack([G[0][j] * x + G[1][j] * y + G[2][j] * z for j in range(3)])
    eps = el.strain(u, cell, (0, 0, 0))
    np.testing.assert_allclose(eps["xy"], 0.5 * (G[0][1] + G[1][0]), rtol=1e-10)
    sig = el.stress(eps, C11, C12, C44)
    S = np.array([[sig[el._SIG[(i, j)]].flat[0] for j in range(3)] for i in range(3)])
    tr = {}
    for name, (i, sgn) in el._FACES.items():
        n = np.zeros(3)
        n[i] = sgn
        tr[name] = S @ n
    f = el.elastic_force(sig, cell, (0, 0, 0), tr)
    assert np.abs(f).max() < 1e-9 * np.abs(S).max() / min(cell)
    # without the tractions the boundary cells feel the missing stress
    f0 = el.elastic_force(sig, cell, (0, 0, 0), {})
    assert np.abs(f0[:, 1:-1, 1:-1, 1:-1]).max() < 1e-9 * np.abs(S).max() / min(cell)
    assert np.abs(f0[:, :, :, 0]).max() > 0.1 * np.abs(S).max() / max(cell)


def test_P15_plane_wave_dispersion():
    """Periodic transverse plane wave: u_tt = -(C44/rho) k_eff^2 u with k_eff of the 4th-order stencil
    applied twice (gradient then divergence)."""
    n, h = 48, 3e-9
    C11, C12, C44, rho = 3.3e11, 0.6e11, 1.1e11, 6853.0
    k = 2 * np.pi * 2 / (n * h)
    x = np.arange(n) * h
    u = np.zeros((3, 1, 1, n))
    u[2, 0, 0] = 1e-12 * np.sin(k * x)   # shear: u_z(x)
    u[0, 0, 0] = 2e-12 * np.cos(k * x)   # longitudinal: u_x(x)
    sig = el.stress(el.strain(u, (h, h, h), (1, 0, 0)), C11, C12, C44)
    f = el.elastic_force(sig, (h, h, h), (1, 0, 0))
    keff = (8 * np.sin(k * h) - np.sin(2 * k * h)) / (6 * h)
    np.testing.assert_allclose(f[2], -C44 * keff ** 2 * u[2], atol=1e-10 * np.abs(f).max())
    np.testing.assert_allclose(f[0], -C11 * keff ** 2 * u[0], atol=1e-10 * np.abs(f).max())
    assert np.abs(f[1]).max() == 0


def test_P15_paper_pulse_speed_and_strain():
    """The paper's NiO numbers (Table 1): one period of an 8 GHz, 0.3 GPa out-of-plane
    shear traction on the left edge launches a pulse travelling at about 4 km/s with a strain
    amplitude of approximately 0.14 % (gamma_xz = 2 eps_xz = t0/C44 = 0.27 %, eps_xz = 0.136 %)."""
    want = _paper_numbers()
    nx, h = 400, 3e-9
    C11, C12, C44, rho = 3.3e11, 0.6e11, 1.1e11, 6853.0
    f0, t0 = 8e9, 0.3e9
    zeros = np.zeros((3, 1, 1, nx), np.float32)
    spec = wl.WorldSpec(name="nio", grid=(nx, 1, 1), cell=(h, h, h), demag=False,
                        mat=wl.make_mat(1, Ms=4.25e5), coupling=wl.default_coupling(),
                        elastic=dict(C11=C11, C12=C12, C44=C44, rho=rho,
                                     traction=dict(face="x-", vec=(0, 0, 1), amp=t0, freq=f0)),
                        m=[np.tile(np.array([1, 0, 0], np.float32).reshape(3, 1, 1, 1), (1, 1, 1, nx))],
                        u=zeros.copy(), v=zeros.copy())
    w = World(spec)
    dt = 1e-13
    n_on = int(round(1 / f0 / dt))
    w.step_rk4(dt, n_on)            # one period of traction
    w.elastic["traction"] = None    # then traction free
    w.step_rk4(dt, 500)
    x = (np.arange(nx) + 0.5) * h
    eps1 = w.strain()["xz"][0, 0]
    amp = np.abs(eps1).max()
    c1 = (np.abs(eps1) * x).sum() / np.abs(eps1).sum()
    w.step_rk4(dt, 600)
    eps2 = w.strain()["xz"][0, 0]
    c2 = (np.abs(eps2) * x).sum() / np.abs(eps2).sum()
    speed = (c2 - c1) / (600 * dt)
    v, tol = want["pulse_speed_m_per_s"]
    assert abs(speed - v) < tol * v, speed
    assert abs(speed - np.sqrt(C44 / rho)) < 0.01 * np.sqrt(C44 / rho)
    v, tol = want["strain_amplitude"]
    assert abs(amp - v) < tol * v, amp
    assert abs(amp - t0 / (2 * C44)) < 0.02 * t0 / (2 * C44)


def test_P20_rayleigh_damping_ratio_of_the_paper():
    """Table 1: Rayleigh stiffness coefficient 0.1 ps, "chosen to yield a damping ratio of
    about 5% for shear waves with a wavelength of 24 nm" (C44 = 110 GPa, rho = 6853 kg/m^3).  A
    periodic standing shear wave of that wavelength is integrated with the oracle; the decay of its
    modal energy gives zeta.  Pins reading S31 (sigma_visc = beta C : strain rate): zeta = beta w0 / 2."""
    want = _paper_numbers()
    beta = want["rayleigh_beta_s"][0]
    n, h = 48, 3e-9                      # wavelength 24 nm = 8 cells
    C11, C12, C44, rho = 3.3e11, 0.6e11, 1.1e11, 6853.0
    k = 2 * np.pi / 24e-9
    x = np.arange(n) * h
    u = np.zeros((3, 1, 1, n), np.float32)
    u[2, 0, 0] = 1e-12 * np.sin(k * x)
    spec = wl.WorldSpec(name="nio", grid=(n, 1, 1), cell=(h, h, h), pbc=(1, 0, 0), demag=False,
                        mat=wl.make_mat(1, Ms=4.25e5), coupling=wl.default_coupling(),
                        elastic=dict(C11=C11, C12=C12, C44=C44, rho=rho, beta=beta, traction=None),
                        m=[np.tile(np.array([1, 0, 0], np.float32).reshape(3, 1, 1, 1), (1, 1, 1, n))],
                        u=u, v=np.zeros_like(u))
    w = World(spec)
    keff = (8 * np.sin(k * h) - np.sin(2 * k * h)) / (6 * h)
    w0 = keff * np.sqrt(C44 / rho)

    def modal_energy():
        a = 2.0 / n * (w.u[2, 0, 0] * np.sin(k * x)).sum()
        adot = 2.0 / n * (w.v[2, 0, 0] * np.sin(k * x)).sum()
        return w0 ** 2 * a ** 2 + adot ** 2

    e0 = modal_energy()
    dt = 5e-14                           # 121 steps per period: RK4 phase error ~ (w0 dt)^4 / 120 = 6e-8
    nsteps = int(round(2 * 2 * np.pi / w0 / dt))
    w.step_rk4(dt, nsteps)
    zeta = -np.log(modal_energy() / e0) / (2 * w0 * nsteps * dt)
    v, tol = want["damping_ratio_shear_24nm"]
    assert abs(zeta - v) < tol * v, zeta                      # the paper's "about 5 %"
    assert abs(zeta - 0.5 * beta * w0) < 0.01 * 0.5 * beta * w0, (zeta, 0.5 * beta * w0)
    # and without the viscous term the same wave does not decay
    spec.elastic["beta"] = 0.0
    spec.u, spec.v = u, np.zeros_like(u)
    w = World(spec)
    e0 = modal_energy()
    w.step_rk4(dt, nsteps)
    assert abs(modal_energy() / e0 - 1) < 1e-6


def test_P17_magnetoelastic_closed_forms():
    """Uniform strain, uniform m: Eq.9 closed form and f_mel = 0; f_mel = div sigma_mel with
    sigma_mel,ii = B1 m_i^2, sigma_mel,ij = B2 m_i m_j for a smooth texture."""
    rng = np.random.default_rng(2)
    B1, B2, Ms = -1.5e7, -0.85e7, 4.25e5
    m = np.array([0.36, 0.48, 0.8]).reshape(3, 1, 1, 1) * np.ones((3, 2, 3, 4))
    e = dict(xx=1e-3, yy=-2e-3, zz=0.5e-3, xy=0.7e-3, xz=-0.3e-3, yz=0.2e-3)
    eps = {k: v * np.ones((2, 3, 4)) for k, v in e.items()}
    one = np.ones((2, 3, 4))
    B = fl.magnetoelastic_field(m, Ms * one, B1 * one, B2 * one, eps)
    E = np.array([[e["xx"], e["xy"], e["xz"]], [e["xy"], e["yy"], e["yz"]], [e["xz"], e["yz"], e["zz"]]])
    mv = np.array([0.36, 0.48, 0.8])
    want = -2 / Ms * (B1 * np.diag(E) * mv + B2 * ((E - np.diag(np.diag(E))) @ mv))
    np.testing.assert_allclose(B[:, 0, 0, 0], want, rtol=1e-13)
    assert np.abs(el.magnetoelastic_force(m, B1 * one, B2 * one, (1e-9,) * 3, (0, 0, 0))).max() < 1e-12 * abs(B1) / 1e-9
    # smooth periodic texture: compare with the divergence of sigma_mel taken spectrally
    n, h = 48, 2e-9
    L = n * h
    Z, Y, X = np.meshgrid(*(np.arange(n) * h,) * 3, indexing="ij")
    th = 1.0 + 0.3 * np.sin(2 * np.pi * X / L) * np.cos(2 * np.pi * Y / L) + 0.2 * np.sin(2 * np.pi * Z / L)
    ph = 0.5 + 0.4 * np.cos(2 * np.pi * X / L) + 0.3 * np.sin(2 * np.pi * (Y + Z) / L)
    m = np.stack([np.sin(th) * np.cos(ph), np.sin(th) * np.sin(ph), np.cos(th)])
    one = np.ones((n, n, n))
    f = el.magnetoelastic_force(m, B1 * one, B2 * one, (h, h, h), (1, 1, 1))

    def d(a, axis):
        kk = 2j * np.pi * np.fft.fftfreq(n, h)
        shape = [1, 1, 1]
        shape[2 - axis] = n
        return np.real(np.fft.ifft(np.fft.fft(a, axis=2 - axis) * kk.reshape(shape), axis=2 - axis))
    want = np.zeros_like(m)
    for j in range(3):
        for i in range(3):
            s = (B1 if i == j else B2) * m[i] * m[j]
            want[j] += d(s, i)
    assert np.abs(f - want).max() < 2e-4 * np.abs(want).max()  # 4th-order stencil error


def test_elastic_energy_error_converges_traction_free():
    """Free vibration of an open block: the scheme (4th-order bulk, 2nd-order boundary closure)
    is not exactly energy conserving, but E_el + E_kin must become constant under refinement
    (measured: -38 %, -12 %, -2.7 % at 8, 16, 32 cells: second order)."""
    errs = []
    for nx, ny in ((8, 6), (16, 12), (32, 24)):
        grid, cell = (nx, ny, 1), (16e-9 / nx, 12e-9 / ny, 2e-9)
        u0 = np.zeros((3, 1, ny, nx))
        y, x = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
        u0[0, 0] = 1e-12 * np.cos(np.pi * (x + 0.5) / nx)
        u0[1, 0] = 0.5e-12 * np.cos(np.pi * (y + 0.5) / ny)
        u0[2, 0] = 0.7e-12 * np.cos(np.pi * (x + 0.5) / nx) * np.cos(np.pi * (y + 0.5) / ny)
        spec = wl.WorldSpec(name="blk", grid=grid, cell=cell, demag=False, mat=wl.make_mat(1, Ms=4e5),
                            coupling=wl.default_coupling(),
                            elastic=dict(C11=2.5e11, C12=1.5e11, C44=1.0e11, rho=6800.0),
                            m=[np.tile(np.array([0, 0, 1], np.float32).reshape(3, 1, 1, 1), (1, 1, ny, nx))],
                            u=u0.astype(np.float32), v=np.zeros_like(u0, dtype=np.float32))
        w = World(spec)
        w.u = u0.copy()
        E0 = sum(w.elastic_energy())
        w.step_rk4(2e-14 * 8 / nx, 300 * nx // 8)
        Ee, Ek = w.elastic_energy()
        assert Ek > 0.1 * E0                    # energy really sloshes between the two forms
        errs.append(abs(Ee + Ek - E0) / E0)
    assert errs[1] < errs[0] / 2.5 and errs[2] < errs[1] / 2.5 and errs[2] < 0.04
