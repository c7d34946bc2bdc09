"""Thin ctypes binding of libmmx.so (include/mmx.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of the library; PyTorch is used for
device memory (tensors whose data_ptr() crosses the ABI) and the CUDA stream.  There is no
CPU fallback: if the library is missing, or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libmmx.so")

HOST, DEVICE = 0, 1
ABI_VERSION = 3   # MMX_ABI_VERSION of include/mmx.h
T_EXCH, T_DMI, T_ANIS_U, T_ANIS_C, T_ZEEMAN, T_DEMAG, T_A12, T_A0, T_DMI_INTER, T_MEL, T_DMI_HOMO = (
    1, 2, 4, 8, 16, 32, 64, 128, 256, 512, 1024)
T_ALL = 2047
F_M0, F_M1, F_U, F_V, F_M2 = 0, 1, 2, 3, 4
F_M = (F_M0, F_M1, F_M2)   # state field id of sublattice s
DMI_INTER = -1
RK4, DP45, HEUN12, BS23, CK45, RKF45 = 0, 1, 2, 3, 4, 5
FACES = {"x-": 0, "x+": 1, "y-": 2, "y+": 3, "z-": 4, "z+": 5}


PROFILE_CATEGORIES = ("demag_x_fwd", "demag_mid_fwd", "demag_inner", "demag_mid_inv", "demag_x_inv",
                      "local", "combine", "controller", "strain", "elastic", "energy")


class MmxError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("mmx status %d: %s" % (code, msg))
        self.code = code


class Material(C.Structure):
    _fields_ = [(k, C.c_double) for k in
                ("Ms", "A", "alpha", "Ku1", "Kc1", "D", "B1", "B2", "pol", "xi", "gamma")] + [
        ("u", C.c_double * 3), ("c1", C.c_double * 3), ("c2", C.c_double * 3)]


class Coupling(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("A0", "A12", "latcon", "D_inter", "scale_A11", "scale_A12")] + [
        ("d_homo", C.c_double * 3)]


class Slonczewski(C.Structure):
    _fields_ = [("jz", C.c_double), ("mp", C.c_double * 3), ("lambda_", C.c_double), ("eps_prime", C.c_double),
                ("thickness", C.c_double)]


class Elastic(C.Structure):
    _fields_ = [("C11", C.c_double), ("C12", C.c_double), ("C44", C.c_double), ("rho", C.c_double),
                ("traction_face", C.c_int), ("traction_vec", C.c_double * 3),
                ("traction_amp", C.c_double), ("traction_freq", C.c_double), ("rayleigh_beta", C.c_double)]


class RkOpts(C.Structure):
    _fields_ = [("method", C.c_int), ("fixed_dt", C.c_int), ("dt0", C.c_double), ("tol", C.c_double),
                ("nsteps", C.c_longlong), ("t_end", C.c_double), ("torque_stop", C.c_double),
                ("max_attempts", C.c_longlong), ("dt_max", C.c_double)]


class RkStats(C.Structure):
    _fields_ = [("accepted", C.c_longlong), ("rejected", C.c_longlong), ("t", C.c_double),
                ("dt", C.c_double), ("last_err", C.c_double), ("max_torque", C.c_double),
                ("launches", C.c_longlong)]


# name -> (restype, argtypes): every symbol include/mmx.h declares
_I3 = C.POINTER(C.c_int)
_D3 = C.POINTER(C.c_double)
_W = C.c_void_p
PROTOTYPES = {
    "mmx_last_error": (C.c_char_p, []),
    "mmx_version": (C.c_char_p, []),
    "mmx_abi_version": (C.c_int, []),
    "mmx_world_create": (C.c_int, [_I3, _D3, _I3, C.c_int, C.c_void_p, C.POINTER(_W)]),
    "mmx_world_destroy": (C.c_int, [_W]),
    "mmx_set_regions": (C.c_int, [_W, C.c_void_p, C.c_int, C.c_int]),
    "mmx_set_material": (C.c_int, [_W, C.c_int, C.c_int, C.POINTER(Material)]),
    "mmx_set_coupling": (C.c_int, [_W, C.POINTER(Coupling)]),
    "mmx_set_bext": (C.c_int, [_W, _D3]),
    "mmx_set_current": (C.c_int, [_W, _D3]),
    "mmx_set_dmi_tensor": (C.c_int, [_W, C.c_int, C.POINTER(C.c_double)]),
    "mmx_set_boundary": (C.c_int, [_W, C.c_int]),
    "mmx_set_slonczewski": (C.c_int, [_W, C.POINTER(Slonczewski)]),
    "mmx_set_elastic": (C.c_int, [_W, C.POINTER(Elastic)]),
    "mmx_enable_demag": (C.c_int, [_W, C.c_int]),
    "mmx_set_state": (C.c_int, [_W, C.c_int, C.c_void_p, C.c_int]),
    "mmx_get_state": (C.c_int, [_W, C.c_int, C.c_void_p, C.c_int]),
    "mmx_set_time": (C.c_int, [_W, C.c_double]),
    "mmx_get_time": (C.c_int, [_W, _D3]),
    "mmx_demag_kernel_init": (C.c_int, [_W, C.c_double]),
    "mmx_newell_tensor_host": (C.c_int, [_I3, _D3, _I3, C.c_double, C.c_void_p, C.c_longlong]),
    "mmx_kernel_spectrum_host": (C.c_int, [_I3, _D3, _I3, C.c_double, C.c_void_p, C.c_longlong,
                                           C.POINTER(C.c_longlong)]),
    "mmx_eval_heff": (C.c_int, [_W, C.c_int, C.c_uint, C.c_void_p, C.c_int]),
    "mmx_eval_torque": (C.c_int, [_W, C.c_int, C.c_void_p, C.c_int]),
    "mmx_eval_accel": (C.c_int, [_W, C.c_void_p, C.c_int]),
    "mmx_energy": (C.c_int, [_W, C.c_uint, _D3]),
    "mmx_elastic_energy": (C.c_int, [_W, _D3, _D3]),
    "mmx_max_torque": (C.c_int, [_W, _D3]),
    "mmx_step_rk4": (C.c_int, [_W, C.c_double, C.c_longlong]),
    "mmx_step_rk45": (C.c_int, [_W, C.POINTER(RkOpts), C.POINTER(RkStats)]),
    "mmx_rk_imag_stability_limit": (C.c_int, [C.c_int, C.c_double, _D3]),
    "mmx_stray_field": (C.c_int, [_W, C.c_double, C.c_void_p, C.c_int]),
    "mmx_stray_field_static": (C.c_int, [_I3, C.c_int, _D3, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "mmx_stray_table_host": (C.c_int, [_I3, _D3, C.c_double, C.c_void_p, C.c_longlong]),
    "mmx_relax": (C.c_int, [_W, C.c_double, C.c_double, C.c_longlong, C.POINTER(RkStats)]),
    "mmx_get_err_history": (C.c_int, [_W, _D3, C.c_int, _I3]),
    "mmx_profile_enable": (C.c_int, [_W, C.c_int]),
    "mmx_profile_read": (C.c_int, [_W, _D3, C.POINTER(C.c_longlong), C.c_int]),
    "mmx_device_bytes": (C.c_int, [_W, C.POINTER(C.c_longlong)]),
    "mmx_graph_enable": (C.c_int, [_W, C.c_int]),
    "mmx_graph_info": (C.c_int, [_W, C.POINTER(C.c_longlong)]),
}

_lib = None


def load(path: str | None = None):
    """dlopen libmmx.so and attach prototypes.  Raises if the library is not built."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or LIB_PATH
    if not os.path.exists(p):
        raise FileNotFoundError(
            "%s not found: build it with `python -m paper_2411_18194_b200.build` "
            "(there is no CPU fallback)" % p)
    lib = C.CDLL(p)
    for name, (res, args) in PROTOTYPES.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    if lib.mmx_abi_version() != ABI_VERSION:
        raise RuntimeError("%s was built from another revision of include/mmx.h (library %d, binding %d): rebuild it"
                           % (p, lib.mmx_abi_version(), ABI_VERSION))
    if path is None:
        _lib = lib
    return lib


def _check(rc):
    if rc != 0:
        raise MmxError(rc, load().mmx_last_error().decode())


def _arr(ctype, vals):
    return (ctype * len(vals))(*vals)


def _ptr_mem(buf):
    """(address, mem kind) of a numpy array (host) or a torch tensor (host or cuda)."""
    if isinstance(buf, np.ndarray):
        assert buf.flags["C_CONTIGUOUS"]
        return buf.ctypes.data, HOST
    assert buf.is_contiguous()
    return buf.data_ptr(), (DEVICE if buf.is_cuda else HOST)


def newell_tensor_host(grid, cell, pbc=(0, 0, 0), cutoff_cells=32.0) -> np.ndarray:
    """mmx_newell_tensor_host: fp64 [6][n2][n1][n0] (xx,yy,zz,xy,xz,yz); needs no GPU."""
    n = [(g // 2 + 1) if p > 0 else g for g, p in zip(grid, pbc)]
    out = np.empty((6, n[2], n[1], n[0]), dtype=np.float64)
    _check(load().mmx_newell_tensor_host(_arr(C.c_int, list(grid)), _arr(C.c_double, list(cell)),
                                         _arr(C.c_int, list(pbc)), float(cutoff_cells),
                                         out.ctypes.data, out.size))
    return out


def kernel_spectrum_host(grid, cell, pbc=(0, 0, 0), cutoff_cells=32.0):
    """mmx_kernel_spectrum_host: (khat fp32 [6][KZ][KY][XP], (Px, Py, Pz)); needs no GPU."""
    lib = load()
    dims = (C.c_longlong * 5)()
    a = (_arr(C.c_int, list(grid)), _arr(C.c_double, list(cell)), _arr(C.c_int, list(pbc)))
    _check(lib.mmx_kernel_spectrum_host(*a, float(cutoff_cells), None, 0, dims))
    px, py, pz, xp, total = (int(x) for x in dims)
    kz, ky = (pz // 2 + 1 if pz > 1 else 1), (py // 2 + 1 if py > 1 else 1)
    out = np.empty((6, kz, ky, xp), dtype=np.float32)
    _check(lib.mmx_kernel_spectrum_host(*a, float(cutoff_cells), out.ctypes.data, out.size, dims))
    return out, (px, py, pz)


def rk_imag_stability_limit(method, growth=0.0) -> float:
    """mmx_rk_imag_stability_limit: largest omega*dt of an undamped oscillation the method advances with an amplification
    of at most 1 + growth per step; needs no GPU."""
    y = C.c_double()
    _check(load().mmx_rk_imag_stability_limit(int(method), float(growth), C.byref(y)))
    return y.value


STRAY_STATIC_MAX_CELLS = 262144


def stray_table_host(grid, cell, height) -> np.ndarray:
    """mmx_stray_table_host: fp32 [Nz][6][Ny][Nx], the table mmx_stray_field_static takes; needs no GPU."""
    out = np.empty((grid[2], 6, grid[1], grid[0]), dtype=np.float32)
    _check(load().mmx_stray_table_host(_arr(C.c_int, list(grid)), _arr(C.c_double, list(cell)), float(height),
                                       out.ctypes.data, out.size))
    return out


def stray_field_static(grid, Ms, m, table, out, stream=None):
    """mmx_stray_field_static: the probe-layer field without any allocation inside the library (see include/mmx.h for
    who needs that, the cell limit and the sharing rules).  m [S][3][Nz][Ny][Nx], table [Nz][6][Ny][Nx] and
    out [3][Ny][Nx] are contiguous fp32 CUDA tensors the caller owns; Ms has one value per sublattice.  The result is in
    `out` in stream order; nothing is returned and nothing is synchronised."""
    for t in (m, table, out):
        assert t.is_cuda and t.is_contiguous() and t.element_size() == 4
    Ms = [float(v) for v in Ms]
    _check(load().mmx_stray_field_static(_arr(C.c_int, list(grid)), len(Ms), _arr(C.c_double, Ms), m.data_ptr(),
                                         table.data_ptr(), out.data_ptr(), C.c_void_p(stream) if stream else None))


class World:
    """Python face of an mmx_world: one method per C entry point, same names without the prefix."""

    def __init__(self, grid, cellsize, pbc=(0, 0, 0), n_sublattices=1, stream=None):
        self.lib = load()
        self.grid = tuple(int(g) for g in grid)
        self.S = int(n_sublattices)
        self.N = self.grid[0] * self.grid[1] * self.grid[2]
        h = _W()
        sp = C.c_void_p(stream) if stream else None
        _check(self.lib.mmx_world_create(_arr(C.c_int, list(self.grid)), _arr(C.c_double, list(cellsize)),
                                         _arr(C.c_int, list(pbc)), self.S, sp, C.byref(h)))
        self.h = h

    def destroy(self):
        if getattr(self, "h", None):
            self.lib.mmx_world_destroy(self.h)
            self.h = None

    __del__ = destroy

    @property
    def shape(self):
        return (3, self.grid[2], self.grid[1], self.grid[0])

    # ---- parameters
    def set_regions(self, regions, n_regions):
        if regions is None:
            _check(self.lib.mmx_set_regions(self.h, None, HOST, 1))
            return
        if isinstance(regions, np.ndarray):
            regions = np.ascontiguousarray(regions, dtype=np.uint16)
        p, mem = _ptr_mem(regions)
        _check(self.lib.mmx_set_regions(self.h, p, mem, int(n_regions)))

    def set_material(self, sublattice, region, **kw):
        m = Material()
        m.gamma = 0.0
        m.u[:] = (0.0, 0.0, 1.0)
        m.c1[:] = (1.0, 0.0, 0.0)
        m.c2[:] = (0.0, 1.0, 0.0)
        for k, v in kw.items():
            if k in ("u", "c1", "c2"):
                getattr(m, k)[:] = [float(x) for x in v]
            else:
                setattr(m, k, float(v))
        _check(self.lib.mmx_set_material(self.h, sublattice, region, C.byref(m)))

    def set_coupling(self, A0=0.0, A12=0.0, latcon=0.35e-9, D_inter=0.0, scale_A11=1.0, scale_A12=1.0,
                     d_homo=(0.0, 0.0, 0.0)):
        c = Coupling(A0, A12, latcon, D_inter, scale_A11, scale_A12)
        c.d_homo[:] = [float(x) for x in d_homo]
        _check(self.lib.mmx_set_coupling(self.h, C.byref(c)))

    def set_bext(self, B):
        _check(self.lib.mmx_set_bext(self.h, _arr(C.c_double, [float(x) for x in B])))

    def set_dmi_tensor(self, sublattice, q):
        """q: [3][3] per-axis DMI vectors of Eq.4 (J/m^2) or None to clear."""
        if q is None:
            _check(self.lib.mmx_set_dmi_tensor(self.h, int(sublattice), None))
            return
        flat = [float(x) for x in np.asarray(q, dtype=np.float64).reshape(9)]
        _check(self.lib.mmx_set_dmi_tensor(self.h, int(sublattice), _arr(C.c_double, flat)))

    def set_boundary(self, kind):
        """kind: "open" (default) or "neumann" (Eq.5)."""
        _check(self.lib.mmx_set_boundary(self.h, {"open": 0, "neumann": 1}[kind]))

    def set_slonczewski(self, jz=0.0, mp=(0.0, 0.0, 1.0), thickness=0.0, eps_prime=0.0, **kw):
        """Slonczewski torque parameters (keyword `lambda`: Slonczewski Lambda, default 1); jz = 0 clears."""
        sl = Slonczewski(float(jz), (C.c_double * 3)(*[float(x) for x in mp]), float(kw.get("lambda", 1.0)),
                         float(eps_prime), float(thickness or 0.0))
        _check(self.lib.mmx_set_slonczewski(self.h, C.byref(sl)))

    def set_current(self, J):
        _check(self.lib.mmx_set_current(self.h, _arr(C.c_double, [float(x) for x in J])))

    def set_elastic(self, e):
        if e is None:
            _check(self.lib.mmx_set_elastic(self.h, None))
            return
        s = Elastic()
        s.C11, s.C12, s.C44, s.rho = e["C11"], e["C12"], e["C44"], e["rho"]
        s.rayleigh_beta = float(e.get("beta", 0.0))
        tr = e.get("traction")
        s.traction_face = -1
        if tr:
            s.traction_face = FACES[tr["face"]]
            s.traction_vec[:] = [float(x) for x in tr["vec"]]
            s.traction_amp, s.traction_freq = tr["amp"], tr["freq"]
        _check(self.lib.mmx_set_elastic(self.h, C.byref(s)))

    def enable_demag(self, on):
        _check(self.lib.mmx_enable_demag(self.h, 1 if on else 0))

    def set_state(self, field, buf):
        p, mem = _ptr_mem(buf)
        _check(self.lib.mmx_set_state(self.h, field, p, mem))

    def get_state(self, field, out=None):
        if out is None:
            out = np.empty(self.shape, dtype=np.float32)
        p, mem = _ptr_mem(out)
        _check(self.lib.mmx_get_state(self.h, field, p, mem))
        return out

    def set_time(self, t):
        _check(self.lib.mmx_set_time(self.h, float(t)))

    def get_time(self):
        t = C.c_double()
        _check(self.lib.mmx_get_time(self.h, C.byref(t)))
        return t.value

    # ---- demag / evaluation
    def demag_kernel_init(self, cutoff_cells=32.0):
        _check(self.lib.mmx_demag_kernel_init(self.h, float(cutoff_cells)))

    def eval_heff(self, sublattice=0, term_mask=T_ALL, out=None):
        if out is None:
            out = np.empty(self.shape, dtype=np.float32)
        p, mem = _ptr_mem(out)
        _check(self.lib.mmx_eval_heff(self.h, sublattice, term_mask, p, mem))
        return out

    def eval_torque(self, sublattice=0, out=None):
        if out is None:
            out = np.empty(self.shape, dtype=np.float32)
        p, mem = _ptr_mem(out)
        _check(self.lib.mmx_eval_torque(self.h, sublattice, p, mem))
        return out

    def eval_accel(self, out=None):
        if out is None:
            out = np.empty(self.shape, dtype=np.float32)
        p, mem = _ptr_mem(out)
        _check(self.lib.mmx_eval_accel(self.h, p, mem))
        return out

    def energy(self, term_mask=T_ALL):
        e = C.c_double()
        _check(self.lib.mmx_energy(self.h, term_mask, C.byref(e)))
        return e.value

    def elastic_energy(self):
        a, b = C.c_double(), C.c_double()
        _check(self.lib.mmx_elastic_energy(self.h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def max_torque(self):
        t = C.c_double()
        _check(self.lib.mmx_max_torque(self.h, C.byref(t)))
        return t.value

    # ---- stepping
    def step_rk4(self, dt, nsteps=1):
        _check(self.lib.mmx_step_rk4(self.h, float(dt), int(nsteps)))

    def step_rk45(self, method=DP45, fixed_dt=False, dt0=0.0, tol=1e-5, nsteps=0, t_end=0.0,
                  torque_stop=0.0, max_attempts=0, dt_max=0.0):
        o = RkOpts(int(method), 1 if fixed_dt else 0, float(dt0), float(tol), int(nsteps), float(t_end),
                   float(torque_stop), int(max_attempts), float(dt_max))
        st = RkStats()
        _check(self.lib.mmx_step_rk45(self.h, C.byref(o), C.byref(st)))
        return {k: getattr(st, k) for k, _ in RkStats._fields_}

    def stray_field(self, height):
        """B [3, Ny, Nx] (tesla, fp32) in a probe layer `height` metres above the top surface."""
        out = np.empty((3, self.grid[1], self.grid[0]), dtype=np.float32)
        p, mem = _ptr_mem(out)
        _check(self.lib.mmx_stray_field(self.h, float(height), p, mem))
        return out

    def relax(self, torque_stop, tol=1e-5, max_attempts=0):
        st = RkStats()
        _check(self.lib.mmx_relax(self.h, float(torque_stop), float(tol), int(max_attempts), C.byref(st)))
        return {k: getattr(st, k) for k, _ in RkStats._fields_}

    def get_err_history(self, n=4096):
        buf = (C.c_double * n)()
        got = C.c_int()
        _check(self.lib.mmx_get_err_history(self.h, buf, n, C.byref(got)))
        return np.array(buf[:got.value])

    def profile_enable(self, on=True):
        _check(self.lib.mmx_profile_enable(self.h, 1 if on else 0))

    def profile_read(self):
        """dict category -> (total ms, launches) since profile_enable / the last read."""
        n = len(PROFILE_CATEGORIES)
        ms = (C.c_double * n)()
        cnt = (C.c_longlong * n)()
        _check(self.lib.mmx_profile_read(self.h, ms, cnt, n))
        return {k: (ms[i], cnt[i]) for i, k in enumerate(PROFILE_CATEGORIES)}

    def device_bytes(self):
        b = C.c_longlong()
        _check(self.lib.mmx_device_bytes(self.h, C.byref(b)))
        return b.value

    def graph_enable(self, on=True):
        _check(self.lib.mmx_graph_enable(self.h, 1 if on else 0))

    def graph_info(self):
        """Kernels inside the live step graph (0: stepping uses plain launches)."""
        b = C.c_longlong()
        _check(self.lib.mmx_graph_info(self.h, C.byref(b)))
        return b.value

    # ---- convenience: marshal a workloads.WorldSpec (plain data) through the calls above
    @classmethod
    def from_spec(cls, spec, stream=None, demag=None):
        w = cls(spec.grid, spec.cell, spec.pbc, spec.S, stream)
        R = int(spec.mat["Ms"].shape[1])
        if spec.regions is not None:
            w.set_regions(np.ascontiguousarray(spec.regions, dtype=np.uint16), R)
        scal = [k for k, v in spec.mat.items() if v.ndim == 2]
        vecs = [k for k, v in spec.mat.items() if v.ndim == 3]
        for s in range(spec.S):
            for r in range(R):
                kw = {k: spec.mat[k][s, r] for k in scal}
                kw.update({k: spec.mat[k][s, r] for k in vecs})
                w.set_material(s, r, **kw)
        cpl = dict(spec.coupling)
        dmi_q = cpl.pop("dmi_q", None)
        dmi_q12 = cpl.pop("dmi_q12", None)
        sl = cpl.pop("slonczewski", None)
        bc = cpl.pop("bc", None)
        w.set_coupling(**cpl)
        if dmi_q is not None:
            for s in range(spec.S):
                w.set_dmi_tensor(s, np.asarray(dmi_q)[s])
        if dmi_q12 is not None:
            w.set_dmi_tensor(DMI_INTER, np.asarray(dmi_q12))
        if sl:
            w.set_slonczewski(**sl)
        if bc:
            w.set_boundary(bc)
        w.set_bext(spec.bext)
        w.set_current(spec.J)
        if spec.elastic is not None:
            w.set_elastic(spec.elastic)
        for s in range(spec.S):
            w.set_state(F_M[s], np.ascontiguousarray(spec.m[s], dtype=np.float32))
        if spec.elastic is not None:
            w.set_state(F_U, np.ascontiguousarray(spec.u, dtype=np.float32))
            w.set_state(F_V, np.ascontiguousarray(spec.v, dtype=np.float32))
        use_demag = spec.demag if demag is None else demag
        if use_demag:
            w.demag_kernel_init(spec.cutoff_cells)
        w.enable_demag(bool(use_demag))
        return w
