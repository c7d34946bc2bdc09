"""ORACLE (test infrastructure): one simulation world -- fields, RHS, stepping, energies.

Follows SURVEY 8c steps 1-11 in order; every formula is in fields.py /
elastic.py / demag.py / rk.py with its citation.  State: m[s] (S sublattices),
optional u, v; everything float64 (inputs are the float32 blobs of `workloads`
widened).
"""
from __future__ import annotations

import numpy as np

from . import demag as dm
from . import elastic as el
from . import fields as fl
from . import newell as nw
from . import rk
from .constants import (T_A0, T_A12, T_ALL, T_ANIS_C, T_ANIS_U, T_DEMAG, T_DMI, T_DMI_HOMO, T_DMI_INTER,
                        T_EXCH, T_MEL, T_ZEEMAN)


class World:
    def __init__(self, spec, demag_mode="fft"):
        self.spec = spec
        self.grid = tuple(spec.grid)
        self.cell = tuple(float(c) for c in spec.cell)
        self.pbc = tuple(spec.pbc)
        self.S = spec.S
        nx, ny, nz = self.grid
        self.reg = (np.zeros((nz, ny, nx), dtype=np.int64) if spec.regions is None
                    else spec.regions.astype(np.int64))
        # expand the region table to per-cell arrays
        self.p = []
        for s in range(self.S):
            d = {}
            for k, tab in spec.mat.items():
                if tab.ndim == 2:
                    d[k] = tab[s][self.reg]
                else:
                    d[k] = np.moveaxis(tab[s][self.reg], -1, 0)
            self.p.append(d)
        self.cpl = dict(spec.coupling)
        self.bext = tuple(spec.bext)
        self.J = tuple(spec.J)
        self.elastic = spec.elastic
        self.m = [np.asarray(a, dtype=np.float64).copy() for a in spec.m]
        self.u = None if spec.u is None else np.asarray(spec.u, dtype=np.float64).copy()
        self.v = None if spec.v is None else np.asarray(spec.v, dtype=np.float64).copy()
        self.t = 0.0
        self.use_demag = bool(spec.demag)
        self.demag_mode = demag_mode
        self._octant = None
        self._spectrum = None
        self._k1 = None
        self._k1_tab = None
        self.precession = True   # False: relaxation mode (reading S39), torque() drops the m x B term
        self.V = self.cell[0] * self.cell[1] * self.cell[2]

    # ------------------------------------------------------------------ demag
    def octant(self):
        if self._octant is None:
            self._octant = nw.kernel_octant(self.grid, self.cell, self.pbc, self.spec.cutoff_cells)
        return self._octant

    def magnetisation(self, m):
        """vector sum of the sublattice moments in a cell, M = sum_s Ms^(s) m^(s) (S15)."""
        return sum(self.p[s]["Ms"][None] * m[s] for s in range(self.S))

    def demag_field(self, m, targets=None):
        M = self.magnetisation(m)
        if self.demag_mode == "direct" or targets is not None:
            return dm.demag_direct(M, self.octant(), self.grid, self.pbc, targets)
        if self._spectrum is None:
            self._spectrum = dm.kernel_spectrum(self.octant(), self.grid, self.pbc)
        return dm.demag_fft(M, self._spectrum, self.grid, self.pbc)

    def stray_field(self, height, m=None):
        """B [3, Ny, Nx] in a probe layer `height` above the top surface (reading S40), of M = sum_s Ms m_s."""
        return dm.stray_field_at_height(self.magnetisation(self.m if m is None else m), self.grid, self.cell, height,
                                        self.spec.cutoff_cells)

    def ghosts(self, m):
        """Ghost values of Eq.5's Neumann boundary condition for every sublattice (reading S41)."""
        q = self.cpl.get("dmi_q")

        def qn_of(s, axis, d):
            D = self.p[s]["D"]
            qa = np.zeros((3,) + D.shape)
            if axis == 0:
                qa[1] = D          # interfacial D: q_x = D y^
            elif axis == 1:
                qa[0] = -D         #                q_y = -D x^
            if q is not None:
                qa = qa + np.asarray(q, float)[s][axis].reshape(3, 1, 1, 1)
            return d * qa

        return fl.neumann_ghosts(m, [self.p[s]["A"] for s in range(self.S)], qn_of, float(self.cpl.get("A12", 0.0)), self.cell)

    # ------------------------------------------------------------------ fields
    def strain(self, u=None):
        u = self.u if u is None else u
        return el.strain(u, self.cell, self.pbc)

    def field_terms(self, s, m=None, u=None, terms=T_ALL, b_demag=None):
        """dict term-bit -> B_term for sublattice s (tesla)."""
        m = self.m if m is None else m
        p = self.p[s]
        # partner sublattices: the inter-sublattice terms of Eq.3 / Eq.4 act between s and every other sublattice
        # (two of them: the paper's s'; "adding a third sublattice with the same interaction terms as the
        # first two" -- reading S38: the terms are summed over both partners)
        others = [t for t in range(self.S) if t != s]
        out = {}
        # P:L161 "The Neumann boundary conditions as given in Eq. (5) are the default in mumax+.  Alternatively, open or
        # periodic boundary conditions can be used": Eq.5 unless the world asks for "open"; three sublattices are open
        # (Eq.5 is written for a sublattice and its partner, reading S41)
        bc = self.cpl.get("bc") or ("neumann" if self.S <= 2 else "open")
        gh = self.ghosts(m) if bc == "neumann" else None   # Eq.5 (reading S41); None: open
        G = (lambda t: None) if gh is None else (lambda t: gh[t])
        if terms & T_EXCH:
            out[T_EXCH] = fl.pair_laplacian(m[s], p["Ms"], p["A"], self.reg, self.cpl["scale_A11"],
                                            self.cell, self.pbc, 2.0, G(s))
        if terms & T_DMI:
            out[T_DMI] = fl.dmi_interfacial(m[s], p["Ms"], p["D"], self.cell, self.pbc, G(s))
            q = self.cpl.get("dmi_q")
            if q is not None and np.any(np.asarray(q)[s]):   # general tensor of Eq.4, same term bit
                out[T_DMI] = out[T_DMI] + fl.dmi_tensor(m[s], p["Ms"], np.asarray(q)[s], self.cell, self.pbc, G(s))
        if terms & T_ANIS_U:
            out[T_ANIS_U] = fl.uniaxial(m[s], p["Ms"], p["Ku1"], p["u"])
        if terms & T_ANIS_C:
            out[T_ANIS_C] = fl.cubic(m[s], p["Ms"], p["Kc1"], p["c1"], p["c2"])
        if terms & T_ZEEMAN:
            out[T_ZEEMAN] = fl.zeeman(m[s], p["Ms"], self.bext)
        if (terms & T_DEMAG) and self.use_demag:
            out[T_DEMAG] = self.demag_field(m) if b_demag is None else b_demag
        if self.S >= 2:
            if terms & T_A12:
                A12 = np.full_like(p["Ms"], self.cpl["A12"])
                out[T_A12] = sum(fl.pair_laplacian(m[o], p["Ms"], A12, self.reg, self.cpl["scale_A12"],
                                                   self.cell, self.pbc, 1.0, G(o)) for o in others)
            if terms & T_A0:
                out[T_A0] = sum(fl.homogeneous_exchange(m[o], p["Ms"], self.cpl["A0"], self.cpl["latcon"])
                                for o in others)
            if terms & T_DMI_INTER:
                Di = np.full_like(p["Ms"], self.cpl["D_inter"])
                out[T_DMI_INTER] = sum(fl.dmi_interfacial(m[o], p["Ms"], Di, self.cell, self.pbc, G(o)) for o in others)
                q12 = self.cpl.get("dmi_q12")
                if q12 is not None and np.any(np.asarray(q12)):
                    # Eq.4 with s != s' ("a third DMI tensor is used to describe the intersublattice
                    # interaction", D^(s,s') = D^(s',s)): eps = sum_i q12_i . (m x d_i m' + m' x d_i m), whose
                    # variation gives B^(s) = (2/Ms^(s)) sum_i q12_i x d_i m^(s') -- the intra-sublattice
                    # expression with the partner's magnetisation (reading S33 for the tensor <-> q_i mapping)
                    for o in others:
                        out[T_DMI_INTER] = out[T_DMI_INTER] + fl.dmi_tensor(m[o], p["Ms"], np.asarray(q12, float),
                                                                            self.cell, self.pbc, G(o))
            if terms & T_DMI_HOMO:
                # Eq.6 between the pairs (first, second) of reading S32: (0,1) for two sublattices, the cyclic
                # pairs (0,1), (1,2), (2,0) for three (reading S38); s is the first spin of the pair (s, s+1)
                # and the second spin of the pair (s-1, s)
                d = self.cpl.get("d_homo", (0.0, 0.0, 0.0))
                B = np.zeros_like(m[s])
                if self.S == 3 or s == 0:
                    B = B + fl.dmi_homogeneous(m[(s + 1) % self.S], p["Ms"], d, 0)
                if self.S == 3 or s == 1:
                    B = B + fl.dmi_homogeneous(m[(s - 1) % self.S], p["Ms"], d, 1)
                out[T_DMI_HOMO] = B
        if (terms & T_MEL) and self.elastic is not None:
            u = self.u if u is None else u
            out[T_MEL] = fl.magnetoelastic_field(m[s], p["Ms"], p["B1"], p["B2"], self.strain(u))
        return out

    def heff(self, s, m=None, u=None, terms=T_ALL, b_demag=None):
        parts = self.field_terms(s, m, u, terms, b_demag)
        B = np.zeros_like(self.m[s])
        for v in parts.values():
            B = B + v
        return B

    def torque(self, s, m=None, u=None, terms=T_ALL, b_demag=None):
        """Eq.1-2 (+ Zhang-Li when J != 0): tau for sublattice s, 1/s."""
        m = self.m if m is None else m
        p = self.p[s]
        tau = fl.llg_torque(m[s], self.heff(s, m, u, terms, b_demag), p["alpha"], p["gamma"], self.precession)
        if any(j != 0.0 for j in self.J):
            tau = tau + fl.zhang_li_torque(m[s], p["Ms"], p["alpha"], p["pol"], p["xi"], self.J,
                                           self.cell, self.pbc)
        sl = self.cpl.get("slonczewski")
        if sl and sl["jz"] != 0.0:   # reading S37
            d = sl.get("thickness") or self.grid[2] * self.cell[2]
            tau = tau + fl.slonczewski_torque(m[s], p["Ms"], p["alpha"], p["gamma"], p["pol"], sl["jz"], sl["mp"],
                                              sl.get("lambda", 1.0), sl.get("eps_prime", 0.0), d)
        return tau * (p["Ms"] > 0)[None]

    # ------------------------------------------------------------------ elastic
    def tractions(self, t):
        tr = (self.elastic or {}).get("traction")
        if not tr:
            return {}
        amp = tr["amp"] * np.sin(2 * np.pi * tr["freq"] * t)
        return {tr["face"]: amp * np.asarray(tr["vec"], float)}

    def acceleration(self, m, u, t, v=None):
        e = self.elastic
        sig = el.stress(el.strain(u, self.cell, self.pbc), e["C11"], e["C12"], e["C44"])
        beta = e.get("beta", 0.0)
        if beta and v is not None:  # viscous (Rayleigh, stiffness-proportional) term
            sv = el.viscous_stress(v, beta, e["C11"], e["C12"], e["C44"], self.cell, self.pbc)
            sig = {k: sig[k] + sv[k] for k in sig}
        f = el.elastic_force(sig, self.cell, self.pbc, self.tractions(t))
        for s in range(self.S):
            f = f + el.magnetoelastic_force(m[s], self.p[s]["B1"], self.p[s]["B2"], self.cell, self.pbc)
        return f / e["rho"]

    # ------------------------------------------------------------------ ODE system
    def get_state(self):
        y = [a.copy() for a in self.m]
        if self.elastic is not None:
            y += [self.u.copy(), self.v.copy()]
        return y

    def set_state(self, y):
        self.m = [a.copy() for a in y[:self.S]]
        if self.elastic is not None:
            self.u, self.v = y[self.S].copy(), y[self.S + 1].copy()
        self._k1 = None

    def rhs(self, y, t):
        m = y[:self.S]
        u = y[self.S] if self.elastic is not None else None
        bd = self.demag_field(m) if self.use_demag else None
        k = [self.torque(s, m, u, T_ALL, bd) for s in range(self.S)]
        if self.elastic is not None:
            k += [y[self.S + 1].copy(), self.acceleration(m, u, t, y[self.S + 1])]
        return k

    def project(self, y):
        out = []
        for i, a in enumerate(y):
            if i < self.S:
                n = np.sqrt((a * a).sum(axis=0, keepdims=True))
                a = np.where(n > 0, a / np.where(n > 0, n, 1.0), a)
            out.append(a)
        return out

    def mag_norm(self, vec):
        """max over sublattices and cells of the Euclidean norm of a per-cell 3-vector (S21, S22)."""
        return max(float(np.sqrt((vec[s] ** 2).sum(axis=0)).max()) for s in range(self.S))

    def step_rk4(self, dt, nsteps=1):
        for _ in range(nsteps):
            y, _, _ = rk.rk_step(self.rhs, self.project, self.get_state(), self.t, dt, rk.RK4)
            self.set_state(y)
            self.t += dt

    def step_embedded_fixed(self, dt, nsteps=1, tab=rk.DP45):
        """Forced-accept steps of an embedded pair of Table 2; returns the list of error
        estimates dt max_c |sum_j e_j k_j|_2 (S29 protocol).  FSAL pairs reuse k_last as the next k_1."""
        errs = []
        for _ in range(nsteps):
            k1 = self._k1 if (tab.fsal and self._k1_tab is tab) else None
            y, ks, err = rk.rk_step(self.rhs, self.project, self.get_state(), self.t, dt, tab, k1)
            self.set_state(y)
            if tab.fsal:
                self._k1, self._k1_tab = ks[-1], tab
            self.t += dt
            errs.append(self.mag_norm(err))
        return errs

    def step_dp45_fixed(self, dt, nsteps=1):
        return self.step_embedded_fixed(dt, nsteps, rk.DP45)

    def max_torque(self):
        k = self.rhs(self.get_state(), self.t)
        return self.mag_norm(k)

    def relax(self, torque_stop, tab=rk.DP45, tol=1e-5, max_attempts=100000):
        """Relaxation (reading S39): damping-only torque, adaptive steps, until max_c |tau_c| < torque_stop [1/s].
        The spin-transfer torques stay as they are (callers relax without currents).  Time is not advanced."""
        t0, self.precession, self._k1 = self.t, False, None
        try:
            out = self.run_adaptive(tab, tol, max_attempts=max_attempts, torque_stop=torque_stop)
        finally:
            self.precession, self._k1, self.t = True, None, t0
        return out

    def run_adaptive(self, tab=rk.DP45, tol=1e-5, dt0=None, nsteps=None, t_end=None, max_attempts=100000,
                     log=None, dt_max=None, torque_stop=None):
        """Adaptive stepping with an embedded pair (controller S21; the step-size exponent is
        1/convergence order).  Returns dict(accepted, rejected, dt, t, last_err); `log`, when a list,
        receives one (dt, err, accepted) tuple per attempt.  dt_max: no step above it is proposed
        or taken (the error norm covers the magnetic variables only, S22; with elastodynamics the
        caller bounds dt by the elastic stability limit)."""
        if self._k1 is None or self._k1_tab is not tab:
            self._k1, self._k1_tab = self.rhs(self.get_state(), self.t), tab
        dt = dt0 if dt0 else 0.01 / self.mag_norm(self._k1)
        acc = rej = 0
        last = 0.0
        for _ in range(max_attempts):
            if dt_max is not None:
                dt = min(dt, dt_max)
            if nsteps is not None and acc >= nsteps:
                break
            if t_end is not None and self.t >= t_end:
                break
            if torque_stop is not None and self.mag_norm(self._k1) < torque_stop:
                break
            if t_end is not None and self.t + dt > t_end:
                dt = t_end - self.t
            y, ks, err = rk.rk_step(self.rhs, self.project, self.get_state(), self.t, dt, tab, self._k1)
            last = self.mag_norm(err)
            ok, dt_new = rk.controller(dt, last, tol, tab.order)
            if log is not None:
                log.append((dt, last, bool(ok)))
            if ok:
                self.set_state(y)
                self._k1 = ks[-1] if tab.fsal else self.rhs(self.get_state(), self.t + dt)
                self._k1_tab = tab
                self.t += dt
                acc += 1
            else:
                rej += 1
            dt = dt_new
        return dict(accepted=acc, rejected=rej, dt=dt, t=self.t, last_err=last)

    def run_dp45(self, tol=1e-5, dt0=None, nsteps=None, t_end=None, max_attempts=100000, log=None):
        return self.run_adaptive(rk.DP45, tol, dt0, nsteps, t_end, max_attempts, log)

    # ------------------------------------------------------------------ energies (step 11, S28)
    def energy(self, terms=T_ALL):
        """Sum of the selected magnetic term energies in joule:
        -1/2 sum Ms V m.B for the bilinear terms, -sum Ms V m.B_ext, -1/4 sum Ms V m.B for Kc1."""
        E = 0.0
        bd = self.demag_field(self.m) if (terms & T_DEMAG and self.use_demag) else None
        for s in range(self.S):
            parts = self.field_terms(s, terms=terms, b_demag=bd)
            for bit, B in parts.items():
                c = 1.0 if bit == T_ZEEMAN else (0.25 if bit == T_ANIS_C else 0.5)
                E += -c * self.V * float((self.p[s]["Ms"][None] * self.m[s] * B).sum())
        return E

    def elastic_energy(self):
        """(1/2 sum sigma:eps V, 1/2 sum rho |v|^2 V)."""
        e = self.elastic
        eps = self.strain()
        sig = el.stress(eps, e["C11"], e["C12"], e["C44"])
        w = 0.0
        for k in el.EPS_KEYS:
            w += (1.0 if k in ("xx", "yy", "zz") else 2.0) * float((sig[k] * eps[k]).sum())
        return 0.5 * w * self.V, 0.5 * e["rho"] * float((self.v ** 2).sum()) * self.V
