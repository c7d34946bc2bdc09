"""ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

A plain, slow, obviously-correct fp64 (numpy) CPU implementation of what the
mmx hot path computes: the finite-difference effective field, the
Landau-Lifshitz-Gilbert right-hand side and its Runge-Kutta advance, written
from /root/reference/PAPER.md (cited as P:L<line>) with the readings listed in
DESIGN.md ("S-list") wherever the paper is silent.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline /
`--impl reference` legs may import this package.  It shares no code with
`paper_2411_18194_b200/` (the CUDA path); only the seeded input generators in
`workloads/` serve both sides.

Pin status (see tests/test_oracle_*.py and DESIGN.md section "Oracle pins"):
  newell / demag .......... pinned (P1-P5, P19, mpmath spot values, dipole limit)
  exchange, DMI, anisotropy pinned (P6, P10, P11; general DMI tensor of Eq.4: P22; uniaxial: P12; cubic: P28 textbook energy
                            values along <100>, <110>, <111> and the precession frequency gamma 2 Kc1/Ms about an easy axis)
  sublattice exchange ..... pinned (A12 term: P6b two-sublattice spin waves, factor and partner wiring;
                            A0 term: P12); homogeneous DMI Eq.6 pinned (P21)
  LLG torque, integrators . pinned (P7, P8, P9; P14: rooted-tree order conditions of RK4 and of all five
                            embedded pairs of Table 2, observed orders, estimate scaling)
  Zhang-Li torque ......... pinned (P13: Gilbert-form identity, rigid translation at -u)
  elastic / magnetoelastic  pinned (P15 paper numbers, P16 patch test, P17; viscous term P20 paper numbers)
  inter-sublattice DMI tensor pinned (P22b); three sublattices pinned (P25: pair-energy gradients, 120-degree state)
  Slonczewski torque ...... pinned (P23: macrospin closed form, switching current, eps at three angles; reading S37)
  relaxation mode ......... pinned (P24: closed form without precession, energy descent); the path it takes: unpinned
  stray field at height ... pinned (P26: on-axis closed form, dipole limit, tie to the in-magnet kernel; reading S40)
  Neumann boundary (Eq.5) . pinned (P27: Eq.5 as printed, collinear-AFM closed form, exact 1/h cancellation); which of the
                            two continuum-equivalent discretisations (open S9 / ghost cells S41) mumax+ shows at finite
                            cell size: parity unpinned
  adaptive-step controller constants (S21), PBC image window (S13), which config switches c3 uses (S8, S14), Zhang-Li
  with two sublattices (S18), the error norm with (u, v) (S22), the DMI chirality sign (S7), the cell-averaged probe of
  S40: parity unpinned -- definitions shared by both sides, stated in DESIGN.md.
"""
