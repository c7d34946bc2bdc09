"""ORACLE (test infrastructure): explicit Runge-Kutta steppers.

Table 2 P:L122-131 lists the embedded pairs with their convergence order and
error-estimate order: Heun (RK12) 2/1, Bogacki-Shampine (RK23) 3/2, Cash-Karp
5/4, Fehlberg (RKF45) 5/4, Dormand-Prince (RK45) 5/4.  The paper names the
methods (refs [51-55]) and prints no coefficients; the tableaux below are the
published ones of those references, restated as exact fractions, and pinned by
the order conditions they must satisfy (tests/test_oracle_dynamics.py, P14).
In every pair the solution of the CONVERGENCE order is propagated and
e = b - b* (b* the weights of the lower, error-estimate order).  Classical RK4
is the textbook method (reading S19).

A state is a list of arrays; `rhs(state, t)` returns the list of derivatives;
`project(state)` is applied to every stage state and to the result (S20: each
m^(s) renormalised to |m| = 1; u, v untouched).
"""
from __future__ import annotations

from fractions import Fraction as Fr

import numpy as np


class Tableau:
    def __init__(self, c, a, b, e=None, fsal=False, order=0):
        self.c = [float(x) for x in c]
        self.a = [[float(x) for x in row] for row in a]
        self.b = [float(x) for x in b]
        self.e = None if e is None else [float(x) for x in e]
        self.fsal = fsal
        self.order = order
        self.stages = len(c)


RK4 = Tableau(c=[0, Fr(1, 2), Fr(1, 2), 1],
              a=[[], [Fr(1, 2)], [0, Fr(1, 2)], [0, 0, 1]],
              b=[Fr(1, 6), Fr(1, 3), Fr(1, 3), Fr(1, 6)], order=4)

_b5 = [Fr(35, 384), 0, Fr(500, 1113), Fr(125, 192), Fr(-2187, 6784), Fr(11, 84), 0]
_e = [Fr(71, 57600), 0, Fr(-71, 16695), Fr(71, 1920), Fr(-17253, 339200), Fr(22, 525), Fr(-1, 40)]
DP45 = Tableau(
    c=[0, Fr(1, 5), Fr(3, 10), Fr(4, 5), Fr(8, 9), 1, 1],
    a=[[],
       [Fr(1, 5)],
       [Fr(3, 40), Fr(9, 40)],
       [Fr(44, 45), Fr(-56, 15), Fr(32, 9)],
       [Fr(19372, 6561), Fr(-25360, 2187), Fr(64448, 6561), Fr(-212, 729)],
       [Fr(9017, 3168), Fr(-355, 33), Fr(46732, 5247), Fr(49, 176), Fr(-5103, 18656)],
       _b5[:6]],
    b=_b5, e=_e, fsal=True, order=5)


# Heun 2(1): explicit trapezoid rule with the Euler step as the embedded solution (ref [51])
HEUN12 = Tableau(c=[0, 1], a=[[], [1]], b=[Fr(1, 2), Fr(1, 2)],
                 e=[Fr(1, 2) - 1, Fr(1, 2)], order=2)

# Bogacki-Shampine 3(2), FSAL (ref [52])
_b3 = [Fr(2, 9), Fr(1, 3), Fr(4, 9), 0]
_b3s = [Fr(7, 24), Fr(1, 4), Fr(1, 3), Fr(1, 8)]
BS23 = Tableau(c=[0, Fr(1, 2), Fr(3, 4), 1],
               a=[[], [Fr(1, 2)], [0, Fr(3, 4)], _b3[:3]],
               b=_b3, e=[x - y for x, y in zip(_b3, _b3s)], fsal=True, order=3)

# Cash-Karp 5(4) (ref [53])
_bck = [Fr(37, 378), 0, Fr(250, 621), Fr(125, 594), 0, Fr(512, 1771)]
_bcks = [Fr(2825, 27648), 0, Fr(18575, 48384), Fr(13525, 55296), Fr(277, 14336), Fr(1, 4)]
CK45 = Tableau(
    c=[0, Fr(1, 5), Fr(3, 10), Fr(3, 5), 1, Fr(7, 8)],
    a=[[],
       [Fr(1, 5)],
       [Fr(3, 40), Fr(9, 40)],
       [Fr(3, 10), Fr(-9, 10), Fr(6, 5)],
       [Fr(-11, 54), Fr(5, 2), Fr(-70, 27), Fr(35, 27)],
       [Fr(1631, 55296), Fr(175, 512), Fr(575, 13824), Fr(44275, 110592), Fr(253, 4096)]],
    b=_bck, e=[x - y for x, y in zip(_bck, _bcks)], order=5)

# Fehlberg 4(5) with the 5th-order solution propagated (Table 2: convergence order 5; ref [54])
_bf = [Fr(16, 135), 0, Fr(6656, 12825), Fr(28561, 56430), Fr(-9, 50), Fr(2, 55)]
_bfs = [Fr(25, 216), 0, Fr(1408, 2565), Fr(2197, 4104), Fr(-1, 5), 0]
RKF45 = Tableau(
    c=[0, Fr(1, 4), Fr(3, 8), Fr(12, 13), 1, Fr(1, 2)],
    a=[[],
       [Fr(1, 4)],
       [Fr(3, 32), Fr(9, 32)],
       [Fr(1932, 2197), Fr(-7200, 2197), Fr(7296, 2197)],
       [Fr(439, 216), -8, Fr(3680, 513), Fr(-845, 4104)],
       [Fr(-8, 27), 2, Fr(-3544, 2565), Fr(1859, 4104), Fr(-11, 40)]],
    b=_bf, e=[x - y for x, y in zip(_bf, _bfs)], order=5)

# embedded weights b* = b - e of each pair and the error-estimate order of Table 2
EMBEDDED = {"heun12": (HEUN12, 1), "bs23": (BS23, 2), "ck45": (CK45, 4), "rkf45": (RKF45, 4), "dp45": (DP45, 4)}


def _axpy(y, dt, coefs, ks):
    out = [yi.copy() for yi in y]
    for cj, k in zip(coefs, ks):
        if cj != 0.0:
            for o, kj in zip(out, k):
                o += (dt * cj) * kj
    return out


def rk_step(rhs, project, y, t, dt, tab, k1=None):
    """One explicit RK step.  Returns (y_new, ks, err_vec) where err_vec is the list
    dt * sum_j e_j k_j (None when the tableau has no embedded estimate).  With an
    FSAL tableau ks[-1] = rhs(y_new) can be passed as k1 of the next step."""
    ks = [k1 if k1 is not None else rhs(y, t)]
    Y = y
    for i in range(1, tab.stages):
        Y = project(_axpy(y, dt, tab.a[i], ks))
        ks.append(rhs(Y, t + tab.c[i] * dt))
    y_new = Y if tab.fsal else project(_axpy(y, dt, tab.b, ks))
    err = None
    if tab.e is not None:
        zero = [np.zeros_like(yi) for yi in y]
        err = _axpy(zero, dt, tab.e, ks)
    return y_new, ks, err


# step-size controller (reading S21)
SAFETY, FAC_MIN, FAC_MAX = 0.8, 0.5, 2.0


def controller(dt, err, tol, order=5):
    """accept iff err <= tol;  dt <- dt * 0.8 * clip((tol/err)^(1/order), 0.5, 2)."""
    accept = err <= tol
    fac = FAC_MAX if err == 0.0 else min(FAC_MAX, max(FAC_MIN, (tol / err) ** (1.0 / order)))
    return accept, dt * SAFETY * fac
