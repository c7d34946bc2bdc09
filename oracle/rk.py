"""ORACLE (test infrastructure): explicit Runge-Kutta steppers.

Table 2 P:L122-131 lists the embedded pairs; Dormand-Prince (RK45) has
convergence order 5 and error-estimate order 4.  Classical RK4 is the textbook
method (reading S19).  Tableaux as restated in SURVEY 8c step 9.

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
