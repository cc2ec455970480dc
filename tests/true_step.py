"""One Dormand-Prince 5(4) step of the atom-ion ODE in 40-digit arithmetic (mpmath): the value both the
CUDA path and the FP64 oracle approximate.  TEST INFRASTRUCTURE: it lets the parity tests measure how far
each of the two is from the exactly evaluated step (eq. (3)-(10); tableau of paper ref. [5]
typed as rationals), instead of assuming that the oracle's rounding is the truth.  Imports neither the
oracle nor the product."""
from fractions import Fraction as F

import mpmath as mp
import numpy as np

mp.mp.dps = 40

C = [F(0), F(1, 5), F(3, 10), F(4, 5), F(8, 9), F(1), F(1)]
A = [[],
     [F(1, 5)],
     [F(3, 40), F(9, 40)],
     [F(44, 45), F(-56, 15), F(32, 9)],
     [F(19372, 6561), F(-25360, 2187), F(64448, 6561), F(-212, 729)],
     [F(9017, 3168), F(-355, 33), F(46732, 5247), F(49, 176), F(-5103, 18656)],
     [F(35, 384), F(0), F(500, 1113), F(125, 192), F(-2187, 6784), F(11, 84)]]


def _q(fr):
    return mp.mpf(fr.numerator) / mp.mpf(fr.denominator)


def rhs(kw, t, y):
    """eq. (3)-(10) with every parameter taken as the exact value of its double."""
    mi, ma = mp.mpf(kw["m_ion"]), mp.mpf(kw["m_atom"])
    n, m = kw.get("n_att", 0) or 4, kw.get("n_rep", 0) or 8
    Cn, Cm = mp.mpf(kw["C4"]), mp.mpf(kw["C8"])
    om = mp.mpf(kw["omega_rf"])
    d = [y[k] - y[6 + k] for k in range(3)]
    r = mp.sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2])
    dV = n * Cn / r ** (n + 1) - m * Cm / r ** (m + 1)
    cw = mp.cos(om * t)
    f = [None] * 12
    for k in range(3):
        f[k] = y[3 + k]
        f[6 + k] = y[9 + k]
        f[3 + k] = -dV * d[k] / r / mi - (mp.mpf(kw["a"][k]) + 2 * mp.mpf(kw["q"][k]) * cw) * om * om / 4 * y[k]
        f[9 + k] = dV * d[k] / r / ma
    return f


def step(kw, t, y, h):
    """ynew (the 5th-order solution) of one step of size h from (t, y[12]) as a list of mpf."""
    t, h = mp.mpf(float(t)), mp.mpf(float(h))
    y = [mp.mpf(float(v)) for v in y]
    k = [rhs(kw, t, y)]
    for s in range(1, 7):
        ys = [y[i] + h * sum(_q(A[s][j]) * k[j][i] for j in range(s)) for i in range(12)]
        if s == 6:
            return ys
        k.append(rhs(kw, t + _q(C[s]) * h, ys))


def step_errors(kw, t, y, h, candidates):
    """max over the four 3-vector blocks of |cand - true| / |true|_inf for each candidate ynew[12]."""
    yt = step(kw, t, y, h)
    out = []
    for c in candidates:
        worst = mp.mpf(0)
        for b in range(4):
            scale = max(max(abs(yt[3 * b + k]) for k in range(3)), max(abs(mp.mpf(float(y[3 * b + k]))) for k in range(3)))
            if scale == 0:
                scale = mp.mpf(1)
            worst = max(worst, max(abs(mp.mpf(float(c[3 * b + k])) - yt[3 * b + k]) for k in range(3)) / scale)
        out.append(float(worst))
    return out
