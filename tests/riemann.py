"""Exact solution of the Riemann problem for a gamma-law gas (textbook construction: pressure function
solved by bisection, then sampling in the similarity variable).  Test-side reference for the Sod
pins; shares nothing with oracle/ or the CUDA path."""
import math

import numpy as np


def _f(p, rho, pk, g):
    a = math.sqrt(g * pk / rho)
    if p > pk:   # shock
        A, B = 2.0 / ((g + 1) * rho), (g - 1) / (g + 1) * pk
        return (p - pk) * math.sqrt(A / (p + B))
    return 2 * a / (g - 1) * ((p / pk) ** ((g - 1) / (2 * g)) - 1.0)   # rarefaction


def star(rl, ul, pl, rr, ur, pr, g):
    lo, hi = 1e-12, 10 * max(pl, pr)
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if _f(mid, rl, pl, g) + _f(mid, rr, pr, g) + (ur - ul) > 0:
            hi = mid
        else:
            lo = mid
    p = 0.5 * (lo + hi)
    u = 0.5 * (ul + ur) + 0.5 * (_f(p, rr, pr, g) - _f(p, rl, pl, g))
    return p, u


def sample(xi, rl, ul, pl, rr, ur, pr, g):
    """(rho, u, p) at similarity coordinate xi = (x - x0)/t, for a left rarefaction + right shock
    or any other combination."""
    ps, us = star(rl, ul, pl, rr, ur, pr, g)
    out = np.empty((3, len(xi)))
    al, ar = math.sqrt(g * pl / rl), math.sqrt(g * pr / rr)
    for n, s in enumerate(xi):
        if s <= us:   # left of the contact
            if ps > pl:
                sl = ul - al * math.sqrt((g + 1) / (2 * g) * ps / pl + (g - 1) / (2 * g))
                if s <= sl:
                    out[:, n] = rl, ul, pl
                else:
                    out[:, n] = rl * ((ps / pl + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * ps / pl + 1)), us, ps
            else:
                head, asl = ul - al, al * (ps / pl) ** ((g - 1) / (2 * g))
                tail = us - asl
                if s <= head:
                    out[:, n] = rl, ul, pl
                elif s >= tail:
                    out[:, n] = rl * (ps / pl) ** (1 / g), us, ps
                else:
                    c = 2 / (g + 1) + (g - 1) / ((g + 1) * al) * (ul - s)
                    out[:, n] = rl * c ** (2 / (g - 1)), 2 / (g + 1) * (al + (g - 1) / 2 * ul + s), pl * c ** (2 * g / (g - 1))
        else:
            if ps > pr:
                sr = ur + ar * math.sqrt((g + 1) / (2 * g) * ps / pr + (g - 1) / (2 * g))
                if s >= sr:
                    out[:, n] = rr, ur, pr
                else:
                    out[:, n] = rr * ((ps / pr + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * ps / pr + 1)), us, ps
            else:
                head, asr = ur + ar, ar * (ps / pr) ** ((g - 1) / (2 * g))
                tail = us + asr
                if s >= head:
                    out[:, n] = rr, ur, pr
                elif s <= tail:
                    out[:, n] = rr * (ps / pr) ** (1 / g), us, ps
                else:
                    c = 2 / (g + 1) - (g - 1) / ((g + 1) * ar) * (ur - s)
                    out[:, n] = rr * c ** (2 / (g - 1)), 2 / (g + 1) * (-ar + (g - 1) / 2 * ur + s), pr * c ** (2 * g / (g - 1))
    return out


def sod_speeds(g=1.4):
    """Shock and contact speeds of the Sod problem."""
    ps, us = star(1.0, 0.0, 1.0, 0.125, 0.0, 0.1, g)
    ar = math.sqrt(g * 0.1 / 0.125)
    shock = ar * math.sqrt((g + 1) / (2 * g) * ps / 0.1 + (g - 1) / (2 * g))
    return shock, us, ps
