"""Exact solution of the 1-D Riemann problem for a calorically perfect gas.

Textbook construction (two-shock/two-rarefaction pressure function, Newton iteration on
f_L(p) + f_R(p) + u_R - u_L = 0, then sampling of the self-similar wave pattern).  Used only
to pin the oracle on the paper's Sod case.
"""
import math

import numpy as np


def _f(p, rho_k, p_k, g):
    a_k = math.sqrt(g * p_k / rho_k)
    if p > p_k:   # shock
        A = 2.0 / ((g + 1.0) * rho_k)
        B = (g - 1.0) / (g + 1.0) * p_k
        f = (p - p_k) * math.sqrt(A / (p + B))
        df = math.sqrt(A / (p + B)) * (1.0 - 0.5 * (p - p_k) / (p + B))
    else:         # rarefaction
        f = 2.0 * a_k / (g - 1.0) * ((p / p_k) ** ((g - 1.0) / (2.0 * g)) - 1.0)
        df = 1.0 / (rho_k * a_k) * (p / p_k) ** (-(g + 1.0) / (2.0 * g))
    return f, df


def star_state(rl, ul, pl, rr, ur, pr, g):
    p = 0.5 * (pl + pr)
    for _ in range(100):
        fl, dfl = _f(p, rl, pl, g)
        fr, dfr = _f(p, rr, pr, g)
        dp = -(fl + fr + ur - ul) / (dfl + dfr)
        p = max(p + dp, 1e-12)
        if abs(dp) <= 1e-14 * p:
            break
    fl, _ = _f(p, rl, pl, g)
    fr, _ = _f(p, rr, pr, g)
    u = 0.5 * (ul + ur) + 0.5 * (fr - fl)
    return p, u


def sample(xi, rl, ul, pl, rr, ur, pr, g):
    """Solution (rho, u, p) at similarity coordinates xi = x/t (array)."""
    ps, us = star_state(rl, ul, pl, rr, ur, pr, g)
    al, ar = math.sqrt(g * pl / rl), math.sqrt(g * pr / rr)
    gm, gp = g - 1.0, g + 1.0
    out = np.zeros((3, len(xi)))
    for n, s in enumerate(xi):
        if s <= us:   # left of contact
            if ps > pl:
                sl = ul - al * math.sqrt(gp / (2 * g) * ps / pl + gm / (2 * g))
                if s <= sl:
                    w = (rl, ul, pl)
                else:
                    w = (rl * ((ps / pl + gm / gp) / (gm / gp * ps / pl + 1.0)), us, ps)
            else:
                shl = ul - al
                asl = al * (ps / pl) ** (gm / (2 * g))
                stl = us - asl
                if s <= shl:
                    w = (rl, ul, pl)
                elif s >= stl:
                    w = (rl * (ps / pl) ** (1.0 / g), us, ps)
                else:
                    c = 2.0 / gp + gm / (gp * al) * (ul - s)
                    w = (rl * c ** (2.0 / gm), 2.0 / gp * (al + gm / 2.0 * ul + s), pl * c ** (2.0 * g / gm))
        else:
            if ps > pr:
                sr = ur + ar * math.sqrt(gp / (2 * g) * ps / pr + gm / (2 * g))
                if s >= sr:
                    w = (rr, ur, pr)
                else:
                    w = (rr * ((ps / pr + gm / gp) / (gm / gp * ps / pr + 1.0)), us, ps)
            else:
                shr = ur + ar
                asr = ar * (ps / pr) ** (gm / (2 * g))
                str_ = us + asr
                if s >= shr:
                    w = (rr, ur, pr)
                elif s <= str_:
                    w = (rr * (ps / pr) ** (1.0 / g), us, ps)
                else:
                    c = 2.0 / gp - gm / (gp * ar) * (ur - s)
                    w = (rr * c ** (2.0 / gm), 2.0 / gp * (-ar + gm / 2.0 * ur + s), pr * c ** (2.0 * g / gm))
        out[:, n] = w
    return out
