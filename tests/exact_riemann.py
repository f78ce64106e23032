"""Exact solution of the 1D Riemann problem for the ideal-gas Euler equations
(textbook Newton iteration on the star pressure).  Test-side reference only:
it is what pin P3 compares the oracle with, and is itself pinned by the
classical Sod values in tests/golden/sod_star.txt."""
from __future__ import annotations

import numpy as np


def _f(p, rho_k, p_k, g):
    a_k = np.sqrt(g * p_k / rho_k)
    if p > p_k:  # shock
        A = 2.0 / ((g + 1.0) * rho_k)
        B = (g - 1.0) / (g + 1.0) * p_k
        q = np.sqrt(A / (p + B))
        return (p - p_k) * q, q * (1.0 - 0.5 * (p - p_k) / (p + B))
    pr = p / p_k  # rarefaction
    return 2.0 * a_k / (g - 1.0) * (pr ** ((g - 1.0) / (2.0 * g)) - 1.0), 1.0 / (rho_k * a_k) * pr ** (-(g + 1.0) / (2.0 * g))


def star_state(left, right, g):
    (rl, ul, pl), (rr, ur, pr) = left, right
    p = max(1e-8, 0.5 * (pl + pr))
    for _ in range(100):
        fl, dfl = _f(p, rl, pl, g)
        fr, dfr = _f(p, rr, pr, g)
        dp = (fl + fr + (ur - ul)) / (dfl + dfr)
        pn = max(1e-12, p - dp)
        if abs(pn - p) < 1e-15 * (pn + p):
            p = pn
            break
        p = pn
    fl, _ = _f(p, rl, pl, g)
    fr, _ = _f(p, rr, pr, g)
    return p, 0.5 * (ul + ur) + 0.5 * (fr - fl)


def sample(left, right, g, xi):
    """(rho, u, p) at similarity coordinates xi = (x - x0)/t (array)."""
    (rl, ul, pl), (rr, ur, pr) = left, right
    ps, us = star_state(left, right, g)
    al, ar = np.sqrt(g * pl / rl), np.sqrt(g * pr / rr)
    xi = np.asarray(xi, dtype=np.float64)
    rho = np.empty_like(xi)
    u = np.empty_like(xi)
    p = np.empty_like(xi)
    gm, gp = g - 1.0, g + 1.0
    for n, s in np.ndenumerate(xi):
        if s <= us:  # left of contact
            if ps > pl:  # left shock
                sl = ul - al * np.sqrt(gp / (2 * g) * ps / pl + gm / (2 * g))
                if s <= sl:
                    r_, u_, p_ = rl, ul, pl
                else:
                    r_ = rl * ((ps / pl + gm / gp) / (gm / gp * ps / pl + 1.0))
                    u_, p_ = us, ps
            else:  # left rarefaction
                shl = ul - al
                asl = al * (ps / pl) ** (gm / (2 * g))
                stl = us - asl
                if s <= shl:
                    r_, u_, p_ = rl, ul, pl
                elif s >= stl:
                    r_, u_, p_ = rl * (ps / pl) ** (1.0 / g), us, ps
                else:
                    c = 2.0 / gp + gm / (gp * al) * (ul - s)
                    r_ = rl * c ** (2.0 / gm)
                    u_ = 2.0 / gp * (al + gm / 2.0 * ul + s)
                    p_ = pl * c ** (2.0 * g / gm)
        else:
            if ps > pr:  # right shock
                sr = ur + ar * np.sqrt(gp / (2 * g) * ps / pr + gm / (2 * g))
                if s >= sr:
                    r_, u_, p_ = rr, ur, pr
                else:
                    r_ = rr * ((ps / pr + gm / gp) / (gm / gp * ps / pr + 1.0))
                    u_, p_ = us, ps
            else:
                shr = ur + ar
                asr = ar * (ps / pr) ** (gm / (2 * g))
                strr = us + asr
                if s >= shr:
                    r_, u_, p_ = rr, ur, pr
                elif s <= strr:
                    r_, u_, p_ = rr * (ps / pr) ** (1.0 / g), us, ps
                else:
                    c = 2.0 / gp - gm / (gp * ar) * (ur - s)
                    r_ = rr * c ** (2.0 / gm)
                    u_ = 2.0 / gp * (-ar + gm / 2.0 * ur + s)
                    p_ = pr * c ** (2.0 * g / gm)
        rho[n], u[n], p[n] = r_, u_, p_
    return rho, u, p
