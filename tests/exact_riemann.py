"""Exact solution of the 1-D Riemann problem for an ideal gas (the pin of the oracle's sweep).

Own implementation of the classical construction: Newton iteration on the pressure function
f(p) = f_L(p) + f_R(p) + (u_R - u_L) = 0 (shock branch from Rankine-Hugoniot, rarefaction branch from the
isentropic relations and Riemann invariants), then sampling of the self-similar solution at xi = x/t.
Independent of oracle/ and of the CUDA path.
"""
import numpy as np


def _f(p, rho, pk, g):
    c = np.sqrt(g * pk / rho)
    if p > pk:   # shock
        A = 2.0 / ((g + 1.0) * rho)
        B = (g - 1.0) / (g + 1.0) * pk
        f = (p - pk) * np.sqrt(A / (p + B))
        df = np.sqrt(A / (p + B)) * (1.0 - 0.5 * (p - pk) / (p + B))
    else:        # rarefaction
        f = 2.0 * c / (g - 1.0) * ((p / pk) ** ((g - 1.0) / (2.0 * g)) - 1.0)
        df = 1.0 / (rho * c) * (p / pk) ** (-(g + 1.0) / (2.0 * g))
    return f, df


def star_state(rl, ul, pl, rr, ur, pr, g):
    p = 0.5 * (pl + pr)
    for _ in range(100):
        fl, dfl = _f(p, rl, pl, g)
        fr, dfr = _f(p, rr, pr, g)
        dp = (fl + fr + ur - ul) / (dfl + dfr)
        p_new = max(p - dp, 1e-14)
        if abs(p_new - p) < 1e-15 * p:
            p = p_new
            break
        p = p_new
    fl, _ = _f(p, rl, pl, g)
    fr, _ = _f(p, rr, pr, g)
    u = 0.5 * (ul + ur) + 0.5 * (fr - fl)
    return p, u


def sample(xi, rl, ul, pl, rr, ur, pr, g):
    """(rho, u, p) at similarity coordinates xi = x/t (array)."""
    ps, us = star_state(rl, ul, pl, rr, ur, pr, g)
    cl = np.sqrt(g * pl / rl); cr = np.sqrt(g * pr / rr)
    xi = np.asarray(xi, dtype=float)
    rho = np.empty_like(xi); u = np.empty_like(xi); p = np.empty_like(xi)
    gm, gp = g - 1.0, g + 1.0
    for i, s in enumerate(xi):
        if s <= us:   # left of contact
            if ps > pl:   # left shock
                sl = ul - cl * np.sqrt(gp / (2 * g) * ps / pl + gm / (2 * g))
                if s < sl:
                    rho[i], u[i], p[i] = rl, ul, pl
                else:
                    rho[i] = rl * ((ps / pl + gm / gp) / (gm / gp * ps / pl + 1.0)); u[i] = us; p[i] = ps
            else:         # left rarefaction
                shl = ul - cl
                csl = cl * (ps / pl) ** (gm / (2 * g))
                stl = us - csl
                if s < shl:
                    rho[i], u[i], p[i] = rl, ul, pl
                elif s > stl:
                    rho[i] = rl * (ps / pl) ** (1.0 / g); u[i] = us; p[i] = ps
                else:
                    c = 2.0 / gp * (cl + 0.5 * gm * (ul - s))
                    u[i] = 2.0 / gp * (cl + 0.5 * gm * ul + s)
                    rho[i] = rl * (c / cl) ** (2.0 / gm)
                    p[i] = pl * (c / cl) ** (2.0 * g / gm)
        else:         # right of contact
            if ps > pr:   # right shock
                sr = ur + cr * np.sqrt(gp / (2 * g) * ps / pr + gm / (2 * g))
                if s > sr:
                    rho[i], u[i], p[i] = rr, ur, pr
                else:
                    rho[i] = rr * ((ps / pr + gm / gp) / (gm / gp * ps / pr + 1.0)); u[i] = us; p[i] = ps
            else:
                shr = ur + cr
                csr = cr * (ps / pr) ** (gm / (2 * g))
                str_ = us + csr
                if s > shr:
                    rho[i], u[i], p[i] = rr, ur, pr
                elif s < str_:
                    rho[i] = rr * (ps / pr) ** (1.0 / g); u[i] = us; p[i] = ps
                else:
                    c = 2.0 / gp * (cr - 0.5 * gm * (ur - s))
                    u[i] = 2.0 / gp * (-cr + 0.5 * gm * ur + s)
                    rho[i] = rr * (c / cr) ** (2.0 / gm)
                    p[i] = pr * (c / cr) ** (2.0 * g / gm)
    return rho, u, p


def shock_speed_right(rr, ur, pr, ps, g):
    cr = np.sqrt(g * pr / rr)
    return ur + cr * np.sqrt((g + 1) / (2 * g) * ps / pr + (g - 1) / (2 * g))
