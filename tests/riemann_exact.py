"""Exact solution of the 1-D Riemann problem for an ideal gas (textbook iterative solver: Newton iteration on the
star-region pressure, then sampling along x/t).  Test helper: it pins the oracle (PAPER.md:460-482 validates GAMER
against this solution); it shares nothing with oracle/ or the CUDA path."""
import numpy as np


def _f_and_df(p, rho_k, p_k, a_k, g):
    if p > p_k:     # shock
        A = 2.0 / ((g + 1.0) * rho_k)
        B = (g - 1.0) / (g + 1.0) * p_k
        s = np.sqrt(A / (p + B))
        return (p - p_k) * s, s * (1.0 - 0.5 * (p - p_k) / (B + p))
    pr = p / p_k    # rarefaction
    return 2.0 * a_k / (g - 1.0) * (pr ** ((g - 1.0) / (2.0 * g)) - 1.0), (1.0 / (rho_k * a_k)) * pr ** (-(g + 1.0) / (2.0 * g))


def star_state(rl, ul, pl, rr, ur, pr, g):
    al, ar = np.sqrt(g * pl / rl), np.sqrt(g * pr / rr)
    p = max(1e-12, 0.5 * (pl + pr))
    for _ in range(200):
        fl, dfl = _f_and_df(p, rl, pl, al, g)
        fr, dfr = _f_and_df(p, rr, pr, ar, g)
        dp = (fl + fr + (ur - ul)) / (dfl + dfr)
        p_new = max(1e-14, p - dp)
        if abs(p_new - p) <= 1e-15 * (p_new + p):
            p = p_new
            break
        p = p_new
    fl, _ = _f_and_df(p, rl, pl, al, g)
    fr, _ = _f_and_df(p, rr, pr, ar, g)
    u = 0.5 * (ul + ur) + 0.5 * (fr - fl)
    return p, u


def sample(xi, rl, ul, pl, rr, ur, pr, g):
    """Solution (rho, u, p) at similarity coordinates xi = (x - x0)/t (array)."""
    xi = np.asarray(xi, np.float64)
    ps, us = star_state(rl, ul, pl, rr, ur, pr, g)
    al, ar = np.sqrt(g * pl / rl), np.sqrt(g * pr / rr)
    rho, u, p = np.empty_like(xi), np.empty_like(xi), np.empty_like(xi)
    gm, gp = g - 1.0, g + 1.0
    for i, s in enumerate(xi.ravel()):
        if s <= us:      # left of the contact
            if ps <= pl:     # left rarefaction
                shl = ul - al
                asl = al * (ps / pl) ** (gm / (2 * g))
                stl = us - asl
                if s <= shl:
                    r, v, q = rl, ul, pl
                elif s >= stl:
                    r, v, q = rl * (ps / pl) ** (1 / g), us, ps
                else:
                    v = 2 / gp * (al + gm / 2 * ul + s)
                    a = 2 / gp * (al + gm / 2 * (ul - s))
                    r = rl * (a / al) ** (2 / gm)
                    q = pl * (a / al) ** (2 * g / gm)
            else:            # left shock
                sl = ul - al * np.sqrt(gp / (2 * g) * ps / pl + gm / (2 * g))
                if s <= sl:
                    r, v, q = rl, ul, pl
                else:
                    r, v, q = rl * ((ps / pl + gm / gp) / (gm / gp * ps / pl + 1)), us, ps
        else:
            if ps > pr:      # right shock
                sr = ur + ar * np.sqrt(gp / (2 * g) * ps / pr + gm / (2 * g))
                if s >= sr:
                    r, v, q = rr, ur, pr
                else:
                    r, v, q = rr * ((ps / pr + gm / gp) / (gm / gp * ps / pr + 1)), us, ps
            else:            # right rarefaction
                shr = ur + ar
                asr = ar * (ps / pr) ** (gm / (2 * g))
                strr = us + asr
                if s >= shr:
                    r, v, q = rr, ur, pr
                elif s <= strr:
                    r, v, q = rr * (ps / pr) ** (1 / g), us, ps
                else:
                    v = 2 / gp * (-ar + gm / 2 * ur + s)
                    a = 2 / gp * (ar - gm / 2 * (ur - s))
                    r = rr * (a / ar) ** (2 / gm)
                    q = pr * (a / ar) ** (2 * g / gm)
        rho.ravel()[i], u.ravel()[i], p.ravel()[i] = r, v, q
    return rho, u, p
