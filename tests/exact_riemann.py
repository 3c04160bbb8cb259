"""Exact solution of the Riemann problem for the ideal-gas Euler equations (textbook: Newton iteration
on the pressure function f_L(p) + f_R(p) + u_R - u_L = 0 with the shock / rarefaction branches).
Used only as a PIN for the oracle; independent of oracle/ and of the CUDA path.
"""
import numpy as np


def _f(p, rho, pk, g):
    a = np.sqrt(g * pk / rho)
    if p > pk:   # shock
        A = 2.0 / ((g + 1.0) * rho)
        B = (g - 1.0) / (g + 1.0) * pk
        return (p - pk) * np.sqrt(A / (p + B)), np.sqrt(A / (p + B)) * (1.0 - 0.5 * (p - pk) / (B + p))
    return 2.0 * a / (g - 1.0) * ((p / pk) ** ((g - 1.0) / (2.0 * g)) - 1.0), 1.0 / (rho * a) * (p / pk) ** (-(g + 1.0) / (2.0 * g))


def star_state(rl, ul, pl, rr, ur, pr, g):
    p = 0.5 * (pl + pr)
    for _ in range(100):
        fl, dfl = _f(p, rl, pl, g)
        fr, dfr = _f(p, rr, pr, g)
        dp = (fl + fr + ur - ul) / (dfl + dfr)
        p = max(1e-14, p - dp)
        if abs(dp) < 1e-15 * p:
            break
    fl, _ = _f(p, rl, pl, g)
    fr, _ = _f(p, rr, pr, g)
    u = 0.5 * (ul + ur) + 0.5 * (fr - fl)
    gm = (g - 1.0) / (g + 1.0)
    rsl = rl * ((p / pl + gm) / (gm * p / pl + 1.0)) if p > pl else rl * (p / pl) ** (1.0 / g)
    rsr = rr * ((p / pr + gm) / (gm * p / pr + 1.0)) if p > pr else rr * (p / pr) ** (1.0 / g)
    return p, u, rsl, rsr


def sample(xi, rl, ul, pl, rr, ur, pr, g):
    """(rho, u, p) at similarity coordinate xi = (x - x0)/t (array)."""
    ps, us, rsl, rsr = star_state(rl, ul, pl, rr, ur, pr, g)
    xi = np.asarray(xi, dtype=np.float64)
    rho = np.empty_like(xi)
    u = np.empty_like(xi)
    p = np.empty_like(xi)
    al, ar = np.sqrt(g * pl / rl), np.sqrt(g * pr / rr)
    for n, s in enumerate(xi.flat):
        if s <= us:     # left of the contact
            if ps > pl:
                sl = ul - al * np.sqrt((g + 1.0) / (2.0 * g) * ps / pl + (g - 1.0) / (2.0 * g))
                w = (rl, ul, pl) if s < sl else (rsl, us, ps)
            else:
                asl = al * (ps / pl) ** ((g - 1.0) / (2.0 * g))
                if s < ul - al:
                    w = (rl, ul, pl)
                elif s > us - asl:
                    w = (rsl, us, ps)
                else:
                    c = 2.0 / (g + 1.0) + (g - 1.0) / ((g + 1.0) * al) * (ul - s)
                    w = (rl * c ** (2.0 / (g - 1.0)), 2.0 / (g + 1.0) * (al + (g - 1.0) / 2.0 * ul + s), pl * c ** (2.0 * g / (g - 1.0)))
        else:
            if ps > pr:
                sr = ur + ar * np.sqrt((g + 1.0) / (2.0 * g) * ps / pr + (g - 1.0) / (2.0 * g))
                w = (rr, ur, pr) if s > sr else (rsr, us, ps)
            else:
                asr = ar * (ps / pr) ** ((g - 1.0) / (2.0 * g))
                if s > ur + ar:
                    w = (rr, ur, pr)
                elif s < us + asr:
                    w = (rsr, us, ps)
                else:
                    c = 2.0 / (g + 1.0) - (g - 1.0) / ((g + 1.0) * ar) * (ur - s)
                    w = (rr * c ** (2.0 / (g - 1.0)), 2.0 / (g + 1.0) * (-ar + (g - 1.0) / 2.0 * ur + s), pr * c ** (2.0 * g / (g - 1.0)))
        rho.flat[n], u.flat[n], p.flat[n] = w
    return rho, u, p
