"""Exact solution of the Riemann problem for the 1-D Euler equations with an ideal gas
(textbook closed form: Newton iteration on the star pressure, then sampling; e.g. Toro 1999,
cited at PAPER.md:346).  Used only to pin the oracle (pins P4, P5)."""
import numpy as np


def _f(p, rho, pk, g):
    a = np.sqrt(g * pk / rho)
    if p > pk:      # shock
        A, B = 2.0 / ((g + 1.0) * rho), (g - 1.0) / (g + 1.0) * pk
        f = (p - pk) * np.sqrt(A / (p + B))
        df = np.sqrt(A / (p + B)) * (1.0 - 0.5 * (p - pk) / (p + B))
    else:           # rarefaction
        f = 2.0 * a / (g - 1.0) * ((p / pk) ** ((g - 1.0) / (2.0 * g)) - 1.0)
        df = 1.0 / (rho * a) * (p / pk) ** (-(g + 1.0) / (2.0 * g))
    return f, df


def star(rl, ul, pl, rr, ur, pr, g):
    p = max(1e-8, 0.5 * (pl + pr))
    for _ in range(200):
        fl, dl = _f(p, rl, pl, g)
        fr, dr = _f(p, rr, pr, g)
        pn = max(1e-12, p - (fl + fr + ur - ul) / (dl + dr))
        if abs(pn - p) <= 1e-15 * (pn + p):
            p = pn
            break
        p = pn
    fl, _ = _f(p, rl, pl, g)
    fr, _ = _f(p, rr, pr, g)
    return p, 0.5 * (ul + ur) + 0.5 * (fr - fl)


def sample(xi, rl, ul, pl, rr, ur, pr, g):
    """rho, u, p at similarity coordinate xi = (x - x0)/t (array)."""
    ps, us = star(rl, ul, pl, rr, ur, pr, g)
    xi = np.asarray(xi, dtype=np.float64)
    rho, u, p = np.empty_like(xi), np.empty_like(xi), np.empty_like(xi)
    al, ar = np.sqrt(g * pl / rl), np.sqrt(g * pr / rr)
    for i, s in enumerate(xi):
        if s <= us:   # left of contact
            if ps > pl:
                sl = ul - al * np.sqrt((g + 1) / (2 * g) * ps / pl + (g - 1) / (2 * g))
                if s <= sl:
                    rho[i], u[i], p[i] = rl, ul, pl
                else:
                    rho[i] = rl * ((ps / pl + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * ps / pl + 1))
                    u[i], p[i] = us, ps
            else:
                shl, stl = ul - al, us - al * (ps / pl) ** ((g - 1) / (2 * g))
                if s <= shl:
                    rho[i], u[i], p[i] = rl, ul, pl
                elif s >= stl:
                    rho[i], u[i], p[i] = rl * (ps / pl) ** (1 / g), us, ps
                else:
                    c = 2 / (g + 1) + (g - 1) / ((g + 1) * al) * (ul - s)
                    rho[i], u[i], p[i] = rl * c ** (2 / (g - 1)), 2 / (g + 1) * (al + (g - 1) / 2 * ul + s), pl * c ** (2 * g / (g - 1))
        else:
            if ps > pr:
                sr = ur + ar * np.sqrt((g + 1) / (2 * g) * ps / pr + (g - 1) / (2 * g))
                if s >= sr:
                    rho[i], u[i], p[i] = rr, ur, pr
                else:
                    rho[i] = rr * ((ps / pr + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * ps / pr + 1))
                    u[i], p[i] = us, ps
            else:
                shr, str_ = ur + ar, us + ar * (ps / pr) ** ((g - 1) / (2 * g))
                if s >= shr:
                    rho[i], u[i], p[i] = rr, ur, pr
                elif s <= str_:
                    rho[i], u[i], p[i] = rr * (ps / pr) ** (1 / g), us, ps
                else:
                    c = 2 / (g + 1) - (g - 1) / ((g + 1) * ar) * (ur - s)
                    rho[i], u[i], p[i] = rr * c ** (2 / (g - 1)), 2 / (g + 1) * (-ar + (g - 1) / 2 * ur + s), pr * c ** (2 * g / (g - 1))
    return rho, u, p
