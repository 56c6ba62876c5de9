"""Exact solution of the 1-D Riemann problem for the ideal-gas Euler equations (test helper, pin P5).

Textbook construction (Toro's textbook ch. 4, PAPER.md ref [30]): Newton iteration on the pressure
function f(p) = f_L(p) + f_R(p) + (u_R - u_L), then sampling of the self-similar solution.
Independent of oracle/ and of the CUDA path.
"""
import numpy as np


def _f(p, rho, pk, g):
    A = 2.0 / ((g + 1.0) * rho)
    B = (g - 1.0) / (g + 1.0) * pk
    c = np.sqrt(g * pk / rho)
    if p > pk:  # shock
        f = (p - pk) * np.sqrt(A / (p + B))
        df = np.sqrt(A / (B + p)) * (1.0 - (p - pk) / (2.0 * (B + p)))
    else:  # rarefaction
        f = 2.0 * c / (g - 1.0) * ((p / pk) ** ((g - 1.0) / (2.0 * g)) - 1.0)
        df = 1.0 / (rho * c) * (p / pk) ** (-(g + 1.0) / (2.0 * g))
    return f, df


def star_state(L, R, g):
    (rl, ul, pl), (rr, ur, pr) = L, R
    p = 0.5 * (pl + pr)
    for _ in range(100):
        fl, dfl = _f(p, rl, pl, g)
        fr, dfr = _f(p, rr, pr, g)
        pn = max(1e-14, p - (fl + fr + ur - ul) / (dfl + dfr))
        if abs(pn - p) < 1e-15 * max(p, pn):
            p = pn
            break
        p = pn
    fl, _ = _f(p, rl, pl, g)
    fr, _ = _f(p, rr, pr, g)
    u = 0.5 * (ul + ur) + 0.5 * (fr - fl)
    return p, u


def sample(xi, L, R, g):
    """Primitive state (rho, u, p) on the ray x/t = xi (array)."""
    (rl, ul, pl), (rr, ur, pr) = L, R
    ps, us = star_state(L, R, g)
    cl, cr = np.sqrt(g * pl / rl), np.sqrt(g * pr / rr)
    xi = np.asarray(xi, np.float64)
    rho, u, p = np.empty_like(xi), np.empty_like(xi), np.empty_like(xi)
    gm, gp = g - 1.0, g + 1.0
    left = xi <= us
    # ---- left of the contact
    if ps > pl:  # left shock
        rs = rl * (ps / pl + gm / gp) / (gm / gp * ps / pl + 1.0)
        sl = ul - cl * np.sqrt(gp / (2 * g) * ps / pl + gm / (2 * g))
        m = left & (xi < sl)
        rho[m], u[m], p[m] = rl, ul, pl
        m = left & (xi >= sl)
        rho[m], u[m], p[m] = rs, us, ps
    else:  # left rarefaction
        rs = rl * (ps / pl) ** (1.0 / g)
        cs = cl * (ps / pl) ** (gm / (2 * g))
        head, tail = ul - cl, us - cs
        m = left & (xi < head)
        rho[m], u[m], p[m] = rl, ul, pl
        m = left & (xi >= head) & (xi <= tail)
        fac = 2.0 / gp + gm / (gp * cl) * (ul - xi[m])
        rho[m] = rl * fac ** (2.0 / gm)
        u[m] = 2.0 / gp * (cl + gm / 2.0 * ul + xi[m])
        p[m] = pl * fac ** (2.0 * g / gm)
        m = left & (xi > tail)
        rho[m], u[m], p[m] = rs, us, ps
    # ---- right of the contact
    right = ~left
    if ps > pr:  # right shock
        rs = rr * (ps / pr + gm / gp) / (gm / gp * ps / pr + 1.0)
        sr = ur + cr * np.sqrt(gp / (2 * g) * ps / pr + gm / (2 * g))
        m = right & (xi > sr)
        rho[m], u[m], p[m] = rr, ur, pr
        m = right & (xi <= sr)
        rho[m], u[m], p[m] = rs, us, ps
    else:
        rs = rr * (ps / pr) ** (1.0 / g)
        cs = cr * (ps / pr) ** (gm / (2 * g))
        head, tail = ur + cr, us + cs
        m = right & (xi > head)
        rho[m], u[m], p[m] = rr, ur, pr
        m = right & (xi <= head) & (xi >= tail)
        fac = 2.0 / gp - gm / (gp * cr) * (ur - xi[m])
        rho[m] = rr * fac ** (2.0 / gm)
        u[m] = 2.0 / gp * (-cr + gm / 2.0 * ur + xi[m])
        p[m] = pr * fac ** (2.0 * g / gm)
        m = right & (xi < tail)
        rho[m], u[m], p[m] = rs, us, ps
    return rho, u, p


def cell_averaged_density(n, t, L, R, g, x0=0.5, sub=64):
    """Cell averages of the exact density on n cells of [0,1] (midpoint rule on `sub` sub-cells)."""
    xs = (np.arange(n * sub) + 0.5) / (n * sub)
    rho, _, _ = sample((xs - x0) / t, L, R, g)
    return rho.reshape(n, sub).mean(axis=1)
