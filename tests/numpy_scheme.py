"""Independent definition-level restatement of the scheme in vectorised NumPy (test helper, pin P11).

Written from PAPER.md Eq. 13-27 and DESIGN.md §3's readings, NOT from oracle/euler_oracle.cpp: it
works on whole arrays with np.roll / edge padding instead of per-face loops, uses no fused
multiply-add, and evaluates the HLLC star flux in the OTHER textbook form
    F*K = [ S*(SK UK - FK) + SK (pK + rhoK (SK - uK)(S* - uK)) D* ] / (SK - S*),  D* = (0, e_a, S*)
(Toro's textbook §10.4, PAPER.md ref [30]) which is algebraically identical to the
F*K = FK + SK(U*K - UK) form the oracle and the CUDA path use.  Agreement is therefore to rounding
(~1e-14 relative in fp64), not bitwise — which is what makes it a pin rather than a copy.
Only for tiny grids.
"""
import numpy as np


def prim(U, g):
    d = U.shape[0] - 2
    rho = U[0]
    v = [U[1 + b] / rho for b in range(d)]
    q = sum(c * c for c in v)
    p = (g - 1.0) * (U[d + 1] - 0.5 * rho * q)
    return np.stack([rho] + v + [p])


def _shift(A, s, ax, boundary):
    """A sampled at index i+s along array axis ax (ghosts by wrap or by clamping the index)."""
    if boundary == "periodic":
        return np.roll(A, -s, axis=ax)
    n = A.shape[ax]
    idx = np.clip(np.arange(n) + s, 0, n - 1)
    return np.take(A, idx, axis=ax)


def _minbee(y0, y1, y2):
    d01, d12 = y1 - y0, y2 - y1
    dy = np.where(d01 * d12 < 0, 0.0, np.where(np.abs(d01) < np.abs(d12), d01, d12))
    return y1 - 0.5 * dy, y1 + 0.5 * dy


def _mc(y0, y1, y2):
    """Monotonized-central limiter in the textbook form (van Leer 1977): sign(d) max(0, min(2|a|, 2|b|, |c|)) when the
    one-sided differences a, b agree in sign, else 0 (c = their mean) — written through np.sign, not the product test."""
    a, b = y1 - y0, y2 - y1
    c = 0.5 * (a + b)
    same = np.sign(a) * np.sign(b) > 0
    dy = np.where(same, np.sign(c) * np.minimum(np.minimum(2 * np.abs(a), 2 * np.abs(b)), np.abs(c)), 0.0)
    return y1 - 0.5 * dy, y1 + 0.5 * dy


def _none(y0, y1, y2):
    return y1, y1


LIMITERS = {"minbee": _minbee, "none": _none, "mc": _mc}


def _flux_phys(V, a, g):
    d = V.shape[0] - 2
    rho, p, vn = V[0], V[d + 1], V[1 + a]
    q = sum(V[1 + b] ** 2 for b in range(d))
    E = p / (g - 1.0) + 0.5 * rho * q
    Uc = np.stack([rho] + [rho * V[1 + b] for b in range(d)] + [E])
    F = np.stack([rho * vn] + [rho * vn * V[1 + b] + (p if b == a else 0.0) for b in range(d)] + [vn * (E + p)])
    return Uc, F


def riemann(VL, VR, a, g, kind):
    d = VL.shape[0] - 2
    UL, FL = _flux_phys(VL, a, g)
    UR, FR = _flux_phys(VR, a, g)
    cL, cR = np.sqrt(g * VL[d + 1] / VL[0]), np.sqrt(g * VR[d + 1] / VR[0])
    uL, uR = VL[1 + a], VR[1 + a]
    SL = np.minimum(uL - cL, uR - cR)
    SR = np.maximum(uL + cL, uR + cR)
    if kind == "hll":
        Fs = (SR * FL - SL * FR + SL * SR * (UR - UL)) / (SR - SL)
        return np.where(SL >= 0, FL, np.where(SR <= 0, FR, Fs))
    pL, pR, rL, rR = VL[d + 1], VR[d + 1], VL[0], VR[0]
    Ss = (pR - pL + rL * uL * (SL - uL) - rR * uR * (SR - uR)) / (rL * (SL - uL) - rR * (SR - uR))
    Dstar = np.zeros_like(FL)
    Dstar[1 + a] = 1.0
    Dstar[d + 1] = Ss
    FsL = (Ss * (SL * UL - FL) + SL * (pL + rL * (SL - uL) * (Ss - uL)) * Dstar) / (SL - Ss)
    FsR = (Ss * (SR * UR - FR) + SR * (pR + rR * (SR - uR) * (Ss - uR)) * Dstar) / (SR - Ss)
    return np.where(SL >= 0, FL, np.where(SR <= 0, FR, np.where(Ss >= 0, FsL, FsR)))


def stage(Uin, Ubase, tau, dr, g, boundary, kind, limiter="minbee"):
    d = Uin.shape[0] - 2
    V = prim(Uin, g)
    out = Ubase.copy()
    for a in range(d):
        ax = V.ndim - 1 - a  # array axes are [f][z][y][x]
        lo, hi = LIMITERS[limiter](_shift(V, -1, ax, boundary), V, _shift(V, 1, ax, boundary))
        # flux at face i+1/2: left state hi(i), right state lo(i+1)
        Fp = riemann(hi, _shift(lo, 1, ax, boundary), a, g, kind)
        if boundary == "periodic":
            Fm = np.roll(Fp, 1, axis=ax)
        else:
            # face -1/2: both ghost cells equal cell 0 -> zero slopes -> VL = V[0]; VR = lo(cell 0)
            first = np.take(V, [0], axis=ax)
            lo0 = np.take(lo, [0], axis=ax)
            F0 = riemann(first, lo0, a, g, kind)
            Fm = np.concatenate([F0, np.take(Fp, np.arange(Fp.shape[ax] - 1), axis=ax)], axis=ax)
        out = out + (tau / dr[a]) * (Fm - Fp)
    return out


def step(U, dt, dr, g, boundary="periodic", kind="hllc", limiter="minbee"):
    U1 = stage(U, U, 0.5 * dt, dr, g, boundary, kind, limiter)
    return stage(U1, U, dt, dr, g, boundary, kind, limiter)


def cfl_dt(U, cfl, dr, g):
    d = U.shape[0] - 2
    V = prim(U, g)
    c = np.sqrt(g * V[d + 1] / V[0])
    S = max(((np.abs(V[1 + a]) + c) / dr[a]).max() for a in range(d))
    return cfl / S
