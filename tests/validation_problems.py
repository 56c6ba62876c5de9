"""The paper's validation procedure (Eq. 28-31, Fig. 10): entropy wave, sound wave and Sod's shock
tube on the unit square, "coaxial" and "oblique" (rotated by 60 degrees about the centre), the analytic solution
substituted into the ghost cells all the time, L1 error of the density against the analytic solution at t = 1 (waves) /
t = 0.125 (shock tube), N = 16^2 ... 1024^2.  Test helper shared by the oracle pins (P16) and the GPU tests; it holds the
analytic solutions and the driver loop, none of the scheme's arithmetic.

Ghost cells: the outermost two cells of every axis (R23), so an N^2 run has (N-4)^2 evolved cells on the same
mesh; the error is taken over the evolved cells.  The time step is fixed from the analytic maximum signal speed
(CFL 0.4) so that every implementation takes the same steps.
"""
import math

import numpy as np

import exact_riemann

GAMMA = 1.4
T_END = {"entropy": 1.0, "sound": 1.0, "sod": 0.125}
SOD_L, SOD_R = (1.0, 0.0, 1.0), (0.125, 0.0, 0.1)  # Eq. 30-31 with R15: p = 0.1 on the right


def primitives(problem, theta, X, Y, t):
    """(rho, vx, vy, p) of the analytic solution at time t; theta = rotation angle about (0.5, 0.5)."""
    c, s = math.cos(theta), math.sin(theta)
    xi = 0.5 + (X - 0.5) * c + (Y - 0.5) * s  # coordinate along the rotated x axis
    if problem == "entropy":      # Eq. 28: a density profile carried at v = 1
        rho, u, p = 2.0 + np.sin(2 * np.pi * (xi - t)), np.ones_like(xi), np.ones_like(xi)
    elif problem == "sound":      # Eq. 29: right-going acoustic wave on rho0 = gamma, p0 = 1 (c0 = 1), amplitude 1e-5
        A = 1e-5
        w = np.sin(2 * np.pi * (xi - t))
        rho, u, p = GAMMA * (1 + A * w), A * w, 1 + GAMMA * A * w
    else:                         # Eq. 30-31: Sod, the exact Riemann solution on rays from xi = 0.5
        if t <= 0:
            left = xi < 0.5
            rho, u, p = (np.where(left, SOD_L[k], SOD_R[k]) for k in range(3))
        else:
            rho, u, p = exact_riemann.sample((xi - 0.5) / t, SOD_L, SOD_R, GAMMA)
    return rho, u * c, u * s, p


def conserved(problem, theta, X, Y, t, dtype):
    rho, vx, vy, p = primitives(problem, theta, X, Y, t)
    E = p / (GAMMA - 1.0) + 0.5 * rho * (vx * vx + vy * vy)
    return np.ascontiguousarray(np.stack([rho, rho * vx, rho * vy, E]).astype(dtype))


def max_speed(problem):
    if problem == "entropy":
        return 1.0 + math.sqrt(GAMMA * 1.0 / 1.0)     # |v| + c at the density minimum rho = 1
    if problem == "sound":
        return 1.0 + 2e-5
    return 2.2                                        # Sod: shock speed 1.75, |u*| + c* < 2.2


def run(stepper, problem, n, theta, dtype=np.float64):
    """Drive `stepper` (set_state / set_ghosts / step_ghosts / get_state: the oracle or the CUDA handle) through the
    whole test; returns (L1 density error over the evolved cells, final state, steps)."""
    x = (np.arange(n) + 0.5) / n
    X, Y = np.meshgrid(x, x)  # arrays are [y][x]
    T = T_END[problem]
    steps = int(math.ceil(T / (0.4 / (max_speed(problem) * n))))
    dt = T / steps
    stepper.set_state(conserved(problem, theta, X, Y, 0.0, dtype))
    G = np.empty((4, n, n), dtype)
    ring = np.ones((n, n), bool)
    ring[2:-2, 2:-2] = False
    Xr, Yr = X[ring], Y[ring]

    def ghosts(t):  # only the ghost cells are read by the solver: fill just those
        G[:, ring] = conserved(problem, theta, Xr, Yr, t, dtype)
        return G

    for k in range(steps):
        t = k * dt
        stepper.set_ghosts(ghosts(t))
        stepper.step_ghosts(dt, ghosts(t + 0.5 * dt))
    U = stepper.get_state()
    rho_exact = primitives(problem, theta, X, Y, T)[0]
    err = np.abs(U[0].astype(np.float64) - rho_exact)[2:-2, 2:-2].mean()
    return err, U, steps
