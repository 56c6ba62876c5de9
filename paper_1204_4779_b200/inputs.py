"""Seeded synthetic inputs: the five BASELINE.json configs and scaled-down / ragged variants.

This module serves BOTH the CUDA path's callers (tests, bench.py, smoke) and the oracle's callers.
It holds none of the method's arithmetic: it only states initial conditions.  Everything is
generated once on the host in fp64 with NumPy `default_rng(seed)` (PCG64), converted to conserved
variables with the definitions of PAPER.md:694 (m_a = rho v_a, E = p/(gamma-1) + rho v^2/2) in fp64,
and cast once to the workload dtype; the identical bits are handed to the GPU library and to the
oracle.  The paper does not say which initial condition its scores were measured on (only grid
sizes and precisions); BASELINE.json's configs are the workloads and no public
dataset is involved.  Recipes: DESIGN.md §5.

Array layout: (nf, [nz,] [ny,] nx), C order, x fastest; fields rho, m_x[, m_y[, m_z]], E.
"""
from dataclasses import dataclass, field

import numpy as np


@dataclass
class Workload:
    name: str
    n: tuple  # cells per axis, x first
    extent: tuple
    gamma: float
    dtype: np.dtype
    boundary: str  # "periodic" | "outflow"
    cfl: float
    steps: int  # number of steps of the config (upper bound when t_end > 0)
    t_end: float = 0.0
    U: np.ndarray = field(default=None, repr=False)  # conserved variables, cast to dtype

    @property
    def dims(self):
        return len(self.n)

    @property
    def nf(self):
        return self.dims + 2

    @property
    def cells(self):
        return int(np.prod(self.n))


def conserved_from_primitive(rho, v, p, gamma):
    """(rho, [v_x, ...], p) -> stacked (rho, m_x.., E) in fp64.  Definitions of PAPER.md:694."""
    rho = np.asarray(rho, np.float64)
    v = [np.asarray(c, np.float64) for c in v]
    q = sum(c * c for c in v)
    E = np.asarray(p, np.float64) / (gamma - 1.0) + 0.5 * rho * q
    return np.stack([rho] + [rho * c for c in v] + [E])


def _centres(n, extent=1.0):
    return (np.arange(n, dtype=np.float64) + 0.5) * (extent / n)


def sod(n=256, dtype=np.float64, axis=0, dims=1, n_other=4):
    """Config 0: 1-D Sod tube on [0,1], gamma 1.4, outflow, CFL 0.4, t_end 0.2.

    dims > 1 embeds the same 1-D problem along `axis` of a dims-D grid (other axes uniform, n_other
    cells, extent n_other/n so that cells stay cubic)."""
    x = _centres(n)
    left = x < 0.5
    rho1, p1 = np.where(left, 1.0, 0.125), np.where(left, 1.0, 0.1)
    shape_n = [n_other] * dims
    shape_n[axis] = n
    ext = [n_other / n] * dims
    ext[axis] = 1.0
    bshape = [1] * dims
    bshape[dims - 1 - axis] = n  # arrays are indexed [z][y][x]
    full = tuple(reversed(shape_n))
    rho = np.broadcast_to(rho1.reshape(bshape), full)
    p = np.broadcast_to(p1.reshape(bshape), full)
    v = [np.zeros(full) for _ in range(dims)]
    U = conserved_from_primitive(rho, v, p, 1.4)
    return Workload(f"sod{dims}d_n{n}_axis{axis}", tuple(shape_n), tuple(ext), 1.4, np.dtype(dtype), "outflow",
                    0.4, 100000, 0.2, np.ascontiguousarray(U.astype(dtype)))


def kelvin_helmholtz(nx=1024, ny=None, dtype=np.float32, seed=0, steps=100):
    """Configs 1 and 2: 2-D Kelvin-Helmholtz on [0,1]^2, periodic, gamma 1.4, CFL 0.4."""
    ny = nx if ny is None else ny
    y = _centres(ny)[:, None]
    inner = np.abs(y - 0.5) < 0.25
    rho = np.broadcast_to(np.where(inner, 2.0, 1.0), (ny, nx)).copy()
    vx = np.broadcast_to(np.where(inner, 0.5, -0.5), (ny, nx)).copy()
    vy = np.zeros((ny, nx))
    p = np.full((ny, nx), 2.5)
    rng = np.random.default_rng(seed)
    vx += 0.01 * rng.uniform(-1.0, 1.0, (ny, nx))
    vy += 0.01 * rng.uniform(-1.0, 1.0, (ny, nx))
    U = conserved_from_primitive(rho, [vx, vy], p, 1.4)
    return Workload(f"kh2d_{nx}x{ny}_{np.dtype(dtype).name}_seed{seed}", (nx, ny), (1.0, 1.0), 1.4, np.dtype(dtype),
                    "periodic", 0.4, steps, 0.0, np.ascontiguousarray(U.astype(dtype)))


def blast(n=256, dtype=np.float32, seed=2, steps=50, shape=None):
    """Configs 3 and 4: 3-D blast in a clumpy medium on [0,1]^3, periodic, gamma 5/3, CFL 0.3.

    rho = exp(0.5 g~), g~ = periodic 3x3x3 box mean of i.i.d. N(0,1); v = 0;
    p = 1 + 100 exp(-r^2 / 0.05^2) centred on the cube.  `shape` = (nx, ny, nz) for ragged variants."""
    nx, ny, nz = (n, n, n) if shape is None else shape
    rng = np.random.default_rng(seed)
    g = rng.standard_normal((nz, ny, nx))
    for ax in range(3):  # separable periodic 3-point mean along each axis = 27-point box mean
        g = (np.roll(g, 1, ax) + g + np.roll(g, -1, ax)) / 3.0
    rho = np.exp(0.5 * g)
    del g
    z = _centres(nz)[:, None, None]
    y = _centres(ny)[None, :, None]
    x = _centres(nx)[None, None, :]
    r2 = (x - 0.5) ** 2 + (y - 0.5) ** 2 + (z - 0.5) ** 2
    p = 1.0 + 100.0 * np.exp(-r2 / 0.05**2)
    gamma = 5.0 / 3.0
    zero = np.zeros_like(rho)
    U = np.empty((5, nz, ny, nx), dtype)
    U[0] = rho
    U[1] = zero
    U[2] = zero
    U[3] = zero
    U[4] = p / (gamma - 1.0)  # v = 0: E = p/(gamma-1)
    return Workload(f"blast3d_{nx}x{ny}x{nz}_{np.dtype(dtype).name}_seed{seed}", (nx, ny, nz), (1.0, 1.0, 1.0), gamma,
                    np.dtype(dtype), "periodic", 0.3, steps, 0.0, U)


def random_smooth(n, dtype=np.float64, seed=0, gamma=1.4, boundary="periodic", jump=True):
    """Generic test state on an arbitrary (possibly ragged, non-cubic) grid: smooth random modes plus,
    optionally, a density/pressure jump so that limiter branches and all Riemann-fan cases occur."""
    n = tuple(int(v) for v in n)
    dims = len(n)
    rng = np.random.default_rng(seed)
    shape = tuple(reversed(n))
    grids = np.meshgrid(*[_centres(m) for m in reversed(n)], indexing="ij")  # [z][y][x] order
    phase = rng.uniform(0, 2 * np.pi, (dims + 2, dims))
    amp = rng.uniform(0.1, 0.4, dims + 2)

    def mode(f):
        s = np.zeros(shape)
        for d in range(dims):
            s = s + np.sin(2 * np.pi * (d + 1) * grids[d] + phase[f, d])
        return amp[f] * s / dims

    rho = 1.0 + mode(0)
    p = 1.0 + mode(dims + 1)
    v = [1.5 * mode(1 + b) + 0.3 * rng.uniform(-1, 1) for b in range(dims)]
    if jump:
        box = np.ones(shape, bool)
        for d in range(dims):
            box &= np.abs(grids[d] - 0.5) < 0.2
        rho = np.where(box, 3.0 * rho, rho)
        p = np.where(box, 8.0 * p, p)
    rho = rho + 0.01 * rng.uniform(-1, 1, shape)
    U = conserved_from_primitive(rho, v, p, gamma)
    ext = tuple(1.0 for _ in n)
    return Workload(f"random{dims}d_{'x'.join(map(str, n))}_seed{seed}", n, ext, gamma, np.dtype(dtype), boundary, 0.4,
                    10, 0.0, np.ascontiguousarray(U.astype(dtype)))


def hypersonic(n, dtype=np.float32, mach=50.0, seed=3):
    """Edge-case state (not a BASELINE config): a slab 0.25 < x < 0.75 of (rho, p) = (1, 1) gas in a medium of
    (1e-6, 1e-6), 1 % noise on both, v_x = +mach c for x < 0.5 and -mach c beyond (c = sqrt(gamma)): supersonic faces of
    both signs, a 10^6 density jump swept at Mach `mach`, a head-on collision in the middle.  Transverse velocities are
    0.3 Uniform(-1, 1).  gamma 1.4, periodic, CFL 0.4."""
    n = tuple(int(v) for v in n)
    dims = len(n)
    shape = tuple(reversed(n))
    rng = np.random.default_rng(seed)
    gamma = 1.4
    X = np.broadcast_to(_centres(n[0]), shape)
    dense = (X > 0.25) & (X < 0.75)
    rho = np.where(dense, 1.0, 1e-6) * (1.0 + 0.01 * rng.uniform(-1, 1, shape))
    p = np.where(dense, 1.0, 1e-6) * (1.0 + 0.01 * rng.uniform(-1, 1, shape))
    c = np.sqrt(gamma)
    v = [np.where(X < 0.5, mach * c, -mach * c) * np.ones(shape)] + [0.3 * rng.uniform(-1, 1, shape) for _ in range(dims - 1)]
    U = conserved_from_primitive(rho, v, p, gamma)
    return Workload(f"hypersonic{dims}d_{'x'.join(map(str, n))}_mach{mach:g}", n, tuple(1.0 for _ in n), gamma,
                    np.dtype(dtype), "periodic", 0.4, 3, 0.0, np.ascontiguousarray(U.astype(dtype)))


def baseline_config(i, scale=1.0):
    """BASELINE.json configs[i]; scale < 1 shrinks the grid (same recipe) for quick parity runs."""
    s = lambda m: max(8, int(round(m * scale)))
    if i == 0:
        return sod(s(256))
    if i == 1:
        return kelvin_helmholtz(s(1024), dtype=np.float32, seed=0, steps=100)
    if i == 2:
        return kelvin_helmholtz(s(4096), dtype=np.float64, seed=1, steps=50)
    if i == 3:
        return blast(s(256), np.float32, seed=2, steps=50)
    if i == 4:
        return blast(s(512), np.float32, seed=3, steps=20)
    if i == 11:  # not a BASELINE config: config 1's recipe at 4096^2 (fp32), the 2-D fp32 case that is NOT L2-resident
        return kelvin_helmholtz(s(4096), dtype=np.float32, seed=0, steps=50)
    if i == 13:  # not a BASELINE config: config 3's recipe in fp64 (the 3-D fp64 case)
        return blast(s(256), np.float64, seed=2, steps=20)
    raise ValueError(i)
