"""ctypes loader for the CPU oracle (TEST INFRASTRUCTURE — see oracle/euler_oracle.cpp header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import
this package.  It imports nothing from paper_1204_4779_b200 (the CUDA path) and vice versa.
"""
import ctypes
import os

import numpy as np

from . import build as _build

_LIBS = {}
_DT = {np.dtype(np.float32): 0, np.dtype(np.float64): 1}
LIMITER = {"minbee": 0, "none": 1, "mc": 2}


def _lib(kind="serial"):
    if kind not in _LIBS:
        path = _build.build()[kind]
        L = ctypes.CDLL(path)
        vp, i64, dbl, cint = ctypes.c_void_p, ctypes.c_int64, ctypes.c_double, ctypes.c_int
        L.oracle_create.restype = vp
        L.oracle_create.argtypes = [cint, ctypes.POINTER(i64), ctypes.POINTER(dbl), dbl, cint]
        L.oracle_destroy.argtypes = [vp]
        L.oracle_destroy.restype = None
        L.oracle_set_option.argtypes = [vp, ctypes.c_char_p, i64]
        L.oracle_set_state.argtypes = [vp, vp]
        L.oracle_get_state.argtypes = [vp, vp]
        L.oracle_set_primitive.argtypes = [vp, vp]
        L.oracle_get_primitive.argtypes = [vp, vp]
        L.oracle_cfl_dt.argtypes = [vp, dbl]
        L.oracle_cfl_dt.restype = dbl
        L.oracle_step.argtypes = [vp, dbl]
        L.oracle_stage.argtypes = [vp, dbl, vp]
        L.oracle_run.argtypes = [vp, dbl, i64, dbl, ctypes.POINTER(i64), ctypes.POINTER(dbl)]
        L.oracle_riemann.argtypes = [cint, cint, cint, cint, dbl, vp, vp, vp]
        L.oracle_minbee.argtypes = [cint, dbl, dbl, dbl, ctypes.POINTER(dbl), ctypes.POINTER(dbl)]
        L.oracle_limited.argtypes = [cint, cint, dbl, dbl, dbl, ctypes.POINTER(dbl), ctypes.POINTER(dbl)]
        L.oracle_set_ghosts.argtypes = [vp, vp]
        L.oracle_step_ghosts.argtypes = [vp, dbl, vp]
        L.oracle_num_threads.restype = cint
        _LIBS[kind] = L
    return _LIBS[kind]


class Oracle:
    """One oracle solver instance.  State arrays are (nf, [nz,] [ny,] nx), x fastest."""

    def __init__(self, n, extent, gamma, dtype, boundary="periodic", riemann="hllc", threads="serial", integrator="midpoint",
                 limiter="minbee"):
        self.n = tuple(int(v) for v in n)  # x first
        self.dims = len(self.n)
        self.dtype = np.dtype(dtype)
        self.nf = self.dims + 2
        self.shape = (self.nf,) + tuple(reversed(self.n))
        self._L = _lib(threads)
        narr = (ctypes.c_int64 * self.dims)(*self.n)
        earr = (ctypes.c_double * self.dims)(*[float(e) for e in extent])
        self._h = self._L.oracle_create(self.dims, narr, earr, float(gamma), _DT[self.dtype])
        if not self._h:
            raise ValueError("oracle_create failed")
        self._opt("boundary", {"periodic": 0, "outflow": 1}[boundary])
        self._opt("riemann", {"hllc": 0, "hll": 1}[riemann])
        self._opt("integrator", {"midpoint": 0, "heun": 1}[integrator])
        self._opt("limiter", LIMITER[limiter])

    def _opt(self, key, val):
        if self._L.oracle_set_option(self._h, key.encode(), val) != 0:
            raise ValueError(f"bad option {key}={val}")

    def set_state(self, U):
        U = np.ascontiguousarray(U, dtype=self.dtype)
        assert U.shape == self.shape, (U.shape, self.shape)
        self._L.oracle_set_state(self._h, U.ctypes.data)

    def get_state(self):
        out = np.empty(self.shape, self.dtype)
        self._L.oracle_get_state(self._h, out.ctypes.data)
        return out

    def set_primitive(self, V):
        """V = (rho, v_a, p), same layout as the state: converted with the EOS of PAPER.md:694 (DESIGN.md §4 "cons")."""
        V = np.ascontiguousarray(V, dtype=self.dtype)
        assert V.shape == self.shape, (V.shape, self.shape)
        self._L.oracle_set_primitive(self._h, V.ctypes.data)

    def get_primitive(self):
        out = np.empty(self.shape, self.dtype)
        self._L.oracle_get_primitive(self._h, out.ctypes.data)
        return out

    def cfl_dt(self, cfl):
        return self._L.oracle_cfl_dt(self._h, float(cfl))

    def step(self, dt):
        self._L.oracle_step(self._h, float(dt))

    def set_ghosts(self, G):
        """Prescribed ghost cells: the outermost two cells of every axis of the current state := G's."""
        G = np.ascontiguousarray(G, dtype=self.dtype)
        assert G.shape == self.shape
        self._L.oracle_set_ghosts(self._h, G.ctypes.data)

    def step_ghosts(self, dt, G_mid):
        """One RK2 step whose intermediate state gets G_mid's ghost cells before the second stage."""
        G_mid = np.ascontiguousarray(G_mid, dtype=self.dtype)
        assert G_mid.shape == self.shape
        self._L.oracle_step_ghosts(self._h, float(dt), G_mid.ctypes.data)

    def stage(self, tau):
        out = np.empty(self.shape, self.dtype)
        self._L.oracle_stage(self._h, float(tau), out.ctypes.data)
        return out

    def run(self, cfl, nsteps, t_end=0.0):
        k = ctypes.c_int64(0)
        t = ctypes.c_double(0)
        self._L.oracle_run(self._h, float(cfl), int(nsteps), float(t_end), ctypes.byref(k), ctypes.byref(t))
        return k.value, t.value

    def close(self):
        if self._h:
            self._L.oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def riemann(VL, VR, axis, gamma, dims, dtype=np.float64, kind="hllc"):
    VL = np.ascontiguousarray(VL, np.float64)
    VR = np.ascontiguousarray(VR, np.float64)
    F = np.empty(dims + 2, np.float64)
    rc = _lib().oracle_riemann(_DT[np.dtype(dtype)], dims, axis, {"hllc": 0, "hll": 1}[kind], float(gamma),
                               VL.ctypes.data, VR.ctypes.data, F.ctypes.data)
    assert rc == 0
    return F


def minbee(y0, y1, y2, dtype=np.float64):
    lo, hi = ctypes.c_double(), ctypes.c_double()
    _lib().oracle_minbee(_DT[np.dtype(dtype)], y0, y1, y2, ctypes.byref(lo), ctypes.byref(hi))
    return lo.value, hi.value


def limited(limiter, y0, y1, y2, dtype=np.float64):
    """(lo, hi) of one interpolation variant ("minbee", "none", "mc")."""
    lo, hi = ctypes.c_double(), ctypes.c_double()
    rc = _lib().oracle_limited(_DT[np.dtype(dtype)], LIMITER[limiter], y0, y1, y2, ctypes.byref(lo), ctypes.byref(hi))
    assert rc == 0
    return lo.value, hi.value


def num_threads(kind="omp"):
    return _lib(kind).oracle_num_threads()


class Wave:
    """The paper's linear-wave example (§2.3, Table 2) as oracle/wave_oracle.cpp states it: fp64, periodic on
    [0, 2 pi), dx = 2 pi / n, dt = dx / c.  step() advances one step and returns the discrete energy of Eq. 8."""

    def __init__(self, n, c=3.43):
        L = ctypes.CDLL(_build.build()["wave"])
        vp, dbl = ctypes.c_void_p, ctypes.c_double
        L.wave_oracle_create.restype = vp
        L.wave_oracle_create.argtypes = [ctypes.c_int64, dbl]
        L.wave_oracle_destroy.argtypes = [vp]
        L.wave_oracle_destroy.restype = None
        L.wave_oracle_set_state.argtypes = [vp, vp, vp]
        L.wave_oracle_get_state.argtypes = [vp, vp, vp]
        L.wave_oracle_step.argtypes = [vp]
        L.wave_oracle_step.restype = dbl
        L.wave_oracle_dx.argtypes = [vp]
        L.wave_oracle_dx.restype = dbl
        L.wave_oracle_dt.argtypes = [vp]
        L.wave_oracle_dt.restype = dbl
        self._L, self.n = L, int(n)
        self._h = L.wave_oracle_create(self.n, float(c))
        if not self._h:
            raise ValueError("wave_oracle_create failed")
        self.dx, self.dt = L.wave_oracle_dx(self._h), L.wave_oracle_dt(self._h)

    def set_state(self, f, g):
        f, g = np.ascontiguousarray(f, np.float64), np.ascontiguousarray(g, np.float64)
        assert f.shape == g.shape == (self.n,)
        self._L.wave_oracle_set_state(self._h, f.ctypes.data, g.ctypes.data)

    def get_state(self):
        f, g = np.empty(self.n), np.empty(self.n)
        self._L.wave_oracle_get_state(self._h, f.ctypes.data, g.ctypes.data)
        return f, g

    def step(self):
        return self._L.wave_oracle_step(self._h)

    def close(self):
        if self._h:
            self._L.wave_oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
