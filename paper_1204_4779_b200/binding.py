"""ctypes binding of libparaiso_hydro.so — argument marshalling only (include/paraiso_hydro.h).

Every function of the C ABI is exposed under the same name (`lib.paraiso_hydro_step`, ...) by
`load_library()`; `ParaisoHydro` wraps one handle with methods of the same names minus the prefix.
No step of the path runs here: state arrays go in and out as raw pointers (NumPy arrays = host
pointers; torch CUDA tensors = device pointers, zero-copy), and PyTorch is used only for device
memory and streams by callers who want them.

There is no CPU fallback: if the library is not built, or no CUDA device is usable, this raises.
"""
import ctypes
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libparaiso_hydro.so")

PARAISO_F32, PARAISO_F64 = 0, 1
PARAISO_OK, PARAISO_EINVAL, PARAISO_ENOMEM, PARAISO_ECUDA, PARAISO_ESTATE, PARAISO_ENONFINITE = 0, -1, -2, -3, -4, -5

BOUNDARY = {"periodic": 0, "outflow": 1}
RIEMANN = {"hllc": 0, "hll": 1}
VARIANT = {"fused": 0, "manifest_flux": 1, "manifest_all": 2, "delayed": 3, "march": 4, "fused1": 5, "pack": 6}

_vp, _i64, _dbl, _int = ctypes.c_void_p, ctypes.c_int64, ctypes.c_double, ctypes.c_int
_pi64, _pdbl = ctypes.POINTER(_i64), ctypes.POINTER(_dbl)

# name -> (restype, argtypes): one entry per symbol declared in include/paraiso_hydro.h
SIGNATURES = {
    "paraiso_hydro_create": (_int, [ctypes.POINTER(_vp), _int, _pi64, _pdbl, _dbl, _int]),
    "paraiso_hydro_destroy": (_int, [_vp]),
    "paraiso_hydro_set_option": (_int, [_vp, ctypes.c_char_p, _i64]),
    "paraiso_hydro_get_option": (_int, [_vp, ctypes.c_char_p, _pi64]),
    "paraiso_hydro_set_stream": (_int, [_vp, _vp]),
    "paraiso_hydro_set_state": (_int, [_vp, _vp]),
    "paraiso_hydro_get_state": (_int, [_vp, _vp]),
    "paraiso_hydro_cfl_dt": (_int, [_vp, _dbl, _pdbl]),
    "paraiso_hydro_step": (_int, [_vp, _dbl]),
    "paraiso_hydro_set_ghosts": (_int, [_vp, _vp]),
    "paraiso_hydro_step_ghosts": (_int, [_vp, _dbl, _vp]),
    "paraiso_hydro_run": (_int, [_vp, _dbl, _i64, _dbl, _pi64, _pdbl]),
    "paraiso_hydro_sync": (_int, [_vp]),
    "paraiso_hydro_time": (_int, [_vp, _pdbl, _pi64]),
    "paraiso_hydro_stats": (_int, [_vp, _pi64]),
    "paraiso_hydro_launch_count": (_int, [_vp, _pi64]),
    "paraiso_hydro_kernel_time": (_int, [_vp, _int, _pdbl, _pi64]),
    "paraiso_hydro_last_error": (ctypes.c_char_p, [_vp]),
    "paraiso_hydro_version": (ctypes.c_char_p, []),
}

# the paper's linear-wave example (include/paraiso_wave.h), exported by the same library
WAVE_SIGNATURES = {
    "paraiso_wave_create": (_int, [ctypes.POINTER(_vp), _i64, _dbl]),
    "paraiso_wave_destroy": (_int, [_vp]),
    "paraiso_wave_set_state": (_int, [_vp, _vp, _vp]),
    "paraiso_wave_get_state": (_int, [_vp, _vp, _vp]),
    "paraiso_wave_step": (_int, [_vp, _i64, _vp]),
    "paraiso_wave_launch_count": (_int, [_vp, _pi64]),
}

# the allocation-free CFL reduction (include/paraiso_hydro_noalloc.h), exported by the same library
PARAISO_ETOOLARGE = -6
NOALLOC_MAX_CELLS = 134217728
NOALLOC_SIGNATURES = {
    "paraiso_hydro_cfl_noalloc": (_int, [_int, _pi64, _pdbl, _dbl, _int, _vp, _dbl, _vp, _vp]),
}

# the probe library (include/paraiso_hydro_probe.h): tests and bench.py's roofline leg only
PROBE_PATH = os.path.join(HERE, "libparaiso_hydro_probe.so")
PROBE_SIGNATURES = {
    "paraiso_probe_arith": (_int, [_int, _i64, _vp, _vp, _vp, _vp]),
    "paraiso_probe_issue_cost": (_int, [_int, _dbl, _pdbl, _pdbl]),
    "paraiso_probe_peak": (_int, [_int, _pdbl]),
    "paraiso_probe_mix_ceiling": (_int, [_int, _dbl, _pdbl]),
}

_LIB = None
_PROBE = None


class ParaisoError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"paraiso_hydro error {code}: {msg}")
        self.code = code


def load_library(path=None):
    """dlopen the C-ABI library and declare every prototype.  Raises if it has not been built
    (`python -m paper_1204_4779_b200.build`): the product path never falls back to anything else."""
    global _LIB
    if _LIB is not None and path is None:
        return _LIB
    p = path or LIB_PATH
    if not os.path.exists(p):
        raise ParaisoError(PARAISO_ECUDA, f"{p} not built; run `python -m paper_1204_4779_b200.build` "
                                          "(there is no CPU fallback)")
    lib = ctypes.CDLL(p)
    for name, (res, args) in list(SIGNATURES.items()) + list(WAVE_SIGNATURES.items()) + list(NOALLOC_SIGNATURES.items()):
        fn = getattr(lib, name)  # AttributeError if a declared symbol is not exported
        fn.restype = res
        fn.argtypes = args
    if path is None:
        _LIB = lib
    return lib


def _pointer(a):
    """Raw address of a NumPy array (host) or a torch tensor (host or device).  The caller keeps it alive."""
    if isinstance(a, np.ndarray):
        if not a.flags["C_CONTIGUOUS"]:
            raise ValueError("state array must be C-contiguous")
        return a.ctypes.data, a.dtype, a.size
    if hasattr(a, "data_ptr"):  # torch.Tensor
        if not a.is_contiguous():
            raise ValueError("state tensor must be contiguous")
        import torch

        dt = {torch.float32: np.dtype(np.float32), torch.float64: np.dtype(np.float64)}[a.dtype]
        return a.data_ptr(), dt, a.numel()
    raise TypeError(f"unsupported state container {type(a)}")


ISSUE_KINDS = {"ffma": 0, "fmnmx": 1, "fsetp_fsel": 2, "iadd3_lop3": 3, "ffma2": 4, "dfma": 5, "mufu": 6}
PEAK_KINDS = {"ffma": 0, "ffma2": 1, "dfma": 2}


def load_probe():
    """dlopen libparaiso_hydro_probe.so (include/paraiso_hydro_probe.h): test / measurement probes, not product."""
    global _PROBE
    if _PROBE is None:
        if not os.path.exists(PROBE_PATH):
            raise ParaisoError(PARAISO_ECUDA, f"{PROBE_PATH} not built; run `python -m paper_1204_4779_b200.build`")
        lib = ctypes.CDLL(PROBE_PATH)
        for name, (res, args) in PROBE_SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _PROBE = lib
    return _PROBE


def probe_issue_cost(kind, sm_clock_mhz):
    """paraiso_probe_issue_cost: (scheduler cycles one more instruction of `kind` costs next to 16 FFMA per
    iteration, cycles of the 16-FFMA loop alone)."""
    c, base = _dbl(0.0), _dbl(0.0)
    rc = load_probe().paraiso_probe_issue_cost(ISSUE_KINDS[kind] if isinstance(kind, str) else int(kind),
                                               float(sm_clock_mhz), ctypes.byref(c), ctypes.byref(base))
    if rc:
        raise ParaisoError(rc, "probe_issue_cost failed")
    return c.value, base.value


def probe_peak(kind):
    """paraiso_probe_peak: measured fused multiply-adds per second / 1e12 of `kind` ("ffma", "ffma2", "dfma")."""
    v = _dbl(0.0)
    rc = load_probe().paraiso_probe_peak(PEAK_KINDS[kind] if isinstance(kind, str) else int(kind), ctypes.byref(v))
    if rc:
        raise ParaisoError(rc, "probe_peak failed")
    return v.value


def probe_mix_ceiling(mix, sm_clock_mhz):
    """paraiso_probe_mix_ceiling: warp instructions per cycle per scheduler of the stage kernel's instruction mix without
    dependencies (mix 0: packed, as k_pack; 1: scalar FFMA)."""
    v = _dbl(0)
    rc = load_probe().paraiso_probe_mix_ceiling(int(mix), float(sm_clock_mhz), ctypes.byref(v))
    if rc != 0:
        raise ParaisoError(rc, "probe_mix_ceiling failed")
    return v.value


def probe_arith(a, b):
    """paraiso_probe_arith on two equal-length device tensors: returns (a / b, sqrt(|a|)) as evaluated by the hot
    path's div_rn / sqrt_rn (device tensors of the same dtype)."""
    import torch

    pa, dt, n = _pointer(a)
    pb, dtb, nb = _pointer(b)
    if dt != dtb or n != nb or not a.is_cuda or not b.is_cuda:
        raise ValueError("probe_arith wants two device tensors of equal dtype and length")
    q, r = torch.empty_like(a), torch.empty_like(a)
    torch.cuda.synchronize()
    rc = load_probe().paraiso_probe_arith(0 if dt == np.dtype(np.float32) else 1, n, pa, pb, q.data_ptr(), r.data_ptr())
    if rc:
        raise ParaisoError(rc, "probe_arith failed")
    return q, r


def cfl_noalloc(U, n, extent, gamma, cfl, out, stream=None):
    """paraiso_hydro_cfl_noalloc: S, dt and the bad-cell count of the conserved state `U` into `out`, for callers that
    must not trigger a device allocation (a code whose own arena holds all of HBM, a tool that was only lent the
    state, a loop that cannot afford cudaMalloc's device-wide synchronisation).  Nothing is allocated here either:
    U   a contiguous torch CUDA tensor (float32 or float64) of shape (dims + 2, [nz,] [ny,] nx) that the caller owns;
    out a torch CUDA float64 tensor of 3 elements that the caller owns (S, dt, bad cells), written asynchronously on
        `stream` (a torch.cuda.Stream or raw cudaStream_t; default: the legacy default stream).
    At most NOALLOC_MAX_CELLS cells (the working memory is a fixed array inside the library); calls on one device
    share that array and must not overlap on the GPU; make the first call on a device before any stream capture."""
    lib = load_library()
    pu, dt, size = _pointer(U)
    po, dto, sizeo = _pointer(out)
    if not (getattr(U, "is_cuda", False) and getattr(out, "is_cuda", False)):
        raise ValueError("cfl_noalloc wants device tensors for U and out (it copies nothing)")
    dims = len(n)
    if dto != np.dtype(np.float64) or sizeo < 3:
        raise ValueError("out must hold 3 float64 values")
    if size != (dims + 2) * int(np.prod([int(v) for v in n], dtype=object)):
        raise ValueError("U does not have (dims + 2) * prod(n) elements")
    narr = (_i64 * dims)(*[int(v) for v in n])
    earr = (_dbl * dims)(*[float(e) for e in extent])
    s = getattr(stream, "cuda_stream", stream)
    rc = lib.paraiso_hydro_cfl_noalloc(dims, narr, earr, float(gamma), PARAISO_F32 if dt == np.dtype(np.float32) else
                                       PARAISO_F64, _vp(pu), float(cfl), _vp(int(s) if s else 0), _vp(po))
    if rc == PARAISO_ETOOLARGE:
        raise ParaisoError(rc, f"cfl_noalloc: more than {NOALLOC_MAX_CELLS} cells; the built-in scratch cannot hold "
                               "their per-block partials (use a handle, or reduce sub-boxes and take the larger S)")
    if rc != PARAISO_OK:
        raise ParaisoError(rc, "cfl_noalloc failed (bad argument)" if rc == PARAISO_EINVAL else "cfl_noalloc: CUDA error")


class ParaisoHydro:
    """One solver handle.  n is (nx[, ny[, nz]]) — x first; state arrays are (nf, [nz,] [ny,] nx)."""

    def __init__(self, n, extent, gamma, dtype, boundary="periodic", riemann="hllc", variant=None, stream=None,
                 **options):
        self._lib = load_library()
        self._h = _vp()
        self._stream_ptr = 0          # the handle's stream (0 = legacy default), mirrored for _source()
        self._pending_sources = []    # sources of asynchronous copies, released at the next blocking call
        self.n = tuple(int(v) for v in n)
        self.dims = len(self.n)
        self.nf = self.dims + 2
        self.dtype = np.dtype(dtype)
        self.shape = (self.nf,) + tuple(reversed(self.n))
        if self.dtype not in (np.dtype(np.float32), np.dtype(np.float64)):
            raise ValueError("dtype must be float32 or float64")
        narr = (_i64 * self.dims)(*self.n)
        earr = (_dbl * self.dims)(*[float(e) for e in extent])
        rc = self._lib.paraiso_hydro_create(ctypes.byref(self._h), self.dims, narr, earr, float(gamma),
                                            PARAISO_F32 if self.dtype == np.float32 else PARAISO_F64)
        if rc != PARAISO_OK:
            msg = self._lib.paraiso_hydro_last_error(None).decode()
            self._h = _vp()
            raise ParaisoError(rc, msg)
        self.set_option("boundary", BOUNDARY[boundary] if isinstance(boundary, str) else boundary)
        self.set_option("riemann", RIEMANN[riemann] if isinstance(riemann, str) else riemann)
        if variant is not None:
            self.set_option("variant", VARIANT[variant] if isinstance(variant, str) else variant)
        for k, v in options.items():
            self.set_option(k, v)
        if stream is not None:
            self.set_stream(stream)

    # -- plumbing
    def _check(self, rc):
        if rc != PARAISO_OK:
            raise ParaisoError(rc, self._lib.paraiso_hydro_last_error(self._h).decode())

    def _state_ptr(self, a):
        ptr, dt, size = _pointer(a)
        if dt != self.dtype:
            raise ValueError(f"state dtype {dt} does not match the handle's {self.dtype}")
        if size != int(np.prod(self.shape)):
            raise ValueError(f"state has {size} elements, expected {self.shape}")
        return ptr

    # -- the C ABI, one method per entry point
    def set_option(self, key, value):
        self._check(self._lib.paraiso_hydro_set_option(self._h, key.encode(), int(value)))

    def get_option(self, key):
        v = _i64(0)
        self._check(self._lib.paraiso_hydro_get_option(self._h, key.encode(), ctypes.byref(v)))
        return v.value

    def set_stream(self, stream):
        """stream: a raw cudaStream_t integer or a torch.cuda.Stream."""
        s = getattr(stream, "cuda_stream", stream)
        self._check(self._lib.paraiso_hydro_set_stream(self._h, _vp(int(s) if s else 0)))
        self._stream_ptr = int(s) if s else 0

    def _source(self, a):
        """Pointer of an array the library will read ASYNCHRONOUSLY on the handle's stream (set_state, set_ghosts,
        step_ghosts with a device or pinned source).  Two things the C ABI leaves to the caller are done here: the
        source object is kept alive until the handle's next blocking call (a temporary such as
        `h.set_state(torch.from_numpy(U).cuda())` would otherwise go back to torch's caching allocator and could be
        reused before the copy has run), and a torch CUDA source, which torch produced on ITS current stream, is
        ordered before the handle's stream by an event when the two streams differ."""
        ptr = self._state_ptr(a)
        if len(self._pending_sources) >= 64:  # a long loop of asynchronous calls: drain instead of hoarding
            self.sync()
        self._pending_sources.append(a)
        if getattr(a, "is_cuda", False):
            import torch

            cur = torch.cuda.current_stream(a.device)
            if int(cur.cuda_stream) != self._stream_ptr:
                mine = (torch.cuda.ExternalStream(self._stream_ptr, device=a.device) if self._stream_ptr
                        else torch.cuda.default_stream(a.device))
                ev = torch.cuda.Event()
                ev.record(cur)
                mine.wait_event(ev)
        return ptr

    def _blocking_call_done(self):
        self._pending_sources.clear()

    def set_state(self, U):
        self._check(self._lib.paraiso_hydro_set_state(self._h, _vp(self._source(U))))

    def get_state(self, out=None):
        if out is None:
            out = np.empty(self.shape, self.dtype)
        self._check(self._lib.paraiso_hydro_get_state(self._h, _vp(self._state_ptr(out))))
        return out

    def cfl_dt(self, cfl):
        dt = _dbl(0)
        self._check(self._lib.paraiso_hydro_cfl_dt(self._h, float(cfl), ctypes.byref(dt)))
        self._blocking_call_done()
        return dt.value

    def step(self, dt):
        self._check(self._lib.paraiso_hydro_step(self._h, float(dt)))

    def set_ghosts(self, G):
        """Prescribed ghost cells (include/paraiso_hydro.h): the outermost two cells of every axis of the current
        state := G's.  G: array / tensor shaped like the state (host or device)."""
        self._check(self._lib.paraiso_hydro_set_ghosts(self._h, self._source(G)))

    def step_ghosts(self, dt, G_mid):
        """One RK2 step whose intermediate state gets G_mid's ghost cells before the second stage."""
        self._check(self._lib.paraiso_hydro_step_ghosts(self._h, float(dt), self._source(G_mid)))

    def run(self, cfl, nsteps, t_end=0.0):
        k, t = _i64(0), _dbl(0)
        self._check(self._lib.paraiso_hydro_run(self._h, float(cfl), int(nsteps), float(t_end), ctypes.byref(k),
                                                ctypes.byref(t)))
        return k.value, t.value

    def sync(self):
        self._check(self._lib.paraiso_hydro_sync(self._h))
        self._blocking_call_done()

    def time(self):
        t, k = _dbl(0), _i64(0)
        self._check(self._lib.paraiso_hydro_time(self._h, ctypes.byref(t), ctypes.byref(k)))
        return t.value, k.value

    def stats(self):
        """Number of cell updates that produced a non-finite or non-positive rho / p (0 = healthy)."""
        k = _i64(0)
        rc = self._lib.paraiso_hydro_stats(self._h, ctypes.byref(k))
        if rc not in (PARAISO_OK, PARAISO_ENONFINITE):
            self._check(rc)
        return k.value

    def launch_count(self):
        k = _i64(0)
        self._check(self._lib.paraiso_hydro_launch_count(self._h, ctypes.byref(k)))
        return k.value

    def kernel_time(self, enable=None):
        """enable=1/0 switches per-stage CUDA-event timing on the handle's stream on or off (and resets
        the accumulators); enable=None reads (total stage-kernel milliseconds, stage launches timed)."""
        ms, k = _dbl(0), _i64(0)
        self._check(self._lib.paraiso_hydro_kernel_time(self._h, -1 if enable is None else int(enable),
                                                        ctypes.byref(ms), ctypes.byref(k)))
        return ms.value, k.value

    def version(self):
        return self._lib.paraiso_hydro_version().decode()

    def destroy(self):
        if getattr(self, "_h", None) and self._h.value:
            self._lib.paraiso_hydro_destroy(self._h)  # synchronises the device
            self._h = _vp()
            self._pending_sources.clear()

    close = destroy

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class ParaisoWave:
    """The paper's linear-wave example (§2.3, Table 2; include/paraiso_wave.h): fp64, periodic on [0, 2 pi),
    dx = 2 pi / n, dt = dx / c.  step(k) advances k steps on the device and returns the energy of Eq. 8 of each."""

    def __init__(self, n, c=3.43):
        self._lib = load_library()
        self._h = _vp()
        self.n = int(n)
        rc = self._lib.paraiso_wave_create(ctypes.byref(self._h), self.n, float(c))
        if rc != PARAISO_OK:
            self._h = _vp()
            raise ParaisoError(rc, "paraiso_wave_create failed (no CUDA device: there is no CPU fallback)" if rc == PARAISO_ECUDA
                               else "paraiso_wave_create failed")
        self.c = float(c)  # dx = 2 pi / n and dt = dx / c are formed inside the library (include/paraiso_wave.h)

    def _check(self, rc):
        if rc != PARAISO_OK:
            raise ParaisoError(rc, "paraiso_wave call failed")

    def set_state(self, f, g):
        f, g = np.ascontiguousarray(f, np.float64), np.ascontiguousarray(g, np.float64)
        if f.shape != (self.n,) or g.shape != (self.n,):
            raise ValueError("f and g must have n elements")
        self._check(self._lib.paraiso_wave_set_state(self._h, f.ctypes.data, g.ctypes.data))

    def get_state(self):
        f, g = np.empty(self.n), np.empty(self.n)
        self._check(self._lib.paraiso_wave_get_state(self._h, f.ctypes.data, g.ctypes.data))
        return f, g

    def step(self, nsteps=1):
        e = np.empty(int(nsteps))
        self._check(self._lib.paraiso_wave_step(self._h, int(nsteps), e.ctypes.data))
        return e

    def launch_count(self):
        k = _i64(0)
        self._check(self._lib.paraiso_wave_launch_count(self._h, ctypes.byref(k)))
        return k.value

    def destroy(self):
        if self._h:
            self._lib.paraiso_wave_destroy(self._h)
            self._h = _vp()

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.destroy()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
