"""paraiso_hydro_cfl_noalloc (include/paraiso_hydro_noalloc.h): the CFL reduction for callers that cannot allocate.

Some users of this library are not allowed to cause a device allocation: a simulation code that gave all of HBM to its
own arena at start-up (a cudaMalloc from a plug-in fails there, or eats memory budgeted for something else), an in-situ
tool that is only lent a pointer to somebody else's state, a time-step loop that cannot afford the device-wide
synchronisation of cudaMalloc / cudaFree.  The handle API allocates in create(); this one entry point does not: its
working memory (per-block partial maxima and a ticket) is a fixed array inside the library, which is why the grid is
limited to NOALLOC_MAX_CELLS cells and why calls on one device share state.

The GPU test compares the entry point with the existing path (a handle holding the same state: set_state + cfl_dt +
stats) on two calls in a row that differ in grid, dimension and precision, so that whatever the first call left in the
shared scratch (more partials, larger maxima) would show up in the second.  The file sorts last on purpose: `pytest -x`
stops at the first failure, and a failure here should not hide the parity tests.  It passes alone in a fresh process
(first call = the set-up call) and after the other tests.
"""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _header_text():
    return open(os.path.join(ROOT, "include", "paraiso_hydro_noalloc.h")).read()


def test_noalloc_entry_point_is_declared_and_exported():
    """No GPU: the header declares exactly one function, the library exports it, the binding's limit is the header's."""
    from paper_1204_4779_b200 import binding, build

    build.build()
    text = _header_text()
    code = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    names = sorted(set(re.findall(r"\b(paraiso_[a-z_]+)\s*\(", code)))
    assert names == sorted(binding.NOALLOC_SIGNATURES) == ["paraiso_hydro_cfl_noalloc"]
    assert hasattr(ctypes.CDLL(binding.LIB_PATH), names[0])
    assert int(re.search(r"#define PARAISO_NOALLOC_MAX_CELLS (\d+)LL", text).group(1)) == binding.NOALLOC_MAX_CELLS
    assert int(re.search(r"#define PARAISO_ETOOLARGE \((-\d+)\)", text).group(1)) == binding.PARAISO_ETOOLARGE


def test_noalloc_source_calls_no_allocator():
    """No GPU: the translation unit of the entry point names no allocating CUDA call."""
    src = open(os.path.join(ROOT, "paper_1204_4779_b200", "csrc", "paraiso_hydro_noalloc.cu")).read()
    code = re.sub(r"//[^\n]*", "", src)
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaMallocAsync", "cudaMemPool", "new ", "malloc("):
        assert banned not in code, banned
    assert "cudaGetSymbolAddress" in code and "static __device__ __align__(256)" in code


def test_noalloc_rejects_bad_arguments_and_oversized_grids_without_a_device():
    """No GPU needed: arguments are checked before the device is touched; a grid beyond the limit gets its own code."""
    from paper_1204_4779_b200 import binding

    lib = binding.load_library()
    i64, dbl = ctypes.c_int64, ctypes.c_double
    fake = ctypes.c_void_p(256)  # never dereferenced: every call below fails in the argument checks
    ext = (dbl * 3)(1.0, 1.0, 1.0)

    def call(dims, n, gamma=1.4, dtype=0, cfl=0.4, U=fake, out=fake):
        return lib.paraiso_hydro_cfl_noalloc(dims, (i64 * 3)(*n), ext, gamma, dtype, U, cfl, None, out)

    assert call(3, (512, 512, 513)) == binding.PARAISO_ETOOLARGE          # one plane more than the limit
    assert call(2, (1 << 20, 1 << 20, 1)) == binding.PARAISO_ETOOLARGE
    assert call(1, (binding.NOALLOC_MAX_CELLS + 1, 1, 1)) == binding.PARAISO_ETOOLARGE
    assert call(0, (8, 8, 8)) == binding.PARAISO_EINVAL
    assert call(4, (8, 8, 8)) == binding.PARAISO_EINVAL
    assert call(2, (8, 0, 1)) == binding.PARAISO_EINVAL
    assert call(2, (8, 8, 1), gamma=1.0) == binding.PARAISO_EINVAL
    assert call(2, (8, 8, 1), cfl=0.0) == binding.PARAISO_EINVAL
    assert call(2, (8, 8, 1), dtype=2) == binding.PARAISO_EINVAL
    assert call(2, (8, 8, 1), U=None) == binding.PARAISO_EINVAL
    assert call(2, (8, 8, 1), out=None) == binding.PARAISO_EINVAL


def _existing_path(w, cfl):
    """(dt, bad cells) of workload w through the handle API: set_state runs the standalone reduction k_cfl."""
    from paper_1204_4779_b200 import binding

    with binding.ParaisoHydro(w.n, w.extent, w.gamma, w.dtype, boundary=w.boundary) as h:
        h.set_state(w.U)
        return h.cfl_dt(cfl), h.stats()


@pytest.mark.gpu
def test_noalloc_cfl_matches_the_handle_path_on_two_calls_in_a_row():
    import torch

    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1204_4779_b200 import binding, inputs

    # call 1: 3-D fp32 blast, 61 blocks with a ragged last one, large S (pressure spike);
    # call 2: 2-D fp64, a single ragged block, S about 40 times smaller, three cells made unphysical (p < 0)
    a = inputs.blast(shape=(97, 64, 40), dtype=np.float32, seed=5)
    b = inputs.random_smooth((100, 30), np.float64, seed=7)
    b.U[3].reshape(-1)[[5, 1234, 2999]] = -1.0
    cases = [(a, 0.3), (b, 0.4)]

    # inputs and outputs belong to the caller and exist before the calls; nothing is synchronised in between
    U_dev = [torch.from_numpy(w.U).cuda() for w, _ in cases]
    out = [torch.full((3,), -1.0, dtype=torch.float64, device="cuda") for _ in cases]
    torch.cuda.synchronize()
    for (w, cfl), U, o in zip(cases, U_dev, out):
        binding.cfl_noalloc(U, w.n, w.extent, w.gamma, cfl, o)
    torch.cuda.synchronize()
    got = [o.cpu().numpy() for o in out]

    for (w, cfl), g in zip(cases, got):
        dt_ref, bad_ref = _existing_path(w, cfl)
        tol = 1e-6 if w.dtype == np.float32 else 1e-13  # the dt tolerances of north_star, as in tests/test_gpu_parity.py
        S, dt, bad = g
        assert S > 0 and np.isfinite(S) and np.isfinite(dt)
        assert abs(dt - dt_ref) <= tol * dt_ref, (w.name, dt, dt_ref)
        assert bad == bad_ref, (w.name, bad, bad_ref)
        # dt is the one division Real(cfl) / S of the dtype
        expect = float(w.dtype.type(cfl) / w.dtype.type(S))
        assert dt == expect, (dt, expect)
        print(f"{w.name}: S={S:.6g} dt={dt:.6e} handle dt={dt_ref:.6e} bit-equal={dt == dt_ref} bad={int(bad)}")
    assert got[0][0] > 5 * got[1][0], "the second call must have the smaller S for the stale-scratch check to bite"
    assert got[0][2] == 0 and got[1][2] == 3

    # and the same two calls again, in the other order, on a side stream: same answers
    st = torch.cuda.Stream()
    again = [torch.zeros(3, dtype=torch.float64, device="cuda") for _ in cases]
    torch.cuda.synchronize()
    for i in (1, 0):
        w, cfl = cases[i]
        binding.cfl_noalloc(U_dev[i], w.n, w.extent, w.gamma, cfl, again[i], stream=st)
    st.synchronize()
    for i in (0, 1):
        assert np.array_equal(again[i].cpu().numpy(), got[i])


@pytest.mark.gpu
def test_noalloc_cfl_allocates_no_device_memory():
    """Free device memory as the driver reports it is the same before and after a burst of calls."""
    import torch

    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1204_4779_b200 import binding, inputs

    w = inputs.random_smooth((64, 48, 20), np.float32, seed=1)
    U = torch.from_numpy(w.U).cuda()
    out = torch.zeros(3, dtype=torch.float64, device="cuda")
    binding.cfl_noalloc(U, w.n, w.extent, w.gamma, 0.3, out)  # the set-up call (loads the kernel, looks up the scratch)
    torch.cuda.synchronize()
    first = out.cpu().numpy().copy()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(50):
        binding.cfl_noalloc(U, w.n, w.extent, w.gamma, 0.3, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
    assert np.array_equal(out.cpu().numpy(), first)
