"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (default variant, device-paced
`run` replaying the CUDA graph).

  configs 1, 2, 3  the oracle (OpenMP build, bit-identical to the serial one) runs the whole config; every cell is
                   compared after the full number of steps with north_star's 100-step tolerance (R17
                   metric) and after one step with the one-step tolerance; t and the step count must agree.
  config 4         test_config4_full_grid_full_length: the OpenMP oracle runs all 20 steps of the 512^3 grid (~3 x 10^9
                   cell-steps, a few minutes on the box's host cores, ~14 GB of host memory); EVERY cell is compared
                   after step 1 (default variant and each end of the Manifest <-> Delayed axis: manifest_all,
                   manifest_flux, delayed, march, pack) and after step 20 (default variant).  The older sampled test is
                   kept as a fast pre-check: (a) dt of the first step against the
                   oracle's CFL reduction over the full state, (b) the first step on SAMPLED sub-boxes: one RK2 step
                   reaches 4 cells, so the oracle advances a sub-box cut (with periodic wrap) from the full initial
                   state with a 6-cell margin and its interior is compared cell by cell with the GPU's full-grid
                   result, (c) properties that hold at any size over the full 20 steps: mass / momentum / energy
                   conserved to round-off on the periodic grid, finite state, positive density and pressure, the
                   device clock equal to the sum of the dt it used.
Inputs never come from the CUDA path: the oracle always starts from the seeded initial state.
"""
import numpy as np
import pytest

from parity_util import TOL, field_errors, own_scale_errors
from paper_1204_4779_b200 import inputs

pytestmark = [pytest.mark.gpu, pytest.mark.slow]


@pytest.fixture(scope="module")
def gpu():
    import torch

    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1204_4779_b200 import binding

    binding.load_library()
    return binding


def oracle_run(oracle_mod, w, nsteps, riemann="hllc"):
    o = oracle_mod.Oracle(w.n, w.extent, w.gamma, w.dtype, w.boundary, riemann, "omp")
    o.set_state(w.U)
    first = None
    t = 0.0
    for k in range(nsteps):
        dt = o.cfl_dt(w.cfl)
        o.step(dt)
        t += dt
        if k == 0:
            first = (o.get_state(), dt)
    out = o.get_state()
    o.close()
    return first, out, t


@pytest.mark.parametrize("cfg,riemann", [(1, "hllc"), (2, "hllc"), (3, "hllc"), (1, "hll"), (3, "hll")])
def test_full_config_matches_oracle(gpu, oracle_mod, cfg, riemann):
    """Configs 1-3 at their stated size and length, HLLC (the paper's solver) and HLL (north_star's fallback; SURVEY A4:
    "parity is required for both"): every conserved field on its own scale max|ref_f| inside north_star's tolerance
    (config 1's m_y, ~0.02 beside m_x ~ 1, is the tight one), and - since the kernels state the oracle's arithmetic
    operation by operation - bit-equal after the first step and after the last."""
    import torch

    w = inputs.baseline_config(cfg)
    (ref1, rdt1), ref, rt = oracle_run(oracle_mod, w, w.steps, riemann)
    tol1, tol100, toldt = TOL[np.dtype(w.dtype)]
    with gpu.ParaisoHydro(w.n, w.extent, w.gamma, w.dtype, w.boundary, riemann) as h:
        h.set_state(torch.from_numpy(w.U).cuda())
        gdt1 = h.cfl_dt(w.cfl)
        assert abs(gdt1 - rdt1) <= toldt * rdt1
        h.run(w.cfl, 1)
        got1 = h.get_state()
        assert np.all(own_scale_errors(got1, ref1) <= tol1), own_scale_errors(got1, ref1)
        assert np.array_equal(got1, ref1), (cfg, riemann, "first step: bit-equal")
        h.run(w.cfl, w.steps - 1)
        got = h.get_state()
        t, k = h.time()
        assert h.stats() == 0 and k == w.steps
    assert abs(t - rt) <= 10 * toldt * rt, (t, rt)
    err = own_scale_errors(got, ref)
    assert np.all(err <= tol100), (cfg, riemann, err)
    assert np.array_equal(got, ref), (cfg, riemann, f"after {w.steps} steps: bit-equal")
    print(f"config {cfg} {riemann}: {w.steps} steps, max own-scale field error {err.max():.2e}, bit-equal True")


def wrapped_box(U, lo, size):
    """U[f][z][y][x]: the box starting at `lo` (x, y, z) with `size` cells per axis, indices wrapped periodically."""
    out = U
    for a, (l, s) in enumerate(zip(lo, size)):
        axis = U.ndim - 1 - a
        out = np.take(out, np.arange(l, l + s), axis=axis, mode="wrap")
    return np.ascontiguousarray(out)


def test_config4_first_step_on_sampled_boxes_and_properties(gpu, oracle_mod):
    import torch

    w = inputs.baseline_config(4)
    n = w.n[0]
    assert w.n == (n, n, n) and w.extent == (1.0, 1.0, 1.0)
    tol1, _, toldt = TOL[np.dtype(w.dtype)]

    # (a) dt of the first step: the oracle's CFL reduction over the full state
    o = oracle_mod.Oracle(w.n, w.extent, w.gamma, w.dtype, w.boundary, "hllc", "omp")
    o.set_state(w.U)
    rdt = o.cfl_dt(w.cfl)
    o.close()

    U0 = w.U.astype(np.float64)
    sums0 = U0.reshape(w.nf, -1).sum(axis=1)
    with gpu.ParaisoHydro(w.n, w.extent, w.gamma, w.dtype, w.boundary, "hllc") as h:
        h.set_state(torch.from_numpy(w.U).cuda())
        gdt = h.cfl_dt(w.cfl)
        assert abs(gdt - rdt) <= toldt * rdt, (gdt, rdt)
        h.run(w.cfl, 1)
        got1 = h.get_state()
        t1, _ = h.time()
        assert abs(t1 - rdt) <= toldt * rdt
        h.run(w.cfl, w.steps - 1)
        got = h.get_state()
        t, k = h.time()
        assert h.stats() == 0 and k == w.steps and t > t1

    # (b) sampled sub-boxes of the first step: the blast centre, a corner that wraps in all three axes, a tile seam
    # of the launch shape (x = 32 k, y = 7 k), the last ragged tile row, and two seeded random boxes
    L, margin = 24, 6
    rng = np.random.default_rng(4)
    corners = [(n // 2 - L // 2,) * 3, (n - L // 2,) * 3, (32 * 5 - L // 2, 7 * 31 - L // 2, 128 - L // 2),
               (n - L, n - L, 0)] + [tuple(int(v) for v in rng.integers(0, n, 3)) for _ in range(2)]
    size = (L + 2 * margin,) * 3
    ext = tuple(s / n for s in size)  # same cell size, exactly (n is a power of two)
    worst = 0.0
    for c in corners:
        lo = tuple(v - margin for v in c)
        sub = wrapped_box(w.U, lo, size)
        o = oracle_mod.Oracle(size, ext, w.gamma, w.dtype, "outflow", "hllc", "omp")
        o.set_state(sub)
        o.step(rdt)
        ref = o.get_state()
        o.close()
        inner = (slice(None),) + (slice(margin, margin + L),) * 3
        g = wrapped_box(got1, c, (L, L, L))
        err = field_errors(g, ref[inner])
        worst = max(worst, err.max())
        assert np.all(err <= tol1), (c, err)
        assert np.array_equal(g, ref[inner]), ("same arithmetic as the oracle: bit-equal", c)
    print(f"config 4 first step: {len(corners)} sampled {L}^3 boxes, worst field error {worst:.2e}")

    # (c) properties over the full run
    assert np.isfinite(got).all()
    G = got.astype(np.float64)
    rho, E = G[0], G[4]
    assert rho.min() > 0
    p = (w.gamma - 1.0) * (E - 0.5 * (G[1] ** 2 + G[2] ** 2 + G[3] ** 2) / rho)
    assert p.min() > 0
    sums = G.reshape(w.nf, -1).sum(axis=1)
    cells = float(n) ** 3
    assert abs(sums[0] - sums0[0]) <= 2e-6 * abs(sums0[0])                 # mass
    assert abs(sums[4] - sums0[4]) <= 2e-6 * abs(sums0[4])                 # energy
    mom_scale = np.abs(G[1:4]).max() * cells
    assert np.all(np.abs(sums[1:4] - sums0[1:4]) <= 2e-6 * mom_scale)      # momentum (zero in total at t = 0)


def test_config4_full_grid_full_length(gpu, oracle_mod):
    """BASELINE config 4 at full size AND full length, every cell (north_star: "on all five configs"; SURVEY §8(c3):
    configs with fewer than 100 steps are checked after 1 step and after their full length).  512^3 is the only config
    whose 32-bit element offsets come near their limit (nf N = 6.7e8)."""
    import torch

    w = inputs.baseline_config(4)
    tol1, tol100, toldt = TOL[np.dtype(w.dtype)]
    (ref1, rdt1), ref, rt = oracle_run(oracle_mod, w, w.steps)

    def first_step(variant):
        with gpu.ParaisoHydro(w.n, w.extent, w.gamma, w.dtype, w.boundary, "hllc", variant) as h:
            h.set_state(torch.from_numpy(w.U).cuda())
            gdt = h.cfl_dt(w.cfl)
            assert abs(gdt - rdt1) <= toldt * rdt1, (variant, gdt, rdt1)
            h.run(w.cfl, 1)
            got1 = h.get_state()
            assert h.stats() == 0
        err = field_errors(got1, ref1)
        assert np.all(err <= tol1), (variant, err)
        assert np.array_equal(got1, ref1), (variant, "same written arithmetic as the oracle: bit-equal")
        return err

    # both ends of the Manifest <-> Delayed axis and both on-chip designs, first step, every cell
    for variant in ("manifest_all", "manifest_flux", "delayed", "march", "pack"):
        first_step(variant)

    # the default variant (what bench.py times): step 1 and the full 20 steps, device-paced run with graph replay
    with gpu.ParaisoHydro(w.n, w.extent, w.gamma, w.dtype, w.boundary, "hllc") as h:
        h.set_state(torch.from_numpy(w.U).cuda())
        h.run(w.cfl, 1)
        got1 = h.get_state()
        assert np.all(field_errors(got1, ref1) <= tol1)
        assert np.array_equal(got1, ref1)
        del got1
        h.run(w.cfl, w.steps - 1)
        got = h.get_state()
        t, k = h.time()
        assert h.stats() == 0 and k == w.steps
    assert abs(t - rt) <= 10 * toldt * rt, (t, rt)
    err = field_errors(got, ref)
    assert np.all(err <= tol100), err
    assert np.all(own_scale_errors(got, ref) <= tol100)
    print(f"config 4: {w.steps} steps on 512^3, max field error {err.max():.2e}, bit-equal {np.array_equal(got, ref)}")
    assert np.array_equal(got, ref)
