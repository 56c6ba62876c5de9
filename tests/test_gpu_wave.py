"""GPU parity of the paper's linear-wave example (§2.3, Table 2; include/paraiso_wave.h) with the oracle
(oracle/wave_oracle.cpp): f and g bit-equal (same operations in the same order, no fused multiply-add), the Reduce Sum
energy equal up to the summation order, and the paper's own observation on the GPU result."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n", [3, 8, 255, 256, 257, 3072, 100003, 1 << 20])
def test_wave_matches_oracle(oracle_mod, n):
    import torch

    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1204_4779_b200 import binding

    steps = 40 if n > 10000 else 3 * n + 5
    o = oracle_mod.Wave(n)
    x = np.arange(n) * o.dx
    f0, g0 = np.sin(x), np.cos(3 * x)
    o.set_state(f0, g0)
    E_ref = np.array([o.step() for _ in range(steps)])
    with binding.ParaisoWave(n) as w:
        w.set_state(f0, g0)
        E = np.concatenate([w.step(steps // 2), w.step(steps - steps // 2)])
        f, g = w.get_state()
        assert w.launch_count() == steps
    fr, gr = o.get_state()
    assert np.array_equal(f, fr) and np.array_equal(g, gr)
    assert np.abs(E - E_ref).max() <= 1e-13 * E_ref.max(), np.abs(E - E_ref).max() / E_ref.max()
    if n >= 8:
        assert (E.max() - E.min()) / E.mean() < 1e-12
