"""The hot path's division and square root (csrc/hydro_math.cuh div_rn / sqrt_rn) against IEEE-754.

DESIGN.md §4: the kernels use the fast path of the IEEE sequences without the range check; inside the
normal range the result must be the correctly rounded one, i.e. identical to what the oracle's `/` and
`std::sqrt` produce on the host.  NumPy's float32 / float64 `/` and `sqrt` are IEEE correctly rounded, so
they are the reference here (no oracle code involved).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _operands(dtype, n, seed, lo_exp, hi_exp):
    rng = np.random.default_rng(seed)
    mant = rng.uniform(1.0, 2.0, n)
    e = rng.integers(lo_exp, hi_exp + 1, n)
    sign = rng.choice([-1.0, 1.0], n)
    return (sign * np.ldexp(mant, e)).astype(dtype)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_div_and_sqrt_are_correctly_rounded_in_the_normal_range(dtype):
    import torch

    from paper_1204_4779_b200 import binding

    n = 1 << 22
    for seed, (lo, hi) in enumerate([(-2, 2), (-20, 20), (-60, 60)]):
        a = _operands(dtype, n, 100 + seed, lo, hi)
        b = _operands(dtype, n, 200 + seed, lo, hi)
        # a few structured cases: equal operands, near-equal mantissas, zero numerators, powers of two
        a[:1000] = b[:1000]
        a[1000:2000] = np.nextafter(b[1000:2000], dtype(np.inf))
        a[2000:3000] = 0.0
        b[3000:4000] = np.ldexp(1.0, np.arange(1000) % 41 - 20).astype(dtype)
        q, r = binding.probe_arith(torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda())
        q, r = q.cpu().numpy(), r.cpu().numpy()
        with np.errstate(all="ignore"):
            qref, rref = a / b, np.sqrt(np.abs(a))
        nz = a != 0
        assert np.array_equal(q[nz], qref[nz]), (dtype, lo, hi, int(np.sum(q[nz] != qref[nz])))
        assert np.all(q[~nz] == 0)
        assert np.array_equal(r[nz], rref[nz]), (dtype, lo, hi, int(np.sum(r[nz] != rref[nz])))


def test_issue_cost_of_the_instruction_classes():
    """DESIGN.md §8 reads the ncu captures with this model: an FFMA costs one scheduler cycle, an ALU-pipe
    instruction (FMNMX, FSETP, FSEL, IADD3, LOP3) about two even with FFMA work to overlap, a packed FFMA2 two
    (two results: half the issue slots per result), a DFMA two.  Measured on the device under test."""
    import subprocess

    from paper_1204_4779_b200 import binding

    try:
        mhz = float(subprocess.run(["nvidia-smi", "--query-gpu=clocks.max.sm", "--format=csv,noheader,nounits", "-i", "0"],
                                   capture_output=True, text=True, timeout=30).stdout.split()[0])
    except Exception:
        mhz = 1965.0
    cost = {k: binding.probe_issue_cost(k, mhz)[0] for k in binding.ISSUE_KINDS}
    base = binding.probe_issue_cost("ffma", mhz)[1]
    print("issue cost in scheduler cycles per instruction:", {k: round(v, 2) for k, v in cost.items()}, "16-FFMA loop:", round(base, 1))
    assert 16.0 <= base <= 30.0            # 16 FFMA + loop control at about one instruction per cycle
    assert 0.8 <= cost["ffma"] <= 1.4
    for k in ("fmnmx", "fsetp_fsel", "iadd3_lop3"):
        assert 1.4 <= cost[k] <= 2.6, (k, cost[k])
    assert 1.6 <= cost["ffma2"] <= 2.6 and 1.6 <= cost["dfma"] <= 2.6
    assert cost["mufu"] >= 1.6


def test_measured_peak_lane_rates():
    """paraiso_probe_peak: the measured denominators of roofline (b).  FFMA2 reaches the nominal FP32 lane rate
    (148 SMs x 128 lanes x clock), scalar FFMA stays below it, DFMA is half the FP32 rate."""
    from paper_1204_4779_b200 import binding

    pk = {k: binding.probe_peak(k) for k in binding.PEAK_KINDS}
    print("measured peak, Tera fused-multiply-adds/s:", {k: round(v, 2) for k, v in pk.items()})
    nominal = 148 * 128 * 1.965e9 / 1e12
    assert 0.5 * nominal <= pk["ffma"] <= 1.05 * nominal
    assert 0.7 * nominal <= pk["ffma2"] <= 1.05 * nominal
    assert 0.25 * nominal <= pk["dfma"] <= 0.55 * nominal


def test_mix_ceiling_probe():
    """paraiso_probe_mix_ceiling: the stage kernel's instruction mix without dependencies issues well below one
    instruction per cycle on four warps per scheduler (the packed FMA and the ALU instructions each hold their pipe for
    two cycles): the ceiling DESIGN.md §8 reads the kernel's 0.51-0.53 against."""
    from paper_1204_4779_b200 import binding

    packed = binding.probe_mix_ceiling(0, 1965.0)
    scalar = binding.probe_mix_ceiling(1, 1965.0)
    print(f"mix ceiling: packed {packed:.3f} IPC (76 instructions), scalar {scalar:.3f} IPC (108 instructions)")
    assert 0.55 < packed < 0.9 and 0.7 < scalar < 1.01
    assert 76.0 / packed < 108.0 / scalar  # the packed mix still finishes the same work sooner
