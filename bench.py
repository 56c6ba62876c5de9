"""bench.py — Gcell-updates/s per full RK2 step of the Euler hot path (BASELINE.json metric) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--variant fused] [--riemann hllc]
                    [--impl reference] [--no-sweep] [--no-cpu]

A "step" = one full RK2 step (both stages a1-a5 + the CFL reduction a0, dt read on the device from the
previous step's fused reduction) of one synthetic workload.  Default workload = BASELINE
config 4 (3-D blast 512^3 fp32, 2.7 GB per state buffer: larger than L2, no flush needed); the other configs
are added to the same JSON line under "all_configs" (short runs; config 1 is L2-resident, said so there).

  value     cells * steps / device time (CUDA events on the handle's stream, max over ranks), state resident in HBM
  e2e       same metric through the C ABI with HOST (pinned) buffers: set_state(host) + cfl_dt + step +
            get_state(host) every step, copies inside the timed region
  roofline  dominant kernel = the RK stage kernel, duration = CUDA events around every stage launch inside the timed
            region.  north_star's roofline is the slower of (a) 2*nf*w*N algorithmic bytes per launch over the measured
            copy bandwidth (MEASURED_PEAKS.json) and (b) the counted arithmetic of DESIGN.md §8 over the NOMINAL FP32 / FP64
            lane rate (`counted_ops_oracle`: the same run against the oracle's mechanical count, profiles/r3_counted_ops.json); the binding one is reported as `bound`, the other under `other_bound`; `traffic` = ncu DRAM
            bytes per launch (profiles/r*_cfg*_ncu_raw.csv); `issue_cost_cycles` = measured issue cost per instruction class
  cpu_baseline  the oracle as it stands, single-threaded and OpenMP, on a bounded sample of the same workload

N > 1: replicas only: every rank advances its own copy of the workload, no data-path collective;
value = all ranks' cell updates / max-over-ranks time, "scaling": "weak".
--impl reference: the oracle (oracle/, OpenMP build) timed on the host cores; rank 0 only.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "Gcell-updates/s per RK2 step"
UNIT = "Gcell/s"
DEFAULT_STEPS = {0: 279, 1: 100, 2: 50, 3: 50, 4: 20, 11: 50, 13: 20}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md clocks line)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc, self.thread = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
        except OSError:
            return self
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [c.strip() for c in line.split(",")]))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [r for t, r in self.rows if t0 <= t <= t1 + 0.1] or [r for _, r in self.rows[-3:]]
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
                pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def algorithmic_bytes_per_cell_step(w):
    """north_star roofline (a): state read and written once per stage, halo excluded = 4*nf*w bytes per cell-step."""
    return 4 * w.nf * w.dtype.itemsize


def make_workload(cfg):
    from paper_1204_4779_b200 import inputs

    return inputs.baseline_config(cfg)


def centred_sample(w, edge):
    """A centred sub-box (edge cells per axis, at most the grid) of the workload's own initial state, as a
    periodic problem of the same mesh size: the bounded sample the oracle is timed on."""
    from paper_1204_4779_b200 import inputs

    sl = [slice(None)]
    n = []
    for a in reversed(range(w.dims)):  # array axes are [f][z][y][x]
        m = min(edge, w.n[a])
        lo = (w.n[a] - m) // 2
        sl.append(slice(lo, lo + m))
        n.append(m)
    n = tuple(reversed(n))
    U = np.ascontiguousarray(w.U[tuple(sl)])
    ext = tuple(w.extent[a] * n[a] / w.n[a] for a in range(w.dims))
    return inputs.Workload(w.name + "_sample" + "x".join(map(str, n)), n, ext, w.gamma, w.dtype, "periodic", w.cfl, 0, 0.0, U)


def oracle_rate(w, steps, warmup, threads):
    """Gcell/s of the oracle (oracle/euler_oracle.cpp as it stands) on workload w; returns (rate, seconds, cores)."""
    import oracle

    o = oracle.Oracle(w.n, w.extent, w.gamma, w.dtype, w.boundary, "hllc", threads)
    o.set_state(w.U)
    for _ in range(warmup):
        o.step(o.cfl_dt(w.cfl))
    t0 = time.perf_counter()
    for _ in range(steps):
        o.step(o.cfl_dt(w.cfl))
    dt = time.perf_counter() - t0
    o.close()
    cores = oracle.num_threads("omp") if threads == "omp" else 1
    return w.cells * steps / dt / 1e9, dt, cores


def cpu_baseline(w):
    edge = {1: 1 << 20, 2: 1536, 3: 144}[w.dims]
    s = centred_sample(w, edge)
    # the serial figure is one warm-up step, then 2 full RK2 steps (+ CFL reduction), pinned to one core
    try:
        allowed = os.sched_getaffinity(0)
        os.sched_setaffinity(0, {min(allowed)})
    except (AttributeError, OSError):
        allowed = None
    try:
        r1, t1, _ = oracle_rate(s, 2, 1, "serial")
    finally:
        if allowed:
            os.sched_setaffinity(0, allowed)
    t1 /= 2.0  # seconds per serial step
    steps = max(2, int(8.0 / max(t1 / 8, 1e-3) / 8))  # ~8 s of OpenMP work if it scales, capped below
    steps = min(steps, 12)
    rn, tn, cores = oracle_rate(s, steps, 1, "omp")
    return {"value": rn, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"centred {'x'.join(map(str, s.n))} sub-box of the workload's initial state, periodic, "
                      f"{steps} RK2 steps (OpenMP build of oracle/euler_oracle.cpp, bit-identical to serial)",
            "serial_value": r1, "serial_cores": 1, "serial_sample": "same sub-box, 1 warm-up + 2 timed RK2 steps pinned to one core",
            "seconds": t1 * 3 + tn}


def reference_arm(args):
    """--impl reference: the oracle timed on the host cores, same metric / config keys; rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = make_workload(args.config)
    edge = {1: 1 << 20, 2: 1024, 3: 128}[w.dims]
    s = centred_sample(w, edge)
    rate, secs, cores = oracle_rate(s, args.steps, args.warmup, "omp")
    sample = (f"each step = one oracle RK2 step (+ CFL reduction) on the centred {'x'.join(map(str, s.n))} sub-box of "
              f"config {args.config}'s initial state, periodic")
    line = {"impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": secs / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32" if w.dtype == np.float32 else "f64", "data": "synthetic",
            "config": {"workload": f"BASELINE config {args.config}: {w.name}", "grid": list(w.n), "riemann": "hllc",
                       "sample": sample},
            "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


WARMUP_SECONDS = 0.5  # device work before anything is timed (clock ramp), on top of the --warmup steps
REPEATS = 30          # every individual is scored by the mean and deviation of 30 runs


def device_run(binding, torch, w, steps, warmup, variant, riemann, per_stage, options=None, repeats=0,
               warmup_seconds=WARMUP_SECONDS):
    """K device-paced steps with the state resident in HBM; returns dict(ms, stage_ms, stage_launches, launches, ...).

    Warm-up: `warmup` steps, then further steps until `warmup_seconds` of device work have run (untimed); the state is
    then set again so that the timed K steps are the first K steps of the workload.  repeats > 0: the same K-step run
    (state set again before each) is timed `repeats` more times; their mean / sample deviation / extremes are returned
    under "repeats" (the headline stays the first run, as the bench contract words it)."""
    s = torch.cuda.Stream()
    with binding.ParaisoHydro(w.n, w.extent, w.gamma, w.dtype, w.boundary, riemann, variant, stream=s,
                              **(options or {})) as h:
        dev = torch.from_numpy(w.U).cuda()
        h.set_state(dev)
        h.run(w.cfl, warmup)
        h.sync()
        t_w = time.perf_counter()
        chunk = max(1, min(steps, 8))
        while time.perf_counter() - t_w < warmup_seconds:
            h.run(w.cfl, chunk)
            h.sync()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

        def timed(first):
            h.set_state(dev)  # device source: stays alive until the handle is closed (the copy is asynchronous)
            h.run(w.cfl, warmup)
            h.sync()
            if first and per_stage:
                h.kernel_time(1)
            torch.cuda.synchronize()
            counted[0] = h.launch_count()
            e0.record(s)
            h.run(w.cfl, steps)
            e1.record(s)
            e1.synchronize()
            torch.cuda.synchronize()
            counted[1] = h.launch_count()
            return e0.elapsed_time(e1)

        counted = [0, 0]  # the library's launch counter before / after the timed region
        ms = timed(True)
        launches = counted[1] - counted[0]
        stage_ms, stage_n = h.kernel_time() if per_stage else (ms, 2 * steps)
        if per_stage:  # the warm-up steps of timed() ran before the stage clock was switched on
            h.kernel_time(0)
        bad = h.stats()
        t, k = h.time()
        if bad or k != steps + warmup:
            raise RuntimeError(f"bench run unhealthy: nonfinite={bad} steps={k}")
        rep = None
        if repeats > 0:
            rates = [w.cells * steps / (timed(False) * 1e-3) / 1e9 for _ in range(repeats)]
            rep = {"n": repeats, "mean": float(np.mean(rates)), "stdev": float(np.std(rates, ddof=1)) if repeats > 1 else 0.0,
                   "min": float(min(rates)), "max": float(max(rates)), "unit": UNIT}
        h.sync()
        del dev
    return {"ms": ms, "stage_ms": stage_ms, "stage_launches": stage_n, "launches": launches, "t": t, "repeats": rep}


def e2e_run(binding, torch, w, steps, warmup, variant, riemann):
    """The same metric through the C ABI with HOST buffers: every step copies the state host -> device
    (set_state from pinned memory), computes dt (cfl_dt), advances one RK2 step and copies the result back."""
    src = torch.from_numpy(w.U).pin_memory()
    dst = torch.empty_like(src).pin_memory()
    s = torch.cuda.Stream()
    with binding.ParaisoHydro(w.n, w.extent, w.gamma, w.dtype, w.boundary, riemann, variant, stream=s) as h:
        def one(inp, out):
            h.set_state(inp)
            h.step(h.cfl_dt(w.cfl))
            h.get_state(out)

        one(src, dst)
        for _ in range(max(0, warmup - 1)):
            one(dst, dst)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        e0.record(s)
        for _ in range(steps):
            one(dst, dst)
        e1.record(s)
        e1.synchronize()
        wall = time.perf_counter() - t0
        ms = max(e0.elapsed_time(e1), wall * 1e3)  # host-blocking calls are part of the end-to-end time
        assert bool(torch.isfinite(dst).all())
    nbytes = w.U.nbytes
    return {"value": w.cells * steps / (ms * 1e-3) / 1e9, "unit": UNIT, "h2d_bytes_per_step": nbytes,
            "d2h_bytes_per_step": nbytes, "ms_per_step": ms / steps, "steps": steps}


# Counted arithmetic of DESIGN.md §4 per cell per RK2 step (HLLC; DESIGN.md §8 derives the table): every + - x fma
# compare select min max abs is one lane-operation, an IEEE division / square root is expanded to the fma sequence the
# kernels execute (fp32: 1 MUFU + 5 / 4 operations, fp64: 1 MUFU + 7 / 9).  Roofline (b) of north_star = these
# operations over the FP32 (128 lanes per SM) or FP64 (64 lanes per SM) lane rate of 148 SMs at 1.965 GHz.
COUNTED_OPS_PER_CELL_STEP = {(1, 4): 299, (2, 4): 638, (3, 4): 1053, (1, 8): 354, (2, 8): 737, (3, 8): 1196}
SM_MAX_GHZ = 1.965


def sm_count():
    """SMs of the device in use (148 on a B200), from the driver."""
    import torch

    return int(torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count)


def alu_peak_tlaneops(itemsize):
    return sm_count() * (128 if itemsize == 4 else 64) * SM_MAX_GHZ * 1e9 / 1e12


# arith = 1 (f32fast): an IEEE division (1 MUFU + 5) / square root (1 MUFU + 4) becomes 1 MUFU + 1 multiplication
COUNTED_OPS_ARITH1 = {(2, 4): 638 - (27 * 4 + 9 * 3), (3, 4): 1053 - (39 * 4 + 13 * 3)}
_MEASURED_ALU_PEAK = {}


def measured_alu_peak(binding, itemsize):
    """Tlaneop/s of the FFMA / FFMA2 (fp32) or DFMA (fp64) pipe measured on this device by the probe library
    (paraiso_probe_peak: 16 independent chains per thread, 8 warps per scheduler, best of 5 short launches), or None."""
    if itemsize not in _MEASURED_ALU_PEAK:
        try:
            # fp32: the better of the scalar and the packed instruction (the packed one reaches the higher lane rate)
            _MEASURED_ALU_PEAK[itemsize] = (max(float(binding.probe_peak("ffma")), float(binding.probe_peak("ffma2")))
                                            if itemsize == 4 else float(binding.probe_peak("dfma")))
        except Exception:
            _MEASURED_ALU_PEAK[itemsize] = None
    return _MEASURED_ALU_PEAK[itemsize]


_ORACLE_COUNTS = None


def oracle_counted_ops(dims, itemsize, riemann):
    """The mechanical count of profiles/r3_counted_ops.json (the oracle instantiated with a counting scalar type,
    `python tests/count_ops.py`; a committed table, nothing under oracle/ is executed here): issue slots per cell per
    RK2 step for this dimension / precision / solver as {"composed": ..., "as_written": ...}, or None."""
    global _ORACLE_COUNTS
    if _ORACLE_COUNTS is None:
        _ORACLE_COUNTS = {}
        try:
            for row in json.load(open(os.path.join(ROOT, "profiles", "r3_counted_ops.json")))["rows"]:
                a = row["after_20_steps"]
                _ORACLE_COUNTS.setdefault((row["dims"], row["itemsize"], row["riemann"]),
                                          {"composed": a["composed"]["slots"], "as_written": a["as_written"]["slots"],
                                           "workload": row["workload"]})
        except Exception:
            pass
    return _ORACLE_COUNTS.get((dims, itemsize, riemann))


def roofline_of(w, r, peak, peak_src, traffic=None, binding=None, counted_ops=None, riemann="hllc"):
    """The slower of north_star's two rooflines is the binding one and is reported as `bound`; the other is kept
    beside it.  (a) HBM: 2*nf*w*N algorithmic bytes per stage launch (state read once, written once; halo excluded)
    over the measured copy bandwidth.  (b) ALU: counted lane-operations per stage launch over the FP32 / FP64 lane
    rate derived from the guide's unit counts and clock."""
    isz = w.dtype.itemsize
    nbytes = 2 * w.nf * isz * w.cells
    avg_ms = r["stage_ms"] / max(1, r["stage_launches"])
    hbm_achieved = nbytes / (avg_ms * 1e-3) / 1e9
    # numerator: HLLC = the hand table of what the kernels execute (upwind side chosen first, selects counted); HLL has
    # no hand table: the oracle's mechanical count (composed: one interpolation per cell and axis) stands in for it
    mech = oracle_counted_ops(w.dims, isz, riemann)
    if counted_ops:
        counted, count_src = counted_ops, "hand table, arith = 1 (DESIGN.md R21)"
    elif riemann == "hll" and mech:
        counted, count_src = mech["composed"], "profiles/r3_counted_ops.json: oracle with a counting scalar, composed, HLL"
    else:
        counted, count_src = COUNTED_OPS_PER_CELL_STEP[(w.dims, isz)], "hand table of DESIGN.md §8 (HLLC, what the kernels execute)"
    ops = counted / 2.0 * w.cells
    alu_achieved = ops / (avg_ms * 1e-3) / 1e12
    alu_nominal = alu_peak_tlaneops(isz)
    alu_measured = measured_alu_peak(binding, isz) if binding is not None else None
    # `frac` divides by the FIXED nominal peak (unit counts x max clock) so that rounds stay comparable; the peak the
    # probe measured on this device in this run (best of 5 short launches: it moves with the power state) is reported
    # beside it as peak_measured / frac_of_measured.  DESIGN.md §8: north_star's 0.70 is read against `frac`.
    alu_peak = alu_nominal
    hbm = {"bound": "hbm", "achieved": hbm_achieved, "peak": peak, "unit": "GB/s", "frac": hbm_achieved / peak,
           "algorithmic_bytes_per_launch": nbytes, "peak_source": peak_src,
           "gcell_per_s_at_peak": peak * 1e9 / (4 * w.nf * isz) / 1e9}
    alu = {"bound": "alu", "achieved": alu_achieved, "peak": alu_peak, "unit": "Tlaneop/s", "frac": alu_achieved / alu_peak,
           "algorithmic_ops_per_launch": ops, "counted_ops_per_cell_step": counted, "counted_ops_source": count_src,
           # the same run read against the oracle's mechanical counts; nominal peak
           "counted_ops_oracle": None if not mech else {
               "composed": mech["composed"], "as_written": mech["as_written"],
               "frac_composed": mech["composed"] / 2.0 * w.cells / (avg_ms * 1e-3) / 1e12 / alu_nominal,
               "frac_as_written": mech["as_written"] / 2.0 * w.cells / (avg_ms * 1e-3) / 1e12 / alu_nominal,
               "source": "profiles/r3_counted_ops.json (python tests/count_ops.py), %s, %s" % (mech["workload"], riemann)},
           "peak_source": "nominal: %d SMs x %d %s lanes x %.3f GHz (B200_PROFILING.md unit counts and clocks.max.sm)"
                          % (sm_count(), 128 if isz == 4 else 64, "FP32" if isz == 4 else "FP64", SM_MAX_GHZ),
           "peak_nominal": alu_nominal, "frac_of_nominal": alu_achieved / alu_nominal,
           "peak_measured": alu_measured, "frac_of_measured": (alu_achieved / alu_measured) if alu_measured else None,
           "peak_measured_source": ("%s fused multiply-adds per second on this device (paraiso_probe_peak)"
                                    % ("max(FFMA, FFMA2)" if isz == 4 else "DFMA")) if alu_measured else None,
           "gcell_per_s_at_peak": alu_peak * 1e12 / counted / 1e9}
    first, other = (alu, hbm) if alu["gcell_per_s_at_peak"] < hbm["gcell_per_s_at_peak"] else (hbm, alu)
    out = dict(first)
    out.update({"traffic": traffic, "kernel": "RK stage kernel(s) (a1-a5 [+a0 in stage 2])", "avg_launch_ms": avg_ms,
                "other_bound": other})
    return out


_UNIT_BYTES = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def ncu_traffic(cfg, variant):
    """dram__bytes_read.sum + dram__bytes_write.sum per STAGE of the RK2 step, parsed from the committed raw ncu export
    profiles/r<round>_cfg<cfg>_<variant>_ncu_raw.csv (newest round first) (`ncu -i ... --page raw --csv` of one `ncu --set full` capture that
    holds exactly the kernels of ONE step, the .md beside it names the command): the sum over every captured launch
    divided by the two stages.  For the one-kernel-per-stage variants that is the mean of the two stage launches.
    Returns (bytes per stage, file name) or (None, None) if that configuration was not captured."""
    import csv

    for rnd in ("r3", "r2"):  # the newest committed capture of this configuration
        name = f"{rnd}_cfg{cfg}_{variant}_ncu_raw.csv"
        p = os.path.join(ROOT, "profiles", name)
        if os.path.exists(p):
            break
    else:
        return None, None
    try:
        rows = list(csv.reader(open(p)))
        hdr, units, data = rows[0], rows[1], rows[2:]
        total = 0.0
        for key in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
            i = hdr.index(key)
            total += sum(float(r[i]) for r in data) * _UNIT_BYTES[units[i]]
        return total / 2.0, name
    except Exception:
        return None, None


def replicas_aggregate(ms_local, cells, steps, world, device=None):
    """Replicas only: every rank advanced its own copy of the workload.  Returns (max-over-ranks
    device time in ms, whole-job Gcell/s = all ranks' cell updates / that time).  The only collective is this
    all-reduce(max) of one timing scalar; it works on any torch.distributed backend (NCCL on GPUs, gloo in tests)."""
    ms = float(ms_local)
    if world > 1:
        import torch
        import torch.distributed as dist

        t = torch.tensor([ms], dtype=torch.float64, device=device if device is not None else "cpu")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    return ms, cells * steps * world / (ms * 1e-3) / 1e9


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--variant", default="fused")
    ap.add_argument("--riemann", default="hllc")
    ap.add_argument("--impl", default="b200")
    ap.add_argument("--no-sweep", action="store_true", help="skip the short runs of the other configs / variants")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--repeats", type=int, default=REPEATS, help="further timed runs of the same K steps (mean +- deviation)")
    ap.add_argument("--warmup-seconds", type=float, default=WARMUP_SECONDS,
                    help="device work before the timed steps, on top of --warmup (0 under ncu: a fixed launch sequence)")
    ap.add_argument("--opt", action="append", default=[], help="key=value launch-shape option (block_x, ...)")
    args = ap.parse_args()
    if args.steps is None:
        args.steps = DEFAULT_STEPS[args.config]
    args.warmup = max(args.warmup, 0)
    if args.impl == "reference":
        return reference_arm(args)

    import torch
    import torch.distributed as dist

    from paper_1204_4779_b200 import binding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    binding.load_library()
    options = {k: int(v) for k, v in (o.split("=") for o in args.opt)}

    w = make_workload(args.config)
    big = w.cells >= (1 << 22)  # per-stage events only where a stage is >> an event record
    peak, peak_src = measured_peaks()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    barrier()
    sampler = ClockSampler(local).start() if rank == 0 else None
    t0 = time.time()
    r = device_run(binding, torch, w, args.steps, args.warmup, args.variant, args.riemann, big, options,
                   repeats=args.repeats, warmup_seconds=args.warmup_seconds)
    t1 = time.time()
    barrier()
    clocks = sampler.stop(t0, t1) if sampler else None
    ms, value = replicas_aggregate(r["ms"], w.cells, args.steps, world, "cuda")

    e2e = None
    if not args.no_e2e:
        e = e2e_run(binding, torch, w, min(args.steps, 5), min(args.warmup, 2), args.variant, args.riemann)
        _, ev = replicas_aggregate(e["ms_per_step"], w.cells, 1, world, "cuda")
        e2e = dict(e, value=ev, h2d_bytes_per_step=e["h2d_bytes_per_step"] * world,
                   d2h_bytes_per_step=e["d2h_bytes_per_step"] * world)

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "warmup_seconds": args.warmup_seconds,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if w.dtype == np.float32 else "f64", "data": "synthetic",
            "config": {"workload": f"BASELINE config {args.config}: {w.name}", "grid": list(w.n), "fields": w.nf,
                       "gamma": w.gamma, "cfl": w.cfl, "boundary": w.boundary, "riemann": args.riemann,
                       "variant": args.variant, "options": options, "parallelism": "replicas" if world > 1 else "1gpu",
                       "l2": "state buffers (2 x %.0f MB) exceed the 126 MB L2; no flush needed" % (w.U.nbytes / 1e6)
                       if 2 * w.U.nbytes > 126e6 else "L2-RESIDENT workload (2 x %.1f MB): not an HBM number" % (w.U.nbytes / 1e6)},
            "roofline": roofline_of(w, r, peak, peak_src, binding=binding if rank == 0 else None, riemann=args.riemann,
                                    counted_ops=COUNTED_OPS_ARITH1.get((w.dims, w.dtype.itemsize)) if options.get("arith") == 1 else None),
            "e2e": e2e, "gpu_launches": r["launches"], "clocks": clocks}
    traffic, traffic_file = ncu_traffic(args.config, args.variant) if not options else (None, None)
    line["roofline"]["traffic"] = traffic
    line["roofline"]["traffic_source"] = ("profiles/" + traffic_file + " (dram__bytes_read.sum + dram__bytes_write.sum of one "
                                          "captured step / 2 stages)") if traffic_file else None
    if r["repeats"]:
        line["repeats"] = dict(r["repeats"], note="rank 0, per GPU: %d further runs of the same %d steps, the state set again "
                                                   "before each (PAPER.md:626 scores by mean and deviation of 30 runs)"
                                                   % (r["repeats"]["n"], args.steps))

    if rank == 0:
        # measured issue cost (scheduler cycles per instruction) of the instruction classes of the stage kernel on
        # this device: the model DESIGN.md §8 reads the ncu captures with
        mhz = (clocks or {}).get("sm_mhz") or 1965.0
        line["roofline"]["issue_cost_cycles"] = {k: round(binding.probe_issue_cost(k, mhz)[0], 3) for k in binding.ISSUE_KINDS}
        # the issue rate the default stage kernel's instruction mix reaches with NO dependencies (4 warps per scheduler):
        # the ceiling its ncu-measured issue rate (profiles/r2_ncu_summary.txt: 0.51-0.53) is to be read against
        line["roofline"]["mix_ceiling_ipc"] = {"k_pack_mix_packed": round(binding.probe_mix_ceiling(0, mhz), 3),
                                               "same_work_scalar_ffma": round(binding.probe_mix_ceiling(1, mhz), 3)}
    if rank == 0 and not args.no_sweep:
        line["all_configs"] = sweep(binding, torch, args, peak, peak_src)
    if rank == 0 and not args.no_cpu:
        line["cpu_baseline"] = cpu_baseline(w)
    if rank == 0 and "all_configs" in line:
        # LAST key on purpose (a reader of the tail of the line sees every config): the default variant of each config,
        # HLLC and HLL, with the fraction of the binding roofline (nominal peak) and its own clock sample
        line["configs_summary"] = [{"config": x["config"], "riemann": x.get("riemann", args.riemann), "gcell_per_s": round(x["value"], 3),
                                    "bound": x["bound"], "frac": round(x["frac"], 4), "sm_mhz": x["clocks"]["sm_mhz"],
                                    "reasons": x["clocks"]["reasons"]}
                                   for x in line["all_configs"] if x.get("variant") == "fused" and "error" not in x]
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line), flush=True)


def sweep(binding, torch, args, peak, peak_src):
    """Short runs of every BASELINE config (and of the 4096^2 fp32 / 256^3 fp64 extras) with every kernel variant (the
    Manifest <-> Delayed axis), same protocol: >= WARMUP_SECONDS of device work before the timed steps, each row with
    its own clock sample."""
    out = []
    local = int(os.environ.get("LOCAL_RANK", "0"))
    for cfg in (0, 1, 2, 3, 4, 11, 13):
        w = make_workload(cfg)
        big = w.cells >= (1 << 22)
        steps = min(DEFAULT_STEPS[cfg], 100 if not big else 10)
        for variant in ("fused", "fused hll", "pack", "march", "fused1", "manifest_flux", "manifest_all", "delayed", "march arith=1"):
            opts, counted = None, None
            riemann = args.riemann
            if variant == "fused hll":  # HLL reported beside HLLC for the default variant of configs 1-4
                if cfg not in (1, 2, 3, 4) or args.riemann == "hll":
                    continue
                riemann = "hll"
            if variant == "march arith=1":  # fp32 only: hardware rcp / rsqrt approximations, inside the tolerances, not bit-equal
                if w.dtype != np.float32 or w.dims == 1:
                    continue
                opts = {"arith": 1}
                counted = COUNTED_OPS_ARITH1[(w.dims, 4)]  # its own counted work, not the IEEE sequences'
            if cfg in (11, 13) and variant in ("manifest_flux", "manifest_all", "delayed", "fused1"):
                continue  # the extras are there for the on-chip kernels
            sampler = ClockSampler(local).start()
            t0 = time.time()
            try:
                r = device_run(binding, torch, w, steps, 3, variant.split()[0], riemann, big, opts)
            except Exception as ex:  # shape not covered, out of memory for manifest_all, ...
                sampler.stop(t0, time.time())
                out.append({"config": cfg, "variant": variant, "error": str(ex)[:120]})
                continue
            clocks = sampler.stop(t0, time.time())
            rl = roofline_of(w, r, peak, peak_src, binding=binding, counted_ops=counted, riemann=riemann)
            out.append({"config": cfg, "workload": w.name, "variant": variant.split()[0] if variant == "fused hll" else variant,
                        "riemann": riemann, "steps": steps,
                        "value": w.cells * steps / (r["ms"] * 1e-3) / 1e9, "unit": UNIT, "ms_per_step": r["ms"] / steps,
                        "bound": rl["bound"], "frac": rl["frac"],
                        "hbm_frac": (rl if rl["bound"] == "hbm" else rl["other_bound"])["frac"],
                        "alu_frac": (rl if rl["bound"] == "alu" else rl["other_bound"])["frac"],
                        "counted_ops_per_cell_step": (rl if rl["bound"] == "alu" else rl["other_bound"])["counted_ops_per_cell_step"],
                        "launches": r["launches"],
                        "clocks": {"sm_mhz": clocks.get("sm_mhz"), "reasons": clocks.get("reasons")}})
        del w
    return out


if __name__ == "__main__":
    main()
