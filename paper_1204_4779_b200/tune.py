"""The paper's Manifest / Delayed search, rebuilt as a measured sweep over this library's variant space.

    python -m paper_1204_4779_b200.tune --config 4 [--repeats 5] [--steps 5] [--riemann hllc] [--json out.json]

Paraiso tunes its generated solvers with a genetic algorithm over per-intermediate Manifest / Delayed choices and
synchronisation points, scoring each individual by the mean and deviation of repeated runs (PAPER.md:610-676, 30
samples per individual PAPER.md:626).  Here the space is small enough to enumerate: kernel variant x launch shape x
cells per thread x staging.  Every candidate advances the same seeded workload with the state resident
in HBM; the score is Gcell-updates/s per RK2 step from CUDA events on the handle's stream, mean and sample deviation
over `--repeats` runs of `--steps` device-paced steps after one warm-up run.  Candidates a grid does not admit (shape
not covered, out of memory) are reported as skipped.  Needs a CUDA device; there is no CPU fallback.
"""
import argparse
import itertools
import json
import statistics
import sys


def candidates(dims, dtype_is_f32):
    """(label, variant, options) for a grid of `dims` dimensions."""
    out = [("manifest_all", "manifest_all", {}), ("manifest_flux", "manifest_flux", {}), ("delayed", "delayed", {})]
    if dims == 1:
        return out
    depths = (0, 32, 128)
    # k_pack (shared-memory window; fp32: packed pairs of cells, fp64: one cell per thread), the default on-chip kernel
    if dims == 3:
        for ty, d in itertools.product((5, 7, 11, 14, 15) if dtype_is_f32 else (7, 14), (0, 64)):
            out.append((f"pack ty={ty}{' two halo warps' if ty == 14 else ''} depth={d or 'auto'}", "pack",
                        {"block_y": ty, "tile_depth": d}))
    else:
        for nwx, d in itertools.product((1, 2, 4, 8) if dtype_is_f32 else (2, 4, 8), (0, 32, 64)):
            out.append((f"pack warps={nwx} overlapping tiles depth={d or 'auto'}", "pack", {"block_x": nwx, "tile_depth": d}))
        for nwx in (4, 7):
            out.append((f"pack warps={nwx} halo warp", "pack", {"block_x": nwx, "block_z": 1}))
    if dims == 3:
        for ty, d in itertools.product((4, 7, 8, 15), depths):
            out.append((f"march ty={ty} depth={d or 'auto'}", "march", {"block_y": ty, "tile_depth": d}))
        for (tx, ty), d in itertools.product(((32, 8), (32, 16), (64, 8)), depths):
            out.append((f"fused1 {tx}x{ty} depth={d or 'auto'}", "fused1", {"block_x": tx, "block_y": ty, "tile_depth": d}))
        if dtype_is_f32:
            for ty in (7, 8):
                out.append((f"march packed f32x2 ty={ty}", "march", {"block_y": ty, "cells_per_thread": 2}))
        out.append(("march ty=7 TMA staging", "march", {"block_y": 7, "staging": 2}))
        out.append(("march ty=7 tensor-map TMA staging", "march", {"block_y": 7, "staging": 3}))
        out.append(("march ty=7 two rows per thread", "march", {"block_y": 7, "block_z": 2}))
        if dtype_is_f32:
            out.append(("march ty=7 arith=1 (not bit-equal)", "march", {"block_y": 7, "arith": 1}))
    else:
        for nwx, d in itertools.product((2, 4, 8), depths):
            out.append((f"march warps={nwx} depth={d or 'auto'}", "march", {"block_x": nwx, "tile_depth": d}))
        for tx, d in itertools.product((64, 128, 256, 512), depths):
            out.append((f"fused1 row={tx} depth={d or 'auto'}", "fused1", {"block_x": tx, "tile_depth": d}))
        if dtype_is_f32:
            out.append(("march packed f32x2 warps=4", "march", {"block_x": 4, "cells_per_thread": 2}))
        out.append(("march warps=4 TMA staging", "march", {"block_x": 4, "staging": 2}))
        out.append(("march warps=4 tensor-map TMA staging", "march", {"block_x": 4, "staging": 3}))
        if dtype_is_f32:
            out.append(("march warps=4 arith=1 (not bit-equal)", "march", {"block_x": 4, "arith": 1}))
    return out


def score(binding, torch, w, variant, options, riemann, steps, repeats):
    s = torch.cuda.Stream()
    with binding.ParaisoHydro(w.n, w.extent, w.gamma, w.dtype, w.boundary, riemann, variant, stream=s, **options) as h:
        dev = torch.from_numpy(w.U).cuda()
        rates = []
        for r in range(repeats + 1):
            h.set_state(dev)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            h.sync()
            e0.record(s)
            h.run(w.cfl, steps)
            e1.record(s)
            e1.synchronize()
            if h.stats():
                raise RuntimeError("non-finite state")
            if r:  # the first run is the warm-up (graph capture, first-touch)
                rates.append(w.cells * steps / (e0.elapsed_time(e1) * 1e-3) / 1e9)
    return statistics.mean(rates), (statistics.stdev(rates) if len(rates) > 1 else 0.0)


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--repeats", type=int, default=5)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--riemann", default="hllc")
    ap.add_argument("--json", default=None)
    args = ap.parse_args()

    import numpy as np
    import torch

    from . import binding, inputs

    if not torch.cuda.is_available():
        raise SystemExit("tune needs a CUDA device: the product path has no CPU fallback")
    binding.load_library()
    w = inputs.baseline_config(args.config)
    rows = []
    for label, variant, options in candidates(w.dims, w.dtype == np.float32):
        try:
            mean, dev = score(binding, torch, w, variant, options, args.riemann, args.steps, args.repeats)
            rows.append({"candidate": label, "variant": variant, "options": options, "gcell_per_s": mean, "stdev": dev})
        except Exception as ex:  # shape not covered by the kernel, out of memory for the Manifest arrays, ...
            rows.append({"candidate": label, "variant": variant, "options": options, "skipped": str(ex)[:100]})
        torch.cuda.empty_cache()
    ok = sorted((r for r in rows if "gcell_per_s" in r), key=lambda r: -r["gcell_per_s"])
    print(f"# config {args.config}: {w.name}, riemann {args.riemann}, {args.repeats} x {args.steps} steps per candidate")
    print(f"# {'candidate':42s} {'Gcell/s':>9s} {'+-':>7s}")
    for r in ok:
        print(f"  {r['candidate']:42s} {r['gcell_per_s']:9.3f} {r['stdev']:7.3f}")
    for r in rows:
        if "skipped" in r:
            print(f"  {r['candidate']:42s}   skipped: {r['skipped']}")
    if args.json:
        json.dump({"config": args.config, "workload": w.name, "rows": rows}, open(args.json, "w"), indent=1)
    return 0


if __name__ == "__main__":
    sys.exit(main())
