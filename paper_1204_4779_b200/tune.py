"""The paper's Manifest / Delayed search, rebuilt as a measured sweep over this library's variant space.

    python -m paper_1204_4779_b200.tune --config 4 [--repeats 5] [--steps 5] [--riemann hllc] [--json out.json]
    python -m paper_1204_4779_b200.tune --config 4 --stochastic 60 [--seed 0]     (the paper's annealing tuner)

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


# ------------------------------------------------------------------------------------------------------------------
# The paper's tuner itself (§3.2-3.3, :612-676): "parallel asynchronous genetic simulated
# annealing".  A database keeps every individual ever measured with the mean mu and sample deviation sigma of its
# repeated benchmark; new individuals are born from parents DRAWN from the database at a random temperature by
# mutation, crossover or triangulation (equal odds).  Host logic only; the fitness function is passed in, so the
# same code runs against a GPU benchmark (main(), --stochastic) or a synthetic landscape (tests/test_tune_host.py).
# One GPU = one worker: the master / worker asynchrony of Fig. 8 has nothing to overlap here and is not rebuilt.
GENES = ("variant", "block_x", "block_y", "block_z", "tile_depth", "cells_per_thread", "staging")


def gene_space(dims, dtype_is_f32):
    """Allowed values per gene (every launch shape some kernel accepts; combinations no kernel covers are
    legal genomes that score 0, like the paper's individuals that fail their test)."""
    space = {
        "variant": ("pack", "march", "fused1", "manifest_flux", "manifest_all", "delayed"),
        "block_x": (0, 1, 2, 4, 7, 8, 64, 128) if dims == 2 else (0, 32, 64),
        "block_y": (0,) if dims == 2 else (0, 4, 5, 7, 8, 11, 14, 15, 16),
        "block_z": (0, 1, 2),
        "tile_depth": (0, 16, 32, 64, 128),
        "cells_per_thread": (0, 2) if dtype_is_f32 else (0,),
        "staging": (0, 2, 3),
    }
    if dims == 1:
        space = {k: ((v if k == "variant" else (0,))) for k, v in space.items()}
    return space


def draw_weight(mu, sigma, mu_top, sigma_top, T):
    """Eq. 12 as DESIGN.md R25 reads it: exp(-(mu_top - mu) / (T + sigma_top + sigma)).  Low temperatures
    strictly prefer high scores, high temperatures hardly care, and a difference small against sigma_top + sigma is
    ignored (the extracted formula lacks the minus sign, which would prefer the WORST individual)."""
    import math

    return math.exp(-(mu_top - mu) / (T + sigma_top + sigma))


def triangulate(base, secondary, primary):
    """Three-parent crossover (Table 4), parents in ascending order of score: for every gene, a change
    of Primary against Base is adopted; else a change of Secondary against Base; else Base's value."""
    return tuple(p if p != b else (s if s != b else b) for b, s, p in zip(base, secondary, primary))


class AnnealingTuner:
    """The database and the birth rules.  `fitness(genome) -> (mu, sigma)`; a failed individual scores (0, 0)."""

    def __init__(self, space, fitness, seed=0, genes=GENES):
        import random

        self.genes = tuple(genes)
        self.space = {g: tuple(space[g]) for g in self.genes}
        self.fitness = fitness
        self.rng = random.Random(seed)
        self.db = {}       # genome -> (mu, sigma)
        self.births = []   # (method, genome) in order of creation

    # -- database
    def measure(self, genome, method="seed"):
        if genome not in self.db:
            self.db[genome] = tuple(float(v) for v in self.fitness(genome))
            self.births.append((method, genome))
        return self.db[genome]

    def top(self):
        return max(self.db.items(), key=lambda kv: kv[1][0])

    def temperature(self):
        """log T uniform between log sigma(I_top) and log mu(I_top)."""
        import math

        (_, (mu_top, sig_top)) = self.top()
        lo = max(sig_top, 1e-6 * max(mu_top, 1e-30), 1e-300)
        hi = max(mu_top, lo)
        return math.exp(self.rng.uniform(math.log(lo), math.log(hi)))

    def draw(self, T):
        (_, (mu_top, sig_top)) = self.top()
        items = list(self.db.items())
        weights = [draw_weight(mu, sig, mu_top, sig_top, T) for _, (mu, sig) in items]
        return self.rng.choices(items, weights=weights, k=1)[0][0]

    # -- birth (§3.3)
    def mutate(self, genome):
        g = list(genome)
        for i in self.rng.sample(range(len(g)), self.rng.randint(1, 2)):  # overwrite one or two genes at random
            g[i] = self.rng.choice(self.space[self.genes[i]])
        return tuple(g)

    def crossover(self, a, b):
        cuts = sorted(self.rng.sample(range(1, len(a)), self.rng.randint(1, min(3, len(a) - 1))))
        out, take_a, last = [], True, 0
        for c in cuts + [len(a)]:
            out.extend((a if take_a else b)[last:c])
            take_a, last = not take_a, c
        return tuple(out)

    def birth(self):
        """One new individual not yet in the database.  Returns (method, genome)."""
        T = self.temperature()
        method = self.rng.choice(("mutation", "crossover", "triangulation"))
        need = {"mutation": 1, "crossover": 2, "triangulation": 3}[method]
        child = None
        if len(self.db) >= need:
            for _ in range(20):  # "if two of the parents are the same the master retries the draws"
                parents = [self.draw(T) for _ in range(need)]
                if len(set(parents)) == need:
                    break
            else:
                parents = None
            if parents:
                if method == "mutation":
                    child = self.mutate(parents[0])
                elif method == "crossover":
                    child = self.crossover(*parents)
                else:
                    child = triangulate(*sorted(parents, key=lambda p: self.db[p][0]))
        # "if the genome ... is already in the DB, the master discards the individual and retries the mutation ...
        #  with each retry, draw temperature T is multiplied by 1.2"
        tries = 0
        while child is None or child in self.db:
            child = self.mutate(self.draw(T))
            method = "mutation"
            T *= 1.2
            tries += 1
            if tries > 10000:
                raise RuntimeError("gene space exhausted")
        return method, child

    def run(self, seeds, budget):
        for g in seeds:
            self.measure(g)
        while len(self.db) < budget:
            method, g = self.birth()
            self.measure(g, method)
        return self.top()


def genome_options(genome, genes=GENES):
    """(variant, options) of a genome for ParaisoHydro."""
    d = dict(zip(genes, genome))
    variant = d.pop("variant")
    return variant, {k: v for k, v in d.items() if v}


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
    ap.add_argument("--stochastic", type=int, default=0,
                    help="run the paper's annealing tuner (PAPER.md §3.2-3.3) for this many individuals instead of the sweep")
    ap.add_argument("--seed", type=int, default=0)
    args = ap.parse_args()

    import numpy as np
    import torch

    from . import binding, inputs

    if not torch.cuda.is_available():
        raise SystemExit("tune needs a CUDA device: the product path has no CPU fallback")
    binding.load_library()
    w = inputs.baseline_config(args.config)
    if args.stochastic:
        return stochastic_main(args, binding, torch, w)
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


def stochastic_main(args, binding, torch, w):
    """The annealing tuner on one GPU: seeds = the three off-chip ends + the default; every individual is benchmarked
    `--repeats` times (mean, deviation); a genome no kernel covers, or a run that ends non-finite, scores 0."""
    import numpy as np

    def fitness(genome):
        variant, options = genome_options(genome)
        try:
            return score(binding, torch, w, variant, options, args.riemann, args.steps, args.repeats)
        except Exception:
            return 0.0, 0.0
        finally:
            torch.cuda.empty_cache()

    space = gene_space(w.dims, w.dtype == np.float32)
    tuner = AnnealingTuner(space, fitness, seed=args.seed)
    zero = tuple(0 for _ in GENES[1:])
    seeds = [(v,) + zero for v in ("delayed", "manifest_flux", "pack" if w.dims > 1 else "delayed")]
    best, (mu, sig) = tuner.run(list(dict.fromkeys(seeds)), args.stochastic)
    print(f"# config {args.config}: {w.name}, annealing tuner (PAPER.md 3.2-3.3), {len(tuner.db)} individuals, "
          f"{args.repeats} x {args.steps} steps each, seed {args.seed}")
    print(f"# {'#':>3s} {'born by':14s} {'Gcell/s':>9s} {'+-':>7s}  genome {GENES}")
    best_so_far = 0.0
    for i, (method, g) in enumerate(tuner.births):
        m, s_ = tuner.db[g]
        best_so_far = max(best_so_far, m)
        print(f"  {i:3d} {method:14s} {m:9.3f} {s_:7.3f}  {g}{'   <- best so far' if m == best_so_far and m > 0 else ''}")
    print(f"# champion: {best}  {mu:.3f} +- {sig:.3f} Gcell/s; failed (score 0): "
          f"{sum(1 for v in tuner.db.values() if v[0] == 0.0)} of {len(tuner.db)}")
    if args.json:
        json.dump({"config": args.config, "workload": w.name, "births": [(m, g, tuner.db[g]) for m, g in tuner.births]},
                  open(args.json, "w"), indent=1)
    return 0


if __name__ == "__main__":
    sys.exit(main())
