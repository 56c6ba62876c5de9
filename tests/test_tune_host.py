"""Host logic of the variant sweep (paper_1204_4779_b200/tune.py): the candidate space it enumerates."""

from paper_1204_4779_b200 import binding, tune



def test_candidate_space():
    for dims in (1, 2, 3):
        for f32 in (True, False):
            c = tune.candidates(dims, f32)
            labels = [l for l, _, _ in c]
            assert len(labels) == len(set(labels)) and len(c) >= 3
            for _, variant, options in c:
                assert variant in binding.VARIANT
                assert all(isinstance(v, int) and v >= 0 for v in options.values())
                assert set(options) <= {"block_x", "block_y", "block_z", "tile_depth", "cells_per_thread", "staging", "arith"}
            packed = [o for _, _, o in c if o.get("cells_per_thread") == 2]
            assert bool(packed) == (f32 and dims > 1)  # packed f32x2 exists for fp32 only
            assert all(v in ("manifest_all", "manifest_flux", "delayed") for _, v, _ in c) == (dims == 1)


# ------------------------------------------------------------------ the paper's annealing tuner (§3.2-3.3)
def test_triangulation_is_the_papers_table_4():
    """PAPER.md:658-664 (Table 4), bit by bit: Base / Secondary / Primary -> Child."""
    base, sec, pri = (0, 0, 0, 0, 1, 1, 1, 1), (0, 0, 1, 1, 0, 0, 1, 1), (0, 1, 0, 1, 0, 1, 0, 1)
    assert tune.triangulate(base, sec, pri) == (0, 1, 1, 1, 0, 0, 0, 1)
    # two independent improvements found by different parents are combined (what triangulation is for)
    assert tune.triangulate(("a", 0, 0), ("a", 5, 0), ("a", 0, 7)) == ("a", 5, 7)


def test_draw_follows_eq_12():
    """Eq. 12 as DESIGN.md R25 reads it: low temperatures prefer the best individual strictly, high temperatures hardly
    care, a difference small against sigma_top + sigma is ignored."""
    w = tune.draw_weight
    assert w(10.0, 0.0, 10.0, 0.0, 0.1) == 1.0                               # the top individual itself
    assert w(9.0, 0.0, 10.0, 0.0, 0.01) < 1e-40                              # T -> 0: only the best survives
    assert w(9.0, 0.0, 10.0, 0.0, 1e6) > 0.999                               # T -> inf: the score does not matter
    assert w(9.9, 0.5, 10.0, 0.5, 1e-9) > 0.9                                # 0.1 apart with sigma 0.5 each: ignored
    assert w(5.0, 0.0, 10.0, 0.0, 1.0) < w(8.0, 0.0, 10.0, 0.0, 1.0) < 1.0   # monotone in the score
    t = tune.AnnealingTuner({"a": (0, 1, 2, 3)}, lambda g: (float(g[0]), 0.1), seed=1, genes=("a",))
    for v in range(4):
        t.measure((v,))
    counts = {v: 0 for v in range(4)}
    for _ in range(4000):
        counts[t.draw(0.05)[0]] += 1
    assert counts[3] > 3500 and counts[0] < 20                               # cold draws: the champion
    for _ in range(200):
        T = t.temperature()
        assert 0.1 * (1 - 1e-9) <= T <= 3.0 * (1 + 1e-9)                     # log-uniform in [sigma_top, mu_top]


def test_annealing_tuner_finds_combined_improvements():
    """A separable landscape with two independent improvements and a trap: the tuner never re-measures a genome, keeps
    every individual, and reaches the optimum well before the space (6 x 8 x 9 x 3 x 5 x 2 x 3 = 38880) is enumerated."""
    space = tune.gene_space(3, True)
    genes = tune.GENES

    def fitness(g):
        d = dict(zip(genes, g))
        if d["variant"] in ("manifest_all",) and d["block_x"]:
            return 0.0, 0.0                                                  # "shape not covered": a failed individual
        s = {"pack": 10.0, "march": 9.0, "fused1": 8.0, "manifest_flux": 4.0, "manifest_all": 3.0, "delayed": 3.5}[d["variant"]]
        s += {14: 1.0, 7: 0.4}.get(d["block_y"], 0.0)                        # improvement 1
        s += {128: 0.5, 64: 0.3}.get(d["tile_depth"], 0.0)                   # improvement 2
        s -= 0.2 * (d["staging"] != 0) + 0.3 * (d["cells_per_thread"] != 0)
        return s, 0.05

    zero = (0,) * (len(genes) - 1)
    best_possible = 10.0 + 1.0 + 0.5
    found = []
    for seed in range(5):
        t = tune.AnnealingTuner(space, fitness, seed=seed)
        best, (mu, sig) = t.run([("delayed",) + zero, ("manifest_flux",) + zero], 250)
        assert len(t.db) == 250 and len({g for _, g in t.births}) == 250    # nothing measured twice, nothing forgotten
        assert {m for m, _ in t.births} >= {"seed", "mutation", "crossover", "triangulation"}
        found.append(mu)
    assert sum(1 for m in found if m >= best_possible - 1e-9) >= 4, found    # the optimum in at least 4 of 5 runs
    assert min(found) >= 11.0, found


def test_genome_options_round_trip():
    v, o = tune.genome_options(("pack", 0, 14, 0, 64, 0, 0))
    assert v == "pack" and o == {"block_y": 14, "tile_depth": 64}
    for dims in (1, 2, 3):
        for f32 in (True, False):
            sp = tune.gene_space(dims, f32)
            assert set(sp) == set(tune.GENES) and all(len(v) >= 1 for v in sp.values())
            assert all(v in binding.VARIANT for v in sp["variant"])
