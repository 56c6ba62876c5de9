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
