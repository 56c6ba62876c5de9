"""Mechanical operation count of one Euler step: the oracle's Solver instantiated with a counting
scalar type (oracle/count_ops.cpp) on the BASELINE recipes at reduced size.  TEST / MEASUREMENT INFRASTRUCTURE: calls
only oracle/ and the seeded input generators; the CUDA path is not involved.  It sits in tests/ because, like the
tests, it brings the oracle and the shared input generators together (oracle/ itself imports nothing of the package).

    python tests/count_ops.py            # prints the table, writes profiles/r3_counted_ops.json and .md

Per config and Riemann solver it reports operations per cell per RK2 step (both stages + the CFL term) by class, for
the state as generated and for the state 20 oracle steps later (the branch mix - supersonic faces, limiter cases -
depends on the data), in two arrangements:
  as_written  cfl_S() + step() run whole: every cell is interpolated twice per axis (once for each of its faces'
              calls) and both sides' U_K, F_K are formed before the upwind test - DESIGN.md §4 as the oracle states it;
  composed    the same member functions, one prim_of per cell and stage, ONE interpolate per cell and axis, one riemann
              per face, the Eq. 23 update - what a kernel that keeps its intermediates has to execute (both sides still
              formed in riemann; the kernels' further saving, choosing the upwind side first in HLLC, is not something
              the oracle's text does and stays a hand count: bench.py's COUNTED_OPS_PER_CELL_STEP).
`slots` weighs a division / square root with the fma sequence the kernels run for it (fp32: 6 / 5, fp64: 8 / 10,
DESIGN.md §8); a negation is an operand modifier (0).  Selects are invisible to the scalar type (they are branches on
the CPU): the hand table counts them, this one cannot.
"""
import ctypes
import json
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HERE = os.path.join(ROOT, "oracle")  # the counting translation unit and its library live beside the oracle
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
SRC = os.path.join(HERE, "count_ops.cpp")
OUT = os.path.join(HERE, "liboracle_count.so")
CLASSES = ["add", "mul", "fma", "div", "sqrt", "cmp", "minmax", "abs", "neg", "copysign"]


def build(force=False):
    deps = [SRC, os.path.join(HERE, "euler_oracle.cpp")]
    if force or not os.path.exists(OUT) or any(os.path.getmtime(d) > os.path.getmtime(OUT) for d in deps):
        # no -fopenmp: the tallies are plain globals; same arithmetic flags as the oracle itself
        subprocess.run(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-mfma", "-shared", "-fPIC", "-Wall",
                        "-Wno-unknown-pragmas", SRC, "-o", OUT], check=True)
    return OUT


def slots(counts, itemsize):
    w = dict.fromkeys(CLASSES, 1)
    w.update(div=6 if itemsize == 4 else 8, sqrt=5 if itemsize == 4 else 10, neg=0)
    return sum(w[k] * counts[k] for k in CLASSES)


def count(w, riemann, U=None):
    L = ctypes.CDLL(build())
    i64, dbl = ctypes.c_int64, ctypes.c_double
    L.oracle_count_ops.argtypes = [ctypes.c_int, ctypes.POINTER(i64), ctypes.POINTER(dbl), dbl, ctypes.c_int, ctypes.c_int,
                                   ctypes.c_int, ctypes.c_void_p, dbl, ctypes.POINTER(ctypes.c_uint64)]
    U = np.ascontiguousarray(w.U if U is None else U)
    out = (ctypes.c_uint64 * 20)()
    L.oracle_count_ops(w.dims, (i64 * w.dims)(*w.n), (dbl * w.dims)(*w.extent), w.gamma, 0 if w.dtype == np.float32 else 1,
                       {"periodic": 0, "outflow": 1}[w.boundary], {"hllc": 0, "hll": 1}[riemann], U.ctypes.data, w.cfl, out)
    res = {}
    for j, name in enumerate(("as_written", "composed")):
        per_cell = {k: out[10 * j + i] / w.cells for i, k in enumerate(CLASSES)}
        res[name] = {"per_cell_step": {k: round(v, 3) for k, v in per_cell.items()},
                     "operations": round(sum(v for k, v in per_cell.items() if k != "neg"), 2),
                     "slots": round(slots(per_cell, w.dtype.itemsize), 2)}
    return res


def main():
    import oracle
    from paper_1204_4779_b200 import inputs  # seeded initial conditions only: serves both sides, holds no arithmetic

    cases = [(0, inputs.sod(256)), (1, inputs.kelvin_helmholtz(128, dtype=np.float32, seed=0)),
             (2, inputs.kelvin_helmholtz(128, dtype=np.float64, seed=1)), (3, inputs.blast(40, np.float32, seed=2)),
             (4, inputs.blast(48, np.float32, seed=3))]
    table = []
    for cfg, w in cases:
        for riemann in ("hllc", "hll"):
            o = oracle.Oracle(w.n, w.extent, w.gamma, w.dtype, w.boundary, riemann, "omp")
            o.set_state(w.U)
            for _ in range(20):
                o.step(o.cfl_dt(w.cfl))
            later = o.get_state()
            o.close()
            row = {"config": cfg, "workload": w.name, "dims": w.dims, "itemsize": w.dtype.itemsize, "riemann": riemann,
                   "initial_state": count(w, riemann), "after_20_steps": count(w, riemann, later)}
            table.append(row)
            a, c = row["after_20_steps"]["as_written"], row["after_20_steps"]["composed"]
            print(f"cfg {cfg} {w.name:34s} {riemann:4s}  as written {a['operations']:8.1f} ops {a['slots']:8.1f} slots | "
                  f"composed {c['operations']:8.1f} ops {c['slots']:8.1f} slots   (t=0: {row['initial_state']['composed']['slots']:.1f})")
    doc = {"command": "python tests/count_ops.py", "classes": CLASSES,
           "slot_weights": "fp32: div 6, sqrt 5; fp64: div 8, sqrt 10; neg 0; everything else 1 (DESIGN.md §8)", "rows": table}
    os.makedirs(os.path.join(ROOT, "profiles"), exist_ok=True)
    with open(os.path.join(ROOT, "profiles", "r3_counted_ops.json"), "w") as f:
        json.dump(doc, f, indent=1)
    with open(os.path.join(ROOT, "profiles", "r3_counted_ops.md"), "w") as f:
        f.write("# Counted arithmetic per cell per RK2 step, from the oracle instantiated with a counting scalar\n\n"
                "Command: `python tests/count_ops.py` (oracle/count_ops.cpp + tests/count_ops.py; calls only oracle/ and "
                "the seeded input generators).  State 20 oracle steps after the recipe's initial condition, reduced grids.\n"
                "`slots` = operations with a division / square root weighted by the kernels' fma sequence "
                "(fp32 6 / 5, fp64 8 / 10); selects are not visible to a scalar type.\n\n"
                "| cfg | workload | solver | as written: ops | slots | composed (one interpolation per cell and axis): ops | slots | div | sqrt |\n"
                "|---|---|---|---|---|---|---|---|---|\n")
        for r in table:
            a, c = r["after_20_steps"]["as_written"], r["after_20_steps"]["composed"]
            f.write(f"| {r['config']} | {r['workload']} | {r['riemann']} | {a['operations']} | {a['slots']} | {c['operations']} | "
                    f"{c['slots']} | {c['per_cell_step']['div']} | {c['per_cell_step']['sqrt']} |\n")
    return 0


if __name__ == "__main__":
    sys.exit(main())
