"""Compile the oracle (test infrastructure) into two shared objects next to its source:

  liboracle_serial.so  single-threaded: the oracle "as it stands" (timed as the CPU baseline on 1 core)
  liboracle_omp.so     the same source with OpenMP over independent cells / grid lines; results are
                       bit-identical (cells are independent, max is order-free) — used where a test
                       needs a long oracle run.

Flags are part of the arithmetic specification: -ffp-contract=off forbids implicit
contraction, -mfma makes the explicit std::fma a hardware instruction.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "euler_oracle.cpp")
WAVE_SRC = os.path.join(HERE, "wave_oracle.cpp")  # the paper's linear-wave example (§2.3), a library of its own
BASE = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-mfma", "-shared", "-fPIC", "-Wall", "-Wno-unknown-pragmas"]


def _stale(out, src=SRC):
    return not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src)


def build(force=False, verbose=False):
    outs = {}
    for name, extra in (("serial", []), ("omp", ["-fopenmp"])):
        out = os.path.join(HERE, f"liboracle_{name}.so")
        if force or _stale(out):
            cmd = BASE + extra + [SRC, "-o", out]
            if verbose:
                print(" ".join(cmd))
            subprocess.run(cmd, check=True)
        outs[name] = out
    out = os.path.join(HERE, "liboracle_wave.so")
    if force or _stale(out, WAVE_SRC):
        cmd = BASE + [WAVE_SRC, "-o", out]
        if verbose:
            print(" ".join(cmd))
        subprocess.run(cmd, check=True)
    outs["wave"] = out
    return outs


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
