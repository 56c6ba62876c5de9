"""Compile the C-ABI library libparaiso_hydro.so (csrc/*.cu) and the probe library libparaiso_hydro_probe.so
(csrc/probe/*.cu: test and measurement probes, include/paraiso_hydro_probe.h) for sm_100a, in-tree (next to this file).

    python -m paper_1204_4779_b200.build [--force] [--verbose] [--keep]

Flags that are part of the arithmetic specification: -fmad=false (no implicit FMA
contraction; the kernels write fma explicitly), default -prec-div=true -prec-sqrt=true -ftz=false.
"""
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "libparaiso_hydro.so")
PROBE_OUT = os.path.join(HERE, "libparaiso_hydro_probe.so")
NVCC = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"

FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-fmad=false", "-prec-div=true", "-prec-sqrt=true", "-ftz=false",
    "--shared", "-Xcompiler", "-fPIC",
    "-cudart", "static",
]


def sources():
    return [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith(".cu")]


def probe_sources():
    d = os.path.join(CSRC, "probe")
    return [os.path.join(d, f) for f in sorted(os.listdir(d)) if f.endswith(".cu")]


def _stale():
    if not (os.path.exists(OUT) and os.path.exists(PROBE_OUT)):
        return True
    t = min(os.path.getmtime(OUT), os.path.getmtime(PROBE_OUT))
    inc = os.path.join(HERE, "..", "include")
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if not os.path.isdir(os.path.join(CSRC, f))] + probe_sources()
    deps += [os.path.join(inc, f) for f in os.listdir(inc)] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False, extra=()):
    """One `nvcc -c` per translation unit, run concurrently, then one link step."""
    if not (force or _stale()):
        return OUT
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    compile_flags = [f for f in FLAGS if f not in ("--shared", "-cudart", "static")]
    procs = []
    probe_objs = []
    for src in sources() + probe_sources():
        obj = os.path.join(objdir, os.path.basename(src)[:-3] + ".o")
        if src in probe_sources():
            probe_objs.append(obj)
        cmd = [NVCC] + compile_flags + list(extra) + ["-c", src, "-o", obj]
        if verbose:
            print(" ".join(cmd), flush=True)
        procs.append((cmd, obj, subprocess.Popen(cmd)))
    objs = []
    for cmd, obj, p in procs:
        if p.wait() != 0:
            raise subprocess.CalledProcessError(p.returncode, cmd)
        if obj not in probe_objs:
            objs.append(obj)
    for group, out in ((objs, OUT), (probe_objs, PROBE_OUT)):
        link = [NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "--shared", "-cudart", "static"] + group + ["-o", out]
        if verbose:
            print(" ".join(link), flush=True)
        subprocess.run(link, check=True)
    return OUT


if __name__ == "__main__":
    extra = ["-Xptxas", "-v"] if "--ptxas" in sys.argv else []
    print(build(force="--force" in sys.argv, verbose=True, extra=extra))
