"""Build step: nvcc-compile csrc/*.cu for sm_100a into libculgt_b200.so next to this file.

    python -m paper_1412_3655_b200.build [--force] [--verbose] [--measure]

The library is built IN-TREE (it is git-ignored but travels with the source snapshot to the
GPU box).  nvcc cross-compiles without a GPU.  Every translation unit is compiled to its own
object (in parallel, rebuilt only when it or a header changed) and the objects are linked into
the shared library.

--measure (or CULGT_MEASURE=1 in the environment) builds a SECOND library,
libculgt_b200_measure.so, with -DCULGT_MEASURE: the measurement-only kernel instantiations
(all-fp32 arithmetic, G = 1, no-solve, the rejected thread-to-site mappings and slab schedules of
DESIGN.md 6.1) are compiled into it and selectable through culgt_set_sweep_variant.  The product
library never contains them; the binding loads the measure library only when CULGT_MEASURE=1.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libculgt_b200.so")
LIB_MEASURE = os.path.join(HERE, "libculgt_b200_measure.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC",
]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _headers():
    return glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) + \
        glob.glob(os.path.join(INCLUDE, "*.h")) + [os.path.abspath(__file__)]


def _measure_flag(measure):
    if measure is None:
        measure = os.environ.get("CULGT_MEASURE", "") not in ("", "0")
    return bool(measure)


def build(force: bool = False, verbose: bool = False, measure=None) -> str:
    measure = _measure_flag(measure)
    lib = LIB_MEASURE if measure else LIB
    obj_dir = os.path.join(HERE, "build", "measure" if measure else "product")
    os.makedirs(obj_dir, exist_ok=True)
    nvcc = os.environ.get("NVCC", "nvcc")
    flags = NVCC_FLAGS + (["-DCULGT_MEASURE"] if measure else []) + (["-Xptxas", "-v"] if verbose else [])
    hdr_time = max(os.path.getmtime(p) for p in _headers())
    jobs = []
    objs = []
    for src in sources():
        obj = os.path.join(obj_dir, os.path.basename(src)[:-3] + ".o")
        objs.append(obj)
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(src), hdr_time):
            jobs.append([nvcc] + flags + ["-c", "-o", obj, src])

    def run(cmd):
        return cmd, subprocess.run(cmd, capture_output=True, text=True)

    if jobs:
        with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 1)) as ex:
            for cmd, res in ex.map(run, jobs):
                if verbose or res.returncode != 0:
                    sys.stderr.write(res.stdout + res.stderr)
                if res.returncode != 0:
                    raise RuntimeError("nvcc failed: " + " ".join(cmd))
    if jobs or not os.path.exists(lib):
        cmd = [nvcc, "-shared", "-o", lib] + objs + ["-ldl"]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
            raise RuntimeError("link failed: " + " ".join(cmd))
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv,
                measure=True if "--measure" in sys.argv else None))
