"""Build libra_mppi.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2209_12842_b200.build [--force] [--checked]

--checked builds libra_mppi_checked.so, the same sources with -DRA_CHECKED: every kernel asserts its own indices
(compute-sanitizer is closed on the GPU pool); tests/test_gpu_checked_build.py runs parity cases through it.

The rollout kernel is instantiated per (dynamics, risk) pair in separate translation units
so they compile in parallel.  No torch headers are involved: the library is plain CUDA.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libra_mppi.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
              "--extended-lambda", "-Xcompiler", "-fPIC", f"-I{INCLUDE}", f"-I{CSRC}"]


def _sources():
    return [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC))] + [os.path.join(INCLUDE, "ra_mppi.h")]


LIB_CHECKED = os.path.join(HERE, "libra_mppi_checked.so")


def source_hash(jobs) -> str:
    """sha256 over every source and header of the library, the compiler flags and the per-object defines."""
    import hashlib
    h = hashlib.sha256()
    for path in _sources():
        with open(path, "rb") as f:
            h.update(os.path.basename(path).encode() + b"\0" + f.read() + b"\0")
    h.update(repr((NVCC_FLAGS[:-2], [(os.path.basename(s), os.path.basename(o), d) for s, o, d in jobs])).encode())
    return h.hexdigest()


def _jobs(obj_dir, defs0):
    jobs = [(os.path.join(CSRC, "ra_mppi.cu"), os.path.join(obj_dir, "ra_mppi.o"), list(defs0)),
            (os.path.join(CSRC, "pipe_peaks.cu"), os.path.join(obj_dir, "pipe_peaks.o"), list(defs0))]
    for d in (0, 1):
        for r in (0, 1, 2, 3):
            jobs.append((os.path.join(CSRC, "rollout_inst.cu"), os.path.join(obj_dir, f"rollout_{d}_{r}.o"),
                         list(defs0) + [f"-DRA_INST_DYN={d}", f"-DRA_INST_RISK={r}"]))
    return jobs


def build(force: bool = False, verbose: bool = False, checked: bool = False) -> str:
    lib = LIB_CHECKED if checked else LIB
    obj_dir = OBJ + "_checked" if checked else OBJ
    jobs = _jobs(obj_dir, ["-DRA_CHECKED"] if checked else [])
    # up to date = the stamp written beside the library by the build that produced it names these very sources and flags
    # (a content hash, not mtimes: a snapshot copied to the GPU box keeps the prebuilt library only if it is of this source)
    stamp, want = lib + ".sha256", source_hash(jobs)
    if not force and os.path.exists(lib) and os.path.exists(stamp) and open(stamp).read().strip() == want:
        return lib
    if os.path.exists(stamp):
        os.remove(stamp)
    os.makedirs(obj_dir, exist_ok=True)
    extra = ["-Xptxas", "-v"] if verbose else []

    def compile_one(job):
        src, obj, defs = job
        cmd = ["nvcc", *NVCC_FLAGS, *extra, *defs, "-c", src, "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed: {' '.join(cmd)}\n{r.stdout}\n{r.stderr}")
        return r.stderr

    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        logs = list(ex.map(compile_one, jobs))
    if verbose:
        with open(os.path.join(obj_dir, "ptxas.log"), "w") as f:
            f.write("\n".join(logs))
    objs = [j[1] for j in jobs]
    cmd = ["nvcc", "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", lib, *objs, "-lcudart"]
    subprocess.run(cmd, check=True)
    with open(stamp, "w") as f:
        f.write(want + "\n")
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, checked="--checked" in sys.argv))
