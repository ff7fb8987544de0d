"""Build libsail_b200.so (the C-ABI product library) in-tree with nvcc for sm_100a.

    python -m paper_1609_07936_b200.build [--force] [--verbose] [--define NAME=VALUE ...]

`--define` passes -DNAME=VALUE to nvcc for every source (diagnostic builds, e.g. SAIL_DIAG_EXTRA_DFMA in csrc/sweep.cu);
it always recompiles, and a later plain build restores the product library (the defines are recorded in build/defines.txt).

Cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with the snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libsail_b200.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
SOURCES = ["sail_api.cu", "sweep.cu", "forward.cu", "branch.cu", "smooth.cu", "selfcool.cu", "microbench.cu"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden", "--expt-relaxed-constexpr"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, defines=None) -> str:
    """defines = None: keep the -D flags of the library that is there (bench.py on a diagnostic build);
    defines = () : the product library; defines = ["NAME=VALUE", ...]: a diagnostic build."""
    os.makedirs(OBJ, exist_ok=True)
    # a library built with other -D flags than the ones asked for now is stale, whatever the time stamps say
    stamp = os.path.join(OBJ, "defines.txt")
    have = open(stamp).read() if os.path.exists(stamp) else ""
    if defines is None:
        defines = have.split()
    want = " ".join(sorted(defines))
    if want != have:
        force = True
    with open(stamp, "w") as f:
        f.write(want)
    headers = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    headers.append(os.path.join(INCLUDE, "sail.h"))
    nvcc = _nvcc()
    jobs = []
    objs = []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(OBJ, src.replace(".cu", ".o"))
        objs.append(o)
        if force or _stale(o, [s] + headers):
            cmd = [nvcc] + NVCC_FLAGS + ["-D" + d for d in defines] + (["-Xptxas", "-v"] if verbose else []) + ["-I", INCLUDE, "-c", s, "-o", o]
            jobs.append(cmd)

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode:
            sys.stderr.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        if r.returncode:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))

    with ThreadPoolExecutor(max_workers=4) as ex:
        list(ex.map(run, jobs))
    if force or jobs or _stale(LIB, objs):
        run([nvcc, "-shared", "-o", LIB] + objs + ["-lcudart"])
    return LIB


if __name__ == "__main__":
    defs = [sys.argv[i + 1] for i, a in enumerate(sys.argv[:-1]) if a == "--define"]
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, defines=defs))
