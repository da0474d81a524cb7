"""Build the C-ABI CUDA library in-tree: paper_1602_07247_b200/libants_recon.so.

nvcc cross-compiles for sm_100a without a GPU; cudart is linked statically so the
library loads (and its symbols can be listed) on a CPU-only box.  Every csrc/*.cu is
one translation unit (the kernel families are instantiated in k_*.cu, one per method);
they are compiled in parallel into build/*.o and linked into one shared object.
"""
from __future__ import annotations

import concurrent.futures
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
OBJ_DIR = os.path.join(_HERE, "build")
LIB = os.path.join(_HERE, "libants_recon.so")

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC"]


def nvcc() -> str:
    cand = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", "nvcc")
    return cand if os.path.exists(cand) else "nvcc"


def _sources():
    names = sorted(os.listdir(CSRC))
    units = [os.path.join(CSRC, f) for f in names if f.endswith(".cu")]
    headers = [os.path.join(CSRC, f) for f in names if not f.endswith(".cu")]
    headers.append(os.path.join(os.path.dirname(_HERE), "include", "ants_recon.h"))
    return units, headers


def _compile(src: str, obj: str, verbose: bool) -> str:
    cmd = [nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src]
    res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed on %s:\n%s" % (os.path.basename(src), res.stdout))
    return res.stdout


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile what is missing or older than its sources; returns the library's path."""
    units, headers = _sources()
    os.makedirs(OBJ_DIR, exist_ok=True)
    newest_header = max(os.path.getmtime(h) for h in headers if os.path.exists(h))
    jobs = []
    for src in units:
        obj = os.path.join(OBJ_DIR, os.path.basename(src)[:-3] + ".o")
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(src), newest_header):
            jobs.append((src, obj))
    objs = [os.path.join(OBJ_DIR, os.path.basename(s)[:-3] + ".o") for s in units]
    if jobs:
        with concurrent.futures.ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as pool:
            for out in pool.map(lambda j: _compile(j[0], j[1], verbose), jobs):
                if verbose and out:
                    print(out)
    if jobs or not os.path.exists(LIB) or any(os.path.getmtime(o) > os.path.getmtime(LIB) for o in objs):
        subprocess.check_call([nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
