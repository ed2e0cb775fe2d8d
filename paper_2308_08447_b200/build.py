"""Build the CUDA library in-tree: nvcc -> paper_2308_08447_b200/libdemag_b200.so (sm_100a only).

The sources are compiled as separate translation units in parallel (plan.cu: C ABI, generic kernel family, tensor
builder; v2_{x,y,z}_{f,d}.cu: the fast-path launchers of one stage and precision each) and linked into one library."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
UNITS = ["plan", "llg"] + [f"v2_{s}_{t}" for s in ("x", "y", "z", "xe") for t in "fd"]
LIB = os.path.join(HERE, "libdemag_b200.so")

ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
NVCC_FLAGS = ARCH + ["-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC"]


def _deps():
    hdrs = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith(".cuh")]
    return hdrs + [os.path.join(os.path.dirname(HERE), "include", "demag.h")]


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)
    newest_hdr = max(os.path.getmtime(d) for d in _deps())
    jobs = []
    for u in UNITS:
        src, obj = os.path.join(CSRC, u + ".cu"), os.path.join(OBJ, u + ".o")
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(newest_hdr, os.path.getmtime(src)):
            jobs.append([nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src])

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        return cmd, r

    if jobs:
        with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 1)) as ex:
            for cmd, r in ex.map(run, jobs):
                if verbose or r.returncode != 0:
                    sys.stderr.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
                if r.returncode != 0:
                    raise RuntimeError("nvcc failed building " + cmd[-1])
    objs = [os.path.join(OBJ, u + ".o") for u in UNITS]
    if jobs or not os.path.exists(LIB):
        r = subprocess.run([nvcc] + ARCH + ["-shared", "-o", LIB] + objs, capture_output=True, text=True)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("nvcc failed linking libdemag_b200.so")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
