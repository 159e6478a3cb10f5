"""Build the CUDA library in-tree: paper_2602_13198_b200/libgpumonty_b200.so (sm_100a only).

nvcc cross-compiles without a GPU.  Called by __graft_entry__.build() and, lazily, by the binding.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgpumonty_b200.so")
LISTINGS = os.path.join(HERE, "build")
SOURCES = ["gm_api.cu", "gm_tables.cu", "gm_transport.cu"]
HEADERS = ["gm_common.cuh", "gm_physics.cuh", "gm_host.h", os.path.join("..", "..", "include", "gpumonty_b200.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _stale(target: str, deps: list[str]) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    hdrs = [os.path.join(CSRC, h) for h in HEADERS] + [os.path.abspath(__file__)]
    objs, jobs = [], []
    for s in SOURCES:
        src = os.path.join(CSRC, s)
        obj = os.path.join(CSRC, s.replace(".cu", ".o"))
        objs.append(obj)
        if force or _stale(obj, [src] + hdrs):
            jobs.append([NVCC] + FLAGS + ["-c", src, "-o", obj])

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode != 0:
            sys.stderr.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
        # registers / spills per kernel: written to the ignored build/ folder (a build must not dirty the checkout;
        # the listing that belongs to a measurement is copied under profiles/ by hand)
        os.makedirs(LISTINGS, exist_ok=True)
        with open(os.path.join(LISTINGS, os.path.basename(cmd[-1]).replace(".o", ".ptxas.txt")), "w") as f:
            # (compile times dropped: the listing then changes only when the code does)
            f.write("".join(l for l in r.stderr.splitlines(True) if "Compile time" not in l))

    if jobs:
        with ThreadPoolExecutor(max_workers=len(jobs)) as ex:
            list(ex.map(run, jobs))
    if jobs or _stale(LIB, objs):
        subprocess.check_call([NVCC, "-shared", "-o", LIB] + objs + ["-gencode", "arch=compute_100a,code=sm_100a"])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
