"""Builds libsgw.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2601_21005_b200.build [--force] [-v]

SGW_XFLAGS in the environment appends extra nvcc flags (e.g. -DNAME for a one-off experiment build; use --force).
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(os.path.dirname(HERE), "build", "sgw")
LIB = os.path.join(HERE, "libsgw.so")
SIZES = [8, 12, 16, 24, 32, 48, 64, 96, 128, 192, 256, 384]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "-Xcompiler", "-fPIC", "--fmad=true"] + os.environ.get("SGW_XFLAGS", "").split()


def _newest(paths):
    return max(os.path.getmtime(p) for p in paths)


def _sources():
    return [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh", ".h"))] + \
           [os.path.join(os.path.dirname(HERE), "include", "sgw.h")]


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= _newest(_sources()):
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    jobs = []
    for n in SIZES:
        jobs.append([NVCC, *FLAGS, f"-DSGW_N={n}", "-c", os.path.join(CSRC, "sgw_pass_inst.cu"),
                     "-o", os.path.join(OBJ, f"pass_{n}.o")])
    for src in ("sgw_core.cu", "sgw_solvers.cu", "sgw_program.cu", "sgw_cut.cu", "sgw_static.cu"):
        jobs.append([NVCC, *FLAGS, "-c", os.path.join(CSRC, src), "-o", os.path.join(OBJ, src[:-3] + ".o")])
    if verbose:
        for j in jobs:
            j.insert(1, "-Xptxas=-v")

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd) + "\n" + r.stdout + r.stderr)
        return r.stderr

    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        logs = list(ex.map(run, jobs))
    if verbose:
        sys.stderr.write("\n".join(logs))
    objs = [j[-1] for j in jobs]
    subprocess.check_call([NVCC, "-shared", "-o", LIB, *objs, "-gencode", "arch=compute_100a,code=sm_100a",
                           "-Xcompiler", "-fPIC"])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
