"""Builds paper_2104_13715_b200/libdia_b200.so with nvcc for sm_100a (in-tree).

The fused kernel is instantiated for every odd kernel size m <= 47 in four variants; each m is its own
translation unit (csrc/dia_eval_inst.cu compiled with -DDIA_INST_M=<m>), so the 24 + 1 compilations run in parallel.
"""
from __future__ import annotations

import concurrent.futures
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "_obj")
LIB = os.path.join(HERE, "libdia_b200.so")
KERNEL_SIZES = list(range(1, 48, 2))
HEADERS = ["dia_eval.cuh", "dia_eval_small.cuh", "dia_fit.cuh", "dia_fit_cluster.cuh", "dia_hess.cuh", "dia_hess_tc.cuh", "dia_tc_probe.cuh", "dia_cov.cuh",
           "dia_probe.cuh"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC"]


def _deps():
    return [os.path.join(CSRC, f) for f in HEADERS + ["dia_api.cu", "dia_eval_inst.cu"]] + \
           [os.path.join(HERE, "..", "include", "dia.h"), os.path.join(HERE, "build.py")]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in _deps())


def _stale(obj: str, deps) -> bool:
    return not os.path.exists(obj) or any(os.path.getmtime(d) > os.path.getmtime(obj) for d in deps)


def _compile(job):
    src, obj, defines, verbose = job
    nvcc = os.environ.get("NVCC", "nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + defines + ["-c", "-o", obj, src]
    r = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
    return r.returncode, " ".join(cmd), r.stdout + r.stderr


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    jobs = [(os.path.join(CSRC, "dia_api.cu"), os.path.join(OBJ, "dia_api.o"), [], verbose)]
    for m in KERNEL_SIZES:
        jobs.append((os.path.join(CSRC, "dia_eval_inst.cu"), os.path.join(OBJ, f"dia_eval_m{m}.o"),
                     [f"-DDIA_INST_M={m}"], verbose))
    # the per-kernel-size units include the kernel headers only; objects newer than their sources are kept
    inst_deps = [os.path.join(CSRC, f) for f in ("dia_eval.cuh", "dia_fit.cuh", "dia_fit_cluster.cuh", "dia_hess_tc.cuh", "dia_eval_inst.cu")] + \
                [os.path.join(HERE, "build.py")]
    todo = [j for j in jobs if force or _stale(j[1], _deps() if j[1].endswith("dia_api.o") else inst_deps)]
    workers = max(1, min(len(todo), os.cpu_count() or 1))
    with concurrent.futures.ThreadPoolExecutor(max_workers=workers) as pool:
        results = list(pool.map(_compile, todo))
    for rc, cmd, out in results:
        if verbose and out:
            print(out)
        if rc != 0:
            raise RuntimeError(f"nvcc failed ({rc}): {cmd}\n{out}")
    nvcc = os.environ.get("NVCC", "nvcc")
    link = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] + [j[1] for j in jobs]
    subprocess.run(link, check=True, cwd=CSRC)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
