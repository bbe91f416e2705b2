"""Build paper_2406_14920_b200/libte_jk.so (C ABI of include/te_jk.h) with nvcc for sm_100a, in-tree.

The per-class kernels are compiled as 10 translation units (te_inst.cu with -DTE_CB=0..9) in parallel.
Objects are cached under paper_2406_14920_b200/build/ and rebuilt when any source is newer.
"""
from __future__ import annotations

import concurrent.futures as cf
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
BUILD = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libte_jk.so")
NVCC = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC",
         "-Xptxas", "-v", "--expt-relaxed-constexpr"]


def _compile(job):
    src, obj, extra = job
    log = obj + ".log"
    cmd = [NVCC] + FLAGS + extra + ["-c", src, "-o", obj]
    with open(log, "w") as fh:
        fh.write(" ".join(cmd) + "\n")
        fh.flush()
        r = subprocess.run(cmd, stdout=fh, stderr=subprocess.STDOUT)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed for {obj}:\n" + open(log).read()[-4000:])
    return obj


# headers every translation unit sees, and the kernel headers only te_inst.cu includes
_COMMON = ["te_internal.h", "te_md.cuh", os.path.join("..", "..", "include", "te_jk.h")]
_KERNELS = ["te_kernels.cuh", "te_jkw.cuh", "te_jkq.cuh", "te_jkb.cuh", "te_jeng.cuh"]


def _newest(names) -> float:
    return max(os.path.getmtime(os.path.join(CSRC, n)) for n in names if os.path.exists(os.path.join(CSRC, n)))


def build(force: bool = False, jobs: int | None = None) -> str:
    """Compile what is stale (an object is stale when one of ITS sources is newer) and link."""
    os.makedirs(BUILD, exist_ok=True)
    work = [(os.path.join(CSRC, "te_lib.cu"), os.path.join(BUILD, "te_lib.o"), [], _newest(["te_lib.cu"] + _COMMON)),
            (os.path.join(CSRC, "te_dispatch.cu"), os.path.join(BUILD, "te_dispatch.o"), [], _newest(["te_dispatch.cu"] + _COMMON)),
            (os.path.join(CSRC, "te_noalloc.cu"), os.path.join(BUILD, "te_noalloc.o"), [],
             _newest(["te_noalloc.cu", "te_kernels.cuh"] + _COMMON))]
    inst_dep = _newest(["te_inst.cu"] + _COMMON + _KERNELS)
    # slowest translation units first so the pool stays busy
    for cb in (1, 4, 2, 0, 3, 5, 6, 7, 9, 8):
        work.append((os.path.join(CSRC, "te_inst.cu"), os.path.join(BUILD, f"te_inst_{cb}.o"), [f"-DTE_CB={cb}"], inst_dep))
    todo = [w[:3] for w in work if force or not os.path.exists(w[1]) or os.path.getmtime(w[1]) < w[3]]
    objs = [w[1] for w in work]
    if not todo and os.path.exists(LIB) and os.path.getmtime(LIB) >= max(os.path.getmtime(o) for o in objs):
        return LIB
    with cf.ThreadPoolExecutor(max_workers=jobs or min(12, os.cpu_count() or 4)) as ex:
        list(ex.map(_compile, todo))
    cmd = [NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB + ".tmp"] + objs
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
