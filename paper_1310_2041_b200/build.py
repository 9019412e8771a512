"""Build libgm.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgm.so")
SOURCES = ["gm_api.cu", "gm_sort.cu", "gm_nlist.cu", "gm_force.cu", "gm_force_dpd.cu", "gm_force_soft.cu", "gm_force_gauss.cu",
           "gm_force_table.cu", "gm_topo.cu", "gm_io.cu", "gm_npt.cu", "gm_static.cu"]
HEADERS = [os.path.join(CSRC, "gm_internal.cuh"), os.path.join(CSRC, "gm_force_impl.cuh"), os.path.join(CSRC, "gm_npt.cuh"), os.path.join(os.path.dirname(HERE), "include", "gm.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC", "-Xcompiler", "-Wall", "-Xptxas", "-v"]
FLAGS += os.environ.get("GM_NVCC_FLAGS", "").split()      # extra -D switches of the kernel sources (e.g. -DNL_COOP=0)


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile every .cu under csrc/ into paper_1310_2041_b200/libgm.so; returns its path."""
    if not force and not stale():
        return LIB
    objs = []
    procs = []
    for src in SOURCES:
        obj = os.path.join(CSRC, src.replace(".cu", ".o"))
        objs.append(obj)
        cmd = [NVCC] + FLAGS + ["-c", os.path.join(CSRC, src), "-o", obj]
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    log = []
    for src, p in procs:
        out, _ = p.communicate()
        log.append(out)
        if p.returncode != 0:
            sys.stderr.write(out)
            raise RuntimeError(f"nvcc failed on {src}")
    # resource usage of every kernel (registers, spills, shared memory): a build log, kept out of the tree's
    # history (_work/ is git-ignored)
    logdir = os.path.join(os.path.dirname(HERE), "_work")
    os.makedirs(logdir, exist_ok=True)
    with open(os.path.join(logdir, "ptxas.log"), "w") as f:
        f.write("\n".join(l for out in log for l in out.splitlines() if "Compile time" not in l) + "\n")
    if verbose:
        print("\n".join(log))
    subprocess.check_call([NVCC, "-shared", "-o", LIB] + objs + ["-gencode", "arch=compute_100a,code=sm_100a"])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
