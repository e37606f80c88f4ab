"""Build liblisa_td.so (the C-ABI CUDA library, sm_100a only) in-tree.

    python -m paper_2501_08261_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with the
repository snapshot.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "liblisa_td.so")
PROBE_LIB = os.path.join(HERE, "liblisa_td_probe.so")  # bench-only fp64 probes (csrc/probe.cu), not product ABI
SOURCES = ["api.cu", "k1_modes_to_pol.cu", "k2_link_response.cu", "k3_tdi.cu", "k5_loglike.cu"]
HEADERS = [os.path.join(CSRC, "common.cuh"), os.path.join(ROOT, "include", "lisa_td.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden"]


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    objs = []
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(HERE, "build", src.replace(".cu", ".o"))
        if force or _stale(o, [s] + HEADERS):
            cmd = [NVCC, *FLAGS, "-c", s, "-o", o]
            if verbose:
                cmd.insert(1, "-Xptxas=-v")
            subprocess.run(cmd, check=True)
        objs.append(o)
    if force or _stale(LIB, objs):
        cmd = [NVCC, "-shared", "-o", LIB, *objs, "-L/usr/local/cuda/lib64", "-lcufft",
               "-Xlinker", "-rpath=/usr/local/cuda/lib64"]
        subprocess.run(cmd, check=True)
    probe_src = os.path.join(CSRC, "probe.cu")
    if force or _stale(PROBE_LIB, [probe_src, os.path.join(CSRC, "lisa_td_probe.h")] + HEADERS):
        subprocess.run([NVCC, *FLAGS, "-shared", probe_src, "-o", PROBE_LIB], check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
