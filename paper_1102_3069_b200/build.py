"""Build the C-ABI library libmm_b200.so in-tree with nvcc for sm_100a (no JIT cache involved).

    python -m paper_1102_3069_b200.build [--force] [-v]

Every kernel family is a translation unit of its own (csrc/kern_*.cu): they compile in parallel, and a change in
one family cannot perturb the code generated for another.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.environ.get("MM_B200_LIB") or os.path.join(HERE, "libmm_b200.so")
OBJDIR = os.path.join(HERE, "build")
SOURCES = ["mm_api.cu", "kern_x.cu", "kern_xq.cu", "kern_y.cu", "kern_mid.cu", "kern_epi.cu", "kern_gen.cu", "kern_static.cu", "demag_host.cpp"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC,-fopenmp,-O2"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    deps.append(os.path.join(os.path.dirname(HERE), "include", "mm.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or _stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        extra = os.environ.get("MM_NVCC_EXTRA", "").split()       # e.g. -DMM_TW_SYM (experiments)
        tag = os.path.splitext(os.path.basename(LIB))[0]
        objdir = os.path.join(OBJDIR, tag)
        os.makedirs(objdir, exist_ok=True)

        def compile_one(src):
            obj = os.path.join(objdir, os.path.splitext(src)[0] + ".o")
            cmd = [nvcc, *NVCC_FLAGS, *extra, "-c", "-o", obj, os.path.join(CSRC, src)]
            if verbose:
                cmd += ["-Xptxas", "-v"]
            subprocess.check_call(cmd)
            return obj

        with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
            objs = list(ex.map(compile_one, SOURCES))
        subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB, *objs, "-lgomp"])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
