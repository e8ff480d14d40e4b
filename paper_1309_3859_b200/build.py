"""Builds paper_1309_3859_b200/libul.so from csrc/ with nvcc for sm_100a (in-tree, no JIT cache).

    python -m paper_1309_3859_b200.build [--force] [--verbose]
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libul.so")
SOURCES = ["ul_api.cu"]
HEADERS = ["ul_math.cuh", "ul_update.cuh", "ul_persist.cuh", "ul_update_tma.cuh", "ul_measure.cuh", os.path.join("..", "..", "include", "ul.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static", "-ldl"]


def _nvcc():
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.sep not in p or os.path.exists(p)):
            return p
    return "nvcc"


def build(force=False, verbose=False):
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    if not force and os.path.exists(SO) and all(os.path.getmtime(SO) >= os.path.getmtime(d) for d in deps):
        return SO
    cmd = [_nvcc()] + NVCC_FLAGS + os.environ.get("UL_NVCC_EXTRA", "").split() + (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", SO + ".tmp"] + [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.run(cmd, check=True, cwd=CSRC)
    os.replace(SO + ".tmp", SO)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
