"""Build libicon_dycore.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2511_02021_b200.build [--force] [--verbose]
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libicon_dycore.so")
SOURCES = ["api.cu", "kernels.cu", "kernels_sc.cu", "kernels_cc.cu", "host_grid.cpp", "sc_tables.cpp", "cc_schedule.cpp", "cc_schedule_check.cpp", "partition.cpp"]
HEADERS = ["device_grid.hpp", "host_grid.hpp", "sc_tables.hpp", "cc_schedule.hpp", "partition.hpp", "kernels.cuh", os.path.join("..", "..", "include", "icon_dycore.h")]
NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC,-fopenmp,-O2", "-shared", "-lgomp",
]


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = os.environ.get("ICON_NVCC_EXTRA", "").split()      # e.g. -DCC_DEBUG (hang reporter of kernels_cc.cu)
    cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if verbose or res.returncode:
        sys.stderr.write(res.stdout)
    if res.returncode:
        raise RuntimeError("nvcc failed:\n" + res.stdout)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
