"""Build libcfgms.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libcfgms.so")
LIB_PROBES = os.path.join(HERE, "libcfgms_probes.so")   # measurement build (-DCFGMS_PROBES): `bench.py --probes` only
SOURCES = ["cfgms.cu"]
HEADERS = ["ptx_sm100.cuh", "head_gemm.cuh", "finalize.cuh", "aux_kernels.cuh"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "--expt-relaxed-constexpr", "-Wno-deprecated-gpu-targets"]


def _stale(lib: str) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS]
    deps.append(os.path.join(HERE, "..", "include", "cfgms.h"))
    return any(os.path.getmtime(p) > t for p in deps)


def build_lib(force: bool = False, verbose: bool = False, probes: bool = False) -> str:
    """probes=True builds the measurement variant with the two DESIGN.md section 7 probes compiled in (a separate
    file; the product library never contains them)."""
    lib = LIB_PROBES if probes else LIB
    if force or _stale(lib):
        nvcc = os.environ.get("NVCC", "nvcc")
        cmd = [nvcc] + NVCC_FLAGS + (["-DCFGMS_PROBES"] if probes else []) + (["-Xptxas", "-v"] if verbose else []) + ["-o", lib] + \
              [os.path.join(CSRC, s) for s in SOURCES]
        subprocess.run(cmd, check=True)
    return lib


if __name__ == "__main__":
    print(build_lib(force="--force" in sys.argv, verbose="-v" in sys.argv, probes="--probes" in sys.argv))
