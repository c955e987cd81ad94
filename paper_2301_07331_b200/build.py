"""Build libhlc2.so (hand-written sm_100a CUDA + the C ABI of include/hlc2.h) in-tree with nvcc.

    python -m paper_2301_07331_b200.build [--force] [-v] [-DHLC2_DEBUG_BOUNDS]

nvcc cross-compiles without a GPU.  The built library is git-ignored but travels with the tree.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libhlc2.so")
SOURCES = ["hlc2_api.cu", "hlc2_build.cu", "hlc2_match.cu", "hlc2_match_same.cu", "hlc2_stream.cu", "hlc2_static.cu"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def _nvcc() -> str:
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.sep not in p or os.path.exists(p)):
            return p
    raise RuntimeError("nvcc not found")


def needs_build() -> bool:
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "hlc2.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, defines=()) -> str:
    """defines: extra -D macros (e.g. HLC2_DEBUG_BOUNDS: device-side index checks in the same-grid match kernel)."""
    if not force and not defines and not needs_build():
        return SO
    tmp = SO + f".tmp{os.getpid()}"
    cmd = [_nvcc()] + NVCC_FLAGS + [f"-D{d}" for d in defines] + (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.run(cmd, check=True)
    os.replace(tmp, SO)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, defines=[a[2:] for a in sys.argv[1:] if a.startswith("-D")]))
