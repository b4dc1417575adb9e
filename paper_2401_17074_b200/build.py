"""Build libtslb.so (the C-ABI library of include/tslb.h) in-tree with nvcc for sm_100a.

    python -m paper_2401_17074_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with gpurun.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtslb.so")
SOURCES = ["tslb_api.cu", "kernels_basic.cu", "kernels_tile.cu"]
HEADERS = [os.path.join(CSRC, "tslb_internal.h"), os.path.join(HERE, "..", "include", "tslb.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static", "--threads", "4"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]
    deps += [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    return any(os.path.getmtime(d) > t for d in deps)


def build_lib(force: bool = False, verbose: bool = False, out: str = LIB, extra_flags=()) -> str:
    """Build the library.  `out` / `extra_flags` (e.g. -DTILE_F32_NS=2) build a variant beside the default one;
    binding.load_library picks it up through the TSLB_LIBRARY environment variable."""
    if out == LIB and not extra_flags and not force and not needs_build():
        return LIB
    tmp = out + ".tmp%d" % os.getpid()
    cmd = [_nvcc()] + NVCC_FLAGS + list(extra_flags) + (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd)
    os.replace(tmp, out)
    return out


if __name__ == "__main__":
    _defs = [a for a in sys.argv[1:] if a.startswith("-D")]
    _out = [a.split("=", 1)[1] for a in sys.argv[1:] if a.startswith("--out=")]
    print(build_lib(force="--force" in sys.argv, verbose="--verbose" in sys.argv, out=_out[0] if _out else LIB, extra_flags=_defs))
