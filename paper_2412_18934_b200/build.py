"""Build step: compiles csrc/ into paper_2412_18934_b200/libdovetail_draft.so for sm_100a.

    python -m paper_2412_18934_b200.build [--force]

nvcc cross-compiles without a GPU. The library links only the CUDA runtime
(statically); it is kept in-tree so that it travels to the GPU box."""
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libdovetail_draft.so")
SOURCES = ["dovetail_draft.cu"]
HEADERS = ["ptx.cuh", "state.cuh", "gemv.cuh", "gemv_mma.cuh", "attention.cuh", "attention_mma.cuh", "tree.cuh", "stream_probe.cuh", "verify.cuh", "epilogue.cuh", "umma.cuh", "gemv_umma.cuh"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS]
    deps += [os.path.join(os.path.dirname(_HERE), "include", f) for f in ("dovetail.h", "dovetail_hooks.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or _stale():
        cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
              ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
