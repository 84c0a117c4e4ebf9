"""Build step of the CUDA library: nvcc -> paper_2606_26268_b200/librt_m1.so (in-tree, sm_100a only).

    python -m paper_2606_26268_b200.build [--force]

nvcc cross-compiles without a GPU.  The library links the static CUDA runtime, so it depends only on
the driver at run time.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
LIB_PATH = os.path.join(HERE, "librt_m1.so")
SOURCES = [os.path.join(HERE, "csrc", "rt_api.cu")]
HEADERS = [os.path.join(HERE, "csrc", f) for f in ("rt_math.cuh", "rt_types.cuh", "rt_kernels_aux.cuh",
                                                    "rt_kernels_step.cuh", "rt_kernels_fused.cuh", "rt_kernels_measure.cuh")] + [os.path.join(ROOT, "include", "rt.h")]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC", "-cudart", "static"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def up_to_date():
    if not os.path.exists(LIB_PATH):
        return False
    t = os.path.getmtime(LIB_PATH)
    return all(os.path.getmtime(f) <= t for f in SOURCES + HEADERS + [os.path.abspath(__file__)])


def build(force=False, verbose=False):
    """Compile the library if it is missing or older than its sources.  Returns the path."""
    if not force and up_to_date():
        return LIB_PATH
    tmp = LIB_PATH + ".tmp%d" % os.getpid()
    cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES
    try:
        subprocess.check_call(cmd)
    except FileNotFoundError as exc:
        raise RuntimeError("nvcc not found: the CUDA library cannot be built (%s)" % exc)
    os.replace(tmp, LIB_PATH)
    return LIB_PATH


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
