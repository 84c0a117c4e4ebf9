"""Build step of the CUDA library: nvcc -> paper_2606_26268_b200/librt_m1.so (in-tree, sm_100a only).

    python -m paper_2606_26268_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The library links the static CUDA runtime, so it depends only on
the driver at run time.  The fused sub-step kernel has 112 instantiations (solver x thick limit x geometry x
feedback x 2-D/3-D x {plain, RK2 average, run-time face fix}); they are compiled as RT_FUSED_PARTS translation units side by side with the
API unit and rt_noalloc.cu (the entry point that allocates nothing), then linked.
"""
import os
import subprocess
import sys
import tempfile
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
LIB_PATH = os.path.join(HERE, "librt_m1.so")
CSRC = os.path.join(HERE, "csrc")
API_SRC = os.path.join(CSRC, "rt_api.cu")
INST_SRC = os.path.join(CSRC, "rt_fused_inst.cu")
NOALLOC_SRC = os.path.join(CSRC, "rt_noalloc.cu")
FUSED_PARTS = 6
SOURCES = [API_SRC, INST_SRC, NOALLOC_SRC]
HEADERS = [os.path.join(CSRC, f) for f in ("rt_math.cuh", "rt_types.cuh", "rt_kernels_aux.cuh", "rt_kernels_step.cuh",
                                           "rt_kernels_fused.cuh", "rt_kernels_measure.cuh", "rt_fused_inst.cuh")] \
    + [os.path.join(ROOT, "include", "rt.h")]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC"]
LINK_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler", "-fPIC", "-cudart", "static"]


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
    nvcc = _nvcc()
    extra = ["-Xptxas", "-v"] if verbose else []
    with tempfile.TemporaryDirectory(prefix="rt_m1_build_") as tmp:
        jobs = [([nvcc] + NVCC_FLAGS + extra + ["-c", API_SRC, "-o", os.path.join(tmp, "rt_api.o")]),
                ([nvcc] + NVCC_FLAGS + extra + ["-c", NOALLOC_SRC, "-o", os.path.join(tmp, "rt_noalloc.o")])]
        for part in range(FUSED_PARTS):
            jobs.append([nvcc] + NVCC_FLAGS + extra + ["-DRT_FUSED_PART=%d" % part, "-c", INST_SRC, "-o",
                                                      os.path.join(tmp, "rt_fused_inst_%d.o" % part)])

        def run(cmd):
            try:
                p = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
            except FileNotFoundError as exc:
                raise RuntimeError("nvcc not found: the CUDA library cannot be built (%s)" % exc)
            return p.returncode, p.stdout

        with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 1)) as ex:
            results = list(ex.map(run, jobs))
        for (rc, out), cmd in zip(results, jobs):
            if verbose or rc != 0:
                sys.stderr.write(out)
            if rc != 0:
                raise RuntimeError("nvcc failed: %s" % " ".join(cmd))
        objs = [j[-1] for j in jobs]
        out_tmp = LIB_PATH + ".tmp%d" % os.getpid()
        subprocess.check_call([nvcc] + LINK_FLAGS + ["-o", out_tmp] + objs)
        os.replace(out_tmp, LIB_PATH)
    return LIB_PATH


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
