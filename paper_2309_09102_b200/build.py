"""Build the C-ABI CUDA library in-tree: paper_2309_09102_b200/liblm_b200.so (sm_100a only).

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with the
gpurun snapshot.  `python -m paper_2309_09102_b200.build [--force] [--verbose]`.
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_ROOT = os.path.dirname(_HERE)
LIB_PATH = os.path.join(_HERE, "liblm_b200.so")
SOURCES = [os.path.join(_CSRC, f) for f in ("lm_api.cu", "lm_inst_specs.cu", "lm_inst_generic_lo.cu",
                                            "lm_inst_generic_hi.cu", "lm_traj_api.cu", "lm_plan_api.cu", "lm_search_api.cu", "lm_inst_traj_spec.cu",
                                            "lm_inst_traj_generic_lo.cu", "lm_inst_traj_generic_hi.cu", "lm_inst_lanegroup.cu")]
DEPS = SOURCES + [os.path.join(_CSRC, f) for f in ("lm_kernels.cuh", "lm_device.cuh", "lm_specs.cuh", "lm_launch.h",
                                                   "lm_ctx.h", "lm_traj.cuh", "lm_traj_launch.h", "lm_coll.cuh")] \
    + [os.path.join(_ROOT, "include", "lm.h")]

# -ftz / -prec-div / -prec-sqrt only affect sqrtf(), rsqrtf() and '/' (MUFU forms); every other
# floating-point operation in the kernels is an explicit round-to-nearest intrinsic.
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-ftz=true", "-prec-div=false", "-prec-sqrt=false", "-Xcompiler", "-fPIC"]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def is_stale() -> bool:
    if not os.path.exists(LIB_PATH):
        return True
    t = os.path.getmtime(LIB_PATH)
    return any(os.path.getmtime(p) > t for p in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile each translation unit (in parallel) and link liblm_b200.so."""
    if not (force or is_stale()):
        return LIB_PATH
    from concurrent.futures import ThreadPoolExecutor
    objdir = os.path.join(_HERE, "build")
    os.makedirs(objdir, exist_ok=True)

    def compile_one(src):
        obj = os.path.join(objdir, os.path.basename(src)[:-3] + f".{os.getpid()}.o")
        cmd = [nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", src, "-o", obj]
        res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + res.stdout)
        return obj, res.stdout

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        results = list(ex.map(compile_one, SOURCES))
    if verbose:
        for _, out in results:
            print(out)
    tmp = LIB_PATH + f".tmp{os.getpid()}"
    cmd = [nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static", "-o", tmp] \
        + [o for o, _ in results]
    res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    for o, _ in results:
        os.remove(o)
    if res.returncode != 0:
        raise RuntimeError("link failed:\n" + " ".join(cmd) + "\n" + res.stdout)
    os.replace(tmp, LIB_PATH)
    return LIB_PATH


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
