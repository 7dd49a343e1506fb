"""Builds paper_2603_03706_b200/libcavmag.so (hand-written CUDA for sm_100a) in-tree with nvcc.

    python -m paper_2603_03706_b200.build [--force]

nvcc cross-compiles without a GPU; the five translation units build in parallel.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libcavmag.so")
SOURCES = ["cavmag_api.cu", "cavmag_batch.cu", "cavmag_noalloc.cu", "demag.cu", "stage_inst_f32_fm.cu", "stage_inst_f32_afm.cu", "stage_inst_f64_fm.cu",
           "stage_inst_f64_afm.cu", "stage_inst_demag_f32_fm.cu", "stage_inst_demag_f32_afm.cu", "stage_inst_demag_f64_fm.cu",
           "stage_inst_demag_f64_afm.cu", "stage_inst_pol_f32_fm.cu", "stage_inst_pol_f32_afm.cu", "stage_inst_pol_f64_fm.cu", "stage_inst_pol_f64_afm.cu", "stage_tma_inst_f32_fm.cu", "stage_tma_inst_f32_afm.cu",
           "stage_tma_inst_f64_fm.cu", "stage_tma_inst_f64_afm.cu", "stage_tma_inst_sweep_f32.cu", "stage_tma_inst_sweep_f64.cu",
           "stage_tma_inst_pol_f32_fm.cu", "stage_tma_inst_pol_f32_afm.cu", "stage_tma_inst_pol_f64_fm.cu", "stage_tma_inst_pol_f64_afm.cu"]
HEADERS = ["cavmag_types.cuh", "stage_kernel.cuh", "stage_tma.cuh", "batch_kernel.cuh", "demag.cuh", os.path.join("..", "..", "include", "cavmag.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "--use_fast_math=false"]


def _nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.sep not in c or os.path.exists(c)):
            return c
    return "nvcc"


def _newest(paths):
    return max(os.path.getmtime(p) for p in paths)


def build(force: bool = False, verbose: bool = False, defines=(), lib: str = LIB, objdir: str = OBJ) -> str:
    LIB, OBJ = lib, objdir
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    deps = srcs + [os.path.join(CSRC, h) for h in HEADERS] + [os.path.abspath(__file__)]
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= _newest(deps):
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    flags = [f for f in NVCC_FLAGS if not f.startswith("--use_fast_math")] + list(defines)
    nvcc = _nvcc()

    def compile_one(src):
        obj = os.path.join(OBJ, os.path.basename(src)[:-3] + ".o")
        hdr = [os.path.join(CSRC, h) for h in HEADERS]
        if (not force) and os.path.exists(obj) and os.path.getmtime(obj) >= _newest([src] + hdr):
            return obj
        cmd = [nvcc] + flags + (["-Xptxas", "-v"] if verbose else []) + ["-c", src, "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
        if verbose:
            sys.stderr.write(r.stderr)
        return obj

    with ThreadPoolExecutor(max_workers=len(srcs)) as ex:
        objs = list(ex.map(compile_one, srcs))
    cmd = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs + ["-ldl"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n" + r.stdout + r.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
