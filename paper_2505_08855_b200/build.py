"""Build libcool_b200.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo).

    python -m paper_2505_08855_b200.build [--force] [-v]

Translation units are compiled in parallel (one nvcc per .cu) and linked into one shared library.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJDIR = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libcool_b200.so")
SOURCES = ["cool_api.cu", "cool_builder.cu", "cool_launch.cu", "cool_inst_f32_m3.cu", "cool_inst_f32_m3f.cu", "cool_inst_f32_m4.cu", "cool_inst_f32_m4f.cu",
           "cool_inst_f64.cu", "cool_inst_analytic.cu", "cool_inst_implicit.cu", "cool_radpress.cu", "cool_fix.cu", "cool_cgs.cu"]
HEADERS = ["cool_internal.h", "cool_physics.cuh", "cool_kernels.cuh", "cool_f32.cuh", "cool_implicit.cuh", os.path.join("..", "..", "include", "cool.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "--use_fast_math", "-fmad=false",     # fast intrinsics, but FMAs only where the source says fmaf
              "-Xcompiler", "-fPIC", "-Xcompiler", "-O2"]


def _nvcc() -> str:
    return os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def _compile(src: str, verbose: bool) -> str:
    obj = os.path.join(OBJDIR, src.replace(".cu", ".o"))
    hdr_t = max(os.path.getmtime(os.path.join(CSRC, h)) for h in HEADERS)
    src_p = os.path.join(CSRC, src)
    if os.path.exists(obj) and os.path.getmtime(obj) > max(hdr_t, os.path.getmtime(src_p), os.path.getmtime(os.path.abspath(__file__))):
        return obj
    extra = os.environ.get("COOL_NVCC_EXTRA", "").split()          # e.g. -DCOOL_SOMETHING=1 for experiments
    cmd = [_nvcc()] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-c", src_p, "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed on {src}")
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or needs_build()):
        return LIB
    os.makedirs(OBJDIR, exist_ok=True)
    if force:
        for f in os.listdir(OBJDIR):
            os.unlink(os.path.join(OBJDIR, f))
    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 4)) as ex:
        objs = list(ex.map(lambda s: _compile(s, verbose), SOURCES))
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.check_call([_nvcc(), "-shared", "-cudart", "shared", "-gencode", "arch=compute_100a,code=sm_100a"] + objs + ["-o", tmp])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
