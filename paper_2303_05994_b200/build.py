"""Build libbsl6d.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2303_05994_b200.build [--force] [-v]

nvcc cross-compiles without a GPU.  Device code is compiled with -fmad=false: every fused multiply-add in the
kernels is an explicit fma(), everything else rounds as written (so the shift/weight arithmetic of steps a1/a2
matches the paper's formulas operation by operation).  Host code uses -ffp-contract=off for the same reason.
The translation units (the API + per-sweep kernels, and the fused-pass kernels once per stencil width) are
compiled in parallel and linked into one shared library.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libbsl6d.so")
OBJDIR = os.path.join(HERE, "_obj")
#: (object name, source, extra flags)
UNITS = [
    ("bsl6d_api.o", "bsl6d_api.cu", []),
    ("bsl6d_fused_q6.o", "bsl6d_fused.cu", ["-DBSL6D_FUSED_Q=6"]),
    ("bsl6d_fused_q8.o", "bsl6d_fused.cu", ["-DBSL6D_FUSED_Q=8"]),
    ("bsl6d_fused_q10.o", "bsl6d_fused.cu", ["-DBSL6D_FUSED_Q=10"]),
    ("bsl6d_pointwise.o", "bsl6d_pointwise.cu", []),
    ("bsl6d_vblock.o", "bsl6d_vblock.cu", []),
    ("bsl6d_ptile_q6.o", "bsl6d_ptile.cu", ["-DBSL6D_PTILE_Q=6"]),
    ("bsl6d_ptile_q8.o", "bsl6d_ptile.cu", ["-DBSL6D_PTILE_Q=8"]),
    ("bsl6d_ptile_q10.o", "bsl6d_ptile.cu", ["-DBSL6D_PTILE_Q=10"]),
    ("bsl6d_static.o", "bsl6d_static.cu", []),
]
HEADERS = ["sweep_kernels.cuh", "density_kernels.cuh", "fused_kernels.cuh", "fused_api.h", "field_kernels.cuh", "pointwise_kernels.cuh", "vblock_kernels.cuh", "ptile_kernels.cuh",
           os.path.join("..", "..", "include", "bsl6d.h")]

NVCC_FLAGS = [
    "-O3", "-std=c++17",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-fmad=false", "-diag-suppress", "128",
    "-Xcompiler", "-fPIC,-ffp-contract=off,-fvisibility=hidden",
]
LINK_FLAGS = ["--shared", "-gencode", "arch=compute_100a,code=sm_100a", "-cudart", "static"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, u[1]) for u in UNITS] + [os.path.join(CSRC, h) for h in HEADERS] + \
           [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, extra_flags=(), lib_path: str = LIB) -> str:
    if not force and lib_path == LIB and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objdir = OBJDIR if lib_path == LIB else lib_path + ".build"
    os.makedirs(objdir, exist_ok=True)

    def compile_unit(u):
        obj, src, flags = u
        cmd = [nvcc] + NVCC_FLAGS + list(extra_flags) + flags + (["-Xptxas", "-v"] if verbose else []) + \
              ["-c", os.path.join(CSRC, src), "-o", os.path.join(objdir, obj)]
        r = subprocess.run(cmd, capture_output=True, text=True)
        return cmd, r

    with ThreadPoolExecutor(max_workers=len(UNITS)) as ex:
        results = list(ex.map(compile_unit, UNITS))
    for cmd, r in results:
        if verbose:
            sys.stderr.write(r.stderr)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    cmd = [nvcc] + LINK_FLAGS + ["-o", lib_path + ".tmp"] + [os.path.join(objdir, u[0]) for u in UNITS]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    os.replace(lib_path + ".tmp", lib_path)
    return lib_path


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
