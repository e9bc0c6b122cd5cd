"""Build paper_2310_14776_b200/libfdham.so (the C-ABI library of include/fdham.h) with nvcc for
sm_100a.  nvcc cross-compiles without a GPU.  `python -m paper_2310_14776_b200.build [-v]`.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
ROOT = os.path.dirname(_HERE)
LIB = os.path.join(_HERE, "libfdham.so")
# the slow units (sweep-kernel instantiations) first, so that the parallel build ends sooner
SOURCES = ["fd_sweep_inst_real.cu", "fd_sweep_inst_real_ex.cu",
           "fd_sweep_inst_cplx_ph0.cu", "fd_sweep_inst_cplx_ph1.cu", "fd_sweep_inst_cplx_ph3.cu",
           "fd_sweep_inst_cplx_ph0_ex.cu", "fd_sweep_inst_cplx_ph1_ex.cu",
           "fd_sweep_inst_cplx_ph3_ex.cu", "fd_sweep_inst_real_jacobi.cu", "fd_sweep_inst_real_ph.cu",
           "fd_sweep_inst_real_hi.cu", "fd_sweep_inst_cplx_hi4.cu", "fd_sweep_inst_cplx_hi5.cu",
           "fd_sweep_inst_cplx_hi6.cu", "fd_sweep_inst_f32.cu",
           "fd_api.cu", "fd_generic.cu", "fd_sweep.cu", "fd_aux.cu", "fd_transfer.cu", "fd_paw.cu", "fd_peaks.cu",
           "fd_noalloc.cu"]
HEADERS = [os.path.join(CSRC, "fd_internal.h"), os.path.join(CSRC, "fd_sweep_kernel.cuh"),
           os.path.join(CSRC, "fd_sweep_inst.h"), os.path.join(ROOT, "include", "fdham.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden"]
OBJDIR = os.path.join(_HERE, "build")


def _nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libfdham cannot be built (there is no CPU fallback)")


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile every translation unit (in parallel) and link libfdham.so; no-op when up to date."""
    if not force and not _stale():
        return LIB
    from concurrent.futures import ThreadPoolExecutor
    os.makedirs(OBJDIR, exist_ok=True)
    nvcc = _nvcc()
    tag = f".tmp{os.getpid()}"

    def compile_one(src: str):
        obj = os.path.join(OBJDIR, tag[1:] + "_" + src.replace(".cu", ".o"))
        cmd = [nvcc, *NVCC_FLAGS, "-c", "-o", obj, os.path.join(CSRC, src)]
        if verbose:
            cmd[1:1] = ["-Xptxas", "-v"]
        return obj, subprocess.run(cmd, capture_output=True, text=True)

    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 1)) as pool:
        results = list(pool.map(compile_one, SOURCES))
    failed = False
    for _, res in results:
        if verbose or res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
        failed |= res.returncode != 0
    objs = [o for o, _ in results]
    try:
        if failed:
            raise RuntimeError("nvcc failed building libfdham.so")
        tmp = LIB + tag
        res = subprocess.run([nvcc, *NVCC_FLAGS, "-shared", "-o", tmp, *objs],
                             capture_output=True, text=True)
        if res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
            raise RuntimeError("nvcc failed linking libfdham.so")
        os.replace(tmp, LIB)
    finally:
        for o in objs:
            if os.path.exists(o):
                os.remove(o)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
