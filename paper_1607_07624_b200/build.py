"""Build libpwfs.so (the C-ABI CUDA library) and libpwfs_peak.so (the FP32-peak micro-benchmark
that only bench.py loads) in-tree with nvcc for sm_100a.

    python -m paper_1607_07624_b200.build [--force] [--verbose] [--tuning]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the
GPU box with the repo snapshot.

--tuning builds a SEPARATE library, libpwfs_tuning.so (objects in build_tuning/), with
-DPWFS_TUNING: it adds the measurement hooks PWFS_DEBUG_T_ALIAS and PWFS_REC_KSPLIT
(include/pwfs.h), which change results or schedules from the environment and therefore
are not compiled into libpwfs.so.  Select it with PWFS_LIB_PATH."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "libpwfs.so")
LIB_PEAK = os.path.join(HERE, "libpwfs_peak.so")          # the FP32-peak micro-benchmark (include/pwfs_peak.h): bench.py only
PEAK_UNIT = (os.path.join(CSRC, "peak_fp32.cu"), [], "peak_fp32.o")
LIB_TUNING = os.path.join(HERE, "libpwfs_tuning.so")      # --tuning: measurement hooks compiled in (never the default)
GRID_R1 = (4, 5, 6, 8, 9, 10, 12, 15, 16, 18, 20, 24, 25, 27, 30, 32, 36, 40, 45, 48, 50, 54, 60, 64)   # PWFS_FOR_EACH_R1 of csrc/pwfs_launch.cuh
# (source, extra flags, object name): the FFT kernels of each grid size M = 32 R1 are their own translation unit
UNITS = [(os.path.join(CSRC, n), [], n[:-3] + ".o")
         for n in ("pwfs_api.cu", "atmo_api.cu", "chain_api.cu", "rec_tc.cu", "psf_api.cu", "sh_api.cu", "dm_api.cu")] + \
        [(os.path.join(CSRC, "pwfs_inst.cu"), [f"-DPWFS_INST_R1={r}"], f"pwfs_inst_r{r}.o") for r in GRID_R1]
SOURCES = sorted({u[0] for u in UNITS} | {PEAK_UNIT[0]})
HEADERS = [os.path.join(CSRC, n) for n in ("pwfs_kernels.cuh", "pwfs_dft.cuh", "pwfs_launch.cuh", "pwfs_small.cuh", "rec_tc.cuh", "device_guard.cuh")] + \
          [os.path.join(ROOT, "include", n) for n in ("pwfs.h", "pwfs_peak.h", "pwfs_atmo.h", "pwfs_chain.h", "pwfs_psf.h", "pwfs_sh.h", "pwfs_dm.h")]
OBJDIR = os.path.join(HERE, "build")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-O2"]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def _newer(target: str, deps) -> bool:
    return os.path.exists(target) and all(os.path.getmtime(target) >= os.path.getmtime(d) for d in deps)


def up_to_date() -> bool:
    return _newer(LIB, SOURCES + HEADERS) and _newer(LIB_PEAK, SOURCES + HEADERS)


def _compile(unit, force: bool, verbose: bool, objdir: str = OBJDIR, flags=()) -> str:
    src, extra, name = unit
    obj = os.path.join(objdir, name)
    if not force and _newer(obj, [src] + HEADERS):
        return obj
    cmd = [nvcc_path()] + NVCC_FLAGS + list(flags) + extra + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src]
    if verbose:
        print(" ".join(cmd), flush=True)
    subprocess.run(cmd, check=True)
    return obj


def build(force: bool = False, verbose: bool = False, tuning: bool = False) -> str:
    """One nvcc -c per source (in parallel; unchanged objects are kept), then one link."""
    lib, objdir, flags = (LIB_TUNING, OBJDIR + "_tuning", ["-DPWFS_TUNING"]) if tuning else (LIB, OBJDIR, [])
    if not force and _newer(lib, SOURCES + HEADERS) and (tuning or _newer(LIB_PEAK, SOURCES + HEADERS)):
        return lib
    os.makedirs(objdir, exist_ok=True)
    units = UNITS + ([] if tuning else [PEAK_UNIT])
    with ThreadPoolExecutor(max_workers=min(len(units), os.cpu_count() or 4)) as pool:
        objs = list(pool.map(lambda u: _compile(u, force, verbose, objdir, flags), units))
    targets = [(lib, objs[:len(UNITS)])] + ([] if tuning else [(LIB_PEAK, objs[len(UNITS):])])
    for target, members in targets:
        tmp = os.path.join(objdir, f"{os.path.basename(target)}.{os.getpid()}")     # link inside the ignored build directory
        try:
            subprocess.run([nvcc_path(), "--shared", "-o", tmp] + members, check=True)
            os.replace(tmp, target)
        finally:
            if os.path.exists(tmp):
                os.remove(tmp)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, tuning="--tuning" in sys.argv))
