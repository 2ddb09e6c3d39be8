"""Builds libkpz_b200.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo snapshot).

The kernel instantiations are split over several translation units (csrc/kpz_launch_*.cu) so that they compile in
parallel; objects go to build/ (git-ignored) and are linked into one shared library.
"""
from __future__ import annotations

import os
import subprocess
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
UNITS = ["kpz.cu", "kpz_launch_update_wide.cu", "kpz_launch_update_narrow.cu", "kpz_launch_resident_wide.cu",
         "kpz_launch_resident_narrow.cu"]
HEADERS = [CSRC / "kpz_device.cuh", CSRC / "kpz_aux_kernels.cuh", CSRC / "kpz_peaks.cuh", CSRC / "kpz_host.h", CSRC / "kpz_launch.cuh",
           HERE.parent / "include" / "kpz.h"]
DEPS = [CSRC / u for u in UNITS] + HEADERS
LIB = HERE / "libkpz_b200.so"
OBJ_DIR = HERE / "build"

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC"]


def needs_build() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    return any(d.stat().st_mtime > t for d in DEPS)


def _compile(nvcc, unit, verbose):
    src = CSRC / unit
    obj = OBJ_DIR / (src.stem + ".o")
    newest = max(d.stat().st_mtime for d in [src] + HEADERS)
    if obj.exists() and obj.stat().st_mtime > newest:
        return obj
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", str(obj), str(src)]
    subprocess.check_call(cmd)
    return obj


def build(force: bool = False, verbose: bool = False) -> Path:
    if force or needs_build():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        OBJ_DIR.mkdir(exist_ok=True)
        if force:
            for o in OBJ_DIR.glob("*.o"):
                o.unlink()
        with ThreadPoolExecutor(max_workers=min(len(UNITS), os.cpu_count() or 1)) as ex:
            objs = list(ex.map(lambda u: _compile(nvcc, u, verbose), UNITS))
        tmp = LIB.with_suffix(".so.tmp%d" % os.getpid())
        subprocess.check_call([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", str(tmp)] + [str(o) for o in objs])
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
