"""Builds libhec.so in-tree with nvcc for sm_100a (explicit arch, -lineinfo so ncu source pages map to csrc/).

Every source is compiled to an object under paper_1805_11991_b200/build/ (git-ignored), in parallel, and only when it or
a header changed; the objects are then linked into libhec.so next to this file."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

PKG = Path(__file__).resolve().parent
ROOT = PKG.parent
CSRC = PKG / "csrc"
OBJ = PKG / "build"
LIB = PKG / "libhec.so"
SOURCES = ["hec_field.cpp", "hec_field_device.cu", "hec_count.cu", "hec_count_g1.cu", "hec_count_g2.cu", "hec_count_g3.cu",
           "hec_count_g4.cu", "hec_count_g5.cu", "hec_histogram.cu", "hec_enum.cu", "hec_gather.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-Wall"]
LINK_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static", "-Xcompiler", "-fPIC"]


def _headers():
    return [p for p in CSRC.iterdir() if p.suffix in (".h", ".cuh")] + [ROOT / "include" / "hec.h", Path(__file__)]


def needs_build() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    return any(d.stat().st_mtime > t for d in list(CSRC.iterdir()) + [ROOT / "include" / "hec.h", Path(__file__)])


def build_lib(force: bool = False, verbose: bool = False) -> Path:
    if not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    OBJ.mkdir(exist_ok=True)
    hdr_time = max(h.stat().st_mtime for h in _headers())

    def compile_one(name: str) -> Path:
        src, obj = CSRC / name, OBJ / (name + ".o")
        if not force and obj.exists() and obj.stat().st_mtime > max(src.stat().st_mtime, hdr_time):
            return obj
        tmp = obj.with_suffix(f".tmp{os.getpid()}.o")
        cmd = [nvcc, *NVCC_FLAGS, "-I", str(ROOT / "include"), "-I", str(CSRC), "-c", str(src), "-o", str(tmp)]
        if verbose:
            cmd += ["-Xptxas", "-v"]
        subprocess.check_call(cmd)
        os.replace(tmp, obj)
        return obj

    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 4)) as pool:
        objs = list(pool.map(compile_one, SOURCES))
    tmp = LIB.with_suffix(f".tmp{os.getpid()}.so")
    subprocess.check_call([nvcc, *LINK_FLAGS, "-o", str(tmp), *[str(o) for o in objs]])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build_lib(force="--force" in sys.argv, verbose="-v" in sys.argv))
