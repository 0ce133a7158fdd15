"""In-tree build of libctr.so (sm_100a only): nvcc cross-compiles without a GPU.

    python -m paper_1009_2288_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIB = PKG / "libctr.so"
SOURCES = ["ctr_api.cu", "ctr_fan.cu", "ctr_si.cu", "ctr_tv.cu", "ctr_cone.cu", "ctr_peaks.cu"]
HEADERS = ["ctr_common.cuh", "ctr_internal.h", "ctr_fan_geom.cuh", "ctr_ell.cuh", "../../include/ctr.h"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC"]
OBJ = PKG / "build"  # object files (git-ignored); one nvcc per source, in parallel


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (cand == "nvcc" or Path(cand).exists()):
            return cand
    return "nvcc"


def needs_build() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    return any((CSRC / f).stat().st_mtime > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not needs_build():
        return LIB
    from concurrent.futures import ThreadPoolExecutor
    OBJ.mkdir(exist_ok=True)
    hdr_t = max((CSRC / f).stat().st_mtime for f in HEADERS)

    def compile_one(src: str):
        obj = OBJ / (src.replace(".cu", f".{os.getpid()}.o") if force else src.replace(".cu", ".o"))
        final = OBJ / src.replace(".cu", ".o")
        if not force and final.exists() and final.stat().st_mtime > max((CSRC / src).stat().st_mtime, hdr_t):
            return final, ""
        cmd = [_nvcc(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-c", "-o", str(obj), str(CSRC / src)]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + res.stdout + res.stderr)
        if obj != final:
            os.replace(obj, final)
        return final, res.stderr

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        done = list(ex.map(compile_one, SOURCES))
    if verbose:
        print("".join(err for _, err in done))
    tmp = LIB.with_name(f"libctr.tmp{os.getpid()}.so")
    cmd = [_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", str(tmp), *[str(o) for o, _ in done]]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("link failed:\n" + " ".join(cmd) + "\n" + res.stdout + res.stderr)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
