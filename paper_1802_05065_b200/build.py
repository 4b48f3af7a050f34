"""Build libfpt_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1802_05065_b200.build [--force]

-fmad=false together with the explicitly rounded intrinsics in csrc/fpt_math.cuh guarantees that the only fused
operations are the written ones; never -use_fast_math.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
INCLUDE = HERE.parent / "include"
LIB = HERE / "libfpt_b200.so"
OBJDIR = HERE / "build"
UNITS = ["fpt_api.cu", "fpt_inst64.cu", "fpt_inst32.cu"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-fmad=false",
    "-prec-div=true", "-prec-sqrt=true", "-ftz=false",
    "-Xcompiler", "-fPIC,-ffp-contract=off,-fno-fast-math,-O2", "-Xptxas", "-v",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def _sources():
    return [p for p in list(CSRC.iterdir()) + [INCLUDE / "fpt.h", INCLUDE / "fpt_dbg.h"] if p.suffix in (".cu", ".cuh", ".h")]


def up_to_date() -> bool:
    return LIB.exists() and all(LIB.stat().st_mtime >= s.stat().st_mtime for s in _sources())


def build(force: bool = False, verbose: bool = False) -> Path:
    if up_to_date() and not force:
        return LIB
    OBJDIR.mkdir(exist_ok=True)
    nvcc = _nvcc()

    def compile_one(unit: str) -> Path:
        obj = OBJDIR / (Path(unit).stem + ".o")
        cmd = [nvcc, *NVCC_FLAGS, "-I", str(INCLUDE), "-c", str(CSRC / unit), "-o", str(obj)]
        r = subprocess.run(cmd, capture_output=True, text=True)
        (OBJDIR / (Path(unit).stem + ".log")).write_text(r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {unit}:\n{r.stdout}\n{r.stderr}")
        if verbose:
            print(r.stderr)
        return obj

    with ThreadPoolExecutor(len(UNITS)) as ex:
        objs = list(ex.map(compile_one, UNITS))
    tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
    cmd = [nvcc, "-shared", "-o", str(tmp), *map(str, objs), "-lcudart_static", "-lpthread", "-ldl", "-lrt"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
