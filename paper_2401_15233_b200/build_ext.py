"""In-tree build of the CUDA library: csrc/*.cu -> paper_2401_15233_b200/libmm.so (sm_100a)."""
from __future__ import annotations

import os
import shutil
import subprocess
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIB = PKG / "libmm.so"                 # the product: include/mm.h
BENCH_LIB = PKG / "libmm_bench.so"     # measurement / self-test hooks: include/mm_bench.h (allocates its own scratch)
SOURCES = ["mm_api.cu"]
BENCH_SOURCES = ["mm_bench.cu"]
DEPS = ["mm_api.cu", "mm_kernels.cuh", "mm_tm14.cuh", "mm_batch5.cuh", "mm_physics.cuh", "../../include/mm.h"]
BENCH_DEPS = ["mm_bench.cu", "mm_kernels.cuh", "mm_physics.cuh", "../../include/mm_bench.h"]
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-shared", "-Xcompiler", "-fPIC"]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and Path(cand).exists():
            return cand
    raise RuntimeError("nvcc not found: the CUDA library cannot be built (there is no CPU fallback)")


def stale(lib: Path = LIB, deps=None) -> bool:
    if not lib.exists():
        return True
    t = lib.stat().st_mtime
    return any((CSRC / d).resolve().stat().st_mtime > t for d in (deps or DEPS))


def _compile(lib: Path, sources, verbose: bool) -> Path:
    cmd = [nvcc_path(), *NVCC_FLAGS]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += ["-o", str(lib), *[str(CSRC / s) for s in sources]]
    subprocess.run(cmd, check=True, cwd=CSRC)
    return lib


def build(force: bool = False, verbose: bool = False) -> Path:
    """libmm.so, the product library."""
    if not force and not stale():
        return LIB
    return _compile(LIB, SOURCES, verbose)


def build_bench(force: bool = False, verbose: bool = False) -> Path:
    """libmm_bench.so, the measurement hooks of include/mm_bench.h."""
    if not force and not stale(BENCH_LIB, BENCH_DEPS):
        return BENCH_LIB
    return _compile(BENCH_LIB, BENCH_SOURCES, verbose)


if __name__ == "__main__":
    print(build(force=True, verbose=True))
    print(build_bench(force=True, verbose=True))


OPCOUNT_TXT = PKG / "opcount.txt"


def opcount(write: bool = True) -> dict:
    """Source-level FP64 operations per cell update of the CUDA path (csrc/opcount_host.cpp:
    mm_physics.cuh compiled on the host with a counting type).  Writes opcount.txt."""
    import tempfile
    with tempfile.TemporaryDirectory() as td:
        exe = Path(td) / "opcount_host"
        subprocess.run(["g++", "-std=c++17", "-O1", "-w", "-o", str(exe), str(CSRC / "opcount_host.cpp")],
                       check=True, cwd=CSRC)
        out = subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout
    vals = {ln.split()[0]: int(ln.split()[1]) for ln in out.splitlines() if ln.strip()}
    if write:
        head = ("# FP64 operations per cell update of the CUDA path, counted at source level by\n"
                "# `python -c 'from paper_2401_15233_b200 import build_ext; build_ext.opcount()'`\n"
                "# (csrc/opcount_host.cpp; each + - * / sqrt exp pow and reciprocal = 1, FMA = 2; no tile overhead).\n"
                "# a(P*), b(P*) of Eq 29c-d are booked as the method's formulas (10 operations per call, SURVEY.md\n"
                "# section 8(d)); the *_executed lines count the kernel's table evaluation (2 x 8 FMA + 2) instead.\n")
        OPCOUNT_TXT.write_text(head + out)
    return vals


def read_opcount() -> dict:
    return {ln.split()[0]: int(ln.split()[1]) for ln in OPCOUNT_TXT.read_text().splitlines()
            if ln.strip() and not ln.startswith("#")}
