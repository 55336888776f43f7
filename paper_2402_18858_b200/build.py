"""Builds libgpuann.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2402_18858_b200.build [--force] [-v]
    python -m paper_2402_18858_b200.build --debug      # libgpuann_debug.so: -DGPUANN_DEBUG_SPIN (csrc/ptx.cuh), i.e. every
                                                       # mbarrier wait traps after 2 s instead of hanging the GPU; the
                                                       # binding loads it when GPUANN_DEBUG_SPIN=1 is in the environment
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIB = PKG / "libgpuann.so"
LIB_DEBUG = PKG / "libgpuann_debug.so"
SOURCES = ["api.cu", "k_aux.cu", "k_fp32.cu", "k_gemm.cu", "k_fused.cu", "k_tail.cu"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-std=c++17", "-O3", "-lineinfo",
    "-shared", "-Xcompiler", "-fPIC",
    # no --use_fast_math: the FP32 / FP64 scalar paths need IEEE division, powf, erff
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and Path(cand).exists():
            return cand
    raise RuntimeError("nvcc not found (set NVCC=/path/to/nvcc)")


def sources() -> list:
    return [CSRC / s for s in SOURCES if (CSRC / s).exists()]


def needs_build(lib: Path = LIB) -> bool:
    if not lib.exists():
        return True
    t = lib.stat().st_mtime
    deps = list(CSRC.glob("*.cu")) + list(CSRC.glob("*.cuh")) + [PKG.parent / "include" / "gpuann.h"]
    return any(d.stat().st_mtime > t for d in deps)


def build(force: bool = False, verbose: bool = False, debug: bool = False) -> Path:
    lib = LIB_DEBUG if debug else LIB
    if not force and not needs_build(lib):
        return lib
    # one nvcc -c per source, in parallel (the tail kernel alone has twelve instantiations), then one link step
    from concurrent.futures import ThreadPoolExecutor
    objdir = PKG / "build" / ("debug" if debug else "release")
    objdir.mkdir(parents=True, exist_ok=True)
    compile_flags = [f for f in NVCC_FLAGS if f != "-shared"] + (["-Xptxas", "-v"] if verbose else [])
    if debug:
        compile_flags.append("-DGPUANN_DEBUG_SPIN")

    def compile_one(src):
        obj = objdir / (src.stem + ".o")
        cmd = [_nvcc()] + compile_flags + ["-c", "-o", str(obj), str(src)]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
        return obj, r.stdout + r.stderr

    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        results = list(ex.map(compile_one, sources()))
    if verbose:
        print("".join(out for _, out in results))
    cmd = [_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler", "-fPIC", "-o", str(lib)] + [str(o) for o, _ in results]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc link failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, debug="--debug" in sys.argv))
