"""Builds librbq_b200.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2606_31519_b200.build [--force]

Cross-compiles without a GPU.  -fmad=false: every fused multiply-add in the kernels is an explicit
fmaf(), so the canonical fp32 order of the encode / query paths is reproducible bit for bit.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
LIB = HERE / "librbq_b200.so"
OBJ = HERE / "build"
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-fmad=false",
         "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def sources():
    return sorted(CSRC.glob("*.cu"))


def _stale(target: Path, deps) -> bool:
    if not target.exists():
        return True
    t = target.stat().st_mtime
    return any(d.stat().st_mtime > t for d in deps)


def build(force: bool = False, verbose: bool = False, probe: bool = False) -> Path:
    """probe=True builds librbq_b200_probe.so with -DRBQ_PROBE (in-kernel timeline stamps, rbq_probe_dump); the
    binding loads it when RBQ_B200_LIB points at it.  The regular library carries no probe code."""
    hdrs = list(CSRC.glob("*.cuh")) + [HERE.parent / "include" / "rbq.h"]
    obj_dir = HERE / ("build_probe" if probe else "build")
    lib = HERE / "librbq_b200_probe.so" if probe else LIB
    flags = FLAGS + (["-DRBQ_PROBE"] if probe else [])
    obj_dir.mkdir(exist_ok=True)

    def compile_one(src: Path):
        obj = obj_dir / (src.stem + ".o")
        if force or _stale(obj, [src] + hdrs):
            r = subprocess.run([NVCC, *flags, "-c", str(src), "-o", str(obj)], capture_output=True, text=True)
            (obj_dir / (src.stem + ".ptxas.log")).write_text(r.stderr)
            if r.returncode != 0:
                raise RuntimeError(f"nvcc failed on {src.name}:\n{r.stderr}")
            if verbose:
                print(r.stderr)
        return obj

    with ThreadPoolExecutor(max_workers=8) as ex:
        objs = list(ex.map(compile_one, sources()))
    if force or _stale(lib, objs):
        r = subprocess.run([NVCC, "-shared", "-o", str(lib), *map(str, objs), "-gencode",
                            "arch=compute_100a,code=sm_100a"], capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"link failed:\n{r.stderr}")
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, probe="--probe" in sys.argv))
