"""Builds libpt_b200.so (the C-ABI library of include/pt_b200.h) in-tree with nvcc for sm_100a.

    python -m paper_1107_3490_b200.build [--force]

nvcc cross-compiles without a GPU.  The library links the static CUDA runtime, so it loads
(and exports its symbols) on a machine without a driver; every compute call then returns
PT_ECUDA -- there is no CPU fallback.
"""
from __future__ import annotations

import shutil
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
ROOT = PKG.parent
CSRC = PKG / "csrc"
LIB = PKG / "libpt_b200.so"
OBJ = PKG / "build"
# the sweep kernels are instantiated in several translation units so that they compile in parallel
SOURCES = ["pt_api.cu", "pt_aux.cu", "pt_sweep.cu", "pt_peak.cu", "pt_sweep_group.cu", "pt_sweep_ws.cu", "pt_sweep_wsg.cu", "pt_noalloc.cu"] + \
          [f"pt_sweep_comp{u}.cu" for u in range(8)]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC",
    "-I", str(ROOT / "include"), "-I", str(CSRC),
]


def _nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and Path(cand).exists():
            return cand
    raise RuntimeError("nvcc not found: libpt_b200.so cannot be built (there is no CPU fallback)")


def _inputs():
    files = [CSRC / s for s in SOURCES]
    files += sorted(CSRC.glob("*.h")) + sorted(CSRC.glob("*.cuh")) + sorted(CSRC.glob("*.inl"))
    files.append(ROOT / "include" / "pt_b200.h")
    return files


def is_stale() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    return any(f.stat().st_mtime > t for f in _inputs())


def _compile(nvcc: str, src: str, verbose: bool) -> Path:
    obj = OBJ / (Path(src).stem + ".o")
    cmd = [nvcc, *NVCC_FLAGS, "-c", "-o", str(obj), str(CSRC / src)]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    res = subprocess.run(cmd, cwd=str(CSRC), capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError(f"nvcc failed on {src}:\n" + res.stderr[-4000:])
    return obj


def build(force: bool = False, verbose: bool = False) -> Path:
    """Compiles every translation unit (in parallel) and links libpt_b200.so."""
    if not force and not is_stale():
        return LIB
    import os
    from concurrent.futures import ThreadPoolExecutor
    nvcc = _nvcc()
    OBJ.mkdir(exist_ok=True)
    workers = max(1, min(len(SOURCES), len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else 4))
    with ThreadPoolExecutor(workers) as pool:
        objs = list(pool.map(lambda s: _compile(nvcc, s, verbose), SOURCES))
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", str(LIB), *map(str, objs)]
    res = subprocess.run(cmd, cwd=str(CSRC), capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed linking libpt_b200.so:\n" + res.stderr[-4000:])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
