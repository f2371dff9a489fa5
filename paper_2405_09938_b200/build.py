"""Build the CUDA library in-tree: nvcc, sm_100a only, -lineinfo (ncu source pages).

    python -m paper_2405_09938_b200.build [--force] [--verbose]

The result, paper_2405_09938_b200/libheeps_sim.so, is git-ignored but travels to the GPU box
with the gpurun snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
INCLUDE = PKG.parent / "include"
LIB = PKG / "libheeps_sim.so"
OBJ = PKG / "build"

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-Xcompiler", "-O2", "--expt-relaxed-constexpr",
]


def sources():
    return sorted(CSRC.glob("*.cu"))


def _stale(target: Path, deps) -> bool:
    if not target.exists():
        return True
    t = target.stat().st_mtime
    return any(d.stat().st_mtime > t for d in deps)


def build_library(force: bool = False, verbose: bool = False, with_checked_object: bool = False) -> Path:
    nvcc = os.environ.get("NVCC", "nvcc")
    headers = list(CSRC.glob("*.cuh")) + list(INCLUDE.glob("*.h")) + [Path(__file__)]
    OBJ.mkdir(exist_ok=True)
    jobs = []
    if with_checked_object:                            # compiled beside the others (it is the longest job of the build)
        src, obj = CSRC / "moments_keyframed.cu", OBJ / "moments_keyframed_checked.o"
        if force or _stale(obj, [src] + headers):
            jobs.append([nvcc, *NVCC_FLAGS, "-DHEEPS_CHECKED", "-I", str(INCLUDE), "-c", str(src), "-o", str(obj)])
    for src in sources():
        obj = OBJ / (src.stem + ".o")
        if force or _stale(obj, [src] + headers):
            cmd = [nvcc, *NVCC_FLAGS, "-I", str(INCLUDE), "-c", str(src), "-o", str(obj)]
            if verbose:
                cmd.insert(1, "-Xptxas=-v")
            jobs.append(cmd)
    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
        return r.stderr
    if jobs:
        with ThreadPoolExecutor(max_workers=min(8, len(jobs))) as ex:
            for log in ex.map(run, jobs):
                if verbose and log:
                    print(log, file=sys.stderr)
    objs = [OBJ / (s.stem + ".o") for s in sources()]
    if force or jobs or _stale(LIB, objs):
        tmp = LIB.with_suffix(f".{os.getpid()}.tmp")
        cmd = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", str(tmp),
               *map(str, objs), "-lcudart"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("link failed:\n" + r.stdout + r.stderr)
        os.replace(tmp, LIB)
    return LIB


CHECKED_LIB = PKG / "libheeps_sim_checked.so"


def build_checked_library() -> Path:
    """libheeps_sim_checked.so: the same library with the keyframed geometry kernel compiled with -DHEEPS_CHECKED (device-side
    bounds checks that trap).  Stands in for compute-sanitizer, which the GPU pool does not offer: run
    `HEEPS_SIM_LIBRARY=paper_2405_09938_b200/libheeps_sim_checked.so python tests/sanitizer_driver.py`."""
    build_library(with_checked_object=True)
    nvcc = os.environ.get("NVCC", "nvcc")
    src = CSRC / "moments_keyframed.cu"
    obj = OBJ / "moments_keyframed_checked.o"
    headers = list(CSRC.glob("*.cuh")) + list(INCLUDE.glob("*.h")) + [Path(__file__)]
    if _stale(obj, [src] + headers):
        r = subprocess.run([nvcc, *NVCC_FLAGS, "-DHEEPS_CHECKED", "-I", str(INCLUDE), "-c", str(src), "-o", str(obj)],
                           capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + r.stdout + r.stderr)
    objs = [OBJ / (s.stem + ".o") for s in sources() if s.stem != "moments_keyframed"] + [obj]
    if _stale(CHECKED_LIB, objs):
        tmp = CHECKED_LIB.with_suffix(f".{os.getpid()}.tmp")
        r = subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", str(tmp), *map(str, objs), "-lcudart"],
                           capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("link failed:\n" + r.stdout + r.stderr)
        os.replace(tmp, CHECKED_LIB)
    return CHECKED_LIB


if __name__ == "__main__":
    if "--checked" in sys.argv:
        print(build_checked_library())
    else:
        print(build_library(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
