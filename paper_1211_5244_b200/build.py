"""In-tree build of the C-ABI library (hand-written CUDA for sm_100a; nvcc cross-compiles without a GPU).

    python -m paper_1211_5244_b200.build [--force] [--jobs N]

Produces paper_1211_5244_b200/libpoisson_b200.so (objects under paper_1211_5244_b200/build/).
The .so is git-ignored but travels to the GPU box with the gpurun snapshot.
"""
from __future__ import annotations

import argparse
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
OBJ = PKG / "build"
LIB = PKG / "libpoisson_b200.so"
INCLUDE = PKG.parent / "include"

NVCC_FLAGS = [
    "-std=c++17", "-O3", "-lineinfo",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden",
]


def _headers_mtime() -> float:
    hs = list(CSRC.glob("*.cuh")) + list(CSRC.glob("*.hpp")) + list(CSRC.glob("*.def")) + [INCLUDE / "poisson.h"]
    return max(h.stat().st_mtime for h in hs)


def build(force: bool = False, jobs: int | None = None, verbose: bool = False, experiments: bool = False) -> Path:
    nvcc = os.environ.get("NVCC", "nvcc")
    OBJ.mkdir(exist_ok=True)
    srcs = sorted(CSRC.glob("*.cu"))
    hdr_t = _headers_mtime()
    # the linked library is newer than every source: nothing to do (also the case on a GPU box, where the
    # library travels with the snapshot and the object files do not, see .gpurunignore)
    if not force and LIB.exists() and LIB.stat().st_mtime >= max(hdr_t, max(s.stat().st_mtime for s in srcs)):
        return LIB
    todo = []
    for s in srcs:
        o = OBJ / (s.stem + ".o")
        if force or not o.exists() or o.stat().st_mtime < max(s.stat().st_mtime, hdr_t):
            todo.append((s, o))

    def compile_one(so):
        s, o = so
        cmd = [nvcc, *NVCC_FLAGS, "-c", str(s), "-o", str(o)]
        if experiments:
            cmd.insert(1, "-DPF_EXPERIMENTS")   # also compile the tuning variants (POISSON_VARIANT=n selects one)
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {s.name}:\n{r.stdout}\n{r.stderr}")
        return s.name, r.stderr

    if todo:
        # biggest translation units first
        todo.sort(key=lambda so: -int("".join(c for c in so[0].stem.split("_")[1] if c.isdigit()) or 0)
                  if so[0].stem.startswith("inst_") else -10 ** 6)
        with ThreadPoolExecutor(max_workers=jobs or os.cpu_count() or 4) as ex:
            for name, err in ex.map(compile_one, todo):
                if verbose and err:
                    print(f"--- {name}\n{err}", file=sys.stderr)
    objs = [str(OBJ / (s.stem + ".o")) for s in srcs]
    if todo or force or not LIB.exists():
        cmd = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-Xcompiler", "-fPIC",
               "-o", str(LIB), *objs, "-cudart", "static"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    return LIB


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--force", action="store_true")
    ap.add_argument("--jobs", type=int, default=None)
    ap.add_argument("--verbose", action="store_true")
    ap.add_argument("--experiments", action="store_true", help="also compile the tuning variants of inst_S*.cu")
    a = ap.parse_args()
    print(build(a.force or a.experiments, a.jobs, a.verbose, a.experiments))
