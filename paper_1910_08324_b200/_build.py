"""In-tree build of ``libspd_b200.so`` (hand-written sm_100a CUDA + the C ABI of include/spd.h).

``build()`` runs nvcc on ``csrc/*.cu`` when the library is missing or older than
its sources.  nvcc cross-compiles without a GPU, so this also runs on the CPU
box; the built ``.so`` is git-ignored but travels to the GPU box with ``gpurun``.
"""
from __future__ import annotations

import glob
import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(_HERE), "include")
LIB_PATH = os.path.join(_HERE, "libspd_b200.so")

NVCC_FLAGS = [
    "-std=c++17", "-O3", "-lineinfo", "--expt-relaxed-constexpr",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-Xcompiler", "-fPIC", "-shared",
]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps():
    return sources() + sorted(glob.glob(os.path.join(CSRC, "*.h"))) + \
        sorted(glob.glob(os.path.join(CSRC, "*.cuh"))) + [os.path.join(INCLUDE, "spd.h")]


def needs_build() -> bool:
    if not os.path.exists(LIB_PATH):
        return True
    t = os.path.getmtime(LIB_PATH)
    return any(os.path.getmtime(p) > t for p in _deps())


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: cannot build libspd_b200.so (there is no CPU fallback)")


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile every CUDA source for sm_100a into ``libspd_b200.so``; returns its path.
    The translation units are compiled in parallel (one nvcc per file), then linked."""
    if force or needs_build():
        from concurrent.futures import ThreadPoolExecutor
        nvcc = nvcc_path()
        objdir = os.path.join(_HERE, "build")
        os.makedirs(objdir, exist_ok=True)
        compile_flags = [f for f in NVCC_FLAGS if f != "-shared"] + (["-Xptxas", "-v"] if verbose else [])

        def compile_one(src):
            obj = os.path.join(objdir, os.path.basename(src)[:-3] + ".o")
            res = subprocess.run([nvcc] + compile_flags + ["-c", "-o", obj, src], cwd=CSRC,
                                 capture_output=True, text=True)
            if res.returncode != 0:
                raise RuntimeError(f"nvcc failed on {src}:\n" + res.stdout[-4000:] + res.stderr[-8000:])
            return obj, res.stderr

        with ThreadPoolExecutor(max_workers=min(8, len(sources()))) as pool:
            done = list(pool.map(compile_one, sources()))
        if verbose:
            print("".join(err for _, err in done))
        link = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB_PATH + ".tmp"] + \
            [obj for obj, _ in done]
        res = subprocess.run(link, cwd=CSRC, capture_output=True, text=True)
        if res.returncode != 0:
            raise RuntimeError("nvcc link failed:\n" + res.stdout[-4000:] + res.stderr[-8000:])
        os.replace(LIB_PATH + ".tmp", LIB_PATH)
    return LIB_PATH
