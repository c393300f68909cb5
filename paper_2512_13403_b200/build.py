"""Build step for the C-ABI library: nvcc -> paper_2512_13403_b200/libdh.so (sm_100a only, in-tree).

    python -m paper_2512_13403_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import concurrent.futures
import glob
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdh.so")
ROOT = os.path.dirname(HERE)

COMPILE_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC",
]
LINK_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static"]
NVCC_FLAGS = COMPILE_FLAGS + LINK_FLAGS[2:]   # the flags of the whole build, for callers that print them


def nvcc_path() -> str | None:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    return None


def sources() -> list[str]:
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps() -> list[str]:
    return sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(ROOT, "include", "dh.h")]


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in _deps())


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile every .cu under csrc/ into libdh.so.  Raises if nvcc is missing or compilation fails."""
    if not force and not is_stale():
        return LIB
    nvcc = nvcc_path()
    if nvcc is None:
        raise RuntimeError("nvcc not found: cannot build libdh.so (there is no CPU fallback)")
    tmp = LIB + f".tmp{os.getpid()}"
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    extra = ["-Xptxas", "-v"] if verbose else []
    extra += os.environ.get("DH_BUILD_DEFINES", "").split()      # e.g. -DDH_TIMING_PROBE (csrc/dh_fused2_impl.cuh)

    def compile_one(src: str):
        obj = os.path.join(objdir, os.path.basename(src)[:-3] + f".{os.getpid()}.o")
        cmd = [nvcc] + COMPILE_FLAGS + extra + ["-c", src, "-o", obj]
        return obj, subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)

    # one nvcc per translation unit, side by side (the stage kernels dominate: the build takes as long as the slowest file)
    with concurrent.futures.ThreadPoolExecutor(max_workers=max(1, min(len(sources()), os.cpu_count() or 1))) as pool:
        results = list(pool.map(compile_one, sources()))
    failed = False
    for _, res in results:
        if verbose or res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
        failed |= res.returncode != 0
    objs = [o for o, _ in results]
    try:
        if failed:
            raise RuntimeError("nvcc failed building libdh.so")
        res = subprocess.run([nvcc] + LINK_FLAGS + objs + ["-o", tmp], cwd=CSRC, capture_output=True, text=True)
        if res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
            raise RuntimeError("nvcc failed linking libdh.so")
    finally:
        for o in objs:
            if os.path.exists(o):
                os.remove(o)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
