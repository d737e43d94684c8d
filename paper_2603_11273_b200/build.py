"""Build libasr_sched.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import glob
import os
import subprocess

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "libasr_sched.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared",
    "-I", os.path.join(ROOT, "include"),
]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    deps = sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(ROOT, "include", "asr_sched.h")]
    return os.path.getmtime(LIB) < max(os.path.getmtime(p) for p in deps)


def _obj_stale(obj: str, src: str, headers) -> bool:
    if not os.path.exists(obj):
        return True
    return os.path.getmtime(obj) < max(os.path.getmtime(p) for p in [src] + headers)


def build(force: bool = False, verbose: bool = False) -> str:
    """one object per .cu (compiled in parallel, only when stale), then one link"""
    if not (force or is_stale()):
        return LIB
    from concurrent.futures import ThreadPoolExecutor
    extra = os.environ.get("ASR_NVCC_EXTRA", "").split()   # e.g. -DSEL_L2_AHEAD=8 for a tuning build
    objdir = os.path.join(PKG, "build")
    os.makedirs(objdir, exist_ok=True)
    headers = glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(ROOT, "include", "asr_sched.h")]
    flags = [f for f in NVCC_FLAGS if f != "-shared"]
    stamp = os.path.join(objdir, "flags.txt")
    flag_text = " ".join(flags + extra)
    if not os.path.exists(stamp) or open(stamp).read() != flag_text:
        force = True

    def compile_one(src):
        obj = os.path.join(objdir, os.path.basename(src)[:-3] + ".o")
        if force or _obj_stale(obj, src, headers):
            cmd = [NVCC] + flags + extra + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src]
            subprocess.check_call(cmd)
        return obj

    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        objs = list(ex.map(compile_one, sources()))
    with open(stamp, "w") as f:
        f.write(flag_text)
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.check_call([NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", tmp] + objs)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
