"""Builds libgq.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "libgq.so")
SOURCES = [os.path.join(HERE, "csrc", f) for f in ("capi.cu", "apps.cu")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-fmad=false",
              "-I" + os.path.join(ROOT, "include"), "-I" + os.path.join(HERE, "csrc"),
              "-shared", "-Xcompiler", "-fPIC"]


def _deps():
    out = list(SOURCES)
    for d in (os.path.join(ROOT, "include"), os.path.join(HERE, "csrc")):
        for dp, _, fs in os.walk(d):
            out += [os.path.join(dp, f) for f in fs if f.endswith((".h", ".cuh", ".cu", ".inc"))]
    return out


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in _deps())


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = os.environ.get("GQ_NVCC_EXTRA", "").split()     # e.g. -DGQ_DEBUG_STUCK=2000000 (livelock detector)
    cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + SOURCES
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
