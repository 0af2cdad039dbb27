"""Builds libgq.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

Variants (same sources, extra -D switches of include/gq/detail/debug.cuh, separate output file):
  ""         libgq.so          the product
  "mutants"  libgq_mutants.so  fault-injection build for tests/test_mutants_gpu.py (every GQ_MUT site compiled in,
                               armed one at a time with gq_set_mutation; livelock detector on, so a broken queue
                               ends its kernel instead of hanging it)
  "dbg"      libgq_dbg.so      event counters, trace ring and latency probes (gq_dbg_sites / gq_dbg_trace)
"""
import os
import subprocess
import tempfile
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "libgq.so")
SOURCES = [os.path.join(HERE, "csrc", f) for f in ("capi.cu", "apps.cu")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-fmad=false",
              "-I" + os.path.join(ROOT, "include"), "-I" + os.path.join(HERE, "csrc"),
              "-Xcompiler", "-fPIC"]
VARIANTS = {"": [], "mutants": ["-DGQ_MUTANTS", "-DGQ_DEBUG_STUCK=4000000"], "dbg": ["-DGQ_DBG_SITES"]}


def lib_path(variant: str = "") -> str:
    return os.path.join(HERE, f"libgq_{variant}.so" if variant else "libgq.so")


def _deps():
    out = list(SOURCES)
    for d in (os.path.join(ROOT, "include"), os.path.join(HERE, "csrc")):
        for dp, _, fs in os.walk(d):
            out += [os.path.join(dp, f) for f in fs if f.endswith((".h", ".cuh", ".cu", ".inc"))]
    return out


def stale(variant: str = "") -> bool:
    lib = lib_path(variant)
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(f) > t for f in _deps())


def build(force: bool = False, verbose: bool = False, variant: str = "") -> str:
    lib = lib_path(variant)
    if not force and not stale(variant):
        return lib
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = VARIANTS[variant] + os.environ.get("GQ_NVCC_EXTRA", "").split()
    flags = NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else [])
    with tempfile.TemporaryDirectory(prefix="gq_build_") as tmp:
        objs = [os.path.join(tmp, os.path.basename(s) + ".o") for s in SOURCES]
        with ThreadPoolExecutor(len(SOURCES)) as ex:       # one nvcc per translation unit, side by side
            list(ex.map(lambda so: subprocess.check_call([nvcc] + flags + ["-c", "-o", so[1], so[0]]), zip(SOURCES, objs)))
        subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", lib + ".tmp"] + objs)
    os.replace(lib + ".tmp", lib)
    return lib


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose=True, variant=sys.argv[1] if len(sys.argv) > 1 else ""))
