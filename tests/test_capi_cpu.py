"""CPU-only checks of the boundary: libgq.so builds, loads without a GPU, exports every
symbol include/gq.h declares, and fails loudly (no CPU fallback) when no device exists."""
import ctypes
import os
import re

import pytest

import paper_2606_01693_b200 as gq

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "gq.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"^\s*(?:int|size_t|const char\*)\s+(\w+)\s*\(", src, flags=re.M)
    return sorted(set(names))


def test_header_symbols_are_exported():
    declared = _declared_symbols()
    assert len(declared) >= 20
    for name in declared:
        assert hasattr(gq.lib, name), f"libgq.so does not export {name}"
    assert sorted(gq.SYMBOLS) == declared


def test_struct_sizes_match_header():
    # sizes implied by the field lists in gq.h (natural alignment)
    assert ctypes.sizeof(gq.gq_opts) == 64
    assert ctypes.sizeof(gq.gq_run_cfg) == 80
    assert ctypes.sizeof(gq.gq_run_result) == 14 * 8 + 16 + 16
    assert gq.HIST_DTYPE.itemsize == 40


def test_storage_bytes_is_pure_host_arithmetic():
    o = gq.gq_opts(max_threads=64)
    b = gq.queue_storage_bytes(gq.GQ_LFQ, 128, o)
    # 16 KiB hot words + two rings of 2N=256 slots * 8 B + Data 128 cells * 8 B
    assert b == 16 * 1024 + 2 * 256 * 8 + 1024
    o.layout = 2
    assert gq.queue_storage_bytes(gq.GQ_LFQ, 128, o) == 16 * 1024 + 2 * 256 * 128 + 1024
    assert gq.queue_storage_bytes(gq.GQ_LFQ, 0, o) == 0           # invalid capacity
    assert gq.queue_storage_bytes(7, 128, o) == 0                 # invalid kind


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(gq.GqError) as ei:
        gq.queue_create(gq.GQ_LFQ, 128)
    assert ei.value.code == gq.GQ_E_CUDA
    with pytest.raises(gq.GqError):
        gq.run_warp_faa_probe(64, 4, 1)
    with pytest.raises(gq.GqError):
        gq.run_faa_ceiling(1, threads=64, ops_per_thread=4)


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2606_01693_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".inc")):
                text = open(os.path.join(dp, f)).read()
                assert "oracle" not in text.replace("ORACLE", ""), f"{f} mentions the oracle"
    for dp, _, fs in os.walk(os.path.join(ROOT, "include")):
        for f in fs:
            assert "oracle" not in open(os.path.join(dp, f)).read()
