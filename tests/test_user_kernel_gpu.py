"""A user kernel, compiled on its own against the public __device__ header, drives the queues through
queue_device_view(): the hand-over litmus of DESIGN.md reading G15 (tests/user_kernel/litmus.cu)."""
import ctypes as C
import os
import sys

import numpy as np
import pytest

import paper_2606_01693_b200 as gq

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "user_kernel"))
pytestmark = pytest.mark.gpu

KINDS = {"G-LFQ": (gq.GQ_LFQ, {}), "G-WFQ": (gq.GQ_WFQ, {}), "G-WFQ-YMC": (gq.GQ_WFQ_YMC, dict(ymc_pool_cells=1 << 24)),
         "G-LFQ-D": (gq.GQ_LFQ_DIRECT, {}),
         "G-WFQ-p1": (gq.GQ_WFQ, dict(enq_patience=1, deq_patience=1, help_delay=2))}


@pytest.fixture(scope="module")
def litmus():
    from build import build          # tests/user_kernel/build.py
    L = C.CDLL(build())
    L.litmus_run.argtypes = [C.c_int, C.c_void_p, C.c_size_t, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_void_p]
    return L


def run(L, kind, capacity, threads, n_prod, ops, fences, flags=0):
    k, extra = KINDS[kind]
    extra = dict(extra)
    extra["flags"] = extra.get("flags", 0) | flags
    q = gq.queue_create_ex(k, capacity, gq.gq_opts(max_threads=threads, **extra))
    try:
        view = gq.queue_device_view(q)
        out = np.zeros(3, np.uint64)
        rc = L.litmus_run(k, view, len(view), threads, n_prod, ops, fences, out.ctypes.data_as(C.c_void_p))
        assert rc == 0, rc
        left = gq.queue_drain(q, 16)
    finally:
        gq.queue_destroy(q)
    assert len(left) == 0
    return int(out[0]), int(out[1]), int(out[2])


@pytest.mark.parametrize("kind", list(KINDS))
@pytest.mark.parametrize("capacity,threads,n_prod,ops", [(1 << 12, 148 * 128, 74 * 128, 64), (64, 2048, 512, 256), (1 << 16, 148 * 256, 32, 4096)])
def test_handover_with_user_fences(litmus, kind, capacity, threads, n_prod, ops):
    # the documented contract: __threadfence() before enqueue publishes the producer's other stores with the item
    consumed, mismatches, foreign = run(litmus, kind, capacity, threads, n_prod, ops, fences=1)
    assert consumed == n_prod * ops and foreign == 0
    assert mismatches == 0


@pytest.mark.parametrize("kind", ["G-LFQ", "G-WFQ-p1"])
@pytest.mark.parametrize("capacity,threads,n_prod,ops", [(1 << 12, 148 * 128, 74 * 128, 64), (64, 2048, 512, 256)])
def test_handover_fenced_build_needs_no_user_fence(litmus, kind, capacity, threads, n_prod, ops):
    # GQ_F_FENCED_PAYLOAD: installing CAS = release, entry load = acquire: the queue itself is the edge (the paper's scheme).
    # G-WFQ's slow path keeps release/acquire in every build; its fast path follows the flag.
    consumed, mismatches, foreign = run(litmus, kind, capacity, threads, n_prod, ops, fences=0, flags=gq.GQ_F_FENCED_PAYLOAD)
    assert consumed == n_prod * ops and foreign == 0
    assert mismatches == 0


def test_handover_default_build_without_fences_is_reported(litmus, capsys):
    # Not a promise of the default build (D6: relaxed installs, the payload cell carries its own handshake): informational.
    consumed, mismatches, foreign = run(litmus, "G-LFQ", 1 << 12, 148 * 128, 74 * 128, 64, fences=0)
    assert consumed == 74 * 128 * 64 and foreign == 0
    with capsys.disabled():
        print(f"\n[litmus] default G-LFQ, no user fences: {mismatches} of {consumed} side words arrived after their item")
