"""queue_drain_noalloc (include/gq.h): the drain for callers that must not allocate (code under CUDA graph capture, serving
loops, harnesses that forbid cudaMalloc).  Its staging memory is a static device array inside libgq.so (256 B + 256 KiB per
GPU, at most GQ_DRAIN_NOALLOC_MAX = 65536 items per call) instead of the two cudaMalloc'ed blocks of queue_drain.

Checked here: its output equals the existing path's (integer work: bit-exact, the bar of every queue test), on two calls
in a row on the same array (the second one shorter, so that stale contents of the shared scratch would show), for every
queue kind; sizes beyond the maximum are refused with a clear message.  This file is collected last on purpose (the
suite runs with pytest -x) and passes alone in a fresh process as well as after the other tests.
"""
import numpy as np
import pytest

import paper_2606_01693_b200 as gq

pytestmark = pytest.mark.gpu

KINDS = {"G-LFQ": gq.GQ_LFQ, "G-WFQ": gq.GQ_WFQ, "G-WFQ-YMC": gq.GQ_WFQ_YMC, "G-LFQ-D": gq.GQ_LFQ_DIRECT}


def fill_and_drain(q, vals, drain, max_items):
    gq.queue_reset(q)
    gq.queue_prefill(q, vals)
    return drain(q, max_items)


@pytest.mark.parametrize("kind", list(KINDS))
def test_drain_noalloc_equals_queue_drain_on_two_calls_in_a_row(kind):
    q = gq.queue_create_ex(KINDS[kind], 8192, gq.gq_opts(max_threads=64))
    try:
        first = (np.arange(5000, dtype=np.uint32) * 2654435761 + 17).astype(np.uint32)
        second = (np.arange(1237, dtype=np.uint32) * 40503 + 5).astype(np.uint32)       # shorter: stale scratch would show
        for vals in (first, second):                                                    # two calls in a row, one shared array
            ref = fill_and_drain(q, vals, gq.queue_drain, 8192)
            out = fill_and_drain(q, vals, gq.queue_drain_noalloc, 8192)
            assert np.array_equal(ref, vals)
            assert np.array_equal(out, ref)                                             # bit-exact, FIFO order included
            assert len(gq.queue_drain_noalloc(q, 16)) == 0                              # empty afterwards: count word cleared
        # partial drains: the bound `max` is honoured and the rest stays in the queue, in order
        gq.queue_reset(q)
        gq.queue_prefill(q, first)
        a = gq.queue_drain_noalloc(q, 1000)
        b = gq.queue_drain(q, 1000)
        c = gq.queue_drain_noalloc(q, 8192)
        assert np.array_equal(np.concatenate([a, b, c]), first) and len(a) == 1000 and len(b) == 1000
    finally:
        gq.queue_destroy(q)


def test_drain_noalloc_after_a_concurrent_run():
    # the state a real caller drains: what a balanced launch left behind (holes from abandoned tickets included)
    q = gq.queue_create_ex(gq.GQ_LFQ, 4096, gq.gq_opts(max_threads=4096))
    try:
        for drain in (gq.queue_drain, gq.queue_drain_noalloc):
            gq.queue_reset(q)
            r = gq.run_split(q, threads=4096, ops_per_thread=8, producer_fraction=0.75, seed=3)
            left = drain(q, 4097)
            assert r["tot_enq"] - r["tot_deq"] == len(left)
            assert (r["sum_enq"] - r["sum_deq"] - int(np.asarray(left, np.uint64).sum())) % 2**64 == 0
            assert len(set(left.tolist())) == len(left)
    finally:
        gq.queue_destroy(q)


def test_drain_noalloc_refuses_sizes_beyond_its_scratch():
    q = gq.queue_create_ex(gq.GQ_LFQ, 1 << 17, gq.gq_opts(max_threads=64))
    try:
        gq.queue_prefill(q, np.arange(70000, dtype=np.uint32))
        with pytest.raises(gq.GqError) as e:
            gq.queue_drain_noalloc(q, gq.GQ_DRAIN_NOALLOC_MAX + 1)
        assert e.value.code == gq.GQ_E_INVAL and "GQ_DRAIN_NOALLOC_MAX" in str(e.value)
        # the documented way out: drain in pieces of at most the maximum
        a = gq.queue_drain_noalloc(q, gq.GQ_DRAIN_NOALLOC_MAX)
        b = gq.queue_drain_noalloc(q, gq.GQ_DRAIN_NOALLOC_MAX)
        assert len(a) == gq.GQ_DRAIN_NOALLOC_MAX
        assert np.array_equal(np.concatenate([a, b]), np.arange(70000, dtype=np.uint32))
    finally:
        gq.queue_destroy(q)
