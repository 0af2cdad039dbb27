"""GPU parity tests: the CUDA queues (through the C ABI) against the oracle.

Several results are correct for a concurrent queue, so parity is membership: the recorded
history must be linearizable w.r.t. the sequential bounded FIFO,
conserve items, and keep per-producer order (L336); single-threaded runs must equal the
sequential model exactly, EMPTY/FULL included.  All integer: bit-exact.
"""
import numpy as np
import pytest

import oracle
import paper_2606_01693_b200 as gq

pytestmark = pytest.mark.gpu

Z = gq.GQ_PATIENCE_ZERO
# (kind, extra gq_opts): the "-p0" variants force every operation onto the slow path, the only
# way to give the helping code real coverage (reading W2 / Y8); "-p1" mixes fast and slow.
VARIANTS = {
    "G-LFQ": (gq.GQ_LFQ, {}),
    "G-WFQ": (gq.GQ_WFQ, {}),
    "G-WFQ-p0": (gq.GQ_WFQ, dict(enq_patience=Z, deq_patience=Z, help_delay=1)),
    "G-WFQ-p1": (gq.GQ_WFQ, dict(enq_patience=1, deq_patience=1, help_delay=2)),
    # G-WFQ-YMC: capacity does not throttle (reading Y3), so its model capacity is "unbounded";
    # the pool is sized per test.  -p0: every enqueue takes the slow path, every dequeue makes one
    # unparked attempt and then takes the slow path (reading Y8).
    "G-WFQ-YMC": (gq.GQ_WFQ_YMC, dict(ymc_pool_cells=1 << 22)),
    "YMC-p0": (gq.GQ_WFQ_YMC, dict(ymc_pool_cells=1 << 22, enq_patience=Z, deq_patience=Z)),
    "YMC-p1": (gq.GQ_WFQ_YMC, dict(ymc_pool_cells=1 << 22, enq_patience=1, deq_patience=1)),
    # ablation builds: "-listed" = the paper's listing order and fences (no D3-D6),
    # "-eager" = polling-consumer mode used by the BFS / tracer drivers
    "G-LFQ-listed": (gq.GQ_LFQ, dict(flags=gq.GQ_F_NO_OPT_CAS | gq.GQ_F_THR_FIRST | gq.GQ_F_NO_PAIRED_FAA | gq.GQ_F_FENCED_PAYLOAD)),
    "G-LFQ-eager": (gq.GQ_LFQ, dict(flags=gq.GQ_F_EAGER_EMPTY)),
    "G-WFQ-eager": (gq.GQ_WFQ, dict(flags=gq.GQ_F_EAGER_EMPTY)),
    "YMC-eager": (gq.GQ_WFQ_YMC, dict(ymc_pool_cells=1 << 22, flags=gq.GQ_F_EAGER_EMPTY)),
    # direct-payload single-ring ablation (include/gq/dlfq.cuh): capacity bound soft, at most n + k items
    "G-LFQ-D": (gq.GQ_LFQ_DIRECT, {}),
    "G-LFQ-D-eager": (gq.GQ_LFQ_DIRECT, dict(flags=gq.GQ_F_EAGER_EMPTY)),
}
KINDS = list(VARIANTS)          # every test below runs for each of these
SMALL = KINDS                   # tiny / single-thread cases
BIG = ["G-LFQ", "G-WFQ", "G-WFQ-YMC", "G-LFQ-D"]        # full-occupancy cases
IDS = KINDS
UNBOUNDED = 1 << 31


def is_ymc(kind):
    return VARIANTS[kind][0] == gq.GQ_WFQ_YMC


def is_direct(kind):
    return VARIANTS[kind][0] == gq.GQ_LFQ_DIRECT


def soft_slack(kind, threads):
    """G-LFQ-D may hold up to n + k items for a moment (dlfq.cuh); every other kind is exact."""
    return threads if is_direct(kind) else 0


def model_capacity(kind, capacity):
    return UNBOUNDED if is_ymc(kind) else capacity


def make(kind, capacity, **opts):
    k, extra = VARIANTS[kind]
    o = gq.gq_opts(**{**extra, **opts})
    return gq.queue_create_ex(k, capacity, o)


def to_history(recs):
    return oracle.History(recs["proc"], recs["op"], recs["arg"], recs["ret_status"], recs["ret_val"],
                          recs["call_ns"], recs["end_ns"])


# ---------------------------------------------------------------- a1: WAVEFAA, Lemma III.1
@pytest.mark.parametrize("threads,rounds,seed", [(32, 8, 1), (5000, 64, 2), (65536 + 17, 16, 3)])
def test_warp_faa_tickets_distinct_and_contiguous(threads, rounds, seed):
    t, final = gq.run_warp_faa_probe(threads, rounds, seed)
    took = t[t != np.uint64(0xFFFFFFFFFFFFFFFF)]
    assert final == len(took)
    assert np.array_equal(np.sort(took), np.arange(len(took), dtype=np.uint64))
    assert 0.3 < len(took) / t.size < 0.7          # the seeded divergence really split the warps


# ---------------------------------------------------------------- single thread == sequential model
@pytest.mark.parametrize("kind", KINDS, ids=IDS)
@pytest.mark.parametrize("capacity", [1, 2, 3, 128])
def test_single_thread_equals_model(kind, capacity):
    rng = np.random.default_rng(capacity)
    n_ops = 6000
    # biased phases so that both FULL and EMPTY are hit repeatedly
    p = np.repeat(rng.choice([0.3, 0.5, 0.7], n_ops // 200), 200)
    ops = (rng.random(n_ops) > p).astype(np.uint32)            # 0 ENQ, 1 DEQ
    args = np.arange(1, n_ops + 1, dtype=np.uint32)
    q = make(kind, capacity, max_threads=64)
    try:
        st, val = gq.queue_run_script(q, ops, args, tid=5)
    finally:
        gq.queue_destroy(q)
    est, eval_ = oracle.fifo_replay(model_capacity(kind, capacity), ops, args)
    assert np.array_equal(st, est)
    ok_deq = (ops == 1) & (est == 0)
    assert np.array_equal(val[ok_deq], eval_[ok_deq])
    assert (est == oracle.ST_EMPTY).any() and (is_ymc(kind) or (est == oracle.ST_FULL).any())


@pytest.mark.parametrize("kind", KINDS, ids=IDS)
def test_fresh_fill_full_drain(kind):
    n = 128
    q = make(kind, n, max_threads=64)
    try:
        ops = [1] + [0] * (n + 1) + [1] * (n + 1)
        args = [0] + list(range(1000, 1000 + n + 1)) + [0] * (n + 1)
        st, val = gq.queue_run_script(q, ops, args)
        assert st[0] == gq.GQ_EMPTY
        if is_ymc(kind):             # no FULL: the (n+1)-th enqueue succeeds and is dequeued last
            assert (st[1:n + 2] == gq.GQ_OK).all()
            assert val[n + 2:2 * n + 3].tolist() == list(range(1000, 1000 + n + 1))
            return
        assert (st[1:n + 1] == gq.GQ_OK).all() and st[n + 1] == gq.GQ_FULL
        assert val[n + 2:2 * n + 2].tolist() == list(range(1000, 1000 + n)) and st[-1] == gq.GQ_EMPTY
    finally:
        gq.queue_destroy(q)


@pytest.mark.parametrize("kind", KINDS, ids=IDS)
@pytest.mark.parametrize("capacity,count", [(1024, 1000), (1024, 77), (1024, 1024), (100, 0), (5, 5)])
def test_prefill_drain_preserves_order(kind, capacity, count):
    q = make(kind, capacity, max_threads=64)
    try:
        vals = (np.arange(count, dtype=np.uint32) * 7 + 3)
        gq.queue_prefill(q, vals)
        out = gq.queue_drain(q, capacity + 10)
        assert np.array_equal(out, vals)
        assert len(gq.queue_drain(q, 10)) == 0
        if count:
            if not is_ymc(kind):
                with pytest.raises(gq.GqError):            # does not fit: GQ_E_STATE
                    gq.queue_prefill(q, np.arange(capacity + 1, dtype=np.uint32))
            else:
                gq.queue_prefill(q, np.arange(7, dtype=np.uint32))
            gq.queue_reset(q)
            assert len(gq.queue_drain(q, 10)) == 0
    finally:
        gq.queue_destroy(q)


# ---------------------------------------------------------------- BJ config 1: tiny history
@pytest.mark.parametrize("kind", KINDS, ids=IDS)
@pytest.mark.parametrize("seed", list(range(1, 9)))
def test_tiny_balanced_history_is_linearizable(kind, seed):
    q = make(kind, 128, max_threads=64, park_ns=2000)
    try:
        r = gq.run_balanced(q, threads=64, block_threads=64, ops_per_thread=16, record_history=1,
                            jitter_ns=200, seed=seed)
        recs = gq.history_dump(q)
        left = gq.queue_drain(q, 256)
    finally:
        gq.queue_destroy(q)
    assert len(recs) == 2048 and r["blocks"] == 1
    # reading H6: neither EMPTY nor FULL can legally occur in this configuration
    assert r["tot_full"] == 0 and r["tot_empty"] == 0 and len(left) == 0
    enq = recs[recs["op"] == 0]
    assert sorted(enq["arg"].tolist()) == sorted(t + i * 64 for t in range(64) for i in range(16))
    ok, msg = oracle.check_history(to_history(recs), model_capacity(kind, 128), relaxed_full=False, leftover=left)
    assert ok, msg


@pytest.mark.parametrize("kind", KINDS, ids=IDS)
@pytest.mark.parametrize("pf,seed", [(0.25, 1), (0.25, 2), (0.75, 3), (0.75, 4), (0.5, 5)])
def test_tiny_split_history_with_empty_and_full(kind, pf, seed):
    # reading H6: n = 16, 64 threads, 16 ops each: EMPTY frequent at 25 % producers, FULL at 75 %
    q = make(kind, 16, max_threads=64, park_ns=1000)
    try:
        r = gq.run_split(q, threads=64, block_threads=64, ops_per_thread=16, record_history=1,
                         jitter_ns=200, seed=seed, producer_fraction=pf)
        recs = gq.history_dump(q)
        left = gq.queue_drain(q, 2048)
    finally:
        gq.queue_destroy(q)
    assert len(recs) == 1024
    assert is_ymc(kind) or len(left) <= 16 + soft_slack(kind, 64)
    assert r["pool_exhausted"] == 0
    if pf < 0.5:
        assert r["tot_empty"] > 0
    if pf > 0.5:
        assert r["tot_full"] > 0 or is_ymc(kind)
    # exact search when it finishes; at 64-way overlap with many EMPTY/FULL returns it may not, and
    # the verdict then rests on the exact OK/EMPTY characterisation + capacity bound + conservation
    ok, msg = oracle.check_history(to_history(recs), model_capacity(kind, 16), relaxed_full=True, leftover=left,
                                   max_steps=3_000_000, accept_unknown=True, soft_slack=soft_slack(kind, 64))
    assert ok, msg


# ---------------------------------------------------------------- conservation at scale
def _conserve(r, left, prefill_vals=()):
    pre = np.asarray(prefill_vals, dtype=np.uint64)
    assert r["tot_enq"] + len(pre) - r["tot_deq"] == len(left)
    s_left = int(np.asarray(left, dtype=np.uint64).sum()) if len(left) else 0
    assert (r["sum_enq"] + int(pre.sum()) - r["sum_deq"] - s_left) % 2**64 == 0


@pytest.mark.parametrize("kind,threads,capacity", [(k, 2048 + 32 + 5, 1 << 12) for k in KINDS] + [(k, 0, 1 << 16) for k in BIG])
def test_balanced_fixed_ops_conserves(kind, threads, capacity):
    q = make(kind, capacity, **(dict(ymc_pool_cells=1 << 26) if is_ymc(kind) else {}))
    try:
        r = gq.run_balanced(q, threads=threads, ops_per_thread=32)
        left = gq.queue_drain(q, (1 << 19) if is_ymc(kind) else capacity + 1 + soft_slack(kind, 1 << 18))
    finally:
        gq.queue_destroy(q)
    assert is_ymc(kind) or len(left) <= capacity + soft_slack(kind, r["threads_launched"])
    assert r["pool_exhausted"] == 0
    assert r["tot_enq"] + r["tot_full"] == r["threads_launched"] * 32
    assert r["tot_deq"] + r["tot_empty"] == r["threads_launched"] * 32
    _conserve(r, left)
    assert len(set(left.tolist())) == len(left)


@pytest.mark.parametrize("kind", BIG)
def test_balanced_timed_full_occupancy(kind):
    # BJ config 2 at full co-residency, shortened window; same launch configuration as bench.py
    q = make(kind, 1 << 16, **(dict(ymc_pool_cells=1 << 31) if is_ymc(kind) else {}))
    try:
        r = gq.run_balanced(q, threads=0, warmup_ms=5, duration_ms=20)
        left = gq.queue_drain(q, (1 << 19) if is_ymc(kind) else (1 << 16) + 1 + soft_slack(kind, 1 << 18))
    finally:
        gq.queue_destroy(q)
    assert r["threads_launched"] == gq.queue_max_coresident_threads(VARIANTS[kind][0], 256)
    assert is_ymc(kind) or len(left) <= (1 << 16) + soft_slack(kind, r["threads_launched"])
    assert r["pool_exhausted"] == 0
    _conserve(r, left)
    assert r["succ_enq"] > 0 and r["succ_deq"] > 0


@pytest.mark.parametrize("kind", BIG)
@pytest.mark.parametrize("pf", [0.1, 0.5, 0.9])
def test_split_timed_conserves(kind, pf):
    # BJ config 3 shape (capacity 2^20 prefilled to 50 %), shortened window
    n = 1 << 20
    pre = np.arange(n // 2, dtype=np.uint32)
    # G-WFQ-YMC never returns FULL, so with more producers than consumers it grows for as long as
    # it runs: fixed-op mode keeps what has to be drained (by one warp, in FIFO order) bounded
    ymc = is_ymc(kind)
    q = make(kind, n, **(dict(ymc_pool_cells=1 << 28) if ymc else {}))
    try:
        gq.queue_prefill(q, pre)
        kw = dict(ops_per_thread=40) if ymc else dict(warmup_ms=2, duration_ms=10)
        r = gq.run_split(q, threads=0, producer_fraction=pf, seed=7, value_base=n // 2, **kw)
        left = gq.queue_drain(q, (1 << 24) if ymc else n + 1 + soft_slack(kind, 1 << 18))
    finally:
        gq.queue_destroy(q)
    assert ymc or len(left) <= n + soft_slack(kind, r["threads_launched"])
    assert r["pool_exhausted"] == 0
    _conserve(r, left, pre)
    # FIFO: what is left of the prefill comes out first and in order
    pre_left = left[left < n // 2]
    assert np.array_equal(pre_left, np.sort(pre_left)) and np.array_equal(left[: len(pre_left)], pre_left)


@pytest.mark.parametrize("kind", KINDS, ids=IDS)
def test_token_protocol_at_scale(kind):
    # exactly once, no foreign token, per-producer monotone — 16384 threads
    q = make(kind, 1 << 14, max_threads=16384)
    try:
        gq.run_split(q, threads=16384, ops_per_thread=24, record_history=1, producer_fraction=0.5, seed=11)
        recs = gq.history_dump(q)
        left = gq.queue_drain(q, 1 << 18)
    finally:
        gq.queue_destroy(q)
    assert len(recs) == 16384 * 24
    h = to_history(recs)
    assert oracle.precheck(h) == ""
    assert oracle.conservation(h, left) == ""


def test_residency_is_enforced():
    q = gq.queue_create(gq.GQ_LFQ, 1024)
    try:
        full = gq.queue_max_coresident_threads(gq.GQ_LFQ, 256)
        with pytest.raises(gq.GqError):
            gq.run_balanced(q, threads=full + 256, ops_per_thread=1)
    finally:
        gq.queue_destroy(q)


# ---------------------------------------------------------------- G-WFQ slow path really runs
@pytest.mark.parametrize("kind", ["G-WFQ-p0", "G-WFQ-p1"])
def test_wfq_slow_path_is_exercised_and_counts_once(kind):
    # Lemma III.7: each logical slow round advances Head/Tail exactly once.  With
    # patience 0 and a quiescent end state every operation took the slow path.
    # parking and the probe switched off, so that fast attempts really fail and patience runs out
    q = make(kind, 256, max_threads=256, flags=gq.GQ_F_NO_DEQ_SPIN | gq.GQ_F_NO_PROBE)
    try:
        r = gq.run_split(q, threads=256, block_threads=64, ops_per_thread=32, producer_fraction=0.5, seed=3) \
            if kind.endswith("p1") else gq.run_balanced(q, threads=256, block_threads=64, ops_per_thread=32)
        left = gq.queue_drain(q, 512)
    finally:
        gq.queue_destroy(q)
    _conserve(r, left)
    if kind.endswith("p0"):
        # 2 ring operations per successful queue op, 1 per FULL/EMPTY that reached the slow path
        assert r["slow_enq"] == r["tot_enq"] + r["tot_deq"]
        assert r["slow_deq"] >= r["tot_enq"] + r["tot_deq"]
    else:
        assert r["slow_enq"] + r["slow_deq"] > 0


@pytest.mark.parametrize("kind", ["YMC-p0", "YMC-p1"])
def test_ymc_slow_paths_are_exercised(kind):
    # parking and the probe off, so that dequeuers really overtake enqueuers and attempts fail
    q = make(kind, 256, max_threads=256, flags=gq.GQ_F_NO_DEQ_SPIN | gq.GQ_F_NO_PROBE)
    try:
        r = gq.run_split(q, threads=256, block_threads=64, ops_per_thread=64, producer_fraction=0.5, seed=3)
        left = gq.queue_drain(q, 1 << 15)
    finally:
        gq.queue_destroy(q)
    assert r["pool_exhausted"] == 0
    _conserve(r, left)
    if kind.endswith("p0"):
        assert r["slow_enq"] == r["tot_enq"]         # every enqueue published a request
    assert r["slow_enq"] > 0 and r["slow_deq"] > 0


@pytest.mark.parametrize("kind", KINDS, ids=IDS)
@pytest.mark.parametrize("pf,seed", [(0.25, 1), (0.75, 2)])
def test_tiny_split_default_parking(kind, pf, seed):
    # same shape with the default (long) parking budget: operations overlap almost entirely, so
    # the exact search is replaced by the bad-pattern refuter + conservation + per-producer order
    q = make(kind, 16, max_threads=64)
    try:
        gq.run_split(q, threads=64, block_threads=64, ops_per_thread=16, record_history=1,
                     jitter_ns=200, seed=seed, producer_fraction=pf)
        recs = gq.history_dump(q)
        left = gq.queue_drain(q, 2048)
    finally:
        gq.queue_destroy(q)
    h = to_history(recs)
    assert oracle.precheck(h) == "" and oracle.conservation(h, left) == ""
    r, why = oracle.poly(h)
    assert r == oracle.LIN_OK, why


# ---------------------------------------------------------------- soak: past every 32-bit wrap
@pytest.mark.parametrize("kind", ["G-LFQ", "G-WFQ"])
def test_soak_past_the_ticket_tag_wrap(kind):
    # G-LFQ's payload cells carry the low 32 bits of the AQ ticket (D6) and payload values are
    # tid + iter*k mod 2^32: 600 ms at full co-residency is ~2.5e10 operations, i.e. more than 2^32 tickets
    # on each ring and more than 2^32 enqueues; G-WFQ's 16-bit cycle field wraps every 2^35 tickets.
    q = make(kind, 1 << 16)
    try:
        r = gq.run_balanced(q, threads=0, warmup_ms=5, duration_ms=600)
        left = gq.queue_drain(q, (1 << 16) + 1)
    finally:
        gq.queue_destroy(q)
    assert r["tot_enq"] + r["tot_deq"] > (1 << 33)
    _conserve(r, left)


# ---------------------------------------------------------------- linearizability beyond the tiny config
@pytest.mark.parametrize("kind,threads,ops,capacity",
                         [(k, 4096, 8, 8192) for k in BIG + ["G-LFQ-listed"]] +
                         # k > n.  Not G-LFQ-D: it answers index starvation with thousands of FULL / EMPTY returns,
                         # and the empty-witness part of the bad-pattern check is not polynomial in those
                         [(k, 4096, 8, 512) for k in ["G-LFQ", "G-WFQ", "G-WFQ-YMC", "G-LFQ-listed"]])
def test_medium_history_bad_pattern_check(kind, threads, ops, capacity):
    # 65 536 recorded operations from 4096 threads (128 warps over several SMs), k <= n and k > n (index
    # starvation: dequeuers of FQ park, D2).  Too large for the exact WGL search at this overlap, but for
    # histories whose returns are all OK / EMPTY with unique values the bad-pattern characterisation
    # (oracle.poly) is exact, so OK here IS a linearizability verdict for the unbounded-FIFO part; FULL
    # returns (possible when k > n) are covered by the capacity lower bound and conservation.
    q = make(kind, capacity, max_threads=threads, **(dict(ymc_pool_cells=1 << 24) if is_ymc(kind) else {}))
    try:
        r = gq.run_balanced(q, threads=threads, ops_per_thread=ops, record_history=1, jitter_ns=100, seed=11)
        recs = gq.history_dump(q)
        left = gq.queue_drain(q, capacity + threads + 1)
    finally:
        gq.queue_destroy(q)
    assert len(recs) == threads * ops * 2
    h = to_history(recs)
    assert oracle.precheck(h) == ""
    assert oracle.conservation(h, left) == ""
    if r["tot_empty"] + r["tot_full"] >= 256:
        # parking (D2) normally absorbs the index starvation; if this run returned many EMPTY / FULL anyway, the
        # empty-witness part of the bad-pattern check would take minutes: keep the exact checks above and stop
        pytest.skip("many EMPTY/FULL returns in this run: bad-pattern check skipped (not polynomial in those)")
    pr, why = oracle.poly(h)
    assert pr == oracle.LIN_OK, why
    if not is_ymc(kind):
        assert oracle.capacity_bound(h, capacity + soft_slack(kind, threads)) == ""


# ---------------------------------------------------------------- split with compacted roles
@pytest.mark.parametrize("kind", ["G-LFQ", "G-WFQ", "G-WFQ-YMC"])
def test_split_role_layout_compact(kind):
    # role_layout = 1 (gq.h): the same seeded Bernoulli roles, but logical threads are placed so that warps are
    # homogeneous.  Same logical behaviour: tiny history through the checker, then BJ config 3 shape conserving.
    q = make(kind, 16, max_threads=64, park_ns=1000)
    try:
        r = gq.run_split(q, threads=64, block_threads=64, ops_per_thread=16, record_history=1, jitter_ns=200, seed=3,
                         producer_fraction=0.5, role_layout=1)
        recs = gq.history_dump(q)
        left = gq.queue_drain(q, 2048)
    finally:
        gq.queue_destroy(q)
    assert len(recs) == 1024 and sorted(set(recs["proc"].tolist())) == list(range(64))
    # a logical thread is a pure producer or a pure consumer, as drawn from the seed
    for t in range(64):
        assert len(set(recs["op"][recs["proc"] == t].tolist())) == 1
    ok, msg = oracle.check_history(to_history(recs), model_capacity(kind, 16), relaxed_full=True, leftover=left,
                                   max_steps=3_000_000, accept_unknown=True)
    assert ok, msg
    if kind == "G-LFQ":
        # role_layout = 2: mixed warps through the fused gq::enqueue_or_dequeue (address-matched WAVEFAA inside a
        # converged warp, reading G10); FULL- and EMPTY-heavy tiny histories through the checker
        for pf, seed in ((0.25, 1), (0.75, 2), (0.5, 3)):
            q = make(kind, 16, max_threads=64, park_ns=1000)
            try:
                r = gq.run_split(q, threads=64, block_threads=64, ops_per_thread=16, record_history=1, jitter_ns=200,
                                 seed=seed, producer_fraction=pf, role_layout=2)
                recs = gq.history_dump(q)
                left = gq.queue_drain(q, 2048)
            finally:
                gq.queue_destroy(q)
            ok, msg = oracle.check_history(to_history(recs), 16, relaxed_full=True, leftover=left, max_steps=3_000_000,
                                           accept_unknown=True)
            assert ok, msg
    else:
        q = make(kind, 16, max_threads=64)
        try:
            with pytest.raises(gq.GqError):                       # the fused operation exists for G-LFQ only
                gq.run_split(q, threads=64, block_threads=64, ops_per_thread=4, producer_fraction=0.5, role_layout=2)
        finally:
            gq.queue_destroy(q)
    n = 1 << 20
    pre = np.arange(n // 2, dtype=np.uint32)
    ymc = is_ymc(kind)
    q = make(kind, n, **(dict(ymc_pool_cells=1 << 28) if ymc else {}))
    try:
        gq.queue_prefill(q, pre)
        kw = dict(ops_per_thread=40) if ymc else dict(warmup_ms=2, duration_ms=10)
        r = gq.run_split(q, threads=0, producer_fraction=0.5, seed=7, value_base=n // 2, role_layout=1, **kw)
        left = gq.queue_drain(q, (1 << 24) if ymc else n + 1)
    finally:
        gq.queue_destroy(q)
    _conserve(r, left, pre)
