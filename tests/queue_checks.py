"""The parity checks of the CUDA queues against the oracle, as plain functions.

tests/test_queues_gpu.py runs them on the product build (they must pass); tests/test_mutants_gpu.py runs the same
functions on the fault-injection build with one fault armed at a time (they must fail): SURVEY.md section 4
"mutation tests: the checker must reject injected bugs".  Every function raises AssertionError (or gq.GqError when
a broken queue trips the watchdog) on a violation and returns a short description of what it established.
"""
import numpy as np

import oracle
import paper_2606_01693_b200 as gq

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
UNBOUNDED = 1 << 31
WGL_TALLY = {"finished": 0, "unknown": 0}      # how often the exact search decided a history (printed by conftest at the end)


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


def conserve(r, left, prefill_vals=()):
    """Counts and checksums of a run balance with what the drain found."""
    pre = np.asarray(prefill_vals, dtype=np.uint64)
    assert r["tot_enq"] + len(pre) - r["tot_deq"] == len(left), "item count not conserved"
    s_left = int(np.asarray(left, dtype=np.uint64).sum()) if len(left) else 0
    assert (r["sum_enq"] + int(pre.sum()) - r["sum_deq"] - s_left) % 2**64 == 0, "payload checksum not conserved"


def history_verdict(h, capacity, relaxed_full, left, max_steps=50_000_000, accept_unknown=False, soft=0):
    ok, msg = oracle.check_history(h, capacity, relaxed_full=relaxed_full, leftover=left, max_steps=max_steps,
                                   accept_unknown=accept_unknown, soft_slack=soft)
    WGL_TALLY["unknown" if "undecided" in msg else "finished"] += 1
    assert ok, msg
    return msg


# ---------------------------------------------------------------- a1: WAVEFAA, Lemma III.1
def check_warp_faa(threads, rounds, seed):
    t, final = gq.run_warp_faa_probe(threads, rounds, seed)
    took = t[t != np.uint64(0xFFFFFFFFFFFFFFFF)]
    assert final == len(took), "counter != tickets handed out"
    assert np.array_equal(np.sort(took), np.arange(len(took), dtype=np.uint64)), "tickets not distinct and contiguous"
    assert 0.3 < len(took) / t.size < 0.7          # the seeded divergence really split the warps
    return f"{len(took)} tickets"


def check_funnel_faa(threads, rounds, seed, window_ns=0):
    """Lemma III.1 through the block-level funnel (D11): distinct, contiguous tickets under seeded nested divergence."""
    t, final, s, n = gq.run_funnel_probe(threads, rounds, seed, window_ns)
    took = t[t != np.uint64(0xFFFFFFFFFFFFFFFF)]
    assert final == len(took) == n, "counter != tickets handed out"
    assert np.array_equal(np.sort(took), np.arange(len(took), dtype=np.uint64)), "funnel tickets not distinct and contiguous"
    assert s == n * (n - 1) // 2
    return f"{len(took)} tickets"


# ---------------------------------------------------------------- single thread == sequential model
def check_single_thread(kind, capacity, n_ops=6000):
    rng = np.random.default_rng(capacity)
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
    assert np.array_equal(st, est), "status sequence differs from the sequential model"
    ok_deq = (ops == 1) & (est == 0)
    assert np.array_equal(val[ok_deq], eval_[ok_deq]), "dequeued values differ from the sequential model"
    assert (est == oracle.ST_EMPTY).any() and (is_ymc(kind) or (est == oracle.ST_FULL).any())
    return "equals the model"


def check_prefill_drain(kind, capacity, count):
    q = make(kind, capacity, max_threads=64)
    try:
        vals = (np.arange(count, dtype=np.uint32) * 7 + 3)
        gq.queue_prefill(q, vals)
        out = gq.queue_drain(q, capacity + 10)
        assert np.array_equal(out, vals), "drain order differs from prefill order"
        assert len(gq.queue_drain(q, 10)) == 0
    finally:
        gq.queue_destroy(q)
    return "FIFO"


# ---------------------------------------------------------------- BJ config 1: tiny history
def check_tiny_balanced(kind, seed, run_kw=None, **opts):
    q = make(kind, 128, max_threads=64, park_ns=8000, **opts)
    try:
        r = gq.run_balanced(q, threads=64, block_threads=64, ops_per_thread=16, record_history=1,
                            jitter_ns=200, seed=seed, **(run_kw or {}))
        recs = gq.history_dump(q)
        left = gq.queue_drain(q, 256)
    finally:
        gq.queue_destroy(q)
    assert len(recs) == 2048 and r["blocks"] == 1
    # reading H6: neither EMPTY nor FULL can legally occur in this configuration
    assert r["tot_full"] == 0 and r["tot_empty"] == 0 and len(left) == 0, "FULL / EMPTY / leftovers in BJ#1"
    enq = recs[recs["op"] == 0]
    # BASELINE.json configs[0]: payload = thread_id << 16 | iter
    assert sorted(enq["arg"].tolist()) == sorted((t << 16) | i for t in range(64) for i in range(16))
    return history_verdict(to_history(recs), model_capacity(kind, 128), False, left)


def check_tiny_split(kind, pf, seed, threads=64, ops=16, capacity=16, exact=False, park_flags=False, **run_kw):
    """reading H6: n = 16, 64 threads, 16 ops each: EMPTY frequent at 25 % producers, FULL at 75 %.
    exact: the WGL search must finish (used with the smaller shapes); otherwise, at 64-way overlap with many EMPTY/FULL
    returns, a search that runs out of budget leaves the verdict to the exact OK/EMPTY characterisation + capacity
    bound + conservation (and is counted in WGL_TALLY)."""
    # park_flags: no parking and no probe, so that dequeuers really invalidate slots under the enqueuers' feet (G6 races)
    extra = dict(flags=VARIANTS[kind][1].get("flags", 0) | gq.GQ_F_NO_DEQ_SPIN | gq.GQ_F_NO_PROBE) if park_flags else {}
    q = make(kind, capacity, max_threads=max(threads, 32), park_ns=4000, **extra)
    try:
        r = gq.run_split(q, threads=threads, block_threads=max(32, min(threads, 64)), ops_per_thread=ops, record_history=1,
                         jitter_ns=200, seed=seed, producer_fraction=pf, **run_kw)
        recs = gq.history_dump(q)
        left = gq.queue_drain(q, 2048)
    finally:
        gq.queue_destroy(q)
    assert len(recs) == threads * ops
    assert is_ymc(kind) or len(left) <= capacity + soft_slack(kind, threads), "more items left than the capacity"
    assert r["pool_exhausted"] == 0
    msg = history_verdict(to_history(recs), model_capacity(kind, capacity), True, left, max_steps=3_000_000 if not exact else 50_000_000,
                          accept_unknown=not exact, soft=soft_slack(kind, threads))
    return r, msg


# ---------------------------------------------------------------- conservation at scale
def check_balanced_fixed_ops(kind, threads, capacity, ops=32):
    q = make(kind, capacity, **(dict(ymc_pool_cells=1 << 26) if is_ymc(kind) else {}))
    try:
        r = gq.run_balanced(q, threads=threads, ops_per_thread=ops)
        left = gq.queue_drain(q, (1 << 19) if is_ymc(kind) else capacity + 1 + soft_slack(kind, 1 << 18))
    finally:
        gq.queue_destroy(q)
    assert is_ymc(kind) or len(left) <= capacity + soft_slack(kind, r["threads_launched"])
    assert r["pool_exhausted"] == 0
    assert r["tot_enq"] + r["tot_full"] == r["threads_launched"] * ops
    assert r["tot_deq"] + r["tot_empty"] == r["threads_launched"] * ops
    conserve(r, left)
    assert len(set(left.tolist())) == len(left), "duplicate values left in the queue"
    return r


def check_token_protocol(kind, threads=16384, ops=24):
    # exactly once, no foreign token, per-producer monotone
    q = make(kind, 1 << 14, max_threads=threads)
    try:
        gq.run_split(q, threads=threads, ops_per_thread=ops, record_history=1, producer_fraction=0.5, seed=11)
        recs = gq.history_dump(q)
        left = gq.queue_drain(q, 1 << 18)
    finally:
        gq.queue_destroy(q)
    assert len(recs) == threads * ops
    h = to_history(recs)
    msg = oracle.precheck(h)
    assert msg == "", msg
    msg = oracle.conservation(h, left)
    assert msg == "", msg
    return "token protocol holds"


# ---------------------------------------------------------------- linearizability beyond the tiny config
def check_medium_history(kind, threads, ops, capacity, max_fail_returns=4096, run_kw=None):
    """65 536 recorded operations from 4096 threads (128 warps over several SMs), k <= n and k > n (index starvation:
    dequeuers of FQ park, D2).  Too large for the exact WGL search at this overlap, but for histories whose returns are
    all OK / EMPTY with unique values the bad-pattern characterisation (oracle.poly) is exact, so OK here IS a
    linearizability verdict for the unbounded-FIFO part; FULL returns (possible when k > n) are covered by the capacity
    lower bound and conservation.  The empty-witness part of that check is not polynomial in EMPTY / FULL returns, so
    a run with more than max_fail_returns of them FAILS (parking, D2, is there to absorb the starvation)."""
    q = make(kind, capacity, max_threads=threads, **(dict(ymc_pool_cells=1 << 24) if is_ymc(kind) else {}))
    try:
        r = gq.run_balanced(q, threads=threads, ops_per_thread=ops, record_history=1, jitter_ns=100, seed=11, **(run_kw or {}))
        recs = gq.history_dump(q)
        left = gq.queue_drain(q, capacity + threads + 1)
    finally:
        gq.queue_destroy(q)
    assert len(recs) == threads * ops * 2
    h = to_history(recs)
    msg = oracle.precheck(h)
    assert msg == "", msg
    msg = oracle.conservation(h, left)
    assert msg == "", msg
    assert r["tot_empty"] + r["tot_full"] <= max_fail_returns, f"{r['tot_empty']} EMPTY + {r['tot_full']} FULL returns: parking did not absorb the starvation"
    pr, why = oracle.poly(h)
    assert pr == oracle.LIN_OK, why
    if not is_ymc(kind):
        msg = oracle.capacity_bound(h, capacity + soft_slack(kind, threads))
        assert msg == "", msg
    return f"{r['tot_empty']} EMPTY, {r['tot_full']} FULL"


# ---------------------------------------------------------------- fast and slow paths mixed, long, on a tiny ring
def check_slow_fast_mix_stress(kind, reps=6, threads=64, capacity=64, ops=40000):
    """Producers and consumers in separate warps (role_layout 1) on a ring as small as the thread count, no parking and no
    probe, patience 1: consumers that poll the empty ring invalidate slots under the producers' feet, so a large share of
    the operations goes through the helping slow paths while the rest stays on the fast path, for millions of tickets and
    thousands of laps.  Checked per launch: items and payload checksums are conserved, and no queue index is lost (a queue
    that ends a launch full must still hold `capacity` items).  This is the run that exposed the shared phase-2 record of
    G-WFQ (D10): a request was handed a ticket nobody drew, and items and indices vanished."""
    q = make(kind, capacity, max_threads=threads, flags=gq.GQ_F_NO_DEQ_SPIN | gq.GQ_F_NO_PROBE,
             **(dict(ymc_pool_cells=1 << 26) if is_ymc(kind) else {}))
    slow = 0
    try:
        for rep in range(reps):
            r = gq.run_split(q, threads=threads, block_threads=32, ops_per_thread=ops, producer_fraction=0.5, seed=7 + rep,
                             role_layout=1, value_base=rep * threads * ops)
            assert r["pool_exhausted"] == 0
            slow += r["slow_enq"] + r["slow_deq"]
            left = gq.queue_drain(q, (threads * ops + 1) if is_ymc(kind) else (capacity + threads + 1))   # YMC is unbounded
            conserve(r, left)
            if not is_ymc(kind):
                # fill it up single-handedly: exactly `capacity` enqueues must succeed, i.e. every index is still in circulation
                st, _ = gq.queue_run_script(q, np.zeros(capacity + 2, np.uint32), np.arange(capacity + 2, dtype=np.uint32), tid=1)
                assert (st == 0).sum() == capacity, f"launch {rep}: only {(st == 0).sum()} of {capacity} indices left in circulation"
                assert np.array_equal(gq.queue_drain(q, capacity + 1), np.arange(capacity, dtype=np.uint32))
    finally:
        gq.queue_destroy(q)
    assert slow > 0 or is_ymc(kind), "the slow paths were never entered"     # (YMC's fast paths hardly ever fail: its slow paths are covered by the all-slow build)
    return f"{slow} slow-path operations"
