"""Mutation tests on the GPU ("mutation tests: the checker must reject injected bugs"; section
8(c.2) G6: "a mutation build without the reload must be caught").

`libgq_mutants.so` is the library built with -DGQ_MUTANTS (paper_2606_01693_b200/build.py variant "mutants"): every fault
of include/gq/detail/debug.cuh is compiled in and gq_set_mutation(n) arms exactly one.  Each fault is a plausible mistake
in one step of the path.  The SAME check functions that tests/test_queues_gpu.py runs on the product build
(tests/queue_checks.py) are run on the broken queue, with the device-recorded histories going through the same oracle:
at least one of them must refuse each fault, which shows that %globaltimer stamps at 64-way overlap leave the checker
its discriminating power.  With no fault armed the instrumented build passes them all.
"""
import pytest

import paper_2606_01693_b200 as gq
import queue_checks as qc

pytestmark = pytest.mark.gpu

# fault -> (queue variants it lives in, what is expected to see it)
MUTANTS = {
    1: ("no reload after a failed TRYDEQ slot CAS (G6)", ["G-LFQ", "G-LFQ-listed"]),
    2: ("payload stored after the index is published, reader does not wait", ["G-LFQ"]),
    3: ("dequeue reads Data[idx ^ 1]", ["G-LFQ"]),
    4: ("emptiness probe off by two: EMPTY with items present", ["G-LFQ", "G-WFQ"]),
    5: ("index recycled before its payload is read", ["G-LFQ"]),
    6: ("WAVEFAA rank off by one: tickets handed out twice", ["G-LFQ", "G-WFQ-YMC"]),
    7: ("Threshold never reset by enqueue", ["G-LFQ", "G-WFQ"]),
    8: ("G-WFQ slow-path install without FIN: item enqueued twice", ["G-WFQ-p0"]),
    9: ("G-WFQ-YMC fast dequeue without claiming the cell", ["YMC-p1", "G-WFQ-YMC"]),
    10: ("ring enqueue installs at slot t ^ 1", ["G-LFQ", "G-WFQ"]),
    11: ("G-WFQ phase-2 helper accepts a record of the other global word (the bug of DESIGN.md D10)", ["G-WFQ-p1"]),
}


def battery(kind):
    """The parity checks of test_queues_gpu.py in the order cheapest first; returns (name, message) of the first
    violation, or None when the queue passed everything."""
    steps = [("warp_faa", lambda: qc.check_warp_faa(5000, 64, 2)),
             ("single_thread[3]", lambda: qc.check_single_thread(kind, 3)),
             ("single_thread[128]", lambda: qc.check_single_thread(kind, 128)),
             ("prefill_drain", lambda: qc.check_prefill_drain(kind, 1024, 1000))]
    steps += [(f"tiny_balanced[{s}]", lambda s=s: qc.check_tiny_balanced(kind, s)) for s in (1, 2, 3, 4)]
    steps += [(f"small_split[{pf},{s}]", lambda pf=pf, s=s: qc.check_tiny_split(kind, pf, s, threads=16, ops=8, capacity=4, exact=True))
              for pf, s in ((0.25, 11), (0.75, 12), (0.5, 14))]
    steps += [(f"tiny_split[{pf},{s}]", lambda pf=pf, s=s: qc.check_tiny_split(kind, pf, s)) for pf, s in ((0.25, 1), (0.75, 3), (0.5, 5))]
    steps += [("no_parking_split", lambda: qc.check_tiny_split(kind, 0.5, 21, threads=64, ops=64, capacity=8, park_flags=True)),
              ("fixed_ops", lambda: qc.check_balanced_fixed_ops(kind, 2048 + 37, 1 << 12)),
              ("medium[k<=n]", lambda: qc.check_medium_history(kind, 4096, 8, 8192, max_fail_returns=256))]
    if "-p" not in kind:        # k > n: only the fast paths park (D2); the all-slow builds answer index starvation with FULL / EMPTY
        steps += [("medium[k>n]", lambda: qc.check_medium_history(kind, 4096, 8, 512, max_fail_returns=256))]
    steps += [("token_protocol", lambda: qc.check_token_protocol(kind, threads=4096, ops=24))]
    if kind.endswith("-p1"):
        steps += [("slow_fast_mix_stress", lambda: qc.check_slow_fast_mix_stress(kind, reps=24))]
    for name, fn in steps:
        try:
            fn()
        except AssertionError as e:
            return name, str(e).splitlines()[0][:200]
        except gq.GqError as e:                      # a broken queue may trip the watchdog / livelock detector
            return name, str(e)
    return None


@pytest.fixture(scope="module")
def mutants():
    with gq.use_variant("mutants"):
        gq.gq_set_mutation(0)
        yield
        gq.gq_set_mutation(0)


@pytest.mark.parametrize("kind", ["G-LFQ", "G-WFQ", "G-WFQ-YMC", "G-WFQ-p0", "G-WFQ-p1", "YMC-p1"])
def test_instrumented_build_without_fault_passes(mutants, kind):
    gq.gq_set_mutation(0)
    assert battery(kind) is None


@pytest.mark.parametrize("mutation", sorted(MUTANTS))
def test_every_fault_is_refused(mutants, mutation):
    what, kinds = MUTANTS[mutation]
    caught = {}
    try:
        for kind in kinds:
            gq.gq_set_mutation(mutation)
            hit = battery(kind)
            if hit:
                caught[kind] = hit
    finally:
        gq.gq_set_mutation(0)
    print(f"\nfault {mutation} ({what}): " + "; ".join(f"{k}: refused by {n}: {m}" for k, (n, m) in caught.items()))
    assert caught, f"fault {mutation} ({what}) passed every parity check on {kinds}"
