#!/usr/bin/env python
"""bench.py — the paper's balanced fixed-duration micro-benchmark on B200.

One "step" = one pass of the whole hot path over one batch of work: queue_reset, then ONE
persistent fully co-resident launch of the balanced kernel (every thread loops
enqueue(unique v); dequeue()) for warmup_ms + duration_ms, on BASELINE.json configs[1]:
G-LFQ, capacity 2^16 uint32 payloads, thread count = full co-residency.

value   = successful enqueues + successful dequeues inside the measurement windows of the K
          timed steps / (K * t_meas)            [Mops/s; eq. (1)-(2), L350-357]
e2e     = the same work through the C ABI with HOST buffers: per step queue_reset +
          run_balanced (config struct in, result struct out) + queue_drain into a host
          array; all successful ops of the launch / host wall time of those calls.
roofline: this path has no contraction and its rings are L2-resident, so the bound is the
          L2 atomic unit, not HBM or tensor: peak = 2 * C1, C1 = the bare warp-batched FAA
          loop on one counter at the same occupancy, measured in this run (DESIGN.md
          "roofline").  The algorithmic-bytes view against the measured HBM copy peak is
          given beside it.
cpu_baseline: the oracle's std::mutex + std::deque queue through the same loop on the host.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--kind lfq|wfq|ymc]
N > 1: replicas only (a linearizable queue is one shared object):
every rank runs the same workload on its own GPU, no data-path collective, scaling "weak".
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

CAPACITY = 1 << 16
WARMUP_MS, DURATION_MS = 20.0, 100.0
# Algorithmic bytes per successful op: what the METHOD must move.  G-LFQ: 2 x 8 B slot
# loads + 2 x 8 B slot atomics + 2 x 8/32 B hot atomics + one 4 B payload access = 36.5 B.  The 8 B ticket-tagged payload cell
# of this implementation (D6) moves 4 B more per op: implementation overhead, reported separately.
ALGO_BYTES_PER_OP = {"lfq": 36.5, "wfq": 37.0, "ymc": 12.0, "lfq_direct": 12.5}
IMPL_EXTRA_BYTES_PER_OP = {"lfq": 4.0, "wfq": 4.0, "ymc": 4.0, "lfq_direct": 0.0}
CEILING_WINDOWS, CEILING_MS = 5, 100.0     # every ceiling: median of 5 windows of 100 ms, spread reported
KINDS = {"lfq": 0, "wfq": 1, "ymc": 2, "lfq_direct": 3}   # lfq_direct: ablation kind (include/gq/dlfq.cuh), sweep context only
# G-WFQ-YMC's pool is a ring (Y10): 0 = the default size pow2ceil(capacity + 4k) = 2^20 cells (16 MiB) for BJ#2,
# 2^21 for BJ#3; every cell is reused every ~45 us of a timed run.  The other kinds ignore the field.
YMC_POOL_CELLS = 0
# The lanes of a warp start every iteration of the benchmark loop together (gq_run_cfg.converged), as the lock-step
# wavefronts of the paper's kernels do: without it a warp that has split once stays split for the rest of the
# launch and draws partial WAVEFAA batches (the two steady states of round 1: 62 vs 79 Gops/s at n >= 2^18).
CONVERGED = 1


def env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


def measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={gpu_index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill()
            out = ""
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------ reference arm
def run_reference(args, rank, world):
    """Tier rule: the reference arm is the oracle, as it stands, on the host cores."""
    if rank != 0:
        return
    import oracle
    cores = oracle.hw_threads()
    for _ in range(args.warmup):
        oracle.mutex_bench("balanced", cores, CAPACITY, warmup_ms=5, duration_ms=20)
    ops = 0
    t0 = time.perf_counter()
    for _ in range(args.steps):
        r = oracle.mutex_bench("balanced", cores, CAPACITY, warmup_ms=WARMUP_MS, duration_ms=DURATION_MS)
        ops += r["succ_enq"] + r["succ_deq"]
    wall = time.perf_counter() - t0
    mops = ops / (args.steps * DURATION_MS * 1e-3) / 1e6
    sample = f"{args.steps} x (20 ms warmup + 100 ms window), {cores} host threads, capacity 2^16"
    line = {"impl": "reference", "metric": "queue Mops/s (balanced)", "value": mops, "unit": "Mops/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": wall / args.steps * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
            "config": {"workload": "BJ#2 balanced, capacity 2^16, std::mutex+std::deque on host threads", "threads": cores},
            "cpu_baseline": {"value": mops, "unit": "Mops/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": mops, "unit": "Mops/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------ replicas
def aggregate_replicas(dist, device, sums, maxes):
    """Replicas only: whole-job units = SUM over ranks, time = MAX over ranks.
    `dist` is torch.distributed (initialised) or None for a single process.  The only
    communication of a multi-GPU run; tests/test_bench_aggregate.py drives it with gloo."""
    import torch
    a = torch.tensor(list(sums), dtype=torch.float64, device=device)
    m = torch.tensor(list(maxes), dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(a, op=dist.ReduceOp.SUM)
        dist.all_reduce(m, op=dist.ReduceOp.MAX)
    return a.tolist(), m.tolist()


# ------------------------------------------------------------------------------ application rows
def run_apps(gq, torch, scale, fast_oracle=True):
    """BASELINE.json configs[3] and [4] (NEXT-1 / NEXT-2 of DESIGN.md section 6): BFS on the seeded R-MAT
    graph and the 1920x1080 tile-queue path tracer, each checked against the oracle on the spot
    (distances bit-exact; image within 1e-3 on >= 99.99 % of pixels) and timed beside it."""
    import numpy as np
    import oracle
    from paper_2606_01693_b200 import inputs
    out = {}
    t0 = time.perf_counter()
    d_rowptr, d_col, src = inputs.rmat_csr_torch(scale, 16, seed=1, device="cuda")   # same arrays as inputs.rmat_csr (tests/test_inputs.py)
    torch.cuda.synchronize()
    gen_s = time.perf_counter() - t0
    rowptr, col = d_rowptr.cpu().numpy().astype(np.uint64), d_col.cpu().numpy().view(np.uint32)
    nv = len(rowptr) - 1
    t0 = time.perf_counter()
    ref, ref_edges = oracle.bfs(rowptr, col, src)
    cpu_s = time.perf_counter() - t0
    d_dist = torch.empty(nv, dtype=torch.int32, device="cuda")
    bfs = {"graph": f"R-MAT scale {scale}, edge factor 16, {nv} vertices, {len(col)} directed edges, source {src}",
           "generate_s": round(gen_s, 1),
           "cpu_oracle": {"ms": round(cpu_s * 1e3, 1), "MTEPS": round(ref_edges / cpu_s / 1e6, 1), "cores": 1}}
    for name, k in KINDS.items():
        best = None
        for _ in range(3):
            st = gq.bfs_run(k, d_rowptr.data_ptr(), d_col.data_ptr(), nv, src, d_dist.data_ptr())
            torch.cuda.synchronize()
            if best is None or st["ms"] < best["ms"]:
                best = st
        exact = bool(np.array_equal(d_dist.cpu().numpy(), ref))
        bfs[name] = {"ms": round(best["ms"], 3), "total_ms": round(best["total_ms"], 3), "levels": best["levels"],
                     "MTEPS": round(best["edges_scanned"] / (best["ms"] * 1e-3) / 1e6, 1),
                     "queue_Mops": round(best["queue_ops"] / (best["ms"] * 1e-3) / 1e6, 1),
                     "threads": best["threads"], "bit_exact": exact}
    out["bfs"] = bfs
    del d_rowptr, d_col, d_dist

    W, H, SPP, B = 1920, 1080, 4, 4
    sph = inputs.sphere_scene(256, seed=1)
    d_sph = torch.from_numpy(np.ascontiguousarray(sph, np.float32)).cuda()
    d_rgb = torch.empty((H, W, 3), dtype=torch.float32, device="cuda")
    t0 = time.perf_counter()
    ref_img, ref_rays = oracle.rt_render(W, H, SPP, B, sph, seed=1)
    cpu_s = time.perf_counter() - t0
    rt = {"scene": "1920x1080, 16x16 tiles, 256 seeded spheres, 4 spp, <= 4 bounces, fp32 no FMA contraction",
          "cpu_oracle": {"ms": round(cpu_s * 1e3, 1), "Mrays": round(ref_rays / cpu_s / 1e6, 2), "cores": oracle.hw_threads()}}
    for name, k in KINDS.items():
        best = None
        for _ in range(3):
            st = gq.rt_render(k, W, H, SPP, B, len(sph), d_sph.data_ptr(), 1, d_rgb.data_ptr())
            torch.cuda.synchronize()
            if best is None or st["ms"] < best["ms"]:
                best = st
        img = d_rgb.cpu().numpy()
        err = np.abs(img.astype(np.float64) - ref_img.astype(np.float64)).max(axis=2)
        rt[name] = {"ms": round(best["ms"], 3), "total_ms": round(best["total_ms"], 3),
                    "Mrays": round(best["rays"] / (best["ms"] * 1e-3) / 1e6, 1),
                    "queue_Mops": round(best["queue_ops"] / (best["ms"] * 1e-3) / 1e6, 3), "items": best["items"],
                    "pixels_within_1e-3": float((err <= 1e-3).mean()), "pixels_bit_exact": float((err == 0).mean()),
                    "rays_match_oracle": bool(best["rays"] == ref_rays)}
    # the paper's own work distribution: one queue per tile, items are rays; must reproduce the image bit for bit
    best = None
    one = d_rgb.clone()
    gq.rt_render(0, W, H, SPP, B, len(sph), d_sph.data_ptr(), 1, one.data_ptr())
    for _ in range(3):
        st = gq.rt_render(0, W, H, SPP, B, len(sph), d_sph.data_ptr(), 1, d_rgb.data_ptr(), mode=1)
        torch.cuda.synchronize()
        if best is None or st["ms"] < best["ms"]:
            best = st
    rt["lfq_one_queue_per_tile"] = {"ms": round(best["ms"], 3), "total_ms": round(best["total_ms"], 3), "queues": best["items"],
                                    "Mrays": round(best["rays"] / (best["ms"] * 1e-3) / 1e6, 1),
                                    "queue_Mops": round(best["queue_ops"] / (best["ms"] * 1e-3) / 1e6, 1),
                                    "identical_to_single_queue": bool(torch.equal(one, d_rgb))}
    out["rt"] = rt
    return out


# ------------------------------------------------------------------------------ our arm
def run_ours(args, rank, world, local_rank):
    import numpy as np
    import torch
    import paper_2606_01693_b200 as gq

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist_
        dist = dist_
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    kind = KINDS[args.kind]
    full = gq.queue_max_coresident_threads(kind, 256)
    threads = args.threads or full
    q = gq.queue_create_ex(kind, CAPACITY, gq.gq_opts(ymc_pool_cells=YMC_POOL_CELLS))
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2
    run_kw = dict(threads=threads, warmup_ms=WARMUP_MS, duration_ms=DURATION_MS, fail_backoff_ns=args.fail_backoff_ns, converged=CONVERGED)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        flush.fill_(1)                       # L2 flushed between iterations (timing rules)
        gq.queue_reset(q)
        return gq.run_balanced(q, **run_kw)

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    t0 = time.perf_counter()
    results = [step() for _ in range(args.steps)]
    barrier()
    wall = time.perf_counter() - t0
    clocks = sampler.stop() if sampler else None

    ops_window = sum(r["succ_enq"] + r["succ_deq"] for r in results)
    ops_all = sum(r["tot_enq"] + r["tot_deq"] for r in results)
    kernel_ms = sum(r["kernel_ms"] for r in results) / len(results)
    meas_s = sum(r["meas_seconds"] for r in results)

    # ---- e2e through the C ABI with host buffers (reset + run + drain to host)
    e2e_ops, e2e_drained = 0, 0
    barrier()
    t1 = time.perf_counter()
    for _ in range(args.steps):
        gq.queue_reset(q)
        r = gq.run_balanced(q, **run_kw)
        left = gq.queue_drain(q, CAPACITY + 1)
        assert r["tot_enq"] - r["tot_deq"] == len(left), "conservation violated"
        e2e_ops += r["tot_enq"] + r["tot_deq"]
        e2e_drained += len(left)
    barrier()
    e2e_wall = time.perf_counter() - t1

    # ---- aggregate over ranks (replicas): ops sum, time max
    (ops_window_all, ops_all_all, e2e_ops_all), (wall_max, e2e_wall_max, kernel_ms_max) = aggregate_replicas(
        dist, "cuda", [ops_window, ops_all, e2e_ops], [wall, e2e_wall, kernel_ms])

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        gq.queue_destroy(q)
        return

    value = ops_window_all / (args.steps * DURATION_MS * 1e-3) / 1e6

    # ---- ceilings at the same occupancy (rank 0, outside the timed region)
    def ceiling(n_counters, per_lane=False):
        """tickets/s of the bare FAA loop: median, min and max over CEILING_WINDOWS windows of CEILING_MS"""
        xs = []
        for _ in range(CEILING_WINDOWS):
            r = gq.run_faa_ceiling(n_counters, per_lane=per_lane, threads=threads, warmup_ms=10, duration_ms=CEILING_MS)
            xs.append(r["succ_enq"] / r["meas_seconds"])
        return statistics.median(xs), min(xs), max(xs)

    c1_tps, c1_min, c1_max = ceiling(1)
    c4_tps, c4_min, c4_max = ceiling(4)
    c1l_tps, _, _ = ceiling(1, per_lane=True)
    peaks, peak_src = measured_peaks()
    ops_per_s_kernel = (ops_all / len(results)) / (kernel_ms * 1e-3)      # whole launch / event duration
    algo_gbps = ops_per_s_kernel * ALGO_BYTES_PER_OP[args.kind] / 1e9
    traffic, traffic_detail = None, None
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:      # written from the committed ncu captures
            traffic_detail = next(r for r in csv.DictReader(f) if r["kind"] == args.kind)
        traffic = float(traffic_detail["dram_bytes_per_launch"])   # dram__bytes_read.sum + dram__bytes_write.sum, one launch
    except Exception:
        pass
    roofline = {"bound": "l2_atomic", "achieved": ops_per_s_kernel / 1e9, "peak": 2 * c1_tps / 1e9, "unit": "Gop/s",
                "frac": ops_per_s_kernel / (2 * c1_tps), "traffic": traffic,
                "traffic_detail": traffic_detail, "traffic_note": "DRAM bytes of the committed ncu --set full capture of this kernel (fixed-op launch, "
                "profiles/r2_balanced_ncu_full.md): the rings are L2-resident, so DRAM sees the cold first touch only; L2 sector bytes per op beside it",
                "kernel": "gqk::bench_kernel", "kernel_ms": kernel_ms,
                "peak_source": "2 x C1; C1 = run_faa_ceiling(1 counter) at the same thread count, measured in this run (median of 5 x 100 ms)",
                "c1_gtickets_s": c1_tps / 1e9, "c1_min_max": [c1_min / 1e9, c1_max / 1e9],
                "c4_gtickets_s": c4_tps / 1e9, "c4_min_max": [c4_min / 1e9, c4_max / 1e9],
                "ceiling_protocol": f"median of {CEILING_WINDOWS} windows of {CEILING_MS:.0f} ms (10 ms warm-up each)",
                "c1_per_lane_faa_gtickets_s": c1l_tps / 1e9, "frac_of_c4_half": ops_per_s_kernel / (c4_tps / 2),
                "frac_min_max": [ops_per_s_kernel / (2 * c1_max), ops_per_s_kernel / (2 * c1_min)],
                "impl_extra_GBps": ops_per_s_kernel * IMPL_EXTRA_BYTES_PER_OP[args.kind] / 1e9,
                "index_cycle_us": (2.0 * CAPACITY / ops_per_s_kernel * 1e6) if threads > CAPACITY else None,
                "index_cycle_note": "k > n: the n indices each go FQ -> enqueuer -> AQ -> dequeuer -> FQ; ops/s = 2n / cycle (DESIGN.md section 5)",
                "algorithmic_GBps": algo_gbps, "hbm_peak_GBps": peaks["hbm_gbs"], "hbm_peak_source": peak_src,
                "hbm_frac": algo_gbps / peaks["hbm_gbs"]}

    # ---- BJ#3 (split, p = 0.5, n = 2^20 prefilled to 2^19) against the same ceiling: the metric names "balanced, split"
    roofline_split = None
    try:
        qs = gq.queue_create_ex(kind, 1 << 20, gq.gq_opts(ymc_pool_cells=YMC_POOL_CELLS))
        pre = np.arange(1 << 19, dtype=np.uint32)
        runs = {}
        for layout in (0, 1, 2):
            xs = []
            for _ in range(3):
                gq.queue_reset(qs)
                gq.queue_prefill(qs, pre)
                r = gq.run_split(qs, threads=threads, warmup_ms=WARMUP_MS, duration_ms=DURATION_MS, producer_fraction=0.5, seed=1,
                                 value_base=1 << 19, role_layout=layout, converged=CONVERGED)
                xs.append((r["succ_enq"] + r["succ_deq"]) / r["meas_seconds"])
            runs[layout] = xs
        gq.queue_destroy(qs)
        a0 = statistics.median(runs[0])
        roofline_split = {"bound": "l2_atomic", "achieved": a0 / 1e9, "peak": 2 * c1_tps / 1e9, "unit": "Gop/s", "frac": a0 / (2 * c1_tps),
                          "workload": "BJ#3 split, p = 0.5, capacity 2^20 prefilled 2^19, seeded Bernoulli roles (mixed warps), median of 3 x 100 ms",
                          "runs_gops": [round(x / 1e9, 2) for x in runs[0]],
                          "same_roles_on_homogeneous_warps_gops": [round(x / 1e9, 2) for x in runs[1]],
                          "mixed_warps_fused_step_gops": [round(x / 1e9, 2) for x in runs[2]],
                          "peak_mixed_warps": c1_tps / 1e9,
                          "frac_of_mixed_peak": a0 / c1_tps,
                          "note": "mixed warps: every WAVEFAA batch holds about 16 tickets instead of 32, so an operation costs the hot "
                                  "counters twice the atomics: their capacity allows 2 x C1 x 16/32 = C1 (peak_mixed_warps).  "
                                  "mixed_warps_fused_step_gops: the same roles through gq::enqueue_or_dequeue_step "
                                  "(gq_run_cfg.role_layout = 2, DESIGN.md D12)"}
    except gq.GqError as e:
        roofline_split = {"error": str(e)}

    # ---- thread sweep of BJ#2 and the producer-fraction sweep of BJ#3 (context, not timed)
    sweep = {}
    if not args.no_sweep:
        for name, k in KINDS.items():
            try:
                fk = gq.queue_max_coresident_threads(k, 256)
                qq = gq.queue_create_ex(k, CAPACITY, gq.gq_opts(ymc_pool_cells=YMC_POOL_CELLS))
            except gq.GqError as e:
                sweep["balanced_" + name] = str(e)
                continue
            pts = {}
            for th in (32, 256, 2048, 16384, 65536, fk):
                gq.queue_reset(qq)
                r = gq.run_balanced(qq, threads=th, warmup_ms=WARMUP_MS, duration_ms=DURATION_MS, fail_backoff_ns=args.fail_backoff_ns, converged=CONVERGED)
                pts[str(th)] = round(r["mops"], 1)
                if r["pool_exhausted"]:
                    pts[str(th) + "_pool_exhausted"] = True      # G-WFQ-YMC ran out of cells inside the run: the number is low
            gq.queue_destroy(qq)
            sweep["balanced_" + name] = pts
            try:
                qq = gq.queue_create_ex(k, 1 << 20, gq.gq_opts(ymc_pool_cells=YMC_POOL_CELLS))
                pre = np.arange(1 << 19, dtype=np.uint32)
                pts = {}
                for pf in (0.1, 0.25, 0.5, 0.75, 0.9):
                    gq.queue_reset(qq)
                    gq.queue_prefill(qq, pre)
                    r = gq.run_split(qq, threads=fk, warmup_ms=WARMUP_MS, duration_ms=DURATION_MS, producer_fraction=pf,
                                     seed=1, value_base=1 << 19, fail_backoff_ns=args.fail_backoff_ns, converged=CONVERGED)
                    pts[str(pf)] = {"enq_mops": round(r["succ_enq"] / r["meas_seconds"] / 1e6, 1),
                                    "deq_mops": round(r["succ_deq"] / r["meas_seconds"] / 1e6, 1),
                                    "full_rate": round(r["full"] / max(1, r["full"] + r["succ_enq"]), 4),
                                    "empty_rate": round(r["empty"] / max(1, r["empty"] + r["succ_deq"]), 4)}
                if name == "lfq":       # the same seeded roles placed on homogeneous warps (gq_run_cfg.role_layout = 1):
                    ptc = {}            # full-size WAVEFAA batches; context for the mixed-warp numbers above
                    for pf in (0.25, 0.5, 0.75):
                        gq.queue_reset(qq)
                        gq.queue_prefill(qq, pre)
                        r = gq.run_split(qq, threads=fk, warmup_ms=WARMUP_MS, duration_ms=DURATION_MS, producer_fraction=pf,
                                         seed=1, value_base=1 << 19, role_layout=1, converged=CONVERGED)
                        ptc[str(pf)] = {"enq_mops": round(r["succ_enq"] / r["meas_seconds"] / 1e6, 1),
                                        "deq_mops": round(r["succ_deq"] / r["meas_seconds"] / 1e6, 1)}
                    sweep["split_lfq_role_layout_1"] = ptc
                    ptf = {}            # mixed warps through the resumable fused operation (role_layout = 2, D12)
                    for pf in (0.1, 0.25, 0.5, 0.75, 0.9):
                        gq.queue_reset(qq)
                        gq.queue_prefill(qq, pre)
                        r = gq.run_split(qq, threads=fk, warmup_ms=WARMUP_MS, duration_ms=DURATION_MS, producer_fraction=pf,
                                         seed=1, value_base=1 << 19, role_layout=2, converged=CONVERGED)
                        ptf[str(pf)] = {"enq_mops": round(r["succ_enq"] / r["meas_seconds"] / 1e6, 1),
                                        "deq_mops": round(r["succ_deq"] / r["meas_seconds"] / 1e6, 1)}
                    sweep["split_lfq_role_layout_2"] = ptf
                gq.queue_destroy(qq)
                sweep["split_" + name] = pts
            except gq.GqError as e:
                sweep["split_" + name] = str(e)

    if not args.no_sweep:
        # capacity sweep at full co-residency (G-LFQ): for n < k the throughput is 2n / (index cycle), DESIGN.md section 5;
        # 5 runs per point: median, min, max (stability: the retry episodes and the two steady states of round 1)
        pts = {}
        for logn in (13, 14, 15, 16, 17, 18, 20):
            qq = gq.queue_create(0, 1 << logn)
            xs = []
            for _ in range(5):
                gq.queue_reset(qq)
                xs.append(gq.run_balanced(qq, threads=full, warmup_ms=WARMUP_MS, duration_ms=DURATION_MS, converged=CONVERGED)["mops"])
            gq.queue_destroy(qq)
            med = statistics.median(xs)
            pts[f"2^{logn}"] = {"mops": round(med, 1), "min": round(min(xs), 1), "max": round(max(xs), 1),
                                "index_cycle_us": round(2.0 * (1 << logn) / (med * 1e6) * 1e6, 2) if (1 << logn) < full else None}
        pts["note"] = "5 runs per point (median, min, max).  n < k: ops/s = 2n / index cycle; n >= 2^18 is bound by the four hot counters"
        sweep["capacity_lfq_full_coresidency"] = pts
        # ablations at the headline point: free-running lanes (converged = 0), block-level ticket funnels (D11)
        abl = {}
        for name, k, n, kw in (("lfq_n2^16_free_running_lanes", 0, CAPACITY, dict(converged=0)),
                               ("lfq_n2^20_free_running_lanes", 0, 1 << 20, dict(converged=0)),
                               ("lfq_n2^20_block_funnels", 0, 1 << 20, dict(converged=1, block_faa=1)),
                               ("ymc_n2^16_block_funnels_window_300ns", 2, CAPACITY, dict(converged=1, block_faa=1, funnel_window_ns=300))):
            qq = gq.queue_create_ex(k, n, gq.gq_opts(ymc_pool_cells=YMC_POOL_CELLS))
            xs = []
            for _ in range(3):
                gq.queue_reset(qq)
                xs.append(gq.run_balanced(qq, threads=full if k == 0 else gq.queue_max_coresident_threads(k, 256), warmup_ms=WARMUP_MS, duration_ms=DURATION_MS, **kw)["mops"])
            gq.queue_destroy(qq)
            abl[name] = {"mops": round(statistics.median(xs), 1), "min": round(min(xs), 1), "max": round(max(xs), 1)}
        sweep["ablations"] = abl

    apps = None
    if args.apps:
        apps = run_apps(gq, torch, args.apps_scale)

    # ---- CPU baseline: the oracle, as it stands, on this box's host cores (bounded sample)
    import oracle
    cores = oracle.hw_threads()
    best = None
    tcount = 1
    cand = []
    while tcount < cores:
        cand.append(tcount); tcount *= 2
    cand.append(cores)
    for t in cand:
        rs = [oracle.mutex_bench("balanced", t, CAPACITY, warmup_ms=WARMUP_MS, duration_ms=DURATION_MS)["mops"] for _ in range(3)]
        m = statistics.median(rs)
        if best is None or m > best[0]:
            best = (m, t)
    cpu_baseline = {"value": best[0], "unit": "Mops/s", "cores": best[1], "kind": "oracle", "host_cores": cores,
                    "sample": f"std::mutex+std::deque, balanced loop, capacity 2^16, 20+100 ms x 3 (median) at threads {cand}; best shown"}

    line = {
        "metric": "queue Mops/s (balanced)", "value": value, "unit": "Mops/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": wall_max / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u64", "data": "synthetic",
        "config": {"workload": f"BJ#2 balanced fixed-duration: {args.kind} capacity 2^16 uint32, {threads} threads "
                               f"(full co-residency = {full}), block 256, 20 ms warmup + 100 ms window per step, lanes of a warp start each iteration together",
                   "kind": args.kind, "threads": threads, "capacity": CAPACITY, "fail_backoff_ns": args.fail_backoff_ns, "converged": CONVERGED,
                   "l2": "256 MiB device buffer written between steps (L2 flush); rings are L2-resident by design",
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "e2e": {"value": e2e_ops_all / e2e_wall_max / 1e6, "unit": "Mops/s", "h2d_bytes_per_step": 64,   # the gq_run_cfg struct
                "d2h_bytes_per_step": 128 + 8 + 4 * (e2e_drained // args.steps),
                "what": "queue_reset + run_balanced + queue_drain(host array) per step; all successful ops of the launch / host wall time"},
        "gpu_launches": args.steps * 3,      # per step: 2 format kernels (queue_reset) + 1 bench kernel
        "clocks": clocks, "roofline": roofline, "roofline_split": roofline_split, "cpu_baseline": cpu_baseline, "sweep": sweep,
        "reference_arm_note": "--impl reference runs the mutex oracle on ALL host threads (contended: a few Mops/s); its best point is 1 thread "
                              "(cpu_baseline.value), so the driver's ours/reference ratio is several times larger than value / cpu_baseline.value",
        "conservation": "checked every e2e step: tot_enq - tot_deq == drained",
        # P:L359 protocol ("5 runs, median"): the timed steps one by one (rank 0's replica) and their median
        "per_step_mops": [round((r["succ_enq"] + r["succ_deq"]) / (DURATION_MS * 1e-3) / 1e6, 1) for r in results],
        "median_step_mops": round(statistics.median((r["succ_enq"] + r["succ_deq"]) / (DURATION_MS * 1e-3) / 1e6 for r in results), 1),
    }
    if apps is not None:
        line["apps"] = apps
    print(json.dumps(line), flush=True)
    gq.queue_destroy(q)
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--kind", default="lfq", choices=list(KINDS))
    ap.add_argument("--threads", type=int, default=0, help="0 = full co-residency")
    ap.add_argument("--fail-backoff-ns", type=int, default=0)
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--apps", action="store_true", help="also run BASELINE.json configs 4/5 (BFS, path tracer) against the oracle; adds minutes of host time")
    ap.add_argument("--apps-scale", type=int, default=22, help="R-MAT scale of the BFS graph (BASELINE.json: 22)")
    args = ap.parse_args()
    rank, world, local_rank = env_int("RANK", 0), env_int("WORLD_SIZE", 1), env_int("LOCAL_RANK", 0)
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
