"""Fixed-op-count run of the balanced / split kernel for ncu (every replay pass does the same
work, unlike the time-terminated benchmark).  Prints the kernel's own counters so that
ncu metrics can be normalised per successful op (instr/op, stall/op; Tables II-III).

  python -m paper_2606_01693_b200.profile_run --kind lfq --threads 65536 --capacity 65536 --ops 64
"""
import argparse
import json

import numpy as np

from . import (GQ_LFQ, GQ_LFQ_DIRECT, GQ_WFQ, GQ_WFQ_YMC, gq_opts, queue_create_ex, queue_destroy, queue_drain, queue_prefill,
               run_balanced, run_split)

KINDS = {"lfq": GQ_LFQ, "wfq": GQ_WFQ, "ymc": GQ_WFQ_YMC, "lfq_direct": GQ_LFQ_DIRECT}


def run_app(a):
    """One launch of an application driver on its BASELINE.json recipe (for ncu -k regex:bfs_kernel|rt_kernel)."""
    import torch
    from . import bfs_run, inputs, rt_render
    if a.mode == "bfs":
        rowptr, col, src = inputs.rmat_csr(a.scale, 16, seed=1)
        nv = len(rowptr) - 1
        d_rowptr = torch.from_numpy(rowptr.view(np.int64)).cuda()
        d_col = torch.from_numpy(col.view(np.int32)).cuda()
        d_dist = torch.empty(nv, dtype=torch.int32, device="cuda")
        st = bfs_run(KINDS[a.kind], d_rowptr.data_ptr(), d_col.data_ptr(), nv, src, d_dist.data_ptr())
        torch.cuda.synchronize()
        st["reached"] = int((d_dist >= 0).sum().item())
    else:
        sph = inputs.sphere_scene(256, seed=1)
        d_sph = torch.from_numpy(np.ascontiguousarray(sph, np.float32)).cuda()
        d_rgb = torch.empty((1080, 1920, 3), dtype=torch.float32, device="cuda")
        st = rt_render(KINDS[a.kind], 1920, 1080, 4, 4, len(sph), d_sph.data_ptr(), 1, d_rgb.data_ptr())
        torch.cuda.synchronize()
    print(json.dumps({"args": vars(a), "result": st}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--kind", default="lfq", choices=list(KINDS))
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--capacity", type=int, default=1 << 16)
    ap.add_argument("--ops", type=int, default=64)
    ap.add_argument("--mode", default="balanced", choices=["balanced", "split", "bfs", "rt"])
    ap.add_argument("--scale", type=int, default=20, help="bfs: R-MAT scale")
    ap.add_argument("--producer-fraction", type=float, default=0.5)
    ap.add_argument("--flags", type=int, default=0)
    ap.add_argument("--layout", type=int, default=0)
    ap.add_argument("--fail-backoff-ns", type=int, default=0)
    ap.add_argument("--pool-cells", type=int, default=0)
    ap.add_argument("--converged", type=int, default=1, help="gq_run_cfg.converged (1 = what bench.py runs)")
    ap.add_argument("--role-layout", type=int, default=0, help="split: gq_run_cfg.role_layout")
    a = ap.parse_args()
    if a.mode in ("bfs", "rt"):
        return run_app(a)
    q = queue_create_ex(KINDS[a.kind], a.capacity, gq_opts(flags=a.flags, layout=a.layout, ymc_pool_cells=a.pool_cells))
    try:
        if a.mode == "split":
            queue_prefill(q, np.arange(a.capacity // 2, dtype=np.uint32))
            r = run_split(q, threads=a.threads, ops_per_thread=a.ops, producer_fraction=a.producer_fraction, seed=1,
                          value_base=a.capacity // 2, fail_backoff_ns=a.fail_backoff_ns, converged=a.converged, role_layout=a.role_layout)
        else:
            r = run_balanced(q, threads=a.threads, ops_per_thread=a.ops, fail_backoff_ns=a.fail_backoff_ns, converged=a.converged)
        left = queue_drain(q, a.capacity + 1)
    finally:
        queue_destroy(q)
    r["succ_ops"] = r["tot_enq"] + r["tot_deq"]
    r["drained"] = len(left)
    r["mops_fixed"] = r["succ_ops"] / (r["kernel_ms"] * 1e-3) / 1e6
    print(json.dumps({"args": vars(a), "result": r}))


if __name__ == "__main__":
    main()
