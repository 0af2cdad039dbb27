"""paper_2606_01693_b200 — thin Python binding of libgq.so (include/gq.h).

Argument marshalling only: every step of the queue path runs in the library's CUDA kernels.
There is no CPU fallback; if libgq.so cannot be loaded, importing this package fails, and
on a box without a CUDA device every compute call raises GqError(GQ_E_CUDA).
The names are those of the C ABI.
"""
import ctypes as C
import os

import numpy as np

import contextlib

from .build import LIB, build as _build

GQ_LFQ, GQ_WFQ, GQ_WFQ_YMC, GQ_LFQ_DIRECT = 0, 1, 2, 3
GQ_OK, GQ_FULL, GQ_EMPTY = 0, 1, 2
GQ_OP_ENQ, GQ_OP_DEQ = 0, 1
GQ_E_INVAL, GQ_E_NOMEM, GQ_E_CUDA, GQ_E_RESIDENCY, GQ_E_TIMEOUT, GQ_E_STATE, GQ_E_POOL = -1, -2, -3, -4, -5, -6, -7
GQ_PATIENCE_ZERO = 0xFFFFFFFF
GQ_F_PER_LANE_FAA, GQ_F_NO_PROBE, GQ_F_NO_DEQ_SPIN, GQ_F_NO_OPT_CAS, GQ_F_PLAIN_THR_STORE = 1, 2, 4, 8, 16
GQ_F_THR_FIRST, GQ_F_NO_PAIRED_FAA, GQ_F_THR_RED_MAX, GQ_F_FENCED_PAYLOAD, GQ_F_EAGER_EMPTY, GQ_F_NO_CELL_PREFETCH, GQ_F_NO_FULL_TEST = 32, 64, 128, 256, 512, 1024, 2048
GQ_F_NO_REPAIR = 4096
GQ_PARK_SPIN_NONE = 0xFFFFFFFF
KIND_NAMES = {GQ_LFQ: "G-LFQ", GQ_WFQ: "G-WFQ", GQ_WFQ_YMC: "G-WFQ-YMC", GQ_LFQ_DIRECT: "G-LFQ-D"}
_ERR = {-1: "INVAL", -2: "NOMEM", -3: "CUDA", -4: "RESIDENCY", -5: "TIMEOUT", -6: "STATE", -7: "POOL"}


TIMED_OUT = False      # set once a call returned GQ_E_TIMEOUT: the kernel is still running, every later CUDA call would block on it


class GqError(RuntimeError):
    def __init__(self, code, where):
        global TIMED_OUT
        self.code = code
        if code == GQ_E_TIMEOUT:
            TIMED_OUT = True
            if os.environ.get("GQ_EXIT_ON_TIMEOUT"):      # test runs: every later CUDA call (frees included) would block on the stuck kernel
                os.write(2, f"\n[gq] {where}: watchdog time-out, kernel still running; exiting (GQ_EXIT_ON_TIMEOUT)\n".encode())
                os._exit(3)
        detail = lib.gq_last_cuda_error().decode() if code in (GQ_E_CUDA, GQ_E_TIMEOUT, GQ_E_NOMEM) or where == "queue_drain_noalloc" else ""
        super().__init__(f"{where}: GQ_E_{_ERR.get(code, code)} {detail}".strip())


class gq_opts(C.Structure):
    _fields_ = [("max_threads", C.c_uint32), ("enq_patience", C.c_uint32), ("deq_patience", C.c_uint32),
                ("help_delay", C.c_uint32), ("ymc_pool_cells", C.c_uint64), ("storage", C.c_void_p),
                ("storage_bytes", C.c_size_t), ("layout", C.c_uint32), ("flags", C.c_uint32),
                ("park_ns", C.c_uint32), ("park_nap_ns", C.c_uint32), ("park_spin_ns", C.c_uint32), ("reserved", C.c_uint32)]


class gq_run_cfg(C.Structure):
    _fields_ = [("threads", C.c_uint32), ("block_threads", C.c_uint32), ("warmup_ms", C.c_double),
                ("duration_ms", C.c_double), ("producer_fraction", C.c_double), ("seed", C.c_uint64),
                ("record_history", C.c_uint32), ("ops_per_thread", C.c_uint32), ("jitter_ns", C.c_uint32),
                ("fail_backoff_ns", C.c_uint32), ("value_base", C.c_uint64),
                ("role_layout", C.c_uint32), ("converged", C.c_uint32), ("block_faa", C.c_uint32), ("funnel_window_ns", C.c_uint32)]


class gq_run_result(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in ("succ_enq", "succ_deq", "full", "empty", "tot_enq", "tot_deq", "tot_full",
                                           "tot_empty", "sum_enq", "sum_deq", "slow_enq", "slow_deq", "helps", "retries")] + \
               [("meas_seconds", C.c_double), ("kernel_ms", C.c_double), ("threads_launched", C.c_uint32),
                ("blocks", C.c_uint32), ("blocks_per_sm", C.c_uint32), ("pool_exhausted", C.c_uint32)]

    def asdict(self):
        d = {n: getattr(self, n) for n, _ in self._fields_}
        d["mops"] = (self.succ_enq + self.succ_deq) / self.meas_seconds / 1e6 if self.meas_seconds > 0 else 0.0
        return d


class gq_bfs_stats(C.Structure):
    _fields_ = [("levels", C.c_uint32), ("threads", C.c_uint32), ("edges_scanned", C.c_uint64),
                ("vertices_visited", C.c_uint64), ("queue_ops", C.c_uint64), ("ms", C.c_double), ("total_ms", C.c_double)]


class gq_bfs_opts(C.Structure):
    _fields_ = [("threads", C.c_uint32), ("block_threads", C.c_uint32), ("huge_degree", C.c_uint32), ("flags", C.c_uint32)]


class gq_rt_scene(C.Structure):
    _fields_ = [("width", C.c_uint32), ("height", C.c_uint32), ("spp", C.c_uint32), ("max_bounce", C.c_uint32),
                ("n_spheres", C.c_uint32), ("threads", C.c_uint32), ("seed", C.c_uint64), ("d_spheres", C.c_void_p)]


class gq_rt_opts(C.Structure):
    _fields_ = [("mode", C.c_uint32), ("reserved", C.c_uint32)]


class gq_rt_stats(C.Structure):
    _fields_ = [("rays", C.c_uint64), ("queue_ops", C.c_uint64), ("ms", C.c_double), ("total_ms", C.c_double),
                ("threads", C.c_uint32), ("items", C.c_uint32)]


HIST_DTYPE = np.dtype([("proc", "<u4"), ("op", "<u4"), ("arg", "<u4"), ("ret_status", "<u4"), ("ret_val", "<u4"),
                       ("_pad", "<u4"), ("call_ns", "<u8"), ("end_ns", "<u8")])

# every symbol include/gq.h declares
SYMBOLS = ("queue_storage_bytes", "queue_create", "queue_create_ex", "queue_destroy", "queue_reset", "queue_prefill",
           "queue_drain", "queue_drain_noalloc", "queue_device_view", "queue_kind", "queue_max_coresident_threads", "run_balanced",
           "run_split", "run_faa_ceiling", "run_slot_atomic_ceiling", "run_warp_faa_probe", "run_funnel_probe", "queue_run_script",
           "history_dump", "bfs_run", "bfs_run_ex", "rt_render", "rt_render_ex", "gq_last_cuda_error", "gq_version",
           "gq_dbg_sites", "gq_dbg_trace", "gq_set_mutation", "queue_debug_counters")


def _load(variant=""):
    path = _build(variant=variant)          # compiles with nvcc when sources are newer than the .so
    L = C.CDLL(path)
    P = C.POINTER
    L.queue_storage_bytes.argtypes = [C.c_int, C.c_uint64, P(gq_opts)]
    L.queue_storage_bytes.restype = C.c_size_t
    L.queue_create.argtypes = [C.c_int, C.c_uint64, P(C.c_void_p)]
    L.queue_create_ex.argtypes = [C.c_int, C.c_uint64, P(gq_opts), P(C.c_void_p)]
    L.queue_destroy.argtypes = [C.c_void_p]
    L.queue_reset.argtypes = [C.c_void_p, C.c_void_p]
    L.queue_prefill.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]
    L.queue_drain.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, P(C.c_uint64), C.c_void_p]
    L.queue_drain_noalloc.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, P(C.c_uint64), C.c_void_p]
    L.queue_device_view.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t]
    L.queue_kind.argtypes = [C.c_void_p]
    L.queue_debug_counters.argtypes = [C.c_void_p, C.c_void_p]
    L.queue_max_coresident_threads.argtypes = [C.c_int, C.c_int, P(C.c_uint32)]
    L.run_balanced.argtypes = [C.c_void_p, P(gq_run_cfg), P(gq_run_result)]
    L.run_split.argtypes = [C.c_void_p, P(gq_run_cfg), P(gq_run_result)]
    L.run_faa_ceiling.argtypes = [P(gq_run_cfg), C.c_uint32, P(gq_run_result)]
    L.run_slot_atomic_ceiling.argtypes = [P(gq_run_cfg), C.c_uint64, P(gq_run_result)]
    L.run_warp_faa_probe.argtypes = [C.c_uint32, C.c_uint32, C.c_uint64, C.c_void_p, P(C.c_uint64)]
    L.run_funnel_probe.argtypes = [C.c_uint32, C.c_uint32, C.c_uint64, C.c_uint32, C.c_void_p, P(C.c_uint64), C.c_void_p]
    L.queue_run_script.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32, C.c_void_p, C.c_void_p]
    L.history_dump.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, P(C.c_uint64)]
    L.bfs_run.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_uint32, C.c_uint32, C.c_void_p, P(gq_bfs_stats), C.c_void_p]
    L.bfs_run_ex.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_uint32, C.c_uint32, C.c_void_p, P(gq_bfs_opts), P(gq_bfs_stats), C.c_void_p]
    L.rt_render.argtypes = [C.c_int, P(gq_rt_scene), C.c_void_p, P(gq_rt_stats), C.c_void_p]
    L.rt_render_ex.argtypes = [C.c_int, P(gq_rt_scene), C.c_void_p, P(gq_rt_opts), P(gq_rt_stats), C.c_void_p]
    L.gq_last_cuda_error.restype = C.c_char_p
    L.gq_version.restype = C.c_char_p
    L.gq_dbg_sites.argtypes = [C.c_void_p]
    L.gq_dbg_trace.argtypes = [C.c_void_p, C.c_uint64, P(C.c_uint64)]
    L.gq_set_mutation.argtypes = [C.c_uint32]
    return L


lib = _load()


@contextlib.contextmanager
def use_variant(variant):
    """Route every call of this module to another build of the same library (build.py VARIANTS: "mutants", "dbg")
    for the duration of the block.  Handles must not cross the boundary."""
    global lib
    saved, lib = lib, _load(variant)
    try:
        yield lib
    finally:
        lib = saved


def _chk(rc, where):
    if rc != 0:
        raise GqError(rc, where)


def _np_ptr(a):
    return a.ctypes.data_as(C.c_void_p)


# ------------------------------------------------------------------ same names as the C ABI
def queue_storage_bytes(kind, capacity, opts=None):
    return lib.queue_storage_bytes(kind, capacity, C.byref(opts) if opts is not None else None)


def queue_create(kind, capacity):
    h = C.c_void_p()
    _chk(lib.queue_create(kind, capacity, C.byref(h)), "queue_create")
    return h


def queue_create_ex(kind, capacity, opts):
    h = C.c_void_p()
    _chk(lib.queue_create_ex(kind, capacity, C.byref(opts), C.byref(h)), "queue_create_ex")
    return h


def queue_destroy(q):
    _chk(lib.queue_destroy(q), "queue_destroy")


def queue_reset(q, stream=None):
    _chk(lib.queue_reset(q, stream), "queue_reset")


def queue_prefill(q, host_vals, stream=None):
    a = np.ascontiguousarray(host_vals, np.uint32)
    _chk(lib.queue_prefill(q, _np_ptr(a), len(a), stream), "queue_prefill")


def queue_drain(q, max_items, stream=None):
    out = np.empty(max(int(max_items), 1), np.uint32)
    n = C.c_uint64(0)
    _chk(lib.queue_drain(q, _np_ptr(out), int(max_items), C.byref(n), stream), "queue_drain")
    return out[: n.value].copy()


GQ_DRAIN_NOALLOC_MAX = 65536


def queue_drain_noalloc(q, max_items, stream=None):
    """queue_drain without any device allocation (static scratch inside the library); max_items <= GQ_DRAIN_NOALLOC_MAX."""
    out = np.empty(max(int(max_items), 1), np.uint32)
    n = C.c_uint64(0)
    _chk(lib.queue_drain_noalloc(q, _np_ptr(out), int(max_items), C.byref(n), stream), "queue_drain_noalloc")
    return out[: n.value].copy()


def queue_device_view(q):
    """The POD device view (gq::LfqView / WfqView / YmcView / DlfqView) as bytes, to hand to a user kernel by value."""
    buf = C.create_string_buffer(512)
    _chk(lib.queue_device_view(q, buf, 512), "queue_device_view")
    return buf.raw


def queue_debug_counters(q):
    """dict of the hot words of a quiescent queue (gq.h)."""
    out = np.zeros(16, np.uint64)
    _chk(lib.queue_debug_counters(q, _np_ptr(out)), "queue_debug_counters")
    k = lib.queue_kind(q)
    if k == GQ_WFQ_YMC:
        return {"head": int(out[0]), "tail": int(out[1]), "N": int(out[6]), "max_threads": int(out[7])}
    d = {"aq_head": int(out[0]), "aq_tail": int(out[1]), "aq_threshold": int(out[2].astype(np.int64)), "N": int(out[6]), "max_threads": int(out[7])}
    if k != GQ_LFQ_DIRECT:
        d.update(fq_head=int(out[3]), fq_tail=int(out[4]), fq_threshold=int(out[5].astype(np.int64)))
    if k == GQ_WFQ:
        names = ("tail_inc", "tail_clr", "head_inc", "head_clr")
        d.update({f"aq_{n}": int(out[8 + i]) for i, n in enumerate(names)})
        d.update({f"fq_{n}": int(out[12 + i]) for i, n in enumerate(names)})
    return d


def queue_max_coresident_threads(kind, block_threads=256):
    out = C.c_uint32(0)
    _chk(lib.queue_max_coresident_threads(kind, block_threads, C.byref(out)), "queue_max_coresident_threads")
    return out.value


def _cfg(**kw):
    cfg = gq_run_cfg()
    for k, v in kw.items():
        setattr(cfg, k, v)
    return cfg


def run_balanced(q, **kw):
    res = gq_run_result()
    rc = lib.run_balanced(q, C.byref(_cfg(**kw)), C.byref(res))
    if rc not in (0, GQ_E_POOL):
        raise GqError(rc, "run_balanced")
    return res.asdict()


def run_split(q, **kw):
    res = gq_run_result()
    rc = lib.run_split(q, C.byref(_cfg(**kw)), C.byref(res))
    if rc not in (0, GQ_E_POOL):
        raise GqError(rc, "run_split")
    return res.asdict()


GQ_CEILING_PER_LANE = 0x100


def run_faa_ceiling(n_counters=1, per_lane=False, **kw):
    res = gq_run_result()
    _chk(lib.run_faa_ceiling(C.byref(_cfg(**kw)), n_counters | (GQ_CEILING_PER_LANE if per_lane else 0), C.byref(res)), "run_faa_ceiling")
    return res.asdict()


def run_slot_atomic_ceiling(slots, **kw):
    res = gq_run_result()
    _chk(lib.run_slot_atomic_ceiling(C.byref(_cfg(**kw)), slots, C.byref(res)), "run_slot_atomic_ceiling")
    return res.asdict()


def run_warp_faa_probe(threads, rounds, seed):
    t = np.empty(threads * rounds, np.uint64)
    fin = C.c_uint64(0)
    _chk(lib.run_warp_faa_probe(threads, rounds, seed, _np_ptr(t), C.byref(fin)), "run_warp_faa_probe")
    return t.reshape(threads, rounds), fin.value


def run_funnel_probe(threads, rounds, seed, window_ns=0, keep_tickets=True):
    """(tickets or None, final counter, sum of tickets, number of tickets)"""
    t = np.empty(threads * rounds, np.uint64) if keep_tickets else None
    fin = C.c_uint64(0)
    sc = np.zeros(2, np.uint64)
    _chk(lib.run_funnel_probe(threads, rounds, seed, window_ns, _np_ptr(t) if keep_tickets else None, C.byref(fin), _np_ptr(sc)), "run_funnel_probe")
    return (t.reshape(threads, rounds) if keep_tickets else None), fin.value, int(sc[0]), int(sc[1])


def queue_run_script(q, ops, args, tid=0):
    ops = np.ascontiguousarray(ops, np.uint32)
    args = np.ascontiguousarray(args, np.uint32)
    st = np.empty(len(ops), np.uint32)
    val = np.empty(len(ops), np.uint32)
    _chk(lib.queue_run_script(q, _np_ptr(ops), _np_ptr(args), len(ops), tid, _np_ptr(st), _np_ptr(val)), "queue_run_script")
    return st, val


def history_dump(q, max_records=1 << 24):
    out = np.empty(max_records, HIST_DTYPE)
    n = C.c_uint64(0)
    _chk(lib.history_dump(q, _np_ptr(out), max_records, C.byref(n)), "history_dump")
    return out[: n.value].copy()


TRACE_DTYPE = np.dtype([("ns", "<u8"), ("site_tid", "<u8"), ("ticket", "<u8"), ("entry", "<u8"), ("head", "<u8"),
                        ("tail", "<u8"), ("thr", "<i8"), ("aux", "<u8")])


def gq_dbg_sites():
    out = np.zeros(80, np.uint64)
    _chk(lib.gq_dbg_sites(_np_ptr(out)), "gq_dbg_sites")
    return out


def gq_dbg_trace(max_records=1 << 16):
    out = np.empty(max_records, TRACE_DTYPE)
    n = C.c_uint64(0)
    _chk(lib.gq_dbg_trace(_np_ptr(out), max_records, C.byref(n)), "gq_dbg_trace")
    return out[: n.value].copy()


def gq_set_mutation(mutation_id):
    _chk(lib.gq_set_mutation(mutation_id), "gq_set_mutation")


def bfs_run(kind, d_rowptr, d_col, nv, src, d_dist, stream=None):
    """d_* are device pointers (ints), e.g. torch_tensor.data_ptr()."""
    st = gq_bfs_stats()
    _chk(lib.bfs_run(kind, d_rowptr, d_col, nv, src, d_dist, C.byref(st), stream), "bfs_run")
    return {n: getattr(st, n) for n, _ in st._fields_}


def bfs_run_ex(kind, d_rowptr, d_col, nv, src, d_dist, stream=None, **opts):
    st = gq_bfs_stats()
    _chk(lib.bfs_run_ex(kind, d_rowptr, d_col, nv, src, d_dist, C.byref(gq_bfs_opts(**opts)), C.byref(st), stream), "bfs_run_ex")
    return {n: getattr(st, n) for n, _ in st._fields_}


def rt_render(kind, width, height, spp, max_bounce, n_spheres, d_spheres, seed, d_rgb, threads=0, stream=None, mode=0):
    """mode 0: one work queue of tile items (rt_render); mode 1: one queue per tile, items are rays (rt_render_ex)."""
    sc = gq_rt_scene(width, height, spp, max_bounce, n_spheres, threads, seed, d_spheres)
    st = gq_rt_stats()
    if mode:
        _chk(lib.rt_render_ex(kind, C.byref(sc), d_rgb, C.byref(gq_rt_opts(mode, 0)), C.byref(st), stream), "rt_render_ex")
    else:
        _chk(lib.rt_render(kind, C.byref(sc), d_rgb, C.byref(st), stream), "rt_render")
    return {n: getattr(st, n) for n, _ in st._fields_}
