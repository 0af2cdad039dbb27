"""ORACLE — TEST INFRASTRUCTURE ONLY.

A plain, slow, obviously-correct CPU statement of what the queue library must compute,
written from PAPER.md before any kernel and sharing no code with the CUDA path:

  (a) sequential bounded-FIFO model            fifo_model.hpp
  (b) linearizability checkers over histories  lincheck.cpp
  (c) std::mutex + std::deque baseline         mutex_queue.cpp
  (+) CPU BFS and CPU ray tracer               apps_cpu.cpp

Only tests/, __graft_entry__.smoke() and bench.py (cpu_baseline / --impl reference) may
import this package.  The product package never does.

Parity pins: every function here is pinned by tests/test_oracle_*.py (brute force on tiny
inputs, hand-written textbook histories, closed forms, cross-agreement of independent
deciders).  Absolute throughput of the mutex baseline is "parity unpinned" by nature (it is
a timing, not a value).
"""
import ctypes as C
import os

import numpy as np

from .build import build as _build

_lib = None

LIN_OK, LIN_VIOLATION, LIN_UNKNOWN, LIN_MALFORMED = 1, 0, -1, -2
ST_OK, ST_FULL, ST_EMPTY = 0, 1, 2
OP_ENQ, OP_DEQ = 0, 1

_u32p = np.ctypeslib.ndpointer(np.uint32, flags="C_CONTIGUOUS")
_u64p = np.ctypeslib.ndpointer(np.uint64, flags="C_CONTIGUOUS")
_HIST = [C.c_uint64, _u32p, _u32p, _u32p, _u32p, _u32p, _u64p, _u64p]


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        L.orc_fifo_replay.argtypes = [C.c_uint64, C.c_uint64, _u32p, _u32p, _u32p, _u32p]
        L.orc_fifo_replay.restype = None
        L.orc_precheck.argtypes = _HIST + [C.c_char_p, C.c_uint64]
        L.orc_brute.argtypes = _HIST + [C.c_uint64, C.c_int]
        L.orc_wgl.argtypes = _HIST + [C.c_uint64, C.c_int, C.c_uint64, C.POINTER(C.c_uint64)]
        L.orc_poly.argtypes = _HIST + [C.c_char_p, C.c_uint64]
        L.orc_capacity.argtypes = _HIST + [C.c_uint64, C.c_char_p, C.c_uint64]
        L.orc_conservation.argtypes = _HIST + [_u32p, C.c_uint64, C.c_char_p, C.c_uint64]
        L.orc_mutex_bench.argtypes = [C.c_int, C.c_uint32, C.c_uint64, C.c_uint64, C.c_double, C.c_uint64,
                                      C.c_double, C.c_double, _u64p, C.POINTER(C.c_double)]
        L.orc_mutex_bench.restype = None
        L.orc_hw_threads.restype = C.c_uint32
        if hasattr(L, "orc_bfs"):
            L.orc_bfs.argtypes = [C.c_uint32, _u64p, _u32p, C.c_uint32,
                                  np.ctypeslib.ndpointer(np.int32, flags="C_CONTIGUOUS"), C.POINTER(C.c_uint64)]
            L.orc_bfs.restype = None
        if hasattr(L, "orc_rt_render"):
            _f32p = np.ctypeslib.ndpointer(np.float32, flags="C_CONTIGUOUS")
            L.orc_rt_render.argtypes = [C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, _f32p,
                                        C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, _f32p, C.POINTER(C.c_uint64)]
            L.orc_rt_render.restype = None
            L.orc_rt_fmix32.argtypes = [C.c_uint32]
            L.orc_rt_fmix32.restype = C.c_uint32
            L.orc_rt_rnd.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32]
            L.orc_rt_rnd.restype = C.c_float
            L.orc_rt_camera_ray.argtypes = [C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_float, C.c_float, _f32p]
            L.orc_rt_camera_ray.restype = None
            L.orc_rt_nearest_hit.argtypes = [C.c_uint32, _f32p, _f32p, _f32p, C.POINTER(C.c_float)]
            L.orc_rt_nearest_hit.restype = C.c_int
            L.orc_rt_scatter.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, _f32p, _f32p]
            L.orc_rt_scatter.restype = None
        _lib = L
    return _lib


class History:
    """Columnar history {proc, op, arg, status, val, call, end}."""

    FIELDS = ("proc", "op", "arg", "status", "val", "call", "end")

    def __init__(self, proc, op, arg, status, val, call, end):
        self.proc = np.ascontiguousarray(proc, np.uint32)
        self.op = np.ascontiguousarray(op, np.uint32)
        self.arg = np.ascontiguousarray(arg, np.uint32)
        self.status = np.ascontiguousarray(status, np.uint32)
        self.val = np.ascontiguousarray(val, np.uint32)
        self.call = np.ascontiguousarray(call, np.uint64)
        self.end = np.ascontiguousarray(end, np.uint64)

    @classmethod
    def from_rows(cls, rows):
        """rows: iterable of (proc, op, arg, status, val, call, end)."""
        rows = list(rows)
        cols = list(zip(*rows)) if rows else [[] for _ in range(7)]
        return cls(*cols)

    def __len__(self):
        return len(self.proc)

    def _args(self):
        return (len(self), self.proc, self.op, self.arg, self.status, self.val, self.call, self.end)


def fifo_replay(capacity, ops, args):
    """Run a sequential script on the model; returns (status[], val[])."""
    ops = np.ascontiguousarray(ops, np.uint32)
    args = np.ascontiguousarray(args, np.uint32)
    st = np.zeros(len(ops), np.uint32)
    val = np.zeros(len(ops), np.uint32)
    lib().orc_fifo_replay(int(capacity), len(ops), ops, args, st, val)
    return st, val


def precheck(h: History) -> str:
    buf = C.create_string_buffer(512)
    lib().orc_precheck(*h._args(), buf, 512)
    return buf.value.decode()


def brute(h: History, capacity, relaxed_full=False) -> int:
    return lib().orc_brute(*h._args(), int(capacity), int(relaxed_full))


def wgl(h: History, capacity, relaxed_full=False, max_steps=50_000_000):
    steps = C.c_uint64(0)
    r = lib().orc_wgl(*h._args(), int(capacity), int(relaxed_full), int(max_steps), C.byref(steps))
    return r, steps.value


def poly(h: History):
    buf = C.create_string_buffer(512)
    r = lib().orc_poly(*h._args(), buf, 512)
    return r, buf.value.decode()


def conservation(h: History, leftover=()) -> str:
    left = np.ascontiguousarray(np.asarray(leftover, dtype=np.uint32))
    buf = C.create_string_buffer(512)
    lib().orc_conservation(*h._args(), left, len(left), buf, 512)
    return buf.value.decode()


def capacity_bound(h: History, capacity) -> str:
    buf = C.create_string_buffer(512)
    lib().orc_capacity(*h._args(), int(capacity), buf, 512)
    return buf.value.decode()


def check_history(h: History, capacity, relaxed_full=True, leftover=(), max_steps=50_000_000, accept_unknown=False,
                  soft_slack=0):
    """The full pipeline of PAPER.md §IV: structural checks, token protocol (L336), the
    bad-pattern characterisation (exact for OK/EMPTY returns of the unbounded FIFO), the capacity
    lower bound, then the exact WGL search against the bounded model (L335).  Returns (ok, msg).

    accept_unknown: when the exact search runs out of budget (histories with ~64-way overlap and
    many FULL/EMPTY returns), accept on the polynomial checks alone and say so in msg.  What is
    then NOT established exactly is only the interplay of FULL returns / the capacity bound with
    the order; FIFO order, EMPTY soundness, conservation and the capacity lower bound are.

    soft_slack > 0: the direct-payload ablation queue (lincheck.hpp, relaxed_full == 2): ENQ->OK
    legal while |S| < n + c_i, and the capacity lower bound is checked against n + soft_slack."""
    msg = precheck(h)
    if msg:
        return False, "precheck: " + msg
    msg = conservation(h, leftover)
    if msg:
        return False, "conservation: " + msg
    r, why = poly(h)
    if r != LIN_OK:
        return False, "poly: " + why
    msg = capacity_bound(h, capacity + int(soft_slack))
    if msg:
        return False, msg
    r, steps = wgl(h, capacity, 2 if soft_slack else relaxed_full, max_steps)
    if r == LIN_OK:
        return True, f"linearizable ({steps} WGL steps)"
    if r == LIN_UNKNOWN:
        if accept_unknown:
            return True, f"bad-pattern + capacity checks pass; exact search undecided after {steps} steps"
        return False, f"WGL budget exhausted after {steps} steps"
    return False, f"WGL: not linearizable ({steps} steps)"


def mutex_bench(mode, threads, capacity, prefill=0, producer_fraction=0.5, seed=1, warmup_ms=20.0, duration_ms=100.0):
    """mode: 'balanced' | 'split'.  Returns a dict with Mops/s and conservation fields."""
    out = np.zeros(10, np.uint64)
    secs = C.c_double(0)
    lib().orc_mutex_bench(0 if mode == "balanced" else 1, int(threads), int(capacity), int(prefill),
                          float(producer_fraction), int(seed), float(warmup_ms), float(duration_ms), out, C.byref(secs))
    keys = ("succ_enq", "succ_deq", "full", "empty", "tot_enq", "tot_deq", "sum_enq", "sum_deq", "sum_left", "left")
    d = {k: int(v) for k, v in zip(keys, out)}
    d["meas_seconds"] = secs.value
    d["mops"] = (d["succ_enq"] + d["succ_deq"]) / secs.value / 1e6
    d["threads"] = int(threads)
    return d


def hw_threads() -> int:
    return int(lib().orc_hw_threads())


def bfs(rowptr, col, src):
    """CPU BFS (apps_cpu.cpp).  Returns (int32 dist[], edges_scanned)."""
    rowptr = np.ascontiguousarray(rowptr, np.uint64)
    col = np.ascontiguousarray(col, np.uint32)
    nv = len(rowptr) - 1
    dist = np.empty(nv, np.int32)
    edges = C.c_uint64(0)
    lib().orc_bfs(nv, rowptr, col, int(src), dist, C.byref(edges))
    return dist, edges.value


def rt_render(width, height, spp, max_bounce, spheres, seed, threads=0, row0=0, row1=None):
    """CPU tracer (apps_cpu.cpp).  spheres: float32 [ns, 8] = cx,cy,cz,r,ar,ag,ab,emissive.
    Renders rows [row0,row1) into a full-size H*W*3 float32 image (other rows zero)."""
    sp = np.ascontiguousarray(spheres, np.float32)
    img = np.zeros((height, width, 3), np.float32)
    rays = C.c_uint64(0)
    if row1 is None:
        row1 = height
    lib().orc_rt_render(width, height, spp, max_bounce, sp.shape[0], sp.reshape(-1), int(seed), int(threads),
                        int(row0), int(row1), img.reshape(-1), C.byref(rays))
    return img, rays.value


# ---- the tracer's steps one by one (apps_cpu.cpp), so that tests can pin each against something other than itself
def rt_fmix32(x) -> int:
    return int(lib().orc_rt_fmix32(int(x) & 0xFFFFFFFF))


def rt_rnd(seed, pixel, sample, bounce, dim) -> float:
    return float(lib().orc_rt_rnd(int(seed), int(pixel), int(sample), int(bounce), int(dim)))


def rt_camera_ray(width, height, px, py, u0, u1):
    """(origin[3], direction[3]) of the primary ray through pixel (px, py) with sub-pixel jitter (u0, u1)."""
    out = np.zeros(6, np.float32)
    lib().orc_rt_camera_ray(int(width), int(height), int(px), int(py), float(u0), float(u1), out)
    return out[:3].copy(), out[3:].copy()


def rt_nearest_hit(spheres, origin, direction):
    """(sphere index or -1, t) of the nearest hit with t > t_min."""
    sp = np.ascontiguousarray(spheres, np.float32)
    t = C.c_float(0)
    i = lib().orc_rt_nearest_hit(sp.shape[0], sp.reshape(-1) if sp.size else np.zeros(8, np.float32),
                                 np.ascontiguousarray(origin, np.float32), np.ascontiguousarray(direction, np.float32), C.byref(t))
    return int(i), float(t.value)


def rt_scatter(seed, pixel, sample, bounce, normal):
    out = np.zeros(3, np.float32)
    lib().orc_rt_scatter(int(seed), int(pixel), int(sample), int(bounce), np.ascontiguousarray(normal, np.float32), out)
    return out
