"""Seeded synthetic inputs for the application drivers (BASELINE.json configs 4 and 5).

Input tooling only: numpy (plus a torch transcription of the graph recipe, so that the scale-22 graph of
config 4 can be generated on the GPU box in seconds instead of minutes), none of the method's arithmetic,
imported neither by the CUDA library nor by the CPU checker.  Tests and bench.py build the arrays here and hand the same arrays
to both sides.  They stand in for the paper's SuiteSparse graphs (Table IV,
L428-440) and its two scenes (L366, L384), which are not available.
"""
import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(x):
    """Counter-based 64-bit mixer (Steele/Lea/Flood splitmix64 finaliser) on a uint64 array."""
    with np.errstate(over="ignore"):
        x = (x + np.uint64(0x9E3779B97F4A7C15)) & _M64
        x = ((x ^ (x >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        x = ((x ^ (x >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        return x ^ (x >> np.uint64(31))


def rmat_edges(scale, edge_factor=16, a=0.57, b=0.19, c=0.19, seed=1, chunk=1 << 22):
    """R-MAT edge pairs: 2^scale vertices, edge_factor * 2^scale generated pairs.  One quadrant
    draw per bit level from a counter-based RNG keyed (seed, edge, level); no noise, no vertex
    permutation.  Returns (src, dst) uint32 arrays."""
    n_edges = edge_factor << scale
    src = np.empty(n_edges, np.uint32)
    dst = np.empty(n_edges, np.uint32)
    key = _splitmix64(np.array([seed], np.uint64))[0]
    for lo in range(0, n_edges, chunk):
        hi = min(lo + chunk, n_edges)
        e = np.arange(lo, hi, dtype=np.uint64)
        u = np.zeros(hi - lo, np.uint32)
        v = np.zeros(hi - lo, np.uint32)
        for level in range(scale):
            with np.errstate(over="ignore"):
                h = _splitmix64((e * np.uint64(64) + np.uint64(level)) ^ key)
            r = (h >> np.uint64(11)).astype(np.float64) * (1.0 / (1 << 53))
            # quadrant 0:(0,0) a | 1:(0,1) b | 2:(1,0) c | 3:(1,1) d
            ubit = r >= a + b
            vbit = ((r >= a) & (r < a + b)) | (r >= a + b + c)
            u = (u << np.uint32(1)) | ubit.astype(np.uint32)
            v = (v << np.uint32(1)) | vbit.astype(np.uint32)
        src[lo:hi] = u
        dst[lo:hi] = v
    return src, dst


def csr_undirected(nv, src, dst):
    """Symmetrise, drop self-loops, sort, deduplicate.  Returns (rowptr uint64[nv+1], col uint32[])."""
    keep = src != dst
    s = src[keep].astype(np.uint64)
    d = dst[keep].astype(np.uint64)
    keys = np.concatenate([(s << np.uint64(32)) | d, (d << np.uint64(32)) | s])
    keys = np.unique(keys)
    rows = (keys >> np.uint64(32)).astype(np.int64)
    col = (keys & np.uint64(0xFFFFFFFF)).astype(np.uint32)
    counts = np.bincount(rows, minlength=nv).astype(np.uint64)
    rowptr = np.zeros(nv + 1, np.uint64)
    np.cumsum(counts, out=rowptr[1:])
    return rowptr, col


def rmat_csr(scale, edge_factor=16, seed=1):
    """BASELINE.json config 4 graph: (rowptr, col, source vertex)."""
    nv = 1 << scale
    src, dst = rmat_edges(scale, edge_factor, seed=seed)
    rowptr, col = csr_undirected(nv, src, dst)
    deg = np.diff(rowptr.astype(np.int64))
    nonisolated = np.flatnonzero(deg > 0)
    source = int(nonisolated[seed % len(nonisolated)])
    return rowptr, col, source


# ---- the same recipe with torch ops (any device): bit-identical arrays, tests/test_inputs.py compares the two on CPU.
# torch has no uint64 arithmetic: int64 with wrapping multiplication, logical shifts written out.
def _i64(c):
    return c - (1 << 64) if c >= (1 << 63) else c


def _lsr(x, s):
    return (x >> s) & ((1 << (64 - s)) - 1)


def _splitmix64_torch(x):
    x = x + _i64(0x9E3779B97F4A7C15)
    x = (x ^ _lsr(x, 30)) * _i64(0xBF58476D1CE4E5B9)
    x = (x ^ _lsr(x, 27)) * _i64(0x94D049BB133111EB)
    return x ^ _lsr(x, 31)


def rmat_csr_torch(scale, edge_factor=16, seed=1, device="cpu", a=0.57, b=0.19, c=0.19, chunk=1 << 24):
    """rmat_csr() computed with torch on `device`.  Returns (rowptr int64[nv+1], col int32[], source) as torch tensors
    on that device; values equal those of rmat_csr (rowptr uint64, col uint32) element for element."""
    import torch
    nv = 1 << scale
    n_edges = edge_factor << scale
    key = int(_splitmix64(np.array([seed], np.uint64))[0])
    key = _i64(key)
    keys = []
    for lo in range(0, n_edges, chunk):
        hi = min(lo + chunk, n_edges)
        e = torch.arange(lo, hi, dtype=torch.int64, device=device)
        u = torch.zeros(hi - lo, dtype=torch.int64, device=device)
        v = torch.zeros(hi - lo, dtype=torch.int64, device=device)
        for level in range(scale):
            h = _splitmix64_torch((e * 64 + level) ^ key)
            r = _lsr(h, 11).to(torch.float64) * (1.0 / (1 << 53))
            ubit = r >= a + b
            vbit = ((r >= a) & (r < a + b)) | (r >= a + b + c)
            u = (u << 1) | ubit.to(torch.int64)
            v = (v << 1) | vbit.to(torch.int64)
        keep = u != v
        u, v = u[keep], v[keep]
        keys.append(torch.unique(torch.cat([(u << 32) | v, (v << 32) | u])))
    keys = torch.unique(torch.cat(keys))
    rows = keys >> 32
    col = (keys & 0xFFFFFFFF).to(torch.int32)
    counts = torch.bincount(rows, minlength=nv)
    rowptr = torch.zeros(nv + 1, dtype=torch.int64, device=device)
    rowptr[1:] = torch.cumsum(counts, 0)
    nonisolated = torch.nonzero(counts > 0).flatten()
    source = int(nonisolated[seed % len(nonisolated)])
    return rowptr, col, source


def sphere_scene(n_spheres=256, seed=1):
    """BASELINE.json config 5 scene: float32 [n, 8] = cx, cy, cz, r, ar, ag, ab, emissive(0/1).
    Centres U[-10,10]^3, radii U[0.2,1.5], albedo U[0,1]^3, 10 % emissive, drawn in this order."""
    rng = np.random.default_rng(seed)
    out = np.empty((n_spheres, 8), np.float32)
    out[:, 0:3] = rng.uniform(-10.0, 10.0, (n_spheres, 3))
    out[:, 3] = rng.uniform(0.2, 1.5, n_spheres)
    out[:, 4:7] = rng.uniform(0.0, 1.0, (n_spheres, 3))
    out[:, 7] = (rng.random(n_spheres) < 0.1).astype(np.float32)
    return out
