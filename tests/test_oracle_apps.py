"""CPU pins of the application oracles (oracle/apps_cpu.cpp) against what mathematics fixes:
closed-form BFS distances on graphs whose distances are known, BFS invariants on a seeded
R-MAT graph, and closed-form images for the tracer (empty scene, one sphere on the axis, an
emissive sphere).  Also the input generators' structural contracts."""
import math

import numpy as np
import pytest

import oracle
from paper_2606_01693_b200 import inputs


def csr_from_edges(nv, edges):
    e = np.asarray(edges, np.uint32).reshape(-1, 2)
    return inputs.csr_undirected(nv, e[:, 0].copy(), e[:, 1].copy())


# ------------------------------------------------------------------------------- BFS
def test_bfs_path_graph_closed_form():
    nv = 50
    rowptr, col = csr_from_edges(nv, [(i, i + 1) for i in range(nv - 1)])
    for src in (0, 17, 49):
        d, edges = oracle.bfs(rowptr, col, src)
        assert d.tolist() == [abs(i - src) for i in range(nv)]
        assert edges == 2 * (nv - 1)                       # every directed edge scanned once


def test_bfs_star_and_ring():
    rowptr, col = csr_from_edges(9, [(0, i) for i in range(1, 9)])
    d, _ = oracle.bfs(rowptr, col, 0)
    assert d.tolist() == [0] + [1] * 8
    d, _ = oracle.bfs(rowptr, col, 3)
    assert d.tolist() == [1, 2, 2, 0, 2, 2, 2, 2, 2]
    n = 11
    rowptr, col = csr_from_edges(n, [(i, (i + 1) % n) for i in range(n)])
    d, _ = oracle.bfs(rowptr, col, 4)
    assert d.tolist() == [min((i - 4) % n, (4 - i) % n) for i in range(n)]


def test_bfs_grid_manhattan_and_disconnected():
    w, h = 7, 5
    edges = [(y * w + x, y * w + x + 1) for y in range(h) for x in range(w - 1)]
    edges += [(y * w + x, (y + 1) * w + x) for y in range(h - 1) for x in range(w)]
    nv = w * h + 3                                         # 3 extra vertices: one isolated, one separate edge
    edges.append((w * h + 1, w * h + 2))
    rowptr, col = csr_from_edges(nv, edges)
    sx, sy = 2, 3
    d, edges_scanned = oracle.bfs(rowptr, col, sy * w + sx)
    expect = [abs(x - sx) + abs(y - sy) for y in range(h) for x in range(w)] + [-1, -1, -1]
    assert d.tolist() == expect
    assert edges_scanned == 2 * ((w - 1) * h + (h - 1) * w)   # the other component is never scanned


def test_bfs_invariants_on_rmat():
    rowptr, col, src = inputs.rmat_csr(12, 16, seed=3)
    d, edges = oracle.bfs(rowptr, col, src)
    nv = len(rowptr) - 1
    assert d[src] == 0 and d.dtype == np.int32
    rows = np.repeat(np.arange(nv), np.diff(rowptr.astype(np.int64)))
    du, dv = d[rows], d[col]
    assert ((du < 0) == (dv < 0)).all()                    # an edge never joins reached and unreached
    reached = du >= 0
    assert (np.abs(du[reached] - dv[reached]) <= 1).all()
    # every reached vertex other than src has a neighbour one hop closer
    has_parent = np.zeros(nv, bool)
    np.logical_or.at(has_parent, rows[reached & (dv == du - 1)], True)
    assert has_parent[(d > 0)].all()
    assert edges == int(np.diff(rowptr.astype(np.int64))[d >= 0].sum())


# ------------------------------------------------------------------------------- generators
def test_rmat_csr_contract():
    rowptr, col, src = inputs.rmat_csr(10, 16, seed=1)
    nv = 1 << 10
    assert rowptr.dtype == np.uint64 and col.dtype == np.uint32 and len(rowptr) == nv + 1
    assert rowptr[0] == 0 and rowptr[-1] == len(col) and (np.diff(rowptr.astype(np.int64)) >= 0).all()
    rows = np.repeat(np.arange(nv), np.diff(rowptr.astype(np.int64)))
    assert (rows != col).all()                             # no self-loops
    key = rows.astype(np.int64) << 32 | col
    assert (np.diff(key) > 0).all()                        # sorted, deduplicated
    assert np.array_equal(np.sort(col.astype(np.int64) << 32 | rows), key)    # symmetric
    assert rowptr[src + 1] > rowptr[src]                   # source is not isolated
    # skew of R-MAT (a = 0.57): the low-id quadrant is much denser than the high-id one
    deg = np.diff(rowptr.astype(np.int64))
    assert deg[: nv // 2].sum() > 2 * deg[nv // 2:].sum()
    r2, c2, s2 = inputs.rmat_csr(10, 16, seed=1)
    assert np.array_equal(rowptr, r2) and np.array_equal(col, c2) and src == s2      # seeded


def test_sphere_scene_contract():
    s = inputs.sphere_scene(256, seed=1)
    assert s.shape == (256, 8) and s.dtype == np.float32
    assert (np.abs(s[:, :3]) <= 10).all() and (s[:, 3] >= 0.2).all() and (s[:, 3] <= 1.5).all()
    assert (s[:, 4:7] >= 0).all() and (s[:, 4:7] <= 1).all()
    assert set(np.unique(s[:, 7]).tolist()) <= {0.0, 1.0} and 10 <= s[:, 7].sum() <= 45
    assert np.array_equal(s, inputs.sphere_scene(256, seed=1))


# ------------------------------------------------------------------------------- tracer
BG = np.array([0.7, 0.8, 1.0], np.float32)


def test_rt_empty_scene_is_background():
    img, rays = oracle.rt_render(64, 48, 4, 4, np.zeros((0, 8), np.float32), seed=5, threads=2)
    assert img.shape == (48, 64, 3)
    assert np.array_equal(img, np.broadcast_to(BG, img.shape))        # (bg*4)/4 is exact
    assert rays == 64 * 48 * 4                                        # one segment per path


def test_rt_emissive_sphere_on_axis():
    # one emissive sphere of radius 5 at the origin, camera at (0,0,35), vertical FOV 40 deg:
    # a pixel sees the sphere iff its ray passes within 5 of the origin (analytic silhouette)
    sph = np.array([[0, 0, 0, 5, 0.25, 0.5, 0.75, 1]], np.float32)
    w, h, spp = 96, 64, 1
    img, rays = oracle.rt_render(w, h, spp, 4, sph, seed=9, threads=1)
    assert rays == w * h                                              # emissive or miss: one segment each
    hit = np.array([1.0, 2.0, 3.0], np.float32)                       # 4 x albedo
    is_hit = (img == hit).all(axis=2)
    is_bg = (img == BG).all(axis=2)
    assert (is_hit | is_bg).all()
    half_h = math.tan(math.radians(20.0))
    ys, xs = np.mgrid[0:h, 0:w]
    # pixel centres at least one pixel inside / outside the silhouette are decided whatever the jitter
    def dist_to_origin(px, py):
        dx = ((px / w) * 2 - 1) * half_h * (w / h)
        dy = (1 - (py / h) * 2) * half_h
        n = np.sqrt(dx * dx + dy * dy + 1)
        # distance from the origin to the line eye + t*d, eye = (0,0,35)
        return 35.0 * np.sqrt(dx * dx + dy * dy) / n
    dmin = np.minimum.reduce([dist_to_origin(xs + a, ys + b) for a in (0, 1) for b in (0, 1)])
    dmax = np.maximum.reduce([dist_to_origin(xs + a, ys + b) for a in (0, 1) for b in (0, 1)])
    assert is_hit[dmax < 4.999].all() and is_bg[dmin > 5.001].all()
    assert is_hit.sum() > 100


def test_rt_diffuse_sphere_centre_pixel_energy_bound():
    # a grey Lambertian sphere in front of a uniform background: every path ends on the background
    # (or is absorbed at the depth limit), so each channel is bg * albedo^j for some j >= 0
    sph = np.array([[0, 0, 0, 6, 0.5, 0.5, 0.5, 0]], np.float32)
    img, rays = oracle.rt_render(32, 32, 1, 4, sph, seed=2, threads=1)
    centre = img[12:20, 12:20].reshape(-1, 3)
    for px in centre:
        # convex sphere, outward hemisphere scatter: exactly one bounce, then the background
        assert np.allclose(px, BG * 0.5, rtol=0, atol=1e-6)
    assert np.array_equal(img[0, 0], BG)
    assert rays >= 32 * 32


def test_rt_threads_and_row_bands_do_not_change_pixels():
    sph = inputs.sphere_scene(64, seed=4)
    a, ra = oracle.rt_render(80, 60, 2, 4, sph, seed=7, threads=1)
    b, rb = oracle.rt_render(80, 60, 2, 4, sph, seed=7, threads=5)
    assert np.array_equal(a, b) and ra == rb
    c, _ = oracle.rt_render(80, 60, 2, 4, sph, seed=7, threads=2, row0=20, row1=31)
    assert np.array_equal(c[20:31], a[20:31]) and not c[:20].any() and not c[31:].any()
    d, _ = oracle.rt_render(80, 60, 2, 4, sph, seed=8, threads=2)
    assert not np.array_equal(a, d)                                   # the seed matters
    assert np.isfinite(a).all() and (a >= 0).all() and a.max() <= 4.0 + 1e-6
