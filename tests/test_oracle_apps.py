"""CPU pins of the application oracles (oracle/apps_cpu.cpp) against what mathematics fixes:
closed-form BFS distances on graphs whose distances are known, BFS invariants on a seeded
R-MAT graph; for the tracer every step on its own (hash against published values and its published
inverse, RNG statistics, camera geometry and nearest hit against float64 formulas, the cosine law of
the scatter direction) and closed-form images (background, emissive silhouette, grey sphere in an
emissive shell, coincident spheres, occlusion, closed diffuse room, sky view factor).
Also the input generators' structural contracts."""
import os
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


# ------------------------------------------------------------------------------- tracer, step by step
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
M32 = 0xFFFFFFFF


def test_rt_fmix32_published_values_and_inverse():
    # tests/golden/fmix32.txt: values of the published MurmurHash3 finaliser (not produced by this repository)
    rows = [l.split() for l in open(os.path.join(GOLDEN, "fmix32.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) >= 5
    for a, b in rows:
        assert oracle.rt_fmix32(int(a, 16)) == int(b, 16), (a, b)
    # fmix32 is a bijection of 32-bit words; its inverse uses the multiplicative inverses of the two constants
    # (x ^= x >> 16 is an involution, x ^= x >> 13 is undone by x ^= x >> 13 ^ x >> 26)
    inv1, inv2 = pow(0x85EBCA6B, -1, 1 << 32), pow(0xC2B2AE35, -1, 1 << 32)
    assert (inv1, inv2) == (0xA5CB9243, 0x7ED1B41D)                   # the published inverse constants

    def unmix(h):
        h ^= h >> 16; h = (h * inv2) & M32; h ^= (h >> 13) ^ (h >> 26); h = (h * inv1) & M32; h ^= h >> 16
        return h
    rng = np.random.default_rng(0)
    for x in [0, 1, 2, M32, 0x80000000] + rng.integers(0, 1 << 32, 2000).tolist():
        assert unmix(oracle.rt_fmix32(x)) == x
    # avalanche: flipping one input bit flips about half of the output bits
    flips = [bin(oracle.rt_fmix32(x) ^ oracle.rt_fmix32(x ^ (1 << b))).count("1") for x in rng.integers(0, 1 << 32, 200).tolist() for b in (0, 7, 16, 31)]
    assert 14.5 < np.mean(flips) < 17.5


def _rnd_spec(seed, pixel, sample, bounce, dim):
    """DESIGN.md section 6 in Python integers (the published finaliser is pinned above)."""
    def fm(h):
        h &= M32; h ^= h >> 16; h = (h * 0x85EBCA6B) & M32; h ^= h >> 13; h = (h * 0xC2B2AE35) & M32; h ^= h >> 16
        return h
    h = fm((seed & M32) ^ ((pixel * 0x9E3779B1) & M32))
    h = fm(h ^ ((sample * 0x85EBCA77 + bounce * 0xC2B2AE3D + dim * 0x27D4EB2F) & M32))
    h = fm(h ^ (seed >> 32))
    return (h >> 8) / float(1 << 24)


def test_rt_rnd_matches_design_and_is_uniform():
    for t in [(1, 0, 0, 0, 0), (1, 1919 + 1079 * 1920, 3, 4, 49), (0x123456789ABCDEF0, 77, 2, 1, 5), (7, 1000, 0, 2, 17)]:
        assert oracle.rt_rnd(*t) == _rnd_spec(*t), t
    # every argument matters (a dropped term changes none of these)
    base = oracle.rt_rnd(5, 10, 1, 2, 3)
    for t in [(6, 10, 1, 2, 3), (5 + (1 << 32), 10, 1, 2, 3), (5, 11, 1, 2, 3), (5, 10, 2, 2, 3), (5, 10, 1, 3, 3), (5, 10, 1, 2, 4)]:
        assert oracle.rt_rnd(*t) != base, t
    # range, grid, uniformity per dimension, independence of neighbouring dimensions / pixels (chi-square, 16 bins)
    n = 20000
    for dim_a, dim_b in ((0, 1), (2, 3), (4, 5)):
        ua = np.array([oracle.rt_rnd(9, p, p % 4, p % 5, dim_a) for p in range(n)])
        ub = np.array([oracle.rt_rnd(9, p, p % 4, p % 5, dim_b) for p in range(n)])
        for u in (ua, ub):
            assert (u >= 0).all() and (u < 1).all() and np.array_equal(u * (1 << 24), np.floor(u * (1 << 24)))
            chi = ((np.bincount((u * 16).astype(int), minlength=16) - n / 16) ** 2 / (n / 16)).sum()
            assert chi < 45, chi                                      # 15 degrees of freedom: P(chi2 > 45) < 1e-4
        joint = np.bincount((ua * 4).astype(int) * 4 + (ub * 4).astype(int), minlength=16)
        assert ((joint - n / 16) ** 2 / (n / 16)).sum() < 45
        assert abs(np.corrcoef(ua, ub)[0, 1]) < 0.03
    seq = np.array([oracle.rt_rnd(9, p, 0, 0, 0) for p in range(n)])
    assert abs(np.corrcoef(seq[:-1], seq[1:])[0, 1]) < 0.03           # neighbouring pixels


def test_rt_camera_ray_is_the_pinhole_of_design_6():
    w, h = 1920, 1080
    for px, py, u0, u1 in [(0, 0, 0.0, 0.0), (959, 539, 0.999, 0.999), (1919, 1079, 0.25, 0.75), (300, 900, 0.5, 0.5)]:
        o, d = oracle.rt_camera_ray(w, h, px, py, u0, u1)
        assert o.tolist() == [0.0, 0.0, 35.0]
        sx = ((px + u0) / w) * 2 - 1
        sy = 1 - ((py + u1) / h) * 2
        v = np.array([sx * math.tan(math.radians(20)) * (w / h), sy * math.tan(math.radians(20)), -1.0])
        assert np.allclose(d, v / np.linalg.norm(v), atol=3e-7)
    _, d = oracle.rt_camera_ray(w, h, 0, 0, 0.0, 0.0)
    assert d[0] < 0 < d[1]                                            # pixel (0,0) is top-left: -x, +y
    # vertical field of view 40 degrees: top and bottom edge rays are 40 degrees apart
    _, top = oracle.rt_camera_ray(w, h, 960, 0, 0.0, 0.0)
    _, bot = oracle.rt_camera_ray(w, h, 960, 1079, 0.0, 1.0)
    assert abs(math.degrees(math.acos(float(np.dot(top.astype(float), bot.astype(float))))) - 40.0) < 1e-3


def _hit_f64(spheres, o, d, t_min=1e-3):
    """Nearest hit by the quadratic formula in float64 (|d| = 1); returns (index, t) or (-1, inf)."""
    best, bt = -1, math.inf
    for i, s in enumerate(np.asarray(spheres, np.float64)):
        oc = np.asarray(o, np.float64) - s[:3]
        b = float(oc @ np.asarray(d, np.float64))
        disc = b * b - (float(oc @ oc) - s[3] * s[3])
        if disc < 0:
            continue
        for t in (-b - math.sqrt(disc), -b + math.sqrt(disc)):
            if t > t_min:
                if t < bt:
                    best, bt = i, t
                break
    return best, bt


def test_rt_nearest_hit_against_float64_quadratic():
    rng = np.random.default_rng(3)
    sph = inputs.sphere_scene(64, seed=6)
    agree = 0
    for _ in range(3000):
        o = rng.uniform(-12, 12, 3).astype(np.float32)
        if rng.random() < 0.3:                                        # origins inside a sphere: the far root
            k = rng.integers(0, 64)
            o = (sph[k, :3] + rng.uniform(-0.5, 0.5, 3) * sph[k, 3]).astype(np.float32)
        d = rng.normal(size=3); d = (d / np.linalg.norm(d)).astype(np.float32)
        d = (d / np.sqrt((d.astype(np.float64) ** 2).sum())).astype(np.float32)
        i, t = oracle.rt_nearest_hit(sph, o, d)
        j, tj = _hit_f64(sph, o, d)
        if i == j:
            agree += 1
            if i >= 0:
                assert abs(t - tj) <= 2e-4 * max(1.0, tj)
        else:                                                         # only near-degenerate cases may differ (grazing, t ~ t_min, near ties)
            ti = _hit_f64(sph[[i]], o, d)[1] if i >= 0 else math.inf
            assert min(abs(ti - tj), abs(tj - 1e-3), abs(ti - 1e-3)) < 1e-3 or not math.isfinite(min(ti, tj))
    assert agree >= 2990
    # exact special cases: axis-aligned unit sphere, ray along -z from z = 35
    unit = np.array([[0, 0, 0, 1, 1, 1, 1, 0]], np.float32)
    assert oracle.rt_nearest_hit(unit, [0, 0, 35], [0, 0, -1]) == (0, 34.0)
    assert oracle.rt_nearest_hit(unit, [0, 0, 0], [0, 0, -1]) == (0, 1.0)              # inside: far root
    assert oracle.rt_nearest_hit(unit, [0, 0, -1], [0, 0, -1])[0] == -1                # on the surface, leaving: t = 0 < t_min
    assert oracle.rt_nearest_hit(unit, [0, 0, 1], [0, 0, -1]) == (0, 2.0)              # on the surface, entering: the far side
    assert oracle.rt_nearest_hit(unit, [0, 2, 35], [0, 0, -1])[0] == -1                # miss
    # ties -> lowest index; occlusion -> nearest, whatever the order in the array
    two = np.array([[0, 0, 0, 1, 0, 0, 0, 0], [0, 0, 0, 1, 1, 1, 1, 0]], np.float32)
    assert oracle.rt_nearest_hit(two, [0, 0, 35], [0, 0, -1])[0] == 0
    assert oracle.rt_nearest_hit(two[::-1].copy(), [0, 0, 35], [0, 0, -1])[0] == 0
    far_first = np.array([[0, 0, -5, 3, 0, 0, 0, 0], [0, 0, 5, 1, 1, 1, 1, 0]], np.float32)
    assert oracle.rt_nearest_hit(far_first, [0, 0, 35], [0, 0, -1]) == (1, 29.0)


def test_rt_scatter_follows_the_cosine_law():
    rng = np.random.default_rng(8)
    for trial in range(4):
        n = rng.normal(size=3); n = (n / np.linalg.norm(n)).astype(np.float32)
        dirs = np.array([oracle.rt_scatter(11, p, p % 4, 1 + trial, n) for p in range(6000)], np.float64)
        assert np.allclose(np.linalg.norm(dirs, axis=1), 1.0, atol=1e-5)
        cos = dirs @ n.astype(np.float64)
        assert (cos >= -1e-6).all()                                   # hemisphere of the normal
        # normalize(n + uniform unit vector) is cosine-weighted: pdf(cos) = 2 cos, E[cos] = 2/3, P(cos < 1/2) = 1/4
        assert abs(cos.mean() - 2 / 3) < 0.012                        # a uniform-hemisphere sampler would give 1/2
        assert abs((cos < 0.5).mean() - 0.25) < 0.02
        # azimuth around n is uniform: the component orthogonal to n has zero mean
        ortho = dirs - np.outer(cos, n)
        assert np.abs(ortho.mean(axis=0)).max() < 0.02
    a = oracle.rt_scatter(11, 5, 0, 1, [0, 1, 0]); b = oracle.rt_scatter(11, 5, 0, 2, [0, 1, 0])
    assert not np.array_equal(a, b)                                   # the bounce index enters the stream


# ------------------------------------------------------------------------------- tracer, whole images with closed forms
def f32(*v):
    return np.array(v, np.float32)


def test_rt_grey_sphere_inside_emissive_shell_is_one_bounce():
    # camera inside an emissive shell of radius 100 (the far root of the quadratic), a convex grey sphere in the middle:
    # a path either sees the shell (4 * a_e) or bounces once off the grey sphere and then sees the shell (a_g * 4 * a_e).
    # Two bounces (a_g^2) would mean a self-intersection at t ~ 0 that t_min failed to exclude.
    a_e, a_g = f32(0.25, 0.5, 0.75), f32(0.5, 0.25, 0.125)
    sph = np.array([[0, 0, 0, 100, *a_e, 1], [0, 0, 0, 6, *a_g, 0]], np.float32)
    img, rays = oracle.rt_render(48, 32, 1, 4, sph, seed=4, threads=2)
    direct, once = a_e * np.float32(4), a_g * (a_e * np.float32(4))
    is_direct, is_once = (img == direct).all(axis=2), (img == once).all(axis=2)
    assert (is_direct | is_once).all() and is_once[16, 24] and is_direct[0, 0]
    assert rays == int(is_direct.sum()) + 2 * int(is_once.sum())      # one segment, or two
    # the same scene with the shell listed last: the order of the array must not matter
    img2, _ = oracle.rt_render(48, 32, 1, 4, sph[::-1].copy(), seed=4, threads=2)
    assert np.array_equal(img, img2)


def test_rt_coincident_spheres_lowest_index_wins_and_occlusion():
    red, blue = [0, 0, 0, 5, 1.0, 0.0, 0.0, 1], [0, 0, 0, 5, 0.0, 0.0, 1.0, 1]
    a, _ = oracle.rt_render(32, 32, 1, 2, np.array([red, blue], np.float32), seed=1, threads=1)
    b, _ = oracle.rt_render(32, 32, 1, 2, np.array([blue, red], np.float32), seed=1, threads=1)
    assert a[16, 16].tolist() == [4.0, 0.0, 0.0] and b[16, 16].tolist() == [0.0, 0.0, 4.0]
    # a small emissive sphere in front of a large one of another colour, the large one listed first
    sph = np.array([[0, 0, -10, 8, 0.0, 1.0, 0.0, 1], [0, 0, 10, 2, 1.0, 0.0, 0.0, 1]], np.float32)
    img, _ = oracle.rt_render(64, 64, 1, 2, sph, seed=1, threads=1)
    assert img[32, 32].tolist() == [4.0, 0.0, 0.0]                    # centre: the near sphere
    assert (img == f32(0.0, 4.0, 0.0)).all(axis=2).sum() > 50         # a ring of the far sphere around it


@pytest.mark.parametrize("max_bounce", [0, 1, 2])
def test_rt_absorption_at_the_depth_limit_inside_a_diffuse_shell(max_bounce):
    # camera inside a big DIFFUSE shell with a grey sphere in the middle.  Normals point away from the centre of their
    # sphere (n = (p - c) / r, never flipped), so a path that hits the shell from inside scatters
    # outwards and sees the sky at its next segment.  Depths 0 .. max_bounce; a diffuse hit AT the limit is absorbed:
    #   shell pixel : B = 0 -> 0 (1 segment);  B >= 1 -> a_s * sky (2 segments)
    #   inner pixel : B = 0 -> 0 (1);  B = 1 -> 0 (2: inner, shell, absorbed);  B = 2 -> a_g * a_s * sky (3)
    a_s, a_g = np.float32(0.75), np.float32(0.5)
    sph = np.array([[0, 0, 0, 100, a_s, a_s, a_s, 0], [0, 0, 0, 6, a_g, a_g, a_g, 0]], np.float32)
    img, rays = oracle.rt_render(32, 24, 1, max_bounce, sph, seed=3, threads=2)
    inner = np.zeros((24, 32), bool)
    for py in range(24):
        for px in range(32):
            u0, u1 = oracle.rt_rnd(3, py * 32 + px, 0, 0, 0), oracle.rt_rnd(3, py * 32 + px, 0, 0, 1)
            inner[py, px] = oracle.rt_nearest_hit(sph, *oracle.rt_camera_ray(32, 24, px, py, u0, u1))[0] == 1
    assert inner[12, 16] and not inner[0, 0] and 20 < inner.sum() < 32 * 24 - 20
    black = np.zeros(3, np.float32)
    shell_px = black if max_bounce == 0 else a_s * BG
    inner_px = (a_g * a_s) * BG if max_bounce == 2 else black
    assert (img[~inner] == shell_px).all() and (img[inner] == inner_px).all()
    seg_shell = 1 if max_bounce == 0 else 2
    seg_inner = min(max_bounce + 1, 3)
    assert rays == int((~inner).sum()) * seg_shell + int(inner.sum()) * seg_inner


def test_rt_depth_limit_zero_and_one_on_an_open_scene():
    a = np.float32(0.5)
    sph = np.array([[0, 0, 0, 6, a, a, a, 0]], np.float32)
    img0, _ = oracle.rt_render(32, 32, 1, 0, sph, seed=2, threads=1)
    img1, _ = oracle.rt_render(32, 32, 1, 1, sph, seed=2, threads=1)
    assert img0[16, 16].tolist() == [0.0, 0.0, 0.0] and np.array_equal(img0[0, 0], BG)     # a hit at depth 0 = the limit: absorbed
    assert np.array_equal(img1[16, 16], BG * a)                                             # one bounce, then the sky


def test_rt_sky_view_factor_of_a_lambertian_point():
    # A huge emissive sphere above the scene acts as the half space y > 50.  A grey sphere below it: a path that hits the
    # grey sphere at a point with normal n scatters into the light with probability (1 + n_y) / 2 for a cosine-weighted
    # direction (view factor of a tilted element to the half space above a horizontal plane), else into the sky.
    a_g, a_e = np.float32(0.5), f32(1.0, 1.0, 1.0)
    R = 1.0e4
    sph = np.array([[0, R + 50, 0, R, *a_e, 1], [0, 0, 0, 6, a_g, a_g, a_g, 0]], np.float32)
    w, h, spp = 48, 48, 64
    img, _ = oracle.rt_render(w, h, spp, 2, sph, seed=5, threads=0)
    checked = 0
    for py, px in [(24, 24), (14, 24), (34, 24), (24, 16), (20, 30)]:
        o, d = oracle.rt_camera_ray(w, h, px, py, 0.5, 0.5)
        i, t = oracle.rt_nearest_hit(sph, o, d)
        assert i == 1
        ny = float((o.astype(np.float64) + d.astype(np.float64) * t)[1] / 6.0)
        f = (1 + ny) / 2
        expect = float(a_g) * (f * 4.0 * a_e.astype(np.float64) + (1 - f) * BG.astype(np.float64))
        # binomial noise of 64 samples between the two outcomes, on top of the variation of n across the pixel
        tol = float(a_g) * 4.0 * (3.5 * math.sqrt(max(f * (1 - f), 0.02) / spp) + 0.03)
        assert np.all(np.abs(img[py, px].astype(np.float64) - expect) < tol), (py, px, img[py, px], expect)
        checked += 1
    assert checked == 5
