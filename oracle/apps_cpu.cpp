// ORACLE — TEST INFRASTRUCTURE ONLY (see fifo_model.hpp header).
//
// CPU statements of what the two application drivers of PAPER.md §V-B (L365-366) must output.
// Written from the definitions, independent of the CUDA path: no shared code, headers or tables.
//
//  orc_bfs        hop distances from `src` over a CSR graph: the textbook array-queue BFS.
//                 "the current frontier is dequeued, outgoing neighbors are
//                 examined, and newly visited vertices are marked and are enqueued into the next
//                 frontier".  Hop distance is unique, so the GPU result must be bit-exact.
//                 Pins (tests/test_oracle_apps.py): closed forms on path, star, grid, ring and
//                 disconnected graphs; |d[u]-d[v]| <= 1 across every edge; parent at d-1.
//
//  orc_rt_render  the path tracer of BASELINE.json config 5 with the paper-silent constants of
//                 DESIGN.md §6, one pixel at a time.  fp32, every operation individually rounded
//                 (built with -ffp-contract=off, no fast-math).
//                 Pins: empty scene = background; one sphere on the axis: analytic primary hit;
//                 emissive sphere: 4 x albedo where hit.  The full 256-sphere image has no
//                 independent pin: parity unpinned beyond those closed forms.
#include <cmath>
#include <cstdint>
#include <thread>
#include <vector>

extern "C" {

void orc_bfs(uint32_t nv, const uint64_t* rowptr, const uint32_t* col, uint32_t src, int32_t* dist,
             uint64_t* edges_scanned) {
  for (uint32_t i = 0; i < nv; ++i) dist[i] = -1;
  std::vector<uint32_t> queue;
  queue.reserve(nv);
  uint64_t edges = 0;
  if (src < nv) { dist[src] = 0; queue.push_back(src); }
  for (size_t head = 0; head < queue.size(); ++head) {
    const uint32_t u = queue[head];
    for (uint64_t e = rowptr[u]; e < rowptr[u + 1]; ++e) {
      ++edges;
      const uint32_t w = col[e];
      if (dist[w] < 0) { dist[w] = dist[u] + 1; queue.push_back(w); }
    }
  }
  *edges_scanned = edges;
}

}  // extern "C"

// ------------------------------------------------------------------------------------- tracer
namespace {

struct V3 { float x, y, z; };
inline V3 add(V3 a, V3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
inline V3 sub(V3 a, V3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
inline V3 mul(V3 a, V3 b) { return {a.x * b.x, a.y * b.y, a.z * b.z}; }
inline V3 scale(V3 a, float s) { return {a.x * s, a.y * s, a.z * s}; }
inline V3 divs(V3 a, float s) { return {a.x / s, a.y / s, a.z / s}; }
inline float dot(V3 a, V3 b) { return (a.x * b.x + a.y * b.y) + a.z * b.z; }

// murmur3 32-bit finaliser, applied three times over (seed, pixel, sample, bounce, dim)
inline uint32_t fmix32(uint32_t x) {
  x ^= x >> 16; x *= 0x85ebca6bu; x ^= x >> 13; x *= 0xc2b2ae35u; x ^= x >> 16;
  return x;
}
inline float rnd(uint64_t seed, uint32_t pixel, uint32_t sample, uint32_t bounce, uint32_t dim) {
  uint32_t x = fmix32((uint32_t)seed ^ (pixel * 0x9E3779B1u));
  x = fmix32(x ^ (sample * 0x85EBCA77u + bounce * 0xC2B2AE3Du + dim * 0x27D4EB2Fu));
  x = fmix32(x ^ (uint32_t)(seed >> 32));
  return (float)(x >> 8) * (1.0f / 16777216.0f);
}

struct Scene { uint32_t w, h, spp, max_bounce, ns; const float* sp; uint64_t seed; };

constexpr float kTMin = 1e-3f;
constexpr float kHalfH = 0.36397023f;           // tan(20 deg): vertical FOV 40 deg
const V3 kEye = {0.0f, 0.0f, 35.0f};
const V3 kBackground = {0.7f, 0.8f, 1.0f};

// radiance of one (pixel, sample) path; *rays += ray segments traced
V3 trace_path(const Scene& sc, uint32_t px, uint32_t py, uint32_t s, uint64_t* rays) {
  const uint32_t pixel = py * sc.w + px;
  const float aspect = (float)sc.w / (float)sc.h;
  const float u0 = rnd(sc.seed, pixel, s, 0, 0), u1 = rnd(sc.seed, pixel, s, 0, 1);
  const float sx = (((float)px + u0) / (float)sc.w) * 2.0f - 1.0f;
  const float sy = 1.0f - (((float)py + u1) / (float)sc.h) * 2.0f;
  V3 d = {sx * (kHalfH * aspect), sy * kHalfH, -1.0f};
  d = divs(d, std::sqrt(dot(d, d)));
  V3 o = kEye, T = {1.0f, 1.0f, 1.0f}, L = {0.0f, 0.0f, 0.0f};
  for (uint32_t b = 0; b <= sc.max_bounce; ++b) {
    ++*rays;
    float best_t = INFINITY;
    int best = -1;
    for (uint32_t i = 0; i < sc.ns; ++i) {             // brute force, ties -> lowest index
      const float* S = sc.sp + 8 * i;
      const V3 oc = sub(o, V3{S[0], S[1], S[2]});
      const float bq = dot(oc, d);
      const float cq = dot(oc, oc) - S[3] * S[3];
      const float disc = bq * bq - cq;
      if (disc < 0.0f) continue;
      const float sq = std::sqrt(disc);
      float t = -bq - sq;
      if (!(t > kTMin)) { t = -bq + sq; if (!(t > kTMin)) continue; }
      if (t < best_t) { best_t = t; best = (int)i; }
    }
    if (best < 0) { L = add(L, mul(T, kBackground)); break; }
    const float* S = sc.sp + 8 * best;
    const V3 albedo = {S[4], S[5], S[6]};
    if (S[7] != 0.0f) { L = add(L, mul(T, scale(albedo, 4.0f))); break; }   // emissive: 4 x albedo, path ends
    T = mul(T, albedo);
    if (b == sc.max_bounce) break;                                          // absorbed
    const V3 p = add(o, scale(d, best_t));
    const V3 n = divs(sub(p, V3{S[0], S[1], S[2]}), S[3]);
    V3 unit = n;                                                            // fallback after 16 rejections
    for (uint32_t k = 0; k < 16; ++k) {
      const V3 v = {2.0f * rnd(sc.seed, pixel, s, b, 2 + 3 * k) - 1.0f,
                    2.0f * rnd(sc.seed, pixel, s, b, 3 + 3 * k) - 1.0f,
                    2.0f * rnd(sc.seed, pixel, s, b, 4 + 3 * k) - 1.0f};
      const float l2 = dot(v, v);
      if (l2 <= 1.0f && l2 > 1e-12f) { unit = divs(v, std::sqrt(l2)); break; }
    }
    V3 sdir = add(n, unit);
    float l2 = dot(sdir, sdir);
    if (!(l2 > 1e-12f)) { sdir = n; l2 = dot(n, n); }
    d = divs(sdir, std::sqrt(l2));
    o = p;
  }
  return L;
}

void render_rows(const Scene& sc, uint32_t y0, uint32_t y1, float* rgb, uint64_t* rays) {
  uint64_t r = 0;
  for (uint32_t py = y0; py < y1; ++py)
    for (uint32_t px = 0; px < sc.w; ++px) {
      V3 acc = {0.0f, 0.0f, 0.0f};
      for (uint32_t s = 0; s < sc.spp; ++s) acc = add(acc, trace_path(sc, px, py, s, &r));   // fixed order
      const V3 c = divs(acc, (float)sc.spp);
      float* out = rgb + 3 * ((size_t)py * sc.w + px);
      out[0] = c.x; out[1] = c.y; out[2] = c.z;
    }
  *rays = r;
}

}  // namespace

extern "C" void orc_rt_render(uint32_t w, uint32_t h, uint32_t spp, uint32_t max_bounce, uint32_t ns, const float* spheres,
                              uint64_t seed, uint32_t threads, uint32_t row0, uint32_t row1, float* rgb, uint64_t* rays_out) {
  Scene sc{w, h, spp, max_bounce, ns, spheres, seed};
  if (row1 > h) row1 = h;
  if (row0 >= row1) { *rays_out = 0; return; }
  if (threads == 0) threads = std::thread::hardware_concurrency();
  const uint32_t rows = row1 - row0;
  if (threads > rows) threads = rows;
  std::vector<std::thread> pool;
  std::vector<uint64_t> rays(threads, 0);
  for (uint32_t t = 0; t < threads; ++t) {
    const uint32_t y0 = row0 + (uint64_t)rows * t / threads, y1 = row0 + (uint64_t)rows * (t + 1) / threads;
    pool.emplace_back(render_rows, std::cref(sc), y0, y1, rgb, &rays[t]);
  }
  for (auto& th : pool) th.join();
  uint64_t total = 0;
  for (uint64_t r : rays) total += r;
  *rays_out = total;
}
