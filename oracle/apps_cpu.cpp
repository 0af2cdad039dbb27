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
//                 DESIGN.md §6, one (pixel, sample) path at a time, written as the textbook loop
//                 "camera ray; repeat { nearest hit; shade; scatter }" over explicit Ray / Hit records.
//                 fp32, every operation individually rounded (built with -ffp-contract=off, no fast-math).
//                 Each step is exported on its own (orc_rt_fmix32, orc_rt_rnd, orc_rt_camera_ray,
//                 orc_rt_nearest_hit, orc_rt_scatter) so that tests/test_oracle_apps.py can pin it
//                 against something other than itself:
//                   fmix32      published MurmurHash3 finaliser values; its published inverse undoes it
//                   rnd         range, 2^-24 grid, uniformity and independence across dims (chi-square)
//                   camera ray  pinhole geometry in float64
//                   nearest hit float64 quadratic formula over all spheres; t_min; ties -> lowest index
//                   scatter     unit length, hemisphere of the normal, E[cos] = 2/3 (cosine law)
//                   image       closed forms: background, emissive silhouette, grey sphere in an emissive
//                               shell (one bounce), coincident spheres, occlusion, closed diffuse room
//                               (absorption at the depth limit, ray count), sky view factor (1+cos)/2
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

struct Vec { float x, y, z; };
struct Ray { Vec origin, dir; };
struct Hit { int sphere; float t; };                       // sphere < 0: miss
struct Sphere { Vec centre; float radius; Vec albedo; bool emissive; };
struct Scene { uint32_t w, h, spp, max_bounce, ns; const float* sp; uint64_t seed; };

inline Vec operator+(Vec a, Vec b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
inline Vec operator-(Vec a, Vec b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
inline Vec operator*(Vec a, Vec b) { return {a.x * b.x, a.y * b.y, a.z * b.z}; }
inline Vec operator*(Vec a, float s) { return {a.x * s, a.y * s, a.z * s}; }
inline Vec operator/(Vec a, float s) { return {a.x / s, a.y / s, a.z / s}; }
inline float dot(Vec a, Vec b) { return (a.x * b.x + a.y * b.y) + a.z * b.z; }      // (x + y) + z
inline Vec unit(Vec a) { return a / std::sqrt(dot(a, a)); }

inline Sphere sphere_at(const Scene& sc, uint32_t i) {
  const float* S = sc.sp + 8 * i;
  return Sphere{{S[0], S[1], S[2]}, S[3], {S[4], S[5], S[6]}, S[7] != 0.0f};
}

// DESIGN.md §6 RNG: three rounds of the 32-bit MurmurHash3 finaliser over (seed, pixel, sample, bounce, dim)
uint32_t fmix32(uint32_t h) {
  h ^= h >> 16;
  h *= 0x85ebca6bu;
  h ^= h >> 13;
  h *= 0xc2b2ae35u;
  h ^= h >> 16;
  return h;
}
float rnd(uint64_t seed, uint32_t pixel, uint32_t sample, uint32_t bounce, uint32_t dim) {
  const uint32_t seed_lo = (uint32_t)seed, seed_hi = (uint32_t)(seed >> 32);
  const uint32_t key = sample * 0x85EBCA77u + bounce * 0xC2B2AE3Du + dim * 0x27D4EB2Fu;
  uint32_t h = fmix32(seed_lo ^ (pixel * 0x9E3779B1u));
  h = fmix32(h ^ key);
  h = fmix32(h ^ seed_hi);
  return (float)(h >> 8) * (1.0f / 16777216.0f);          // 24 high bits: a multiple of 2^-24 in [0, 1)
}

constexpr float kTMin = 1e-3f;
constexpr float kTanHalfFov = 0.36397023f;                 // tan(20 deg): vertical field of view 40 deg
const Vec kEye = {0.0f, 0.0f, 35.0f};
const Vec kBackground = {0.7f, 0.8f, 1.0f};
constexpr float kEmission = 4.0f;

// pinhole camera at kEye looking down -z, up +y; (u0, u1) = sub-pixel jitter
Ray camera_ray(const Scene& sc, uint32_t px, uint32_t py, float u0, float u1) {
  const float aspect = (float)sc.w / (float)sc.h;
  const float sx = (((float)px + u0) / (float)sc.w) * 2.0f - 1.0f;
  const float sy = 1.0f - (((float)py + u1) / (float)sc.h) * 2.0f;
  return Ray{kEye, unit(Vec{sx * (kTanHalfFov * aspect), sy * kTanHalfFov, -1.0f})};
}

// smallest t > kTMin over all spheres (|d| = 1: t = -b -+ sqrt(b^2 - c)); equal t: the lowest index wins
Hit nearest_hit(const Scene& sc, const Ray& ray) {
  Hit best{-1, INFINITY};
  for (uint32_t i = 0; i < sc.ns; ++i) {
    const Sphere s = sphere_at(sc, i);
    const Vec oc = ray.origin - s.centre;
    const float b = dot(oc, ray.dir);
    const float c = dot(oc, oc) - s.radius * s.radius;
    const float disc = b * b - c;
    if (disc < 0.0f) continue;
    const float root = std::sqrt(disc);
    float t = -b - root;                                   // near root first, else the far one (origin inside)
    if (!(t > kTMin)) t = -b + root;
    if (!(t > kTMin)) continue;
    if (t < best.t) best = Hit{(int)i, t};
  }
  return best;
}

// Lambertian direction: normalize(n + u), u a unit vector by rejection sampling in the unit ball
// (try k uses dims 2+3k .. 4+3k; at most 16 tries, then u = n)
Vec scatter(const Scene& sc, uint32_t pixel, uint32_t sample, uint32_t bounce, Vec n) {
  Vec u = n;
  for (uint32_t k = 0; k < 16; ++k) {
    const Vec v = {2.0f * rnd(sc.seed, pixel, sample, bounce, 2 + 3 * k) - 1.0f,
                   2.0f * rnd(sc.seed, pixel, sample, bounce, 3 + 3 * k) - 1.0f,
                   2.0f * rnd(sc.seed, pixel, sample, bounce, 4 + 3 * k) - 1.0f};
    const float len2 = dot(v, v);
    if (len2 <= 1.0f && len2 > 1e-12f) { u = v / std::sqrt(len2); break; }
  }
  Vec s = n + u;
  float len2 = dot(s, s);
  if (!(len2 > 1e-12f)) { s = n; len2 = dot(n, n); }
  return s / std::sqrt(len2);
}

// One bounce of one path.  Returns true while the path lives; when it ends *radiance is its value.
bool bounce_once(const Scene& sc, uint32_t pixel, uint32_t sample, uint32_t depth, Ray* ray, Vec* throughput, Vec* radiance) {
  const Hit hit = nearest_hit(sc, *ray);
  if (hit.sphere < 0) { *radiance = *throughput * kBackground; return false; }
  const Sphere s = sphere_at(sc, (uint32_t)hit.sphere);
  if (s.emissive) { *radiance = *throughput * (s.albedo * kEmission); return false; }
  *throughput = *throughput * s.albedo;
  if (depth == sc.max_bounce) { *radiance = Vec{0.0f, 0.0f, 0.0f}; return false; }      // absorbed at the depth limit
  const Vec p = ray->origin + ray->dir * hit.t;
  const Vec n = (p - s.centre) / s.radius;
  *ray = Ray{p, scatter(sc, pixel, sample, depth, n)};
  return true;
}

// radiance of one (pixel, sample) path; *rays += ray segments traced
Vec trace_path(const Scene& sc, uint32_t px, uint32_t py, uint32_t sample, uint64_t* rays) {
  const uint32_t pixel = py * sc.w + px;
  Ray ray = camera_ray(sc, px, py, rnd(sc.seed, pixel, sample, 0, 0), rnd(sc.seed, pixel, sample, 0, 1));
  Vec throughput = {1.0f, 1.0f, 1.0f}, radiance = {0.0f, 0.0f, 0.0f};
  for (uint32_t depth = 0;; ++depth) {
    ++*rays;
    if (!bounce_once(sc, pixel, sample, depth, &ray, &throughput, &radiance)) return radiance;
  }
}

void render_rows(const Scene& sc, uint32_t y0, uint32_t y1, float* rgb, uint64_t* rays) {
  uint64_t r = 0;
  for (uint32_t py = y0; py < y1; ++py)
    for (uint32_t px = 0; px < sc.w; ++px) {
      Vec acc = {0.0f, 0.0f, 0.0f};
      for (uint32_t s = 0; s < sc.spp; ++s) acc = acc + trace_path(sc, px, py, s, &r);   // samples in order
      const Vec c = acc / (float)sc.spp;
      float* out = rgb + 3 * ((size_t)py * sc.w + px);
      out[0] = c.x; out[1] = c.y; out[2] = c.z;
    }
  *rays = r;
}

}  // namespace

extern "C" {

uint32_t orc_rt_fmix32(uint32_t x) { return fmix32(x); }
float orc_rt_rnd(uint64_t seed, uint32_t pixel, uint32_t sample, uint32_t bounce, uint32_t dim) { return rnd(seed, pixel, sample, bounce, dim); }
// out6 = origin xyz, direction xyz
void orc_rt_camera_ray(uint32_t w, uint32_t h, uint32_t px, uint32_t py, float u0, float u1, float* out6) {
  Scene sc{w, h, 1, 0, 0, nullptr, 0};
  const Ray r = camera_ray(sc, px, py, u0, u1);
  out6[0] = r.origin.x; out6[1] = r.origin.y; out6[2] = r.origin.z; out6[3] = r.dir.x; out6[4] = r.dir.y; out6[5] = r.dir.z;
}
// returns the sphere index (-1 = miss), *t_out = hit distance
int orc_rt_nearest_hit(uint32_t ns, const float* spheres, const float* origin3, const float* dir3, float* t_out) {
  Scene sc{1, 1, 1, 0, ns, spheres, 0};
  const Hit h = nearest_hit(sc, Ray{{origin3[0], origin3[1], origin3[2]}, {dir3[0], dir3[1], dir3[2]}});
  *t_out = h.t;
  return h.sphere;
}
void orc_rt_scatter(uint64_t seed, uint32_t pixel, uint32_t sample, uint32_t bounce, const float* normal3, float* out3) {
  Scene sc{1, 1, 1, 0, 0, nullptr, seed};
  const Vec d = scatter(sc, pixel, sample, bounce, Vec{normal3[0], normal3[1], normal3[2]});
  out3[0] = d.x; out3[1] = d.y; out3[2] = d.z;
}

void orc_rt_render(uint32_t w, uint32_t h, uint32_t spp, uint32_t max_bounce, uint32_t ns, const float* spheres,
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

}  // extern "C"
