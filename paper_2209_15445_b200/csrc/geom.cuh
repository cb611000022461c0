// Solids, distance-to-boundary with a warp-cooperative BVH, and Locate  (
// §8(c) G1-G5).  Every function that takes an `active` flag must be called by all
// 32 lanes of a warp in converged control flow: lanes whose volume has a BVH are served one after the
// other by the whole warp (each lane tests one child box / one primitive), which turns the paper's
// "quasi-random memory access + divergence" bottleneck into coalesced, uniform work.
#pragma once
#include <type_traits>

#include "types.cuh"

namespace adept {

__device__ __forceinline__ const DevVolume& volume(const DevCtx& c, int v) { return c.vol[v]; }

// The navigator is written once for the precision R of the geometry it reads: double -- the transport path, all
// state fp64 (BASELINE.json:north_star) -- or float, the single-precision geometry mode of PAPER.md:41 (every solid,
// transform and BVH box in fp32), which the ray-cast validator can be pointed at.
template <typename R> struct Geo;
template <> struct Geo<double> {
  static __device__ __forceinline__ const VolT<double>& vol(const DevCtx& c, int v) { return c.vol[v]; }
  static __device__ __forceinline__ const double* rot(const DevCtx& c) { return c.rot; }
  static __device__ __forceinline__ const BvhT<double>& bvh(const DevCtx& c, int i) { return c.bvh[i]; }
  static __device__ __forceinline__ double inf() { return ADEPT_INF; }
};
template <> struct Geo<float> {
  static __device__ __forceinline__ const VolT<float>& vol(const DevCtx& c, int v) { return c.vol32[v]; }
  static __device__ __forceinline__ const float* rot(const DevCtx& c) { return c.rot32; }
  static __device__ __forceinline__ const BvhT<float>& bvh(const DevCtx& c, int i) { return c.bvh32[i]; }
  static __device__ __forceinline__ float inf() { return __int_as_float(0x7f800000); }
};
__device__ __forceinline__ double r_abs(double x) { return fabs(x); }
__device__ __forceinline__ float r_abs(float x) { return fabsf(x); }
__device__ __forceinline__ double r_sqrt(double x) { return sqrt(x); }
__device__ __forceinline__ float r_sqrt(float x) { return sqrtf(x); }
__device__ __forceinline__ double r_min(double a, double b) { return fmin(a, b); }
__device__ __forceinline__ float r_min(float a, float b) { return fminf(a, b); }
__device__ __forceinline__ double r_max(double a, double b) { return fmax(a, b); }
__device__ __forceinline__ float r_max(float a, float b) { return fmaxf(a, b); }

// local = R^T (global - t); R (row-major, local axes as columns) is only read for rotated placements
template <typename R>
__device__ __forceinline__ void to_local(const DevCtx& c, int vi, const VolT<R>& v, R gx, R gy, R gz, R l[3]) {
  const R q0 = gx - v.t[0], q1 = gy - v.t[1], q2 = gz - v.t[2];
  if (v.identity) { l[0] = q0; l[1] = q1; l[2] = q2; return; }
  const R* __restrict__ M = Geo<R>::rot(c) + 9 * static_cast<size_t>(vi);
#pragma unroll
  for (int i = 0; i < 3; ++i) l[i] = __ldg(M + i) * q0 + __ldg(M + 3 + i) * q1 + __ldg(M + 6 + i) * q2;
}
template <typename R>
__device__ __forceinline__ void dir_to_local(const DevCtx& c, int vi, const VolT<R>& v, R gx, R gy, R gz, R l[3]) {
  if (v.identity) { l[0] = gx; l[1] = gy; l[2] = gz; return; }
  const R* __restrict__ M = Geo<R>::rot(c) + 9 * static_cast<size_t>(vi);
#pragma unroll
  for (int i = 0; i < 3; ++i) l[i] = __ldg(M + i) * gx + __ldg(M + 3 + i) * gy + __ldg(M + 6 + i) * gz;
}

// global = t + R local (inverse of to_local)
__device__ __forceinline__ void to_global(const DevCtx& c, int vi, const DevVolume& v, const double l[3], double g[3]) {
  if (v.identity) { g[0] = v.t[0] + l[0]; g[1] = v.t[1] + l[1]; g[2] = v.t[2] + l[2]; return; }
  const double* __restrict__ R = c.rot + 9 * static_cast<size_t>(vi);
#pragma unroll
  for (int j = 0; j < 3; ++j) g[j] = v.t[j] + __ldg(R + 3 * j) * l[0] + __ldg(R + 3 * j + 1) * l[1] + __ldg(R + 3 * j + 2) * l[2];
}

// ---------------------------------------------------------------- G1 solids
template <typename R>
__device__ __forceinline__ bool inside_solid(int solid, const R h[3], const R p[3]) {
  if (solid == ADEPT_BOX) return r_abs(p[0]) <= h[0] && r_abs(p[1]) <= h[1] && r_abs(p[2]) <= h[2];
  const R r2 = p[0] * p[0] + p[1] * p[1];
  return r2 >= h[0] * h[0] && r2 <= h[1] * h[1] && r_abs(p[2]) <= h[2];
}

// min_i (sgn(d_i) h_i - p_i) / d_i over d_i != 0.  The three quotients n_i / |d_i| are compared by
// cross-multiplication and only the smallest is divided (one division instead of three; when two are
// within rounding of each other either is the minimum to 1 ulp).
// `face` receives the exit face, 2 * axis + (d[axis] > 0), or -1.
template <typename R>
__device__ __forceinline__ R box_exit(const R h[3], const R p[3], const R d[3], int& face) {
  R num = R(1), den = R(0);   // +inf as 1/0
  face = -1;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    const R ad = r_abs(d[i]);
    const R ni = h[i] - (d[i] > R(0) ? p[i] : -p[i]);   // distance to the exit plane along the axis
    if (ad != R(0) && ni * den <= num * ad) { num = ni; den = ad; face = 2 * i + (d[i] > R(0) ? 1 : 0); }
  }
  return den != R(0) ? r_max(num / den, R(0)) : Geo<R>::inf();
}

template <typename R>
__device__ __forceinline__ R box_entry(const R h[3], const R p[3], const R d[3]) {
  R tn = -Geo<R>::inf(), tf = Geo<R>::inf();
  bool miss = false;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    if (d[i] != R(0)) {
      const R t1 = (-h[i] - p[i]) / d[i];
      const R t2 = (h[i] - p[i]) / d[i];
      tn = r_max(tn, r_min(t1, t2));
      tf = r_min(tf, r_max(t1, t2));
    } else if (r_abs(p[i]) > h[i]) {
      miss = true;
    }
  }
  if (!miss && tn <= tf && tf > R(0)) return r_max(tn, R(0));
  return Geo<R>::inf();
}

template <typename R>
__device__ __forceinline__ R tube_exit(const R h[3], const R p[3], const R d[3]) {
  R t = Geo<R>::inf();
  if (d[2] != R(0)) t = ((d[2] > R(0) ? h[2] : -h[2]) - p[2]) / d[2];
  const R A = d[0] * d[0] + d[1] * d[1];
  if (A > R(0)) {
    const R B = p[0] * d[0] + p[1] * d[1];
    const R r2 = p[0] * p[0] + p[1] * p[1];
    const R Co = r2 - h[1] * h[1];
    const R disc_o = B * B - A * Co;
    t = r_min(t, (-B + r_sqrt(r_max(disc_o, R(0)))) / A);
    if (h[0] > R(0) && B < R(0)) {
      const R Ci = r2 - h[0] * h[0];
      const R disc_i = B * B - A * Ci;
      if (disc_i > R(0)) t = r_min(t, (-B - r_sqrt(disc_i)) / A);
    }
  }
  return r_max(t, R(0));
}

template <typename R>
__device__ __forceinline__ R tube_entry(const R h[3], const R p[3], const R d[3]) {
  if (inside_solid(ADEPT_TUBE, h, p)) return R(0);
  R best = Geo<R>::inf();
  const R r2 = p[0] * p[0] + p[1] * p[1];
  const R rmin2 = h[0] * h[0], rmax2 = h[1] * h[1];
  if (r_abs(p[2]) > h[2] && p[2] * d[2] < R(0)) {  // (a) end caps
    const R t = (r_abs(p[2]) - h[2]) / r_abs(d[2]);
    const R x = p[0] + t * d[0], y = p[1] + t * d[1];
    const R q2 = x * x + y * y;
    if (q2 >= rmin2 && q2 <= rmax2) best = r_min(best, t);
  }
  const R A = d[0] * d[0] + d[1] * d[1];
  if (A > R(0)) {
    const R B = p[0] * d[0] + p[1] * d[1];
    const R Co = r2 - rmax2;
    if (Co > R(0) && B < R(0)) {  // (b) outer cylinder from outside
      const R disc = B * B - A * Co;
      if (disc > R(0)) {
        const R t = (-B - r_sqrt(disc)) / A;
        if (t >= R(0) && r_abs(p[2] + t * d[2]) <= h[2]) best = r_min(best, t);
      }
    }
    if (h[0] > R(0)) {  // (c) inner cylinder, far root: leaving the hole into the solid
      const R Ci = r2 - rmin2;
      const R disc = B * B - A * Ci;
      if (disc > R(0)) {
        const R t = (-B + r_sqrt(disc)) / A;
        if (t > R(0) && r_abs(p[2] + t * d[2]) <= h[2]) best = r_min(best, t);
      }
    }
  }
  return best;
}

template <typename R>
__device__ __forceinline__ R solid_exit(const VolT<R>& v, const R p[3], const R d[3], int& face) {
  if (v.solid == ADEPT_BOX) return box_exit(v.dims, p, d, face);
  face = -1;
  return tube_exit(v.dims, p, d);
}
template <typename R>
__device__ __forceinline__ R solid_entry(const VolT<R>& v, const R p[3], const R d[3]) {
  return v.solid == ADEPT_BOX ? box_entry(v.dims, p, d) : tube_entry(v.dims, p, d);
}

template <typename R>
__device__ __forceinline__ bool inside_volume(const DevCtx& c, int vol, R x, R y, R z) {
  const VolT<R>& v = Geo<R>::vol(c, vol);
  R l[3];
  to_local(c, vol, v, x, y, z, l);
  return inside_solid(v.solid, v.dims, l);
}

template <typename R>
__device__ __forceinline__ R entry_distance(const DevCtx& c, int vol, R px, R py, R pz, R dx, R dy, R dz) {
  const VolT<R>& v = Geo<R>::vol(c, vol);
  R lp[3], ld[3];
  to_local(c, vol, v, px, py, pz, lp);
  dir_to_local(c, vol, v, dx, dy, dz, ld);
  return solid_entry(v, lp, ld);
}

// Entry distance into daughter `vol` for a segment of length s_max: the exact entry_distance when that is <= s_max,
// else any value > s_max.  For a box the segment's extent along each local axis is compared with the slab first
// (no division): a segment that stays clear of a slab by more than rounding cannot enter the box.
__device__ __forceinline__ double entry_distance_within(const DevCtx& c, int vol, double px, double py, double pz, double dx,
                                                        double dy, double dz, double s_max) {
  const DevVolume& v = volume(c, vol);
  double lp[3], ld[3];
  to_local(c, vol, v, px, py, pz, lp);
  dir_to_local(c, vol, v, dx, dy, dz, ld);
  if (v.solid == ADEPT_BOX && s_max < 1.0e30) {
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      const double a = lp[i], b = lp[i] + s_max * ld[i];
      const double pad = 1.0e-9 * (fabs(a) + fabs(b) + v.dims[i]);
      if (fmin(a, b) > v.dims[i] + pad || fmax(a, b) < -v.dims[i] - pad) return ADEPT_INF;
    }
  }
  return solid_entry(v, lp, ld);
}

// ---------------------------------------------------------------- warp-cooperative BVH
__device__ __forceinline__ double warp_min(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(kFull, v, o));
  return v;
}
__device__ __forceinline__ float warp_min(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fminf(v, __shfl_xor_sync(kFull, v, o));
  return v;
}
__device__ __forceinline__ int warp_min_int(int v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = min(v, __shfl_xor_sync(kFull, v, o));
  return v;
}

// lane tests box `i` (< n valid) of a SoA box array of stride `stride` against the ray; returns hit
template <typename R>
__device__ __forceinline__ bool ray_box(const R* __restrict__ box, int stride, int i, bool valid, R px, R py, R pz, R ix, R iy, R iz,
                                        R best) {
  if (!valid) return false;
  const R lx = __ldg(box + i), ly = __ldg(box + stride + i), lz = __ldg(box + 2 * stride + i);
  const R hx = __ldg(box + 3 * stride + i), hy = __ldg(box + 4 * stride + i), hz = __ldg(box + 5 * stride + i);
  const R ax = (lx - px) * ix, bx = (hx - px) * ix;
  const R ay = (ly - py) * iy, by = (hy - py) * iy;
  const R az = (lz - pz) * iz, bz = (hz - pz) * iz;
  // fmin/fmax drop NaN operands (0 * inf when the ray is parallel to a slab and starts on its plane)
  const R tn = r_max(r_max(r_min(ax, bx), r_min(ay, by)), r_min(az, bz));
  const R tf = r_min(r_min(r_max(ax, bx), r_max(ay, by)), r_max(az, bz));
  return tn <= tf && tf >= R(0) && tn < best;
}

template <typename R>
__device__ __forceinline__ bool point_box(const R* __restrict__ box, int stride, int i, bool valid, R px, R py, R pz) {
  if (!valid) return false;
  return px >= __ldg(box + i) && py >= __ldg(box + stride + i) && pz >= __ldg(box + 2 * stride + i) &&
         px <= __ldg(box + 3 * stride + i) && py <= __ldg(box + 4 * stride + i) && pz <= __ldg(box + 5 * stride + i);
}

// All arguments warp-uniform.  Returns min(best, nearest daughter entry distance).  The traversal
// state is a short stack of one 32-bit child mask per level, shared by the warp.
// `hit` (warp-uniform, out): touchable id of the daughter that gave the returned minimum, -1 if none did
// or two daughters tie.
template <typename R>
__device__ __forceinline__ R bvh_ray(const DevCtx& c, const BvhT<R>& b, R px, R py, R pz, R dx, R dy, R dz, R best, int& hit) {
  hit = -1;
  const int lane = threadIdx.x & 31;
  const R ix = R(1) / dx, iy = R(1) / dy, iz = R(1) / dz;
  const int top = b.n_levels - 1;
  unsigned mask[kBvhMaxLevels];
  int first[kBvhMaxLevels];
  int level = top;
  first[top] = 0;
  mask[top] = __ballot_sync(kFull, ray_box(b.node_box[top], b.n_nodes[top], lane, lane < b.n_nodes[top], px, py, pz,
                                           ix, iy, iz, best));
  for (;;) {
    if (mask[level] == 0) {
      if (level == top) break;
      ++level;
      continue;
    }
    const int ch = __ffs(mask[level]) - 1;
    mask[level] &= mask[level] - 1;
    const int node = first[level] + ch;
    const int base = node << 5;
    if (level == 0) {
      const int i = base + lane;
      R t = Geo<R>::inf();
      int pv = -1;
      if (ray_box(b.prim_box, b.n_prims, i, i < b.n_prims, px, py, pz, ix, iy, iz, best)) {
        pv = __ldg(b.prim_vol + i);
        t = entry_distance<R>(c, pv, px, py, pz, dx, dy, dz);
      }
      const R m = warp_min(t);
      if (m < best) {
        best = m;
        const unsigned w = __ballot_sync(kFull, t == m);
        hit = __shfl_sync(kFull, pv, __ffs(w) - 1);
        if (w & (w - 1)) hit = -1;
      }
    } else {
      const int n = b.n_nodes[level - 1];
      const int i = base + lane;
      first[level - 1] = base;
      mask[level - 1] = __ballot_sync(kFull, ray_box(b.node_box[level - 1], n, i, i < n, px, py, pz, ix, iy, iz, best));
      --level;
    }
  }
  return best;
}

// All arguments warp-uniform.  Lowest touchable id among the daughters containing the point, or -1.
template <typename R>
__device__ __forceinline__ int bvh_point(const DevCtx& c, const BvhT<R>& b, R px, R py, R pz) {
  const int lane = threadIdx.x & 31;
  const int top = b.n_levels - 1;
  unsigned mask[kBvhMaxLevels];
  int first[kBvhMaxLevels];
  int level = top;
  int found = 0x7fffffff;
  first[top] = 0;
  mask[top] = __ballot_sync(kFull, point_box(b.node_box[top], b.n_nodes[top], lane, lane < b.n_nodes[top], px, py, pz));
  for (;;) {
    if (mask[level] == 0) {
      if (level == top) break;
      ++level;
      continue;
    }
    const int ch = __ffs(mask[level]) - 1;
    mask[level] &= mask[level] - 1;
    const int base = (first[level] + ch) << 5;
    const int i = base + lane;
    if (level == 0) {
      int hit = 0x7fffffff;
      if (point_box(b.prim_box, b.n_prims, i, i < b.n_prims, px, py, pz)) {
        const int v = __ldg(b.prim_vol + i);
        if (inside_volume<R>(c, v, px, py, pz)) hit = v;
      }
      found = min(found, warp_min_int(hit));
    } else {
      const int n = b.n_nodes[level - 1];
      first[level - 1] = base;
      mask[level - 1] = __ballot_sync(kFull, point_box(b.node_box[level - 1], n, i, i < n, px, py, pz));
      --level;
    }
  }
  return found == 0x7fffffff ? -1 : found;
}

// ---------------------------------------------------------------- candidate lists
// Most queries in a BVH volume are asked from a place whose surroundings are already known.  A NavCache says:
// "every daughter of `vol` that comes within `reach` of the point q0 is in `list`".  A segment from p of length
// s can then only enter listed daughters if |p - q0| + s <= reach, so the query is a lane-local loop of exact
// entry tests over the list -- no traversal, no warp cooperation -- and because the minimum is taken over a
// superset of the daughters the traversal would test exactly, by the same entry_distance, the result is
// bit-identical.  For a longer ray the list is tried first: a hit closer than reach - |p - q0| is final, else the
// traversal starts from that bound.  Two sources of lists:
//  * per daughter, built once by adept_init (DevBvh::nbr): the siblings within DevBvh::nbr_reach of the daughter's
//    solid (and the daughter itself).  A track that has just left daughter A into the mother is within the push
//    distance of A, so the list of A serves with reach = nbr_reach - margin around its exit point.  This is the
//    crystal -> gap -> crystal passage, i.e. nearly every query of a shower in a barrel of crystals.
//  * per lane, built on the spot by the warp (bvh_candidates) around a track that keeps asking from within a small
//    ball: 16 chords per step, step after step, of the e+- that spiral in the gaps (profiles/r1e_configs34.md:
//    82 % of the instructions of such a step were traversals).
#ifndef ADEPT_CAND_CAP
#define ADEPT_CAND_CAP 12
#endif
#ifndef ADEPT_CAND_MULT
#define ADEPT_CAND_MULT 8.0
#endif
#ifndef ADEPT_CAND_RMAX
#define ADEPT_CAND_RMAX 2.0
#endif
constexpr int kCandCap = ADEPT_CAND_CAP;             // entries of a lane-built list (a gap corner touches 4 crystals)
// (measured on configs 4 / 5, profiles/r2_summary.md: cap 8, ball 4 segments <= 1 cm: 1130 ms / 21.7 events/s; 12, 8, 2 cm: 1084 / 22.6)
constexpr double kCandRadius = 0.25;    // [cm] least radius of the ball a lane-built list covers ...
constexpr double kCandRadiusMax = ADEPT_CAND_RMAX;  // ... and the largest: the ball is sized to serve the next few segments of the track that asks
                                        // (ADEPT_CAND_MULT times the segment that triggered it; a list whose ball the very next chord leaves is
                                        // pure cost -- profiles/r2_summary.md: 18 % of the samples of a config-4 launch were such builds)
constexpr int kNbrCap = 12;             // entries of a per-daughter list
struct NavCache {
  double qx, qy, qz, reach;             // see above (reach <= 0: no list)
  const int32_t* list;
  uint32_t vol;                         // the BVH volume the list belongs to
  int count, queries;                   // entries; traversals made in `vol` since the last list
};
__device__ __forceinline__ void nav_cache_reset(NavCache& k) {
  k.qx = k.qy = k.qz = 0.0; k.reach = -1.0; k.list = nullptr; k.vol = kDeadVolume; k.count = 0; k.queries = 0;
}

// A track has crossed from volume `from` into `into` at (x, y, z): if `from` is a daughter of the BVH volume `into`
// with a neighbour list, that list serves the next queries.
__device__ __forceinline__ void nav_cache_left_daughter(const DevCtx& c, NavCache& k, uint32_t from, int into, double x, double y, double z) {
  if (into < 0) return;
  const DevVolume& m = volume(c, into);
  if (m.bvh < 0 || volume(c, from).mother != into) return;
  const DevBvh& b = c.bvh[m.bvh];
  if (b.nbr_reach <= 0.0) return;
  const int d = static_cast<int>(from) - m.dbegin;
  const int n = __ldg(b.nbr_count + d);
  if (n < 0) return;
  k.qx = x; k.qy = y; k.qz = z;
  k.reach = b.nbr_reach - 1.0e-5;        // the exit point is within the push distance (and rounding) of `from`
  k.list = b.nbr + static_cast<size_t>(d) * kNbrCap;
  k.vol = static_cast<uint32_t>(into); k.count = n; k.queries = 0;
}

// All arguments warp-uniform; list = the requesting lane's kCandCap entries in shared memory.
// Returns the number of daughters within rho of (px, py, pz), or -1 if they do not fit the list.
__device__ __forceinline__ int bvh_candidates(const DevCtx& c, const DevBvh& b, double px, double py, double pz, double rho,
                                              int32_t* list) {
  const int lane = threadIdx.x & 31;
  const unsigned lt = (1u << lane) - 1u;
  const double pad = rho * (1.0 + 1.0e-9) + 1.0e-12;
  const auto near_box = [&](const double* __restrict__ box, int stride, int i, bool valid) {
    if (!valid) return false;
    return px >= __ldg(box + i) - pad && py >= __ldg(box + stride + i) - pad && pz >= __ldg(box + 2 * stride + i) - pad &&
           px <= __ldg(box + 3 * stride + i) + pad && py <= __ldg(box + 4 * stride + i) + pad && pz <= __ldg(box + 5 * stride + i) + pad;
  };
  const int top = b.n_levels - 1;
  unsigned mask[kBvhMaxLevels];
  int first[kBvhMaxLevels];
  int level = top, count = 0;
  first[top] = 0;
  mask[top] = __ballot_sync(kFull, near_box(b.node_box[top], b.n_nodes[top], lane, lane < b.n_nodes[top]));
  for (;;) {
    if (mask[level] == 0) {
      if (level == top) break;
      ++level;
      continue;
    }
    const int ch = __ffs(mask[level]) - 1;
    mask[level] &= mask[level] - 1;
    const int base = (first[level] + ch) << 5;
    const int i = base + lane;
    if (level == 0) {
      bool ok = false;
      int pv = -1;
      if (near_box(b.prim_box, b.n_prims, i, i < b.n_prims)) {
        pv = __ldg(b.prim_vol + i);
        const DevVolume& v = volume(c, pv);
        ok = true;
        if (v.solid == ADEPT_BOX) {   // the oriented box itself, inflated
          double l[3];
          to_local(c, pv, v, px, py, pz, l);
          ok = fabs(l[0]) <= v.dims[0] + pad && fabs(l[1]) <= v.dims[1] + pad && fabs(l[2]) <= v.dims[2] + pad;
        }
      }
      const unsigned m = __ballot_sync(kFull, ok);
      const int at = count + __popc(m & lt);
      if (ok && at < kCandCap) list[at] = pv;
      count += __popc(m);
    } else {
      const int n = b.n_nodes[level - 1];
      first[level - 1] = base;
      mask[level - 1] = __ballot_sync(kFull, near_box(b.node_box[level - 1], n, i, i < n));
      --level;
    }
  }
  __syncwarp();
  return count <= kCandCap ? count : -1;
}

// ---------------------------------------------------------------- G3 distance to boundary
// min(exit distance of the own solid, entry distance of every daughter), capped at s_max.
// Warp-convergent call; lanes with active == false return s_max.
// BVH = false instantiates the pure loop navigator (geometries without a BVH volume): no cooperative code.
// `face` (out) is the relocation hint (nav_relocate): when the returned distance is the exit of the volume's
// own box through one face and no daughter is entered first, the face index 2 * axis + (direction > 0) in
// the volume's frame -- the key of the hint table; when it is the entry into daughter d, -2 - d; -1 when
// neither is known (the cap s_max, a tube, a tie).
// Inlined into the step kernels (3.7 % of a config-2 pass, 5 % of a config-4 pass, 20 % of the ray-cast over
// calls: no argument moves, and the compiler schedules the box test into the surrounding phase), and so are
// the cooperative traversals bvh_ray / bvh_point (another 5 % of a config-4 pass).
// `cache` (BVH only, warp-uniformly null or not): the lane's candidate list (see above); `cand` (may be null): the
// block's shared-memory room for lane-built lists -- with it, a lane that traverses twice in a row in the same
// volume gets a list around its current point.
template <bool BVH, typename R>
__device__ __forceinline__ R nav_distance_body(const DevCtx& c, int nav, bool active, R px, R py, R pz, R dx, R dy, R dz, uint32_t vol,
                                               R s_max, int& face, NavCache* cache = nullptr, int32_t* cand = nullptr,
                                               bool skip_own = false) {
  const int lane = threadIdx.x & 31;
  R s = s_max;
  bool need = false;
  int bvh = -1;
  face = -1;
  if (active) {
    const VolT<R>& v = Geo<R>::vol(c, vol);
    if (!skip_own) {   // (skip_own: the caller knows the segment ends before the volume's own surface, nav_safety)
      R lp[3], ld[3];
      to_local(c, vol, v, px, py, pz, lp);
      dir_to_local(c, vol, v, dx, dy, dz, ld);
      int f;
      const R s_exit = solid_exit(v, lp, ld, f);
      if (s_exit < s_max) { s = s_exit; face = f; }
    }
    if (v.dcount > 0) {
      if (BVH && nav == ADEPT_NAV_BVH && v.bvh >= 0) {
        need = true;
        bvh = v.bvh;
      } else {
        for (int k = 0; k < v.dcount; ++k) {
          const R e = entry_distance<R>(c, v.dbegin + k, px, py, pz, dx, dy, dz);
          if (e <= s) { face = e < s ? -2 - (v.dbegin + k) : -1; s = e; }
        }
      }
    }
  }
  if (!BVH) return s;
  if constexpr (std::is_same<R, double>::value) if (cache) {
    // the lane's candidate list first (lane-local): final if the segment cannot leave its reach
    const auto ask_list = [&]() {
      for (int j = 0; j < cache->count; ++j) {
        const int pv = cache->list[j];
        const double e = entry_distance_within(c, pv, px, py, pz, dx, dy, dz, s);
        if (e <= s) { face = e < s ? -2 - pv : -1; s = e; }   // (a tie between two daughters: no hint, as in bvh_ray)
      }
      const double ox = px - cache->qx, oy = py - cache->qy, oz = pz - cache->qz;
      if (sqrt(ox * ox + oy * oy + oz * oz) + s <= cache->reach * (1.0 - 1.0e-9)) need = false;
    };
    if (need && cache->reach > 0.0 && cache->vol == vol) ask_list();
    // A lane that keeps asking in the same volume -- its list has just run out, or this is its second uncovered
    // query there -- gets a list of its own around where it is, built by the warp (one cooperative walk, the price
    // of one traversal) BEFORE the query is answered, so that the list answers it and the next few: a ball of
    // ADEPT_CAND_MULT segment lengths.  (A longer segment would leave any ball that still fits a list; a first query in a volume
    // is a traversal: most tracks only pass through.)
    bool build = false;
    const double rho = fmax(kCandRadius, ADEPT_CAND_MULT * static_cast<double>(s_max));
    if (need && cand && rho <= kCandRadiusMax) {
      if (cache->vol != vol) { cache->vol = vol; cache->queries = 0; cache->reach = -1.0; }
      build = cache->reach > 0.0 || ++cache->queries >= 2;
    }
    unsigned mb = __ballot_sync(kFull, build);
    while (mb) {
      const int src = __ffs(mb) - 1;
      mb &= mb - 1;
      int32_t* mine = cand + kCandCap * ((threadIdx.x & ~31) + src);
      const int n = bvh_candidates(c, c.bvh[__shfl_sync(kFull, bvh, src)], __shfl_sync(kFull, px, src), __shfl_sync(kFull, py, src),
                                   __shfl_sync(kFull, pz, src), __shfl_sync(kFull, rho, src), mine);
      if (lane == src) {
        cache->qx = px; cache->qy = py; cache->qz = pz;
        cache->reach = n >= 0 ? rho : -1.0;
        cache->list = mine;
        cache->count = n >= 0 ? n : 0;
        cache->queries = n >= 0 ? 0 : -6;  // (did not fit: traverse now, and the next seven times)
      }
    }
    if (build && cache->reach > 0.0) ask_list();
  }
  unsigned m = __ballot_sync(kFull, need);
  while (m) {
    const int src = __ffs(m) - 1;
    m &= m - 1;
    int hit;
    const R r = bvh_ray<R>(c, Geo<R>::bvh(c, __shfl_sync(kFull, bvh, src)), __shfl_sync(kFull, px, src),
                           __shfl_sync(kFull, py, src), __shfl_sync(kFull, pz, src), __shfl_sync(kFull, dx, src),
                           __shfl_sync(kFull, dy, src), __shfl_sync(kFull, dz, src), __shfl_sync(kFull, s, src), hit);
    if (lane == src && r < s) { s = r; face = hit >= 0 ? -2 - hit : -1; }
  }
  return s;
}
template <bool BVH = true, typename R = double>
__device__ __forceinline__ R nav_distance(const DevCtx& c, int nav, bool active, R px, R py, R pz, R dx, R dy, R dz, uint32_t vol, R s_max,
                                          int& face, NavCache* cache = nullptr, int32_t* cand = nullptr, bool skip_own = false) {
  return nav_distance_body<BVH, R>(c, nav, active, px, py, pz, dx, dy, dz, vol, s_max, face, cache, cand, skip_own);
}
template <bool BVH = true>
__device__ __forceinline__ double nav_distance(const DevCtx& c, int nav, bool active, double px, double py, double pz, double dx,
                                               double dy, double dz, uint32_t vol, double s_max) {
  int face;
  return nav_distance<BVH, double>(c, nav, active, px, py, pz, dx, dy, dz, vol, s_max, face);
}

// ---------------------------------------------------------------- safety (reading A)
// A lower bound on the distance from a point inside volume `vol` (and inside none of its daughters) to the
// nearest boundary of the volume: its own surface or any daughter.  Only used to decide that a chord of the
// field propagation shorter than this bound cannot reach a boundary, so that its geometry query can be skipped
// -- the result of the step is the same with or without it (the oracle has no safety at all).  Conservative by
// construction: distances to the own surface are exact or under-estimated, a daughter's is bounded by the
// largest per-axis separation (<= the Euclidean distance); 1e-6 relative and 1e-9 cm are taken off for
// rounding.  Lane-local.  For a volume whose daughters sit in a BVH there is no cheap bound on them: `own_only` is
// set and the value bounds the distance to the volume's own surface only (the query then skips the own solid).
__device__ __forceinline__ double solid_safety_in(const DevVolume& v, const double p[3]) {
  if (v.solid == ADEPT_BOX) return fmin(fmin(v.dims[0] - fabs(p[0]), v.dims[1] - fabs(p[1])), v.dims[2] - fabs(p[2]));
  const double r = sqrt(p[0] * p[0] + p[1] * p[1]);
  double s = fmin(v.dims[1] - r, v.dims[2] - fabs(p[2]));
  if (v.dims[0] > 0.0) s = fmin(s, r - v.dims[0]);
  return s;
}
__device__ __forceinline__ double solid_safety_out(const DevVolume& v, const double p[3]) {
  if (v.solid == ADEPT_BOX) return fmax(fmax(fabs(p[0]) - v.dims[0], fabs(p[1]) - v.dims[1]), fabs(p[2]) - v.dims[2]);
  const double r = sqrt(p[0] * p[0] + p[1] * p[1]);
  return fmax(fmax(r - v.dims[1], v.dims[0] - r), fabs(p[2]) - v.dims[2]);
}
__device__ __forceinline__ double nav_safety(const DevCtx& c, uint32_t vol, double px, double py, double pz, bool& own_only) {
  const DevVolume& v = volume(c, vol);
  double l[3];
  to_local(c, vol, v, px, py, pz, l);
  double s = solid_safety_in(v, l);
  own_only = v.dcount > 0 && v.bvh >= 0;
  for (int k = 0; !own_only && k < v.dcount && s > 0.0; ++k) {
    const DevVolume& d = volume(c, v.dbegin + k);
    to_local(c, v.dbegin + k, d, px, py, pz, l);
    s = fmin(s, solid_safety_out(d, l));
  }
  return s * (1.0 - 1.0e-6) - 1.0e-9;
}

// ---------------------------------------------------------------- G4 Locate
// From the world down, descend into the first daughter (index order) containing the point.
// Warp-convergent call; returns -1 outside the world or for inactive lanes.
template <bool BVH = true, typename R = double>
__device__ __noinline__ int nav_locate(const DevCtx& c, int nav, bool active, R qx, R qy, R qz) {
  const int lane = threadIdx.x & 31;
  int cur = -1;
  bool desc = false;
  if (active && inside_volume<R>(c, 0, qx, qy, qz)) {
    cur = 0;
    desc = true;
  }
  if (!BVH) {  // lane-local descent, no warp cooperation needed
    while (desc) {
      const VolT<R>& v = Geo<R>::vol(c, cur);
      int next = -1;
      for (int k = 0; k < v.dcount; ++k) {
        if (inside_volume<R>(c, v.dbegin + k, qx, qy, qz)) { next = v.dbegin + k; break; }
      }
      if (next < 0) desc = false; else cur = next;
    }
    return cur;
  }
  while (__any_sync(kFull, desc)) {
    bool need = false;
    int bvh = -1;
    if (desc) {
      const VolT<R>& v = Geo<R>::vol(c, cur);
      if (v.dcount == 0) {
        desc = false;
      } else if (nav == ADEPT_NAV_BVH && v.bvh >= 0) {
        need = true;
        bvh = v.bvh;
      } else {
        int next = -1;
        for (int k = 0; k < v.dcount; ++k) {
          if (inside_volume<R>(c, v.dbegin + k, qx, qy, qz)) { next = v.dbegin + k; break; }
        }
        if (next < 0) desc = false; else cur = next;
      }
    }
    unsigned m = __ballot_sync(kFull, need);
    while (m) {
      const int src = __ffs(m) - 1;
      m &= m - 1;
      const int r = bvh_point<R>(c, Geo<R>::bvh(c, __shfl_sync(kFull, bvh, src)), __shfl_sync(kFull, qx, src),
                                 __shfl_sync(kFull, qy, src), __shfl_sync(kFull, qz, src));
      if (lane == src) {
        if (r < 0) desc = false; else cur = r;
      }
    }
  }
  return cur;
}

// ---------------------------------------------------------------- A5 relocation after a boundary
// Same result as nav_locate(q) -- the deepest volume containing q -- found locally: climb from the
// volume the track was in until q is inside, then descend.  Daughters lie inside their mothers and
// siblings are disjoint (adept.h), so at most one daughter contains q and the order in which they are
// tried cannot change the answer: the neighbours (in index order) of the daughter just left are tried
// first, which makes a crossing between consecutive layers of a stack O(1) instead of O(layers)
// (relocation cost and "fewer trial steps").  Warp-convergent call when BVH is true.
// Returns -1 outside the world or for inactive lanes.
//
// Hints (`face`, from nav_distance).  face >= 0: hint table (DevCtx::nbr, built once by adept_init with
// hint_kernel): nbr[6 v + f] = Locate of the point just outside the centre of face f of box volume v.
// face <= -2: the daughter -2 - face the step ended on.  Either way that one candidate is tested first; if the pushed point is inside it, the descent
// starts there -- the deepest volume containing q is unique, so the answer is the same as the climb's --
// and in a stack of slabs a crossing costs one containment test instead of four or five dependent ones.
template <bool BVH, typename R>
__device__ __forceinline__ int nav_relocate_body(const DevCtx& c, int nav, bool active, uint32_t vol_old, R qx, R qy, R qz, int face) {
  int cur = -1, prev = -1;
  bool desc = false, done = false;
  if (active) {
    const int cand = face >= 0 ? __ldg(c.nbr + 6 * static_cast<size_t>(vol_old) + face) : (face <= -2 ? -2 - face : -1);
    if (cand >= 0 && inside_volume<R>(c, cand, qx, qy, qz)) {
      cur = cand;
      // Out of an ISOLATED daughter (adept_init: a box with no sibling within kIsolationMargin of it) into
      // its mother: a point outside the box but within margin / 2 of it along every local axis is nearer
      // than the margin to the box, so no sibling can contain it and the mother is the answer -- no
      // descent, i.e. no BVH point query per crystal-to-gap crossing.  Checked here, not assumed, so the
      // result is Locate(q) for any q and any hint.
      if (face >= 0) {
        const VolT<R>& vo = Geo<R>::vol(c, vol_old);
        if (vo.isolated && vo.mother == cand) {
          R l[3];
          to_local(c, vol_old, vo, qx, qy, qz, l);
          const R a0 = r_abs(l[0]) - vo.dims[0], a1 = r_abs(l[1]) - vo.dims[1], a2 = r_abs(l[2]) - vo.dims[2];
          const R out = r_max(a0, r_max(a1, a2));      // > 0: outside the box; <= margin / 2: within reach of no sibling
          done = out > R(0) && out <= R(0.5 * kIsolationMargin);
        }
      }
    } else {
      cur = static_cast<int>(vol_old);
      while (cur >= 0 && !inside_volume<R>(c, cur, qx, qy, qz)) { prev = cur; cur = Geo<R>::vol(c, cur).mother; }
    }
    desc = cur >= 0 && !done;
  }
  for (;;) {
    if (BVH) { if (!__any_sync(kFull, desc)) break; } else if (!desc) break;
    bool need = false;
    int bvh = -1;
    if (desc) {
      const VolT<R>& v = Geo<R>::vol(c, cur);
      if (v.dcount == 0) {
        desc = false;
      } else if (BVH && nav == ADEPT_NAV_BVH && v.bvh >= 0) {
        need = true;
        bvh = v.bvh;
      } else {
        int next = -1;
        if (prev >= 0) {  // came up from daughter `prev` (q is outside it): try its neighbours first
          const int k0 = prev - v.dbegin;
          if (k0 + 1 < v.dcount && inside_volume<R>(c, prev + 1, qx, qy, qz)) next = prev + 1;
          else if (k0 >= 1 && inside_volume<R>(c, prev - 1, qx, qy, qz)) next = prev - 1;
        }
        for (int k = 0; next < 0 && k < v.dcount; ++k) {
          const int d = v.dbegin + k;
          if (prev >= 0 && (d == prev || d == prev + 1 || d == prev - 1)) continue;
          if (inside_volume<R>(c, d, qx, qy, qz)) next = d;
        }
        if (next < 0) desc = false; else cur = next;
        prev = -1;
      }
    }
    if (BVH) {
      unsigned m = __ballot_sync(kFull, need);
      const int lane = threadIdx.x & 31;
      while (m) {
        const int src = __ffs(m) - 1;
        m &= m - 1;
        const int r = bvh_point<R>(c, Geo<R>::bvh(c, __shfl_sync(kFull, bvh, src)), __shfl_sync(kFull, qx, src),
                                   __shfl_sync(kFull, qy, src), __shfl_sync(kFull, qz, src));
        if (lane == src) {
          if (r < 0) desc = false; else cur = r;
          prev = -1;
        }
      }
    }
  }
  return cur;
}
template <bool BVH = true, typename R = double>
__device__ __forceinline__ int nav_relocate(const DevCtx& c, int nav, bool active, uint32_t vol_old, R qx, R qy, R qz, int face = -1) {
  return nav_relocate_body<BVH, R>(c, nav, active, vol_old, qx, qy, qz, face);
}

}  // namespace adept
