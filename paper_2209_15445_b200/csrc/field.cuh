// Charged-track propagation in a magnetic field by sagitta-limited chords  (SURVEY.md §8 row A6,
// §8(c) F1-F6).  Uniform field: exact helix end points.  Field map: one classical RK4
// step per chord.  The chord loop is warp-convergent (lanes that finished idle inside it) so that the
// geometry query of every chord can use the warp-cooperative BVH; the chord budget (F4) bounds the
// divergence the paper measured.
#pragma once
#include "geom.cuh"

namespace adept {

__device__ __forceinline__ void cross3(const double a[3], const double b[3], double c[3]) {
  c[0] = a[1] * b[2] - a[2] * b[1];
  c[1] = a[2] * b[0] - a[0] * b[2];
  c[2] = a[0] * b[1] - a[1] * b[0];
}

// F6: B = (0, 0, bz(r, z)), bilinear, clamped outside the grid.  FIELD >= 0: the field kind, known at compile time
// (no test of it per evaluation: four evaluations per RK4 chord); -1: read from the context.
template <int FIELD = -1>
__device__ __forceinline__ void field_at(const DevCtx& c, const double p[3], double B[3]) {
  const int kind = FIELD >= 0 ? FIELD : c.field_kind;
  if (kind == ADEPT_FIELD_UNIFORM) { B[0] = c.B[0]; B[1] = c.B[1]; B[2] = c.B[2]; return; }
  B[0] = B[1] = B[2] = 0.0;
  if (kind != ADEPT_FIELD_MAP_RZ) return;
  const double r = sqrt(p[0] * p[0] + p[1] * p[1]);
  // (grid coordinates by multiplication with the inverse spacing: exact for the 1 cm grid of the configs, within
  // an ulp otherwise, and the interpolant is continuous across cells)
  double fr = (r - c.r0) * c.inv_dr, fz = (p[2] - c.z0) * c.inv_dz;
  fr = fmin(fmax(fr, 0.0), c.fr_max);
  fz = fmin(fmax(fz, 0.0), c.fz_max);
  const int ir = min(static_cast<int>(fr), c.nr - 2);
  const int iz = min(static_cast<int>(fz), c.nz - 2);
  const double a = fr - ir, b = fz - iz;
  const double* m = c.bz + iz * c.nr + ir;
  const double v00 = __ldg(m), v01 = __ldg(m + 1), v10 = __ldg(m + c.nr), v11 = __ldg(m + c.nr + 1);
  const double lo = v00 + a * (v01 - v00);
  const double hi = v10 + a * (v11 - v10);
  B[2] = lo + b * (hi - lo);
}

// sin and cos of a small angle by their Maclaurin series (|x| <= 0.8: the terms dropped, x^19/19! and x^20/20!,
// are below 2e-19).  A chord turns the track by omega = sqrt(8 delta / R) about B, half of that is what the helix
// needs; libdevice's sincos spends most of its ~90 instructions on argument reduction that cannot be needed here.
__device__ __forceinline__ void sincos_small(double x, double& sn, double& cs) {
  const double z = x * x;
  double p = -1.0 / 355687428096000.0;          // -1/17!
  p = fma(p, z, 1.0 / 1307674368000.0);         //  1/15!
  p = fma(p, z, -1.0 / 6227020800.0);           // -1/13!
  p = fma(p, z, 1.0 / 39916800.0);              //  1/11!
  p = fma(p, z, -1.0 / 362880.0);               // -1/9!
  p = fma(p, z, 1.0 / 5040.0);                  //  1/7!
  p = fma(p, z, -1.0 / 120.0);                  // -1/5!
  p = fma(p, z, 1.0 / 6.0);                     //  1/3!
  sn = fma(-x * z, p, x);
  double q = 1.0 / 6402373705728000.0;          //  1/18!
  q = fma(q, z, -1.0 / 20922789888000.0);       // -1/16!
  q = fma(q, z, 1.0 / 87178291200.0);           //  1/14!
  q = fma(q, z, -1.0 / 479001600.0);            // -1/12!
  q = fma(q, z, 1.0 / 3628800.0);               //  1/10!
  q = fma(q, z, -1.0 / 40320.0);                // -1/8!
  q = fma(q, z, 1.0 / 720.0);                   //  1/6!
  q = fma(q, z, -1.0 / 24.0);                   // -1/4!
  q = fma(q, z, 0.5);                           //  1/2!
  cs = fma(-z, q, 1.0);
}

// sin and cos of an angle too large for the series: libdevice's routine, out of line (the chord loop is the hottest code
// of the field kernels and misses the instruction cache as it is; a chord turns the track by more than 1.6 rad only
// below ~3 keV at 3.8 T)
__device__ __noinline__ void sincos_large(double x, double* sn, double* cs) { sincos(x, sn, cs); }

// F3: exact helix about the unit vector b; kappa = -q kCB |B| / p is the turning angle per unit path length
// (constant over a step: F1 takes p at the pre-step energy), so omega = kappa h and h / omega = 1 / kappa.
// sin(omega), cos(omega) and 1 - cos(omega) all come from the half angle.
// inlined (as rk4): as calls their array arguments lived in local memory (config 3: 251 -> 227 ms per pass)
__device__ __forceinline__ void helix(const double b[3], double kappa, double inv_kappa, double h, const double p[3],
                                      const double d[3], double p1[3], double d1[3]) {
  const double half = 0.5 * kappa * h;
  double s2, c2;
  if (fabs(half) <= 0.8) sincos_small(half, s2, c2);
  else sincos_large(half, &s2, &c2);
  const double so = 2.0 * s2 * c2, omc = 2.0 * s2 * s2, co = 1.0 - omc;
  const double dpar = d[0] * b[0] + d[1] * b[1] + d[2] * b[2];
  const double dl[3] = {dpar * b[0], dpar * b[1], dpar * b[2]};
  const double dt[3] = {d[0] - dl[0], d[1] - dl[1], d[2] - dl[2]};
  double bxd[3];
  cross3(b, dt, bxd);
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    d1[i] = dl[i] + dt[i] * co + bxd[i] * so;
    p1[i] = p[i] + dl[i] * h + inv_kappa * (dt[i] * so + bxd[i] * omc);
  }
}

// ... and its direction alone (the tangent at a boundary hit): the same arithmetic as helix() for d1
__device__ __forceinline__ void helix_dir(const double b[3], double kappa, double h, const double d[3], double d1[3]) {
  const double half = 0.5 * kappa * h;
  double s2, c2;
  if (fabs(half) <= 0.8) sincos_small(half, s2, c2);
  else sincos_large(half, &s2, &c2);
  const double so = 2.0 * s2 * c2, omc = 2.0 * s2 * s2, co = 1.0 - omc;
  const double dpar = d[0] * b[0] + d[1] * b[1] + d[2] * b[2];
  const double dl[3] = {dpar * b[0], dpar * b[1], dpar * b[2]};
  const double dt[3] = {d[0] - dl[0], d[1] - dl[1], d[2] - dl[2]};
  double bxd[3];
  cross3(b, dt, bxd);
#pragma unroll
  for (int i = 0; i < 3; ++i) d1[i] = dl[i] + dt[i] * co + bxd[i] * so;
}

// F1, F3: one classical RK4 step on (x, d): x' = d, d' = (q kCB / p) d x B(x); B0 = B(p), already known
template <int FIELD = -1>
__device__ __forceinline__ void rk4(const DevCtx& c, int charge, double pmom, double h, const double p[3],
                                    const double d[3], const double B0[3], double p1[3], double d1[3]) {
  const double kap = charge * kCB / pmom;
  double B[3], k1v[3], k2v[3], k3v[3], k4v[3], k2x[3], k3x[3], k4x[3], x[3], v[3], t[3];
  cross3(d, B0, t);
#pragma unroll
  for (int i = 0; i < 3; ++i) { k1v[i] = kap * t[i]; x[i] = p[i] + 0.5 * h * d[i]; v[i] = d[i] + 0.5 * h * k1v[i]; }
  field_at<FIELD>(c, x, B);
  cross3(v, B, t);
#pragma unroll
  for (int i = 0; i < 3; ++i) { k2x[i] = v[i]; k2v[i] = kap * t[i]; x[i] = p[i] + 0.5 * h * k2x[i]; v[i] = d[i] + 0.5 * h * k2v[i]; }
  field_at<FIELD>(c, x, B);
  cross3(v, B, t);
#pragma unroll
  for (int i = 0; i < 3; ++i) { k3x[i] = v[i]; k3v[i] = kap * t[i]; x[i] = p[i] + h * k3x[i]; v[i] = d[i] + h * k3v[i]; }
  field_at<FIELD>(c, x, B);
  cross3(v, B, t);
  double n = 0.0;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    k4x[i] = v[i]; k4v[i] = kap * t[i];
    p1[i] = p[i] + (h / 6.0) * (d[i] + 2.0 * k2x[i] + 2.0 * k3x[i] + k4x[i]);
    d1[i] = d[i] + (h / 6.0) * (k1v[i] + 2.0 * k2v[i] + 2.0 * k3v[i] + k4v[i]);
    n += d1[i] * d1[i];
  }
  n = rsqrt(n);
#pragma unroll
  for (int i = 0; i < 3; ++i) d1[i] *= n;
}

// F2-F4 chord loop.  flag: 0 physics limit reached, 1 boundary (pos = hit point without the push,
// pushdir = chord direction), 2 truncated (chord budget).  Warp-convergent.
// FIELD >= 0 fixes the field kind at compile time (no helix / RK4 code where it cannot run); -1 = runtime.
//
// What the loop does NOT do per chord (measured: config 3 spent 4.5 us per chord of its spiralling tracks, a
// chain of ~900 dependent instructions): the constants of a uniform field (|B|, B / |B|, the turning rate kappa)
// are taken once per step; sines and cosines of the small turning angle come from their series; and the
// geometry query of a chord is skipped while the track is provably farther from every boundary than the chord is
// long (nav_safety; SURVEY.md F5 reading A: "safety only decides whether the chord's geometry query can be
// skipped" -- the outcome of the step is the same, so the oracle has no safety at all).  A safety is computed
// when a step needs more than one chord, and again when it is used up.
template <int FIELD = -1, bool BVH = true>
__device__ __forceinline__ int propagate(const DevCtx& c, int nav, bool active, int charge, double ekin, double pos[3], double dir[3],
                         uint32_t vol, double s_phys, double& s_out, int& chords_out, double pushdir[3], int& face_out,
                         NavCache* cache = nullptr, int32_t* cand = nullptr) {
  const int field_kind = FIELD >= 0 ? FIELD : c.field_kind;
  const double pmom = sqrt(ekin * (ekin + 2.0 * kMe));
  const double kappa = field_kind == ADEPT_FIELD_UNIFORM ? -charge * kCB * c.Bn / pmom : 0.0;
  const double inv_kappa = kappa != 0.0 ? 1.0 / kappa : 0.0;
  double s_done = 0.0;
  double safe = -1.0;   // clearance known to be left around pos (< 0: not known) ...
  bool own_only = false; // ... to the volume's own surface only (its daughters sit in a BVH)
  double h_step = -1.0; // uniform field: the chord length limit of this step (< 0: not yet known)
  int chords = 0, flag = 0, face_hit = -1;
  bool running = active;
#pragma unroll
  for (int i = 0; i < 3; ++i) pushdir[i] = dir[i];
  while (__any_sync(kFull, running)) {
    // --- per-lane: decide the next segment
    bool query = false, straight = false, last = false, chord = false, skip_own = false;
    double h = 0.0, L = 0.0, rest = 0.0;
    double u[3] = {0.0, 0.0, 0.0}, p1[3], d1[3], B[3] = {0.0, 0.0, 0.0};
    if (running) {
      if (s_done >= s_phys) {
        flag = 0; running = false;
      } else {
        // In a uniform field |d x B| is a constant of the motion, so the radius and the chord limit sqrt(8 delta R)
        // are those of the step's first chord (the oracle re-evaluates them per chord and finds the same numbers to
        // rounding).  On a field map they change from chord to chord.
        double bperp = 0.0, h_max = 0.0;
        const bool curved = charge != 0 && field_kind != ADEPT_FIELD_NONE;   // gammas go straight
        if (curved && (field_kind != ADEPT_FIELD_UNIFORM || h_step < 0.0)) {
          field_at<FIELD>(c, pos, B);
          double dxB[3];
          cross3(dir, B, dxB);
          bperp = sqrt(dxB[0] * dxB[0] + dxB[1] * dxB[1] + dxB[2] * dxB[2]);
          if (bperp != 0.0) {
            const double Rcurv = pmom / (kCB * bperp);
            h_max = sqrt(8.0 * c.delta_chord * Rcurv);
            if (field_kind == ADEPT_FIELD_MAP_RZ) {  // F2': at most 0.5 rad of turn per RK4 chord
              const double Bn = sqrt(B[0] * B[0] + B[1] * B[1] + B[2] * B[2]);
              h_max = fmin(h_max, 0.5 * pmom / (kCB * Bn));
            }
          }
          if (field_kind == ADEPT_FIELD_UNIFORM) h_step = h_max;   // 0: the track runs along B
        } else if (curved) {
          h_max = h_step;
        }
        rest = s_phys - s_done;
        if (!curved || h_max == 0.0) {
          straight = true; query = true; L = rest;
          u[0] = dir[0]; u[1] = dir[1]; u[2] = dir[2];
        } else if (chords >= c.chord_budget) {
          flag = 2; running = false;
        } else {
          last = h_max >= rest;
          h = last ? rest : h_max;
          if (field_kind == ADEPT_FIELD_UNIFORM) helix(c.bhat, kappa, inv_kappa, h, pos, dir, p1, d1);
          else rk4<FIELD>(c, charge, pmom, h, pos, dir, B, p1, d1);
          chord = true;
          // the chord needs no geometry query if it is shorter than the clearance left (a chord's length never
          // exceeds its arc's, so h bounds it)
          if (safe < h && !(last && safe < 0.0)) safe = nav_safety(c, vol, pos[0], pos[1], pos[2], own_only);
          const bool clear = h < safe;
          query = !clear || own_only;      // (own_only: the daughters still have to be asked, the own solid not)
          skip_own = clear;
          safe = clear ? safe - h : -1.0;
          if (cache && query && !last && cache->queries < 1) cache->queries = 1;   // a step of several chords: list at once
          if (query) {   // unit chord vector and length
            const double ch[3] = {p1[0] - pos[0], p1[1] - pos[1], p1[2] - pos[2]};
            const double L2 = ch[0] * ch[0] + ch[1] * ch[1] + ch[2] * ch[2];
            const double iL = rsqrt(L2);
            L = L2 * iL;
            u[0] = ch[0] * iL; u[1] = ch[1] * iL; u[2] = ch[2] * iL;
          }
        }
      }
    }
    // --- warp-cooperative geometry query of this segment
    int face;
    const double s_geo = nav_distance<BVH>(c, nav, query, pos[0], pos[1], pos[2], u[0], u[1], u[2], vol, L, face, cache, cand, skip_own);
    if (query) face_hit = face;   // only meaningful when this segment ends on the boundary (flag 1), which ends the loop
    if (straight) {
      pushdir[0] = u[0]; pushdir[1] = u[1]; pushdir[2] = u[2];
      if (s_geo < rest) {
#pragma unroll
        for (int i = 0; i < 3; ++i) pos[i] += s_geo * dir[i];
        s_done += s_geo; flag = 1;
      } else {
#pragma unroll
        for (int i = 0; i < 3; ++i) pos[i] += rest * dir[i];
        s_done = s_phys; flag = 0;
      }
      running = false;
    } else if (chord) {
      ++chords;
      if (query && s_geo < L) {
        const double frac = s_geo / L;
        double dh[3];
        if (field_kind == ADEPT_FIELD_UNIFORM) {
          helix_dir(c.bhat, kappa, h * frac, dir, dh);
        } else {
          double n = 0.0;
#pragma unroll
          for (int i = 0; i < 3; ++i) { dh[i] = dir[i] + frac * (d1[i] - dir[i]); n += dh[i] * dh[i]; }
          n = rsqrt(n);
#pragma unroll
          for (int i = 0; i < 3; ++i) dh[i] *= n;
        }
#pragma unroll
        for (int i = 0; i < 3; ++i) { pos[i] += s_geo * u[i]; dir[i] = dh[i]; pushdir[i] = u[i]; }
        s_done += h * frac; flag = 1; running = false;
      } else {
#pragma unroll
        for (int i = 0; i < 3; ++i) { pos[i] = p1[i]; dir[i] = d1[i]; }
        s_done = last ? s_phys : s_done + h;
      }
    }
  }
  s_out = s_done;
  chords_out = chords;
  face_out = flag == 1 ? face_hit : -1;
  return flag;
}

// ------------------------------------------------------------------------------------------------
// Wide form of the chord loop, for populations so small that a track has W = 8, 16 or 32 lanes of its warp to
// itself (charged.cuh: sparse tiles).  The tracks that outlive a shower by thousands of steps -- e+- spiralling
// in vacuum, 16 chords per step -- are one serial chain of chords each, and in the loop above every link of
// that chain is an integration step AND a geometry query (in a gap between crystals ~1 000 dependent
// instructions over the candidate list; profiles/r2_summary.md).  Only the integration is inherently serial:
// chord k+1 starts where chord k ends, whether or not chord k was tested yet.  So the lanes of the group
// integrate up to W chords ahead (all lanes redundantly, in lockstep; lane j keeps chord j), then lane j asks
// the geometry about chord j, and the first chord that ends on a boundary -- exactly the one the sequential
// loop would have stopped at -- decides the step; what was integrated beyond it is dropped.  On a field map every
// chord and every query is computed by the same arithmetic as in propagate(), so the result is bit-identical.  In a
// uniform field not even the integration is serial: the helix is exact for any arc length, so lane j evaluates the
// end of chord j directly from the start of the round (same chord lengths, accumulated by the same additions; end
// points equal to those of the chord-by-chord composition to rounding).
// All lanes of a group pass the same track; `cache` is the group's candidate list (kept identical in its lanes).
template <int FIELD, bool BVH>
__device__ __forceinline__ int propagate_wide(const DevCtx& c, int nav, int shift, bool active, int charge, double ekin, double pos[3],
                                              double dir[3], uint32_t vol, double s_phys, double& s_out, int& chords_out,
                                              double pushdir[3], int& face_out, NavCache* cache, int32_t* cand) {
  constexpr int field_kind = FIELD;
  const int lane = threadIdx.x & 31;
  const int W = 1 << shift, li = lane & (W - 1), g0 = lane & ~(W - 1);
  const unsigned gmask = (W == 32 ? kFull : ((1u << W) - 1u)) << g0;
  const double pmom = sqrt(ekin * (ekin + 2.0 * kMe));
  const double kappa = field_kind == ADEPT_FIELD_UNIFORM ? -charge * kCB * c.Bn / pmom : 0.0;
  const double inv_kappa = kappa != 0.0 ? 1.0 / kappa : 0.0;
  const bool curved = charge != 0 && field_kind != ADEPT_FIELD_NONE;
  double s_done = 0.0, h_step = -1.0;
  int chords = 0, flag = 0, face_hit = -1;
  bool running = active;
#pragma unroll
  for (int i = 0; i < 3; ++i) pushdir[i] = dir[i];
  if (BVH && cache) {   // the list of the group's first lane (the lane that runs the rest of the step) is the group's
    cache->qx = __shfl_sync(kFull, cache->qx, g0); cache->qy = __shfl_sync(kFull, cache->qy, g0);
    cache->qz = __shfl_sync(kFull, cache->qz, g0); cache->reach = __shfl_sync(kFull, cache->reach, g0);
    cache->list = reinterpret_cast<const int32_t*>(__shfl_sync(kFull, reinterpret_cast<unsigned long long>(cache->list), g0));
    cache->vol = __shfl_sync(kFull, cache->vol, g0); cache->count = __shfl_sync(kFull, cache->count, g0);
    cache->queries = 0;
  }
  while (__any_sync(kFull, running)) {
    // ---- integrate up to W segments ahead; lane li keeps segment li
    double p[3] = {pos[0], pos[1], pos[2]}, d[3] = {dir[0], dir[1], dir[2]};
    double P[3] = {0.0, 0.0, 0.0}, D[3] = {0.0, 0.0, 0.0}, D1[3] = {0.0, 0.0, 0.0}, U[3] = {0.0, 0.0, 0.0};
    double L = 0.0, H = 0.0, Sb = 0.0, reach_end = 0.0;   // reach_end: path from the round's start to the end of my segment
    int kind = 0;                                          // my segment: 0 none, 1 chord, 2 straight
    double sd = s_done, cum = 0.0;
    int ch = chords, nseg = 0, end = -1;                   // end: -1 round full, 0 physics limit, 2 chord budget
    bool integ = running;
    for (int j = 0; j < W; ++j) {
      if (!__any_sync(kFull, integ)) break;
      if (!integ) continue;
      if (sd >= s_phys) { end = 0; integ = false; continue; }
      double B[3] = {0.0, 0.0, 0.0}, h_max = 0.0;
      if (curved && (field_kind != ADEPT_FIELD_UNIFORM || h_step < 0.0)) {
        field_at<FIELD>(c, p, B);
        double dxB[3];
        cross3(d, B, dxB);
        const double bperp = sqrt(dxB[0] * dxB[0] + dxB[1] * dxB[1] + dxB[2] * dxB[2]);
        if (bperp != 0.0) {
          const double Rcurv = pmom / (kCB * bperp);
          h_max = sqrt(8.0 * c.delta_chord * Rcurv);
          if (field_kind == ADEPT_FIELD_MAP_RZ) {
            const double Bn = sqrt(B[0] * B[0] + B[1] * B[1] + B[2] * B[2]);
            h_max = fmin(h_max, 0.5 * pmom / (kCB * Bn));
          }
        }
        if (field_kind == ADEPT_FIELD_UNIFORM) h_step = h_max;
      } else if (curved) {
        h_max = h_step;
      }
      const double rest = s_phys - sd;
      if (!curved || h_max == 0.0) {          // straight to the physics limit: the last segment
        if (li == j) {
          kind = 2; L = rest; Sb = sd; reach_end = cum + rest;
#pragma unroll
          for (int i = 0; i < 3; ++i) { P[i] = p[i]; D[i] = d[i]; U[i] = d[i]; }
        }
        if (field_kind != ADEPT_FIELD_UNIFORM) {
#pragma unroll
          for (int i = 0; i < 3; ++i) p[i] += rest * d[i];
        }
        sd = s_phys; nseg = j + 1; end = 0; integ = false;
      } else if (ch >= c.chord_budget) {
        end = 2; integ = false;
      } else {
        const bool last = h_max >= rest;
        const double h = last ? rest : h_max;
        if (field_kind == ADEPT_FIELD_UNIFORM) {
          // the helix is known in closed form: only the arc lengths are accumulated here (by the same additions as in
          // the sequential loop); every lane evaluates its own chord's end point after the loop, all at once
          if (li == j) { kind = 1; H = h; Sb = sd; reach_end = cum + h; }
        } else {
          double p1[3], d1[3];
          rk4<FIELD>(c, charge, pmom, h, p, d, B, p1, d1);
          if (li == j) {
            kind = 1; H = h; Sb = sd; reach_end = cum + h;
            const double cv[3] = {p1[0] - p[0], p1[1] - p[1], p1[2] - p[2]};
            const double L2 = cv[0] * cv[0] + cv[1] * cv[1] + cv[2] * cv[2];
            const double iL = rsqrt(L2);
            L = L2 * iL;
#pragma unroll
            for (int i = 0; i < 3; ++i) { P[i] = p[i]; D[i] = d[i]; D1[i] = d1[i]; U[i] = cv[i] * iL; }
          }
#pragma unroll
          for (int i = 0; i < 3; ++i) { p[i] = p1[i]; d[i] = d1[i]; }
        }
        sd = last ? s_phys : sd + h;
        cum += h; ++ch; nseg = j + 1;
        if (last) { end = 0; integ = false; }
      }
    }
    if (field_kind == ADEPT_FIELD_UNIFORM) {
      // Exact helix: lane li evaluates the end of chord li from the round's start, arc length = the accumulated
      // chord lengths (F3 holds for any arc; the sequential loop composes the same rotation chord by chord, so
      // the two agree to rounding, not bit for bit); a segment starts where the previous lane's chord ends.
      double E[3] = {pos[0], pos[1], pos[2]}, F[3] = {dir[0], dir[1], dir[2]};
      if (kind == 1) helix(c.bhat, kappa, inv_kappa, reach_end, pos, dir, E, F);
      double Ep[3], Fp[3];
#pragma unroll
      for (int i = 0; i < 3; ++i) { Ep[i] = __shfl_up_sync(kFull, E[i], 1); Fp[i] = __shfl_up_sync(kFull, F[i], 1); }
      if (li == 0) {
#pragma unroll
        for (int i = 0; i < 3; ++i) { Ep[i] = pos[i]; Fp[i] = dir[i]; }
      }
      if (kind == 1) {
        const double cv[3] = {E[0] - Ep[0], E[1] - Ep[1], E[2] - Ep[2]};
        const double L2 = cv[0] * cv[0] + cv[1] * cv[1] + cv[2] * cv[2];
        const double iL = rsqrt(L2);
        L = L2 * iL;
#pragma unroll
        for (int i = 0; i < 3; ++i) { P[i] = Ep[i]; D[i] = Fp[i]; D1[i] = F[i]; U[i] = cv[i] * iL; }
      } else if (kind == 2) {   // the straight last segment (a track along B) starts at the end of the chords before it
#pragma unroll
        for (int i = 0; i < 3; ++i) { P[i] = Ep[i]; D[i] = Fp[i]; U[i] = Fp[i]; E[i] = Ep[i] + L * Fp[i]; F[i] = Fp[i]; }
      }
      // the state after the round's last segment, for every lane of the group
      const int src = g0 + (nseg > 0 ? nseg - 1 : 0);
#pragma unroll
      for (int i = 0; i < 3; ++i) {
        const double e = __shfl_sync(kFull, E[i], src), f = __shfl_sync(kFull, F[i], src);
        if (nseg > 0) { p[i] = e; d[i] = f; }
      }
    }
    // ---- which segments need a geometry query (nav_safety, as in propagate(): one clearance around the round's start)
    double safe = -1.0;
    bool own_only = false;
    if (running && nseg > 1) safe = nav_safety(c, vol, pos[0], pos[1], pos[2], own_only);
    const bool clear = kind == 1 && reach_end < safe;
    const bool query = running && (kind == 2 || (kind == 1 && (!clear || own_only)));
    // ---- the group's candidate list (geom.cuh NavCache): when two or more of the round's segments are not covered by
    // the list the group has, a new one is built around the middle of the round, its ball just large enough for all
    // of them (up to kCandRadiusMax)
    if (BVH && cache && cand) {
      bool uncovered = false;
      const double mx = 0.5 * (pos[0] + p[0]), my = 0.5 * (pos[1] + p[1]), mz = 0.5 * (pos[2] + p[2]);
      double need_r = 0.0;
      if (query && nav == ADEPT_NAV_BVH) {
        const DevVolume& v = volume(c, vol);
        if (v.dcount > 0 && v.bvh >= 0) {
          uncovered = true;
          if (cache->reach > 0.0 && cache->vol == vol) {
            const double ox = P[0] - cache->qx, oy = P[1] - cache->qy, oz = P[2] - cache->qz;
            uncovered = !(sqrt(ox * ox + oy * oy + oz * oz) + L <= cache->reach * (1.0 - 1.0e-9));
          }
          const double ox = P[0] - mx, oy = P[1] - my, oz = P[2] - mz;
          need_r = sqrt(ox * ox + oy * oy + oz * oz) + L;
        }
      }
      const unsigned um = __ballot_sync(kFull, uncovered) & gmask;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {   // largest need of the group (groups are aligned runs of W lanes)
        const double other = __shfl_xor_sync(kFull, need_r, o);
        if (o < W) need_r = fmax(need_r, other);
      }
      const double rho = fmax(kCandRadius, need_r * (1.0 + 1.0e-6) + 1.0e-9);
      const bool rebuild = __popc(um) >= 2 && rho <= kCandRadiusMax;
      unsigned mb = __ballot_sync(kFull, li == 0 && rebuild);
      const int bvh = rebuild ? volume(c, vol).bvh : 0;
      while (mb) {
        const int src = __ffs(mb) - 1;
        mb &= mb - 1;
        int32_t* list = cand + kCandCap * ((threadIdx.x & ~31) + src);
        const int n = bvh_candidates(c, c.bvh[__shfl_sync(kFull, bvh, src)], __shfl_sync(kFull, mx, src), __shfl_sync(kFull, my, src),
                                     __shfl_sync(kFull, mz, src), __shfl_sync(kFull, rho, src), list);
        if (g0 == src) {
          cache->qx = mx; cache->qy = my; cache->qz = mz;
          cache->reach = n >= 0 ? rho : -1.0;
          cache->list = list;
          cache->count = n >= 0 ? n : 0;
          cache->vol = vol; cache->queries = 0;
        }
      }
    }
    int face;
    const double s_geo = nav_distance<BVH>(c, nav, query, P[0], P[1], P[2], U[0], U[1], U[2], vol, L, face, cache, nullptr, clear);
    const unsigned hm = __ballot_sync(kFull, query && s_geo < L) & gmask;
    // the first segment of the group that ends on a boundary decides (its lane computes the end state; the shuffles
    // are unconditional because the groups of a warp differ)
    const int src = hm ? __ffs(hm) - 1 : lane;
    double r[10] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    int rf = -1, rc = 0;
    if (hm && lane == src) {
      double dh[3] = {D[0], D[1], D[2]};
      double s_end = Sb + s_geo;
      if (kind == 1) {
        const double frac = s_geo / L;
        if (field_kind == ADEPT_FIELD_UNIFORM) {
          helix_dir(c.bhat, kappa, H * frac, D, dh);
        } else {
          double n = 0.0;
#pragma unroll
          for (int i = 0; i < 3; ++i) { dh[i] = D[i] + frac * (D1[i] - D[i]); n += dh[i] * dh[i]; }
          n = rsqrt(n);
#pragma unroll
          for (int i = 0; i < 3; ++i) dh[i] *= n;
        }
        s_end = Sb + H * frac;
      }
      // (a straight segment advances along the direction itself, a chord along its unit vector; U is either)
#pragma unroll
      for (int i = 0; i < 3; ++i) { r[i] = P[i] + s_geo * U[i]; r[3 + i] = dh[i]; r[6 + i] = U[i]; }
      r[9] = s_end;
      rf = face;
      rc = chords + li + (kind == 1 ? 1 : 0);
    }
#pragma unroll
    for (int i = 0; i < 10; ++i) r[i] = __shfl_sync(kFull, r[i], src);
    rf = __shfl_sync(kFull, rf, src);
    rc = __shfl_sync(kFull, rc, src);
    if (hm) {    // (only groups that are running have queries)
#pragma unroll
      for (int i = 0; i < 3; ++i) { pos[i] = r[i]; dir[i] = r[3 + i]; pushdir[i] = r[6 + i]; }
      s_done = r[9]; face_hit = rf; chords = rc;
      flag = 1; running = false;
    } else if (running) {
#pragma unroll
      for (int i = 0; i < 3; ++i) { pos[i] = p[i]; dir[i] = d[i]; }
      s_done = sd; chords = ch;
      if (end >= 0) { flag = end; running = false; }
    }
  }
  s_out = s_done;
  chords_out = chords;
  face_out = flag == 1 ? face_hit : -1;
  return flag;
}

}  // namespace adept
