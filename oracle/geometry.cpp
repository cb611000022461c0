/* ORACLE -- TEST INFRASTRUCTURE ONLY (see oracle.h).
 *
 * G1-G5 of SURVEY.md §8(c): box and tube solids, the brute-force 'loop' navigator that searches
 * ALL daughter volumes (the paper's own correctness baseline) and Locate.
 * Pinned by tests/test_oracle_geometry.py: analytic slab boundaries of the calorimeter, ray/solid
 * distances against a dense ray-march with the inside() predicate, Locate against brute force over
 * every touchable.
 */
#include <algorithm>

#include "internal.h"

namespace orc {

void to_local(const Volume& v, const double g[3], double l[3]) {
  const double q[3] = {g[0] - v.t[0], g[1] - v.t[1], g[2] - v.t[2]};
  for (int i = 0; i < 3; ++i) l[i] = v.R[0 + i] * q[0] + v.R[3 + i] * q[1] + v.R[6 + i] * q[2];
}
void dir_to_local(const Volume& v, const double g[3], double l[3]) {
  for (int i = 0; i < 3; ++i) l[i] = v.R[0 + i] * g[0] + v.R[3 + i] * g[1] + v.R[6 + i] * g[2];
}

static bool inside_solid(int solid, const double h[3], const double p[3]) {
  if (solid == ORC_BOX) return std::fabs(p[0]) <= h[0] && std::fabs(p[1]) <= h[1] && std::fabs(p[2]) <= h[2];
  const double r2 = p[0] * p[0] + p[1] * p[1];
  return r2 >= h[0] * h[0] && r2 <= h[1] * h[1] && std::fabs(p[2]) <= h[2];
}

/* G1 box: exit distance from inside = min_i (sgn(d_i) h_i - x_i)/d_i, clamped at 0 */
static double box_exit(const double h[3], const double p[3], const double d[3]) {
  double t = kInf;
  for (int i = 0; i < 3; ++i) {
    if (d[i] != 0.0) {
      const double ti = ((d[i] > 0.0 ? h[i] : -h[i]) - p[i]) / d[i];
      t = std::min(t, ti);
    }
  }
  return std::max(t, 0.0);
}

/* G1 box: entry distance by the slab method; miss = +inf */
static double box_entry(const double h[3], const double p[3], const double d[3]) {
  double tn = -kInf, tf = kInf;
  for (int i = 0; i < 3; ++i) {
    if (d[i] != 0.0) {
      const double t1 = (-h[i] - p[i]) / d[i];
      const double t2 = (h[i] - p[i]) / d[i];
      tn = std::max(tn, std::min(t1, t2));
      tf = std::min(tf, std::max(t1, t2));
    } else if (std::fabs(p[i]) > h[i]) {
      return kInf;
    }
  }
  if (tn <= tf && tf > 0.0) return std::max(tn, 0.0);
  return kInf;
}

/* G1 tube (rmin, rmax, hz), full phi.  A = dx^2+dy^2, B = x dx + y dy, C = r^2 - R^2. */
static double tube_exit(const double h[3], const double p[3], const double d[3]) {
  double t = kInf;
  if (d[2] != 0.0) t = ((d[2] > 0.0 ? h[2] : -h[2]) - p[2]) / d[2];
  const double A = d[0] * d[0] + d[1] * d[1];
  if (A > 0.0) {
    const double B = p[0] * d[0] + p[1] * d[1];
    const double r2 = p[0] * p[0] + p[1] * p[1];
    const double Co = r2 - h[1] * h[1];
    const double disc_o = B * B - A * Co;
    t = std::min(t, (-B + std::sqrt(std::max(disc_o, 0.0))) / A);
    if (h[0] > 0.0 && B < 0.0) {
      const double Ci = r2 - h[0] * h[0];
      const double disc_i = B * B - A * Ci;
      if (disc_i > 0.0) t = std::min(t, (-B - std::sqrt(disc_i)) / A);
    }
  }
  return std::max(t, 0.0);
}

static double tube_entry(const double h[3], const double p[3], const double d[3]) {
  if (inside_solid(ORC_TUBE, h, p)) return 0.0;
  double best = kInf;
  const double r2 = p[0] * p[0] + p[1] * p[1];
  const double rmin2 = h[0] * h[0], rmax2 = h[1] * h[1];
  /* (a) end caps */
  if (std::fabs(p[2]) > h[2] && p[2] * d[2] < 0.0) {
    const double t = (std::fabs(p[2]) - h[2]) / std::fabs(d[2]);
    const double x = p[0] + t * d[0], y = p[1] + t * d[1];
    const double q2 = x * x + y * y;
    if (q2 >= rmin2 && q2 <= rmax2) best = std::min(best, t);
  }
  const double A = d[0] * d[0] + d[1] * d[1];
  if (A > 0.0) {
    const double B = p[0] * d[0] + p[1] * d[1];
    /* (b) outer cylinder from outside */
    const double Co = r2 - rmax2;
    if (Co > 0.0 && B < 0.0) {
      const double disc = B * B - A * Co;
      if (disc > 0.0) {
        const double t = (-B - std::sqrt(disc)) / A;
        if (t >= 0.0 && std::fabs(p[2] + t * d[2]) <= h[2]) best = std::min(best, t);
      }
    }
    /* (c) inner cylinder, far root: the ray leaves the hole into the solid */
    if (h[0] > 0.0) {
      const double Ci = r2 - rmin2;
      const double disc = B * B - A * Ci;
      if (disc > 0.0) {
        const double t = (-B + std::sqrt(disc)) / A;
        if (t > 0.0 && std::fabs(p[2] + t * d[2]) <= h[2]) best = std::min(best, t);
      }
    }
  }
  return best;
}

}  // namespace orc

using namespace orc;

extern "C" double orc_solid_entry(int solid, const double dims[3], const double p[3], const double d[3]) {
  return solid == ORC_BOX ? box_entry(dims, p, d) : tube_entry(dims, p, d);
}
extern "C" double orc_solid_exit(int solid, const double dims[3], const double p[3], const double d[3]) {
  return solid == ORC_BOX ? box_exit(dims, p, d) : tube_exit(dims, p, d);
}

extern "C" int orc_inside(const orc_ctx* c, const double pos[3], uint32_t volume) {
  const Volume& v = c->vol[volume];
  double l[3];
  to_local(v, pos, l);
  return inside_solid(v.solid, v.dims, l) ? 1 : 0;
}

/* G3: loop navigator -- own solid's exit distance and EVERY daughter's entry distance */
extern "C" double orc_distance(const orc_ctx* c, const double pos[3], const double dir[3], uint32_t volume,
                               double s_max) {
  const Volume& v = c->vol[volume];
  double lp[3], ld[3];
  to_local(v, pos, lp);
  dir_to_local(v, dir, ld);
  double s = orc_solid_exit(v.solid, v.dims, lp, ld);
  for (int k = 0; k < v.dcount; ++k) {
    const Volume& dv = c->vol[v.dbegin + k];
    double dp[3], dd[3];
    to_local(dv, pos, dp);
    dir_to_local(dv, dir, dd);
    s = std::min(s, orc_solid_entry(dv.solid, dv.dims, dp, dd));
  }
  return std::min(s, s_max);
}

/* G4: from the world down, descend into the first daughter (index order) containing the point */
extern "C" int64_t orc_locate(const orc_ctx* c, const double pos[3]) {
  if (!orc_inside(c, pos, 0)) return -1;
  int cur = 0;
  for (;;) {
    const Volume& v = c->vol[cur];
    int next = -1;
    for (int k = 0; k < v.dcount; ++k) {
      if (orc_inside(c, pos, static_cast<uint32_t>(v.dbegin + k))) { next = v.dbegin + k; break; }
    }
    if (next < 0) return cur;
    cur = next;
  }
}

/* G5: primaries are placed at Locate(p0 + eps_push d0) */
extern "C" int64_t orc_place(const orc_ctx* c, const double pos[3], const double dir[3]) {
  const double q[3] = {pos[0] + c->cfg.eps_push * dir[0], pos[1] + c->cfg.eps_push * dir[1],
                       pos[2] + c->cfg.eps_push * dir[2]};
  return orc_locate(c, q);
}
