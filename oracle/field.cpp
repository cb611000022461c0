/* ORACLE -- TEST INFRASTRUCTURE ONLY (see oracle.h).
 *
 * F1-F6 of SURVEY.md §8(c): propagation of a charged track in a magnetic field by chords whose
 * sagitta stays below delta_chord, with a chord budget per step (F4).
 * Uniform field: exact helix endpoints.  Field map: one classical RK4 step per chord.
 * Pinned by tests/test_oracle_field.py: helix vs the analytic circle and the return to the start
 * after one turn, RK4 in a uniform map vs the helix with the h^5 error law, |d| = 1; the chord loop of
 * the ORC_FIELD_MAP_RZ branch by its chord count (sagitta limit, and the F2' clamp as the number
 * ceil(s / (0.5 p / (2.998 |B|)))), its end point vs the exact helix within the RK4 bound, a boundary
 * hit (point within delta_chord of the analytic circle, unit interpolated tangent within (h/R)^2 of
 * the exact one, push direction = unit chord) and an adaptive DOP853 integration of F1 in the real,
 * non-uniform solenoid map; tests/test_oracle_stepper.py closes the per-event ledger through it.
 */
#include <algorithm>

#include "internal.h"

using namespace orc;

static inline void cross(const double a[3], const double b[3], double c[3]) {
  c[0] = a[1] * b[2] - a[2] * b[1];
  c[1] = a[2] * b[0] - a[0] * b[2];
  c[2] = a[0] * b[1] - a[1] * b[0];
}

/* F6: B = (0,0,Bz(r,z)), bilinear on the r-z grid, clamped outside */
extern "C" void orc_field_at(const orc_ctx* c, const double p[3], double B[3]) {
  const orc_field& f = c->field;
  if (f.kind == ORC_FIELD_UNIFORM) { B[0] = f.B[0]; B[1] = f.B[1]; B[2] = f.B[2]; return; }
  B[0] = B[1] = B[2] = 0.0;
  if (f.kind != ORC_FIELD_MAP_RZ) return;
  const double r = std::sqrt(p[0] * p[0] + p[1] * p[1]);
  double fr = (r - f.r0) / f.dr, fz = (p[2] - f.z0) / f.dz;
  fr = std::min(std::max(fr, 0.0), static_cast<double>(f.nr - 1));
  fz = std::min(std::max(fz, 0.0), static_cast<double>(f.nz - 1));
  const int ir = std::min(static_cast<int>(std::floor(fr)), f.nr - 2);
  const int iz = std::min(static_cast<int>(std::floor(fz)), f.nz - 2);
  const double a = fr - ir, b = fz - iz;
  const double* m = c->bz.data();
  const double v00 = m[iz * f.nr + ir], v01 = m[iz * f.nr + ir + 1];
  const double v10 = m[(iz + 1) * f.nr + ir], v11 = m[(iz + 1) * f.nr + ir + 1];
  const double lo = v00 + a * (v01 - v00);
  const double hi = v10 + a * (v11 - v10);
  B[2] = lo + b * (hi - lo);
}

/* F3: exact helix in a uniform field. omega = -q kCB |B| h / p. */
extern "C" void orc_helix(const double B[3], int charge, double pmom, double h, const double p[3],
                          const double d[3], double p1[3], double d1[3]) {
  const double Bn = std::sqrt(B[0] * B[0] + B[1] * B[1] + B[2] * B[2]);
  const double b[3] = {B[0] / Bn, B[1] / Bn, B[2] / Bn};
  const double omega = -charge * kCB * Bn * h / pmom;
  const double dpar = d[0] * b[0] + d[1] * b[1] + d[2] * b[2];
  const double dl[3] = {dpar * b[0], dpar * b[1], dpar * b[2]};
  const double dt[3] = {d[0] - dl[0], d[1] - dl[1], d[2] - dl[2]};
  double bxd[3];
  cross(b, dt, bxd);
  const double so = std::sin(omega), co = std::cos(omega);
  const double sh = std::sin(0.5 * omega);
  const double omc = 2.0 * sh * sh; /* 1 - cos(omega) */
  const double hw = h / omega;
  for (int i = 0; i < 3; ++i) {
    d1[i] = dl[i] + dt[i] * co + bxd[i] * so;
    p1[i] = p[i] + dl[i] * h + hw * (dt[i] * so + bxd[i] * omc);
  }
}

/* F1, F3: one classical RK4 step of length h on (x, d): x' = d, d' = (q kCB / p) d x B(x) */
extern "C" void orc_rk4(const orc_ctx* c, int charge, double pmom, double h, const double p[3],
                        const double d[3], double p1[3], double d1[3]) {
  const double kap = charge * kCB / pmom;
  auto deriv = [&](const double x[3], const double v[3], double dx[3], double dv[3]) {
    double B[3], vxB[3];
    orc_field_at(c, x, B);
    cross(v, B, vxB);
    for (int i = 0; i < 3; ++i) { dx[i] = v[i]; dv[i] = kap * vxB[i]; }
  };
  double k1x[3], k1v[3], k2x[3], k2v[3], k3x[3], k3v[3], k4x[3], k4v[3], x[3], v[3];
  deriv(p, d, k1x, k1v);
  for (int i = 0; i < 3; ++i) { x[i] = p[i] + 0.5 * h * k1x[i]; v[i] = d[i] + 0.5 * h * k1v[i]; }
  deriv(x, v, k2x, k2v);
  for (int i = 0; i < 3; ++i) { x[i] = p[i] + 0.5 * h * k2x[i]; v[i] = d[i] + 0.5 * h * k2v[i]; }
  deriv(x, v, k3x, k3v);
  for (int i = 0; i < 3; ++i) { x[i] = p[i] + h * k3x[i]; v[i] = d[i] + h * k3v[i]; }
  deriv(x, v, k4x, k4v);
  for (int i = 0; i < 3; ++i) {
    p1[i] = p[i] + (h / 6.0) * (k1x[i] + 2.0 * k2x[i] + 2.0 * k3x[i] + k4x[i]);
    d1[i] = d[i] + (h / 6.0) * (k1v[i] + 2.0 * k2v[i] + 2.0 * k3v[i] + k4v[i]);
  }
  const double n = std::sqrt(d1[0] * d1[0] + d1[1] * d1[1] + d1[2] * d1[2]);
  for (int i = 0; i < 3; ++i) d1[i] /= n;
}

/* F2-F4: chord loop. On return pos/dir hold the end point and tangent (at a boundary: the hit point
   WITHOUT the push, and pushdir = chord direction). Returns 0 physics, 1 boundary, 2 truncated. */
extern "C" int orc_propagate(const orc_ctx* c, int charge, double ekin, double pos[3], double dir[3],
                             uint32_t volume, double s_phys, double* s_done_out, int* chords_out,
                             double pushdir[3]) {
  const double pmom = std::sqrt(ekin * (ekin + 2.0 * kMe));
  double s_done = 0.0;
  int chords = 0;
  int flag = 0;
  for (int i = 0; i < 3; ++i) pushdir[i] = dir[i];
  for (;;) {
    if (s_done >= s_phys) { flag = 0; break; }
    double B[3] = {0.0, 0.0, 0.0};
    if (c->field.kind != ORC_FIELD_NONE) orc_field_at(c, pos, B);
    double dxB[3];
    cross(dir, B, dxB);
    const double bperp = std::sqrt(dxB[0] * dxB[0] + dxB[1] * dxB[1] + dxB[2] * dxB[2]);
    const double rest = s_phys - s_done;
    if (bperp == 0.0) {
      /* straight line (no field, B = 0 or d parallel to B): not a chord, no budget */
      const double s_geo = orc_distance(c, pos, dir, volume, rest);
      for (int i = 0; i < 3; ++i) pushdir[i] = dir[i];
      if (s_geo < rest) {
        for (int i = 0; i < 3; ++i) pos[i] += s_geo * dir[i];
        s_done += s_geo;
        flag = 1;
      } else {
        for (int i = 0; i < 3; ++i) pos[i] += rest * dir[i];
        s_done = s_phys;
        flag = 0;
      }
      break;
    }
    if (chords >= c->cfg.chord_budget) { flag = 2; break; }
    const double Rcurv = pmom / (kCB * bperp);
    double h_max = std::sqrt(8.0 * c->cfg.delta_chord * Rcurv);
    if (c->field.kind == ORC_FIELD_MAP_RZ) {
      /* F2': an RK4 chord may not turn the direction about B by more than 0.5 rad,
         or the one-step integrator loses accuracy (local error ~ omega^5/120) and conditioning */
      const double Bn = std::sqrt(B[0] * B[0] + B[1] * B[1] + B[2] * B[2]);
      h_max = std::min(h_max, 0.5 * pmom / (kCB * Bn));
    }
    const bool last = h_max >= rest; /* this chord completes the step */
    const double h = last ? rest : h_max;
    double p1[3], d1[3];
    if (c->field.kind == ORC_FIELD_UNIFORM) orc_helix(B, charge, pmom, h, pos, dir, p1, d1);
    else orc_rk4(c, charge, pmom, h, pos, dir, p1, d1);
    double ch[3] = {p1[0] - pos[0], p1[1] - pos[1], p1[2] - pos[2]};
    const double L = std::sqrt(ch[0] * ch[0] + ch[1] * ch[1] + ch[2] * ch[2]);
    const double u[3] = {ch[0] / L, ch[1] / L, ch[2] / L};
    const double s_geo = orc_distance(c, pos, u, volume, L);
    ++chords;
    if (s_geo < L) {
      const double frac = s_geo / L;
      double ph[3], dh[3];
      if (c->field.kind == ORC_FIELD_UNIFORM) {
        orc_helix(B, charge, pmom, h * frac, pos, dir, ph, dh); /* exact tangent at arc h*frac */
      } else {
        double n = 0.0;
        for (int i = 0; i < 3; ++i) { dh[i] = dir[i] + frac * (d1[i] - dir[i]); n += dh[i] * dh[i]; }
        n = std::sqrt(n);
        for (int i = 0; i < 3; ++i) dh[i] /= n;
      }
      for (int i = 0; i < 3; ++i) { pos[i] += s_geo * u[i]; dir[i] = dh[i]; pushdir[i] = u[i]; }
      s_done += h * frac;
      flag = 1;
      break;
    }
    for (int i = 0; i < 3; ++i) { pos[i] = p1[i]; dir[i] = d1[i]; }
    s_done = last ? s_phys : s_done + h; /* exact, so the loop ends on the next test */
  }
  *s_done_out = s_done;
  *chords_out = chords;
  return flag;
}
