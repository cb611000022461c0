// One transport step of one track per lane  (rows A2-A8), in two phases that the
// frozen-step hook chains and the transport kernels run as separate kernels with per-process staging
// queues in between:
//   move      step-start rules, physics step limit, propagation, continuous loss, MSC, push past the
//             boundary + relocation (A5), process choice
//   interact  sample the discrete process, create secondaries (A8)
// move is warp-convergent: every lane of the warp must call it (inactive lanes pass active = false)
// because propagation and relocation use the warp-cooperative navigator.
#pragma once
#include "field.cuh"
#include "physics.cuh"

namespace adept {

enum { MODE_ANY = 0, MODE_GAMMA = 1, MODE_CHARGED = 2 };

// what the move phase leaves to do
enum { NEXT_NONE = 0, NEXT_INTERACT = 2 };

__device__ __forceinline__ double carried_energy(int species, double ekin) {
  return species == ADEPT_POSITRON ? ekin + 2.0 * kMe : ekin;
}

__device__ __forceinline__ void init_out(StepOut& o, const Track& in, bool active) {
  o.post = in;
  o.alive = active ? 1 : 0;
  o.outcome = ADEPT_OUT_BOUNDARY;
  o.chords = 0; o.n_sec = 0;
  o.s = 0.0; o.edep_dep = 0.0; o.edep_cut = 0.0; o.escaped = 0.0; o.killed = 0.0;
  o.sec[0].species = -1; o.sec[1].species = -1;
}

// Phase 1.  On return o.post holds the moved (and, after a boundary, relocated) state, `process` the
// chosen discrete process for NEXT_INTERACT, and `mat` the material of the pre-step volume.
// o.post.step is NOT yet incremented.
template <int MODE, int FIELD = -1, bool BVH = true>
__device__ int step_move(const DevCtx& c, int nav, bool active, const Track& in, StepOut& o, Stream& u, int& process,
                         int& mat) {
  init_out(o, in, active);
  const bool is_gamma = MODE == MODE_GAMMA || (MODE == MODE_ANY && in.species == ADEPT_GAMMA);
  const bool positron = !is_gamma && in.species == ADEPT_POSITRON;
  u.init(in.event, c.seed, in.id, in.step);
  process = 0;
  mat = 0;

  bool go = active;
  bool vacuum = true, lim_disc = false, range_out = false;
  double s_phys = 0.0, stot = 0.0, x0 = 0.0, x1 = 0.0, S = 0.0, R = ADEPT_INF;
  GridPos gp{0, 0.0};
  const double* tab = nullptr;
  int row = 0;
  const double T0 = in.ekin;

  // ---- S4 / step-start rules, physics step limit (A2, A3)
  if (active) {
    if (in.step >= c.max_steps) {
      o.killed += carried_energy(in.species, T0); o.alive = 0; o.outcome = ADEPT_OUT_KILLED; go = false;
    } else if (T0 < kTmin) {
      o.edep_cut += T0; o.alive = 0; o.outcome = ADEPT_OUT_STOPPED; go = false;
      mat = volume(c, in.vol).material;
      if (!is_gamma) o.post.ekin = 0.0;
      if (positron) annihilation_at_rest(c, mat, o, u);
    } else {
      mat = volume(c, in.vol).material;
      vacuum = mat_scalar(c, mat, S_VACUUM) != 0.0;
      if (!vacuum) gp = grid_pos(c, T0);
      if (is_gamma) {
        double se = 0.0;
        if (!vacuum) {
          tab = c.tab_g + static_cast<size_t>(mat) * kNGrid * kRowG; row = kRowG;
          x0 = interp(tab, row, 0, gp);                                   // Compton
          x1 = T0 > 2.0 * kMe ? interp(tab, row, 1, gp) : 0.0;            // pair, exact threshold (P2)
          se = interp(tab, row, 2, gp);                                   // photoelectric
        }
        stot = x0 + x1 + se;
        s_phys = stot > 0.0 ? div_pos(-log_pos(u.uniform(0)), stot) : ADEPT_INF;
      } else {
        double sa = 0.0;
        if (!vacuum) {
          if (positron) {
            tab = c.tab_ep + static_cast<size_t>(mat) * kNGrid * kRowEp; row = kRowEp;
            x0 = interp(tab, row, 0, gp); x1 = interp(tab, row, 1, gp); sa = interp(tab, row, 2, gp);
            S = interp(tab, row, 3, gp); R = interp(tab, row, 4, gp);
          } else {
            tab = c.tab_em + static_cast<size_t>(mat) * kNGrid * kRowEm; row = kRowEm;
            x0 = interp(tab, row, 0, gp); x1 = interp(tab, row, 1, gp);
            S = interp(tab, row, 2, gp); R = interp(tab, row, 3, gp);
          }
        }
        stot = x0 + x1 + sa;
        const double s_disc = stot > 0.0 ? div_pos(-log_pos(u.uniform(0)), stot) : ADEPT_INF;
        range_out = R <= c.rho_R;
        const double s_loss = range_out ? R : c.alpha_R * R + c.rho_R * (1.0 - c.alpha_R) * (2.0 - c.rho_R / R);
        lim_disc = s_disc < s_loss;
        s_phys = lim_disc ? s_disc : s_loss;
      }
    }
  }

  // ---- propagation (A4, A6): straight line for gammas, chords for e-/e+
  double pos[3] = {in.x, in.y, in.z}, dir[3] = {in.dx, in.dy, in.dz}, pushdir[3];
  double s = 0.0;
  int chords = 0;
  const int charge = is_gamma ? 0 : (positron ? +1 : -1);
  int face;
  const int flag = propagate<FIELD, BVH>(c, nav, go, charge, T0, pos, dir, in.vol, s_phys, s, chords, pushdir, face);

  // ---- along-step actions (A7)
  o.s = s; o.chords = chords;
  bool cross = go && flag == 1;
  if (go && !is_gamma) {
    double dE = 0.0;
    if (!vacuum) {
      if (flag == 0 && !lim_disc && range_out) dE = T0;
      else if (s <= 0.01 * R) dE = S * s;
      else dE = T0 - inverse_range(c, tab, row, positron ? 4 : 3, c.rhint + (2 * mat + (positron ? 1 : 0)) * kHintStride, R - s);
      dE = fmin(fmax(dE, 0.0), T0);
    }
    o.edep_dep += dE;
    o.post.ekin = T0 - dE;
    if (o.post.ekin < kTmin) {
      o.edep_cut += o.post.ekin; o.post.ekin = 0.0;
      o.post.x = pos[0]; o.post.y = pos[1]; o.post.z = pos[2];
      o.post.dx = dir[0]; o.post.dy = dir[1]; o.post.dz = dir[2];
      if (positron) annihilation_at_rest(c, mat, o, u);
      o.alive = 0; o.outcome = ADEPT_OUT_STOPPED;
      go = false; cross = false;
    }
    if (go && !vacuum && s > 0.0) {  // P9 Highland MSC at the pre-step energy
      const double X0 = mat_scalar(c, mat, S_X0);
      const double pbeta = T0 * (T0 + 2.0 * kMe) / (T0 + kMe);
      const double beta2 = T0 * (T0 + 2.0 * kMe) / ((T0 + kMe) * (T0 + kMe));
      const double corr = fmax(0.0, 1.0 + 0.038 * log_pos(s / (X0 * beta2)));
      const double th0 = (13.6 / pbeta) * sqrt(s / X0) * corr;
      const double u2 = u.uniform(2), u3 = u.uniform(3);
      const double th = th0 * sqrt(-2.0 * log_pos(u2));
      double sn, cs, dn[3];
      sincos(th, &sn, &cs);
      rotate(dir, cs, sn, 2.0 * u3, dn);
      dir[0] = dn[0]; dir[1] = dn[1]; dir[2] = dn[2];
    }
  }
  if (go) {
    o.post.dx = dir[0]; o.post.dy = dir[1]; o.post.dz = dir[2];
    if (cross) {  // G5: push past the boundary
      pos[0] += c.eps_push * pushdir[0]; pos[1] += c.eps_push * pushdir[1]; pos[2] += c.eps_push * pushdir[2];
    }
    o.post.x = pos[0]; o.post.y = pos[1]; o.post.z = pos[2];
  }
  // ---- relocation (A5), warp-convergent
  const int nv = nav_relocate<BVH>(c, nav, cross, in.vol, pos[0], pos[1], pos[2], face);
  if (!go) return NEXT_NONE;
  if (cross) {
    if (nv < 0) {
      o.escaped += carried_energy(in.species, o.post.ekin); o.alive = 0; o.outcome = ADEPT_OUT_ESCAPED;
    } else {
      o.post.vol = static_cast<uint32_t>(nv); o.outcome = ADEPT_OUT_BOUNDARY;
    }
    return NEXT_NONE;
  }
  if (flag == 2) { o.outcome = ADEPT_OUT_TRUNCATED; return NEXT_NONE; }
  if (!is_gamma && !lim_disc) { o.outcome = ADEPT_OUT_LOSS; return NEXT_NONE; }
  // ---- choice of the discrete process (U1)
  const double u1 = u.uniform(1);
  if (is_gamma) {
    process = ADEPT_OUT_PHOTO;
    if (u1 * stot < x0) process = ADEPT_OUT_COMPTON;
    else if (u1 * stot < x0 + x1) process = ADEPT_OUT_PAIR;
    if (process == ADEPT_OUT_PHOTO) {  // no sampling involved: done here rather than staged (12 % of all steps)
      photoelectric(c, mat, o, in.step);
      o.outcome = ADEPT_OUT_PHOTO;
      return NEXT_NONE;
    }
  } else {
    process = ADEPT_OUT_BREM;
    if (u1 * stot < x0) process = ADEPT_OUT_BREM;
    else if (!positron || u1 * stot < x0 + x1) process = ADEPT_OUT_IONI;
    else process = ADEPT_OUT_ANNI;
  }
  return NEXT_INTERACT;
}

// The whole step in one call (frozen-step hook).
template <int MODE>
__device__ void step_track(const DevCtx& c, int nav, bool active, const Track& in, StepOut& o) {
  Stream u;
  int process, mat;
  const int next = step_move<MODE>(c, nav, active, in, o, u, process, mat);
  if (next == NEXT_INTERACT) run_process(c, process, in.species, mat, o, u);
  if (o.alive) o.post.step = in.step + 1;
}

}  // namespace adept
