/* ORACLE -- TEST INFRASTRUCTURE ONLY (see oracle.h).
 *
 * S1-S4 of SURVEY.md §8(c): the gamma step, the e-/e+ step (step limitation, propagation,
 * continuous loss, Highland MSC (P9), relocation, discrete interaction) and the per-primary LIFO
 * event loop with the energy ledger (S3).  The paper fixes the workflow (one step
 * at a time, secondaries tracked immediately) but none of the formulas; the readings are listed in
 * DESIGN.md §3.  Pinned by tests/test_oracle_stepper.py: per-event energy conservation to 1e-9,
 * the unscattered-photon fraction exp(-sum Sigma t), CSDA range of an electron with discrete
 * processes closed, <theta^2> = 2 theta0^2 of the MSC kick.
 * Parity unpinned by the paper (no worked numbers): A_eff, cut conversion, step-function
 * constants, eps_push, delta_chord, chord budget, draw slots -- see DESIGN.md §3.
 */
#include <algorithm>
#include <cstring>

#include "internal.h"

using namespace orc;

void orc_run_process(const orc_ctx*, int, const orc_track*, int, orc_step_result*, orc_track*);
void orc_annihilate_at_rest(const orc_ctx*, const orc_track*, int, orc_step_result*, orc_track*);

extern "C" orc_ctx* orc_create(const orc_geometry* g, const orc_materials* m, const orc_field* f,
                               const orc_config* cfg) {
  orc_ctx* c = new orc_ctx;
  c->vol.resize(g->n_vol);
  for (int i = 0; i < g->n_vol; ++i) {
    Volume& v = c->vol[i];
    v.solid = g->solid[i];
    v.material = g->material[i];
    v.mother = g->mother[i];
    v.dbegin = g->daughter_begin[i];
    v.dcount = g->daughter_count[i];
    for (int k = 0; k < 3; ++k) { v.dims[k] = g->dims[3 * i + k]; v.t[k] = g->trans[3 * i + k]; }
    for (int k = 0; k < 9; ++k) v.R[k] = g->rot[9 * i + k];
  }
  c->n_mat = m->n_mat;
  c->tables.assign(m->tables, m->tables + static_cast<size_t>(m->n_mat) * N_TAB * kNGrid);
  c->scalars.assign(m->scalars, m->scalars + static_cast<size_t>(m->n_mat) * N_SCAL);
  if (m->n_elem && m->elem_bk && m->pe_cum) {
    c->n_elem.assign(m->n_elem, m->n_elem + m->n_mat);
    c->elem_bk.assign(m->elem_bk, m->elem_bk + static_cast<size_t>(m->n_mat) * ORC_MAX_ELEMENTS);
    c->pe_cum.assign(m->pe_cum, m->pe_cum + static_cast<size_t>(m->n_mat) * kNGrid * ORC_MAX_ELEMENTS);
  }
  c->field = *f;
  if (f->kind == ORC_FIELD_MAP_RZ) c->bz.assign(f->bz, f->bz + static_cast<size_t>(f->nr) * f->nz);
  c->field.bz = nullptr;
  c->cfg = *cfg;
  c->u0 = std::log(1.0e-3);
  c->du = (std::log(1.0e8) - std::log(1.0e-3)) / (kNGrid - 1);
  return c;
}

extern "C" void orc_destroy(orc_ctx* c) { delete c; }

extern "C" void orc_set_recorder(orc_ctx* c, uint32_t mask, uint32_t stride, orc_track* buf, size_t cap) {
  c->rec_mask = mask; c->rec_stride = stride ? stride : 1; c->rec_buf = buf; c->rec_cap = cap;
  c->rec_n = 0; c->rec_counter = 0;
}
extern "C" size_t orc_recorded(const orc_ctx* c) { return c->rec_n; }

static inline double carried(const orc_track& t) { return t.species == ORC_POSITRON ? t.ekin + 2.0 * kMe : t.ekin; }

/* G5: push past the boundary and relocate; returns false if the track left the world */
static bool cross_boundary(const orc_ctx* c, orc_track& t, const double pushdir[3]) {
  for (int i = 0; i < 3; ++i) t.pos[i] += c->cfg.eps_push * pushdir[i];
  const int64_t v = orc_locate(c, t.pos);
  if (v < 0) return false;
  t.volume = static_cast<uint32_t>(v);
  return true;
}

/* S1 */
static void gamma_step(const orc_ctx* c, const orc_track* in, orc_step_result* out, orc_track* sec) {
  orc_track& t = out->post;
  const int mat = c->vol[in->volume].material;
  const double k = in->ekin;
  if (k < kTmin) { out->edep_cut += k; out->alive = 0; out->outcome = ORC_OUT_STOPPED; return; }
  double sc = 0.0, sp = 0.0, se = 0.0;
  if (scalar(c, mat, S_VACUUM) == 0.0) {
    sc = orc_lookup(c, mat, T_G_COMPTON, k);
    /* P2 threshold: the interpolated table is positive in the grid cell that straddles 2m */
    sp = k > 2.0 * kMe ? orc_lookup(c, mat, T_G_PAIR, k) : 0.0;
    se = orc_lookup(c, mat, T_G_PHOTO, k);
  }
  const double stot = sc + sp + se;
  const double u0 = orc_uniform(in->event, c->cfg.seed, in->id, in->step, 0);
  const double s_phys = stot > 0.0 ? -std::log(u0) / stot : kInf;
  const double s_geo = orc_distance(c, in->pos, in->dir, in->volume, s_phys);
  if (s_geo < s_phys) {
    for (int i = 0; i < 3; ++i) t.pos[i] += s_geo * in->dir[i];
    out->s = s_geo;
    if (!cross_boundary(c, t, in->dir)) {
      out->escaped += k; out->alive = 0; out->outcome = ORC_OUT_ESCAPED;
    } else {
      out->outcome = ORC_OUT_BOUNDARY;
    }
    return;
  }
  for (int i = 0; i < 3; ++i) t.pos[i] += s_phys * in->dir[i];
  out->s = s_phys;
  const double u1 = orc_uniform(in->event, c->cfg.seed, in->id, in->step, 1);
  int process = ORC_OUT_PHOTO;
  if (u1 * stot < sc) process = ORC_OUT_COMPTON;
  else if (u1 * stot < sc + sp) process = ORC_OUT_PAIR;
  orc_run_process(c, process, in, mat, out, sec);
}

/* S2 */
static void charged_step(const orc_ctx* c, const orc_track* in, orc_step_result* out, orc_track* sec) {
  orc_track& t = out->post;
  const bool positron = in->species == ORC_POSITRON;
  const int mat = c->vol[in->volume].material;
  const bool vacuum = scalar(c, mat, S_VACUUM) != 0.0;
  const double T0 = in->ekin;
  if (T0 < kTmin) {
    out->edep_cut += T0; t.ekin = 0.0;
    if (positron) orc_annihilate_at_rest(c, in, mat, out, sec);
    out->alive = 0; out->outcome = ORC_OUT_STOPPED;
    return;
  }
  const int tb = positron ? T_EP_BREM : T_EM_BREM, ti = positron ? T_EP_IONI : T_EM_IONI;
  const int td = positron ? T_EP_DEDX : T_EM_DEDX, tr = positron ? T_EP_RANGE : T_EM_RANGE;
  double sb = 0.0, si = 0.0, sa = 0.0, S = 0.0, R = kInf;
  if (!vacuum) {
    sb = orc_lookup(c, mat, tb, T0);
    si = orc_lookup(c, mat, ti, T0);
    if (positron) sa = orc_lookup(c, mat, T_EP_ANNI, T0);
    S = orc_lookup(c, mat, td, T0);
    R = orc_lookup(c, mat, tr, T0);
  }
  const double stot = sb + si + sa;
  const double u0 = orc_uniform(in->event, c->cfg.seed, in->id, in->step, 0);
  const double s_disc = stot > 0.0 ? -std::log(u0) / stot : kInf;
  const double aR = c->cfg.alpha_R, rR = c->cfg.rho_R;
  const bool range_out = R <= rR;
  const double s_loss = range_out ? R : aR * R + rR * (1.0 - aR) * (2.0 - rR / R);
  const bool lim_disc = s_disc < s_loss;
  const double s_phys = lim_disc ? s_disc : s_loss;
  /* propagate */
  double pushdir[3], s = 0.0;
  int chords = 0;
  const int flag = orc_propagate(c, positron ? +1 : -1, T0, t.pos, t.dir, in->volume, s_phys, &s, &chords, pushdir);
  out->s = s; out->chords = chords;
  /* continuous loss */
  double dE = 0.0;
  if (!vacuum) {
    if (flag == 0 && !lim_disc && range_out) dE = T0;
    else if (s <= 0.01 * R) dE = S * s;
    else {
      const double Tn = orc_inverse_range(c, mat, tr, R - s);
      dE = T0 - Tn;
    }
    dE = std::min(std::max(dE, 0.0), T0);
  }
  out->edep_dep += dE;
  t.ekin = T0 - dE;
  if (t.ekin < kTmin) {
    out->edep_cut += t.ekin; t.ekin = 0.0;
    if (positron) { orc_track p = *in; orc_annihilate_at_rest(c, &p, mat, out, sec); }
    out->alive = 0; out->outcome = ORC_OUT_STOPPED;
    return;
  }
  /* P9 Highland MSC at the pre-step energy */
  if (!vacuum && s > 0.0) {
    const double X0 = scalar(c, mat, S_X0);
    const double pbeta = T0 * (T0 + 2.0 * kMe) / (T0 + kMe);
    const double beta2 = T0 * (T0 + 2.0 * kMe) / ((T0 + kMe) * (T0 + kMe));
    const double corr = std::max(0.0, 1.0 + 0.038 * std::log(s / (X0 * beta2)));
    const double th0 = (13.6 / pbeta) * std::sqrt(s / X0) * corr;
    const double u2 = orc_uniform(in->event, c->cfg.seed, in->id, in->step, 2);
    const double u3 = orc_uniform(in->event, c->cfg.seed, in->id, in->step, 3);
    const double th = th0 * std::sqrt(-2.0 * std::log(u2));
    double dn[3];
    orc_rotate(t.dir, std::cos(th), std::sin(th), 2.0 * kPi * u3, dn);
    for (int i = 0; i < 3; ++i) t.dir[i] = dn[i];
  }
  if (flag == 1) {
    if (!cross_boundary(c, t, pushdir)) {
      out->escaped += carried(t); out->alive = 0; out->outcome = ORC_OUT_ESCAPED;
    } else {
      out->outcome = ORC_OUT_BOUNDARY;
    }
    return;
  }
  if (flag == 2) { out->outcome = ORC_OUT_TRUNCATED; return; }
  if (!lim_disc) { out->outcome = ORC_OUT_LOSS; return; }
  const double u1 = orc_uniform(in->event, c->cfg.seed, in->id, in->step, 1);
  int process = ORC_OUT_BREM;
  if (u1 * stot < sb) process = ORC_OUT_BREM;
  else if (!positron || u1 * stot < sb + si) process = ORC_OUT_IONI;
  else process = ORC_OUT_ANNI;
  orc_run_process(c, process, in, mat, out, sec);
}

extern "C" void orc_step(const orc_ctx* c, const orc_track* in, orc_step_result* out, orc_track sec[2]) {
  *out = orc_step_result{};
  out->post = *in;
  out->alive = 1;
  if (in->step >= c->cfg.max_steps) { /* S4 */
    out->killed += carried(*in); out->alive = 0; out->outcome = ORC_OUT_KILLED;
    return;
  }
  if (in->species == ORC_GAMMA) gamma_step(c, in, out, sec);
  else charged_step(c, in, out, sec);
  if (out->alive) out->post.step = in->step + 1;
}

/* PAPER.md:71 describes the CPU workflow this oracle keeps: one track at a time, secondaries on a
   stack.  S3: every step's energy goes into exactly one ledger bucket. */
extern "C" int orc_run(orc_ctx* c, size_t n, const orc_track* primaries, double* edep, orc_ledger* ledger,
                       orc_stats* stats) {
  std::vector<orc_track> stack;
  std::vector<uint64_t> iter; /* population-stepping iteration at which the track would be stepped */
  orc_step_result r;
  orc_track sec[2];
  for (size_t ip = 0; ip < n; ++ip) {
    stack.push_back(primaries[ip]);
    iter.push_back(0);
    ledger->primary += carried(primaries[ip]);
    while (!stack.empty()) {
      const orc_track t = stack.back();
      stack.pop_back();
      const uint64_t it = iter.back();
      iter.pop_back();
      if (stats && it + 1 > stats->iterations) stats->iterations = it + 1;
      if (c->rec_cap && ((c->rec_mask >> t.species) & 1u)) {
        if (c->rec_counter++ % c->rec_stride == 0 && c->rec_n < c->rec_cap) c->rec_buf[c->rec_n++] = t;
      }
      orc_step(c, &t, &r, sec);
      edep[t.volume] += r.edep_dep + r.edep_cut;
      ledger->deposited += r.edep_dep;
      ledger->below_cut += r.edep_cut;
      ledger->escaped += r.escaped;
      ledger->killed += r.killed;
      if (stats) {
        stats->steps[t.species]++;
        stats->outcomes[r.outcome]++;
        stats->chords += static_cast<uint64_t>(r.chords);
        for (int k = 0; k < r.n_sec; ++k) stats->secondaries[sec[k].species]++;
      }
      if (r.alive) { stack.push_back(r.post); iter.push_back(it + 1); }
      for (int k = 0; k < r.n_sec; ++k) { stack.push_back(sec[k]); iter.push_back(it + 1); }
      if (stats && stack.size() > stats->peak_stack) stats->peak_stack = stack.size();
    }
  }
  return 0;
}
