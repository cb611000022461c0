/* ORACLE -- TEST INFRASTRUCTURE ONLY (see oracle.h).
 *
 * M7 table lookup, P10 rotation and the final-state samplers P1-P6, P8 of SURVEY.md §8(c)
 * (PAPER.md:53 delegates all physics to a library; BASELINE.json:north_star names the model set).
 * Pinned by tests/test_oracle_physics.py: chi-square of the sampled spectra against the
 * differential cross sections, energy/momentum balance of every final state, the production-cut
 * rule, and the rotation's orthonormality / polar angle.
 */
#include <algorithm>

#include "internal.h"

using namespace orc;

/* M7: linear interpolation in ln T of the quantity itself */
extern "C" double orc_lookup(const orc_ctx* c, int material, int tab, double ekin) {
  const double* y = table(c, material, tab);
  const double x = (std::log(ekin) - c->u0) / c->du;
  int i = static_cast<int>(std::floor(x));
  i = std::min(std::max(i, 0), kNGrid - 2);
  const double f = x - i;
  return y[i] + f * (y[i + 1] - y[i]);
}

/* M7 inverse range: R_j <= r < R_{j+1}, ln T = u_j + du (r - R_j)/(R_{j+1} - R_j).
   Returns 0 when r lies below the first node (the track stops). */
extern "C" double orc_inverse_range(const orc_ctx* c, int material, int range_table, double r) {
  const double* R = table(c, material, range_table);
  if (r < R[0]) return 0.0;
  int lo = 0, hi = kNGrid - 1; /* invariant: R[lo] <= r, and r < R[hi] or hi is the last node */
  while (hi - lo > 1) {
    const int mid = (lo + hi) / 2;
    if (R[mid] <= r) lo = mid; else hi = mid;
  }
  const double lnT = c->u0 + c->du * lo + c->du * (r - R[lo]) / (R[lo + 1] - R[lo]);
  return std::exp(lnT);
}

/* P10: rotate d by polar (cos_t, sin_t) and azimuth phi */
extern "C" void orc_rotate(const double d[3], double cos_t, double sin_t, double phi, double out[3]) {
  const double rho2 = d[0] * d[0] + d[1] * d[1];
  const double rho = std::sqrt(rho2);
  double e1[3], e2[3];
  if (rho > 0.0) {
    e1[0] = d[0] * d[2] / rho; e1[1] = d[1] * d[2] / rho; e1[2] = -rho2 / rho;
    e2[0] = -d[1] / rho; e2[1] = d[0] / rho; e2[2] = 0.0;
  } else {
    e1[0] = d[2] >= 0.0 ? 1.0 : -1.0; e1[1] = 0.0; e1[2] = 0.0;
    e2[0] = 0.0; e2[1] = 1.0; e2[2] = 0.0;
  }
  const double a = sin_t * std::cos(phi), b = sin_t * std::sin(phi);
  double n = 0.0;
  for (int i = 0; i < 3; ++i) { out[i] = a * e1[i] + b * e2[i] + cos_t * d[i]; n += out[i] * out[i]; }
  n = std::sqrt(n);
  for (int i = 0; i < 3; ++i) out[i] /= n;
}

namespace {

struct Final {
  const orc_ctx* c;
  const orc_track* parent;
  int material;
  orc_step_result* out;
  orc_track* sec;

  /* M5: an e- below T_c or a gamma below k_c is not created; its energy is deposited locally.
     e+ are always created.  Children get id = parent's block 0xFFFFFFFF - child_index (R3). */
  void emit(int species, const double dir[3], double ekin, uint32_t child_index) {
    const double cut = species == ORC_GAMMA ? scalar(c, material, S_KCUT) : scalar(c, material, S_TCUT);
    if (species != ORC_POSITRON && ekin < cut) { out->edep_cut += ekin; return; }
    orc_track& s = sec[out->n_sec++];
    for (int i = 0; i < 3; ++i) { s.pos[i] = out->post.pos[i]; s.dir[i] = dir[i]; }
    s.ekin = ekin;
    s.id = orc_child_id(parent->event, c->cfg.seed, parent->id, parent->step, child_index);
    s.event = parent->event;
    s.step = 0;
    s.volume = out->post.volume;
    s.species = species;
  }
};

inline double pmom(double T) { return std::sqrt(T * (T + 2.0 * kMe)); }

void normalise(double v[3]) {
  const double n = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
  for (int i = 0; i < 3; ++i) v[i] /= n;
}

/* P1 Klein-Nishina */
void compton(Final& f, Stream& u) {
  orc_track& g = f.out->post;
  const double k = g.ekin, kap = k / kMe;
  const double e0 = 1.0 / (1.0 + 2.0 * kap);
  const double a1 = -std::log(e0), a2 = 0.5 * (1.0 - e0 * e0);
  double eps = 1.0, t = 0.0, sin2 = 0.0;
  for (int it = 0; it < 1000; ++it) {
    const double r1 = u.draw(), r2 = u.draw(), r3 = u.draw();
    if (r1 * (a1 + a2) < a1) eps = std::exp(-r2 * a1);
    else eps = std::sqrt(e0 * e0 + (1.0 - e0 * e0) * r2);
    t = (1.0 - eps) / (kap * eps);
    sin2 = t * (2.0 - t);
    if (1.0 - eps * sin2 / (1.0 + eps * eps) >= r3) break;
  }
  const double phi = 2.0 * kPi * u.draw();
  const double cos_t = 1.0 - t, sin_t = std::sqrt(std::max(sin2, 0.0));
  double d1[3];
  orc_rotate(g.dir, cos_t, sin_t, phi, d1);
  const double k1 = eps * k;
  const double Te = k - k1;
  if (Te >= scalar(f.c, f.material, S_TCUT)) {
    double de[3] = {k * g.dir[0] - k1 * d1[0], k * g.dir[1] - k1 * d1[1], k * g.dir[2] - k1 * d1[2]};
    normalise(de);
    f.emit(ORC_ELECTRON, de, Te, 0);
  } else {
    f.out->edep_cut += Te;
  }
  for (int i = 0; i < 3; ++i) g.dir[i] = d1[i];
  g.ekin = k1;
  if (k1 < kTmin) { f.out->edep_cut += k1; f.out->alive = 0; }
}

/* P2 Bethe-Heitler pair, complete screening */
void pair(Final& f, Stream& u) {
  orc_track& g = f.out->post;
  const double k = g.ekin, a = kMe / k;
  const double fmax = 1.0 - (4.0 / 3.0) * a * (1.0 - a);
  double eps = 0.5;
  for (int it = 0; it < 1000; ++it) {
    const double r1 = u.draw(), r2 = u.draw();
    eps = a + (1.0 - 2.0 * a) * r1;
    if (1.0 - (4.0 / 3.0) * eps * (1.0 - eps) >= r2 * fmax) break;
  }
  const double phi = 2.0 * kPi * u.draw();
  const double Ep = eps * k, Em = (1.0 - eps) * k; /* total energies: e+ takes eps */
  const double Tp = std::max(Ep - kMe, 0.0), Tm = std::max(Em - kMe, 0.0);
  const double thm = kMe / Em, thp = kMe / Ep;
  double dm[3], dp[3];
  orc_rotate(g.dir, std::cos(thm), std::sin(thm), phi, dm);
  orc_rotate(g.dir, std::cos(thp), std::sin(thp), phi + kPi, dp);
  f.emit(ORC_ELECTRON, dm, Tm, 0);
  f.emit(ORC_POSITRON, dp, Tp, 1);
  f.out->alive = 0;
}

/* C5 element selector: in a compound the target element of a photoelectric absorption is element j
   with probability n_j sigma_j(k) / Sigma_photo(k).  The cumulative shares are tabulated on the ln T grid and
   interpolated like every table (M7); the choice uses U6 of the step's stream (a spare slot of R3): the first
   j with U6 < c_j(k), else the last element.  Single-element materials draw nothing. */
int select_element(const orc_ctx* c, int material, const orc_track* parent, double k) {
  if (c->n_elem.empty() || c->n_elem[material] <= 1) return 0;
  const int n = c->n_elem[material];
  const double x = (std::log(k) - c->u0) / c->du;
  int i = static_cast<int>(std::floor(x));
  i = std::min(std::max(i, 0), kNGrid - 2);
  const double fr = x - i;
  const double* row0 = c->pe_cum.data() + (static_cast<size_t>(material) * kNGrid + i) * ORC_MAX_ELEMENTS;
  const double* row1 = row0 + ORC_MAX_ELEMENTS;
  const double u6 = orc_uniform(parent->event, c->cfg.seed, parent->id, parent->step, 6);
  for (int j = 0; j < n - 1; ++j) {
    const double cj = row0[j] + fr * (row1[j] - row0[j]);
    if (u6 < cj) return j;
  }
  return n - 1;
}

/* P3 photoelectric, K shell (of the selected element in a compound) */
void photo(Final& f, Stream&) {
  orc_track& g = f.out->post;
  const double k = g.ekin;
  const int el = select_element(f.c, f.material, f.parent, k);
  const double BK = f.c->n_elem.empty() ? scalar(f.c, f.material, S_BK)
                                        : f.c->elem_bk[static_cast<size_t>(f.material) * ORC_MAX_ELEMENTS + el];
  if (k > BK) {
    f.out->edep_cut += BK;
    f.emit(ORC_ELECTRON, g.dir, k - BK, 0);
  } else {
    f.out->edep_cut += k;
  }
  f.out->alive = 0;
}

/* P4 bremsstrahlung; returns false when kinematically closed */
bool brem(Final& f, Stream& u) {
  orc_track& e = f.out->post;
  const double T = e.ekin, kc = scalar(f.c, f.material, S_KCUT);
  if (!(T > kc)) return false;
  const double E = T + kMe, lr = std::log(T / kc);
  double k = kc;
  for (int it = 0; it < 1000; ++it) {
    const double r1 = u.draw(), r2 = u.draw();
    k = kc * std::exp(r1 * lr);
    const double y = k / E;
    if (4.0 / 3.0 - 4.0 * y / 3.0 + y * y >= (4.0 / 3.0) * r2) break;
  }
  k = std::min(k, T);
  const double phi = 2.0 * kPi * u.draw();
  const double th = kMe / E;
  double dg[3];
  orc_rotate(e.dir, std::cos(th), std::sin(th), phi, dg);
  f.emit(ORC_GAMMA, dg, k, 0);
  e.ekin = T - k;
  return true;
}

/* kinematics shared by P5 and P6: delta ray of energy Td off a parent of energy T */
void delta_ray(Final& f, double T, double Td, double phi) {
  orc_track& e = f.out->post;
  const double cos_t = std::min(1.0, std::sqrt(Td * (T + 2.0 * kMe) / (T * (Td + 2.0 * kMe))));
  const double sin_t = std::sqrt(std::max(0.0, 1.0 - cos_t * cos_t));
  double dd[3];
  orc_rotate(e.dir, cos_t, sin_t, phi, dd);
  const double p = pmom(T), pd = pmom(Td);
  double dn[3] = {p * e.dir[0] - pd * dd[0], p * e.dir[1] - pd * dd[1], p * e.dir[2] - pd * dd[2]};
  normalise(dn);
  f.emit(ORC_ELECTRON, dd, Td, 0);
  for (int i = 0; i < 3; ++i) e.dir[i] = dn[i];
  e.ekin = T - Td;
}

/* P5 Moller */
bool moller(Final& f, Stream& u) {
  const double T = f.out->post.ekin, Tc = scalar(f.c, f.material, S_TCUT);
  if (!(T > 2.0 * Tc)) return false;
  const double g = 1.0 + T / kMe, g2 = g * g;
  const double b = (2.0 * g - 1.0) / g2, c0 = (g - 1.0) * (g - 1.0) / g2;
  const double x = Tc / T, hmax = 2.25 - 1.25 * b;
  double eps = x;
  for (int it = 0; it < 1000; ++it) {
    const double r1 = u.draw(), r2 = u.draw();
    eps = x * 0.5 / (x * (1.0 - r1) + 0.5 * r1);
    const double ie = 1.0 / eps, i1 = 1.0 / (1.0 - eps);
    const double h = eps * eps * (c0 + ie * (ie - b) + i1 * (i1 - b));
    if (h >= r2 * hmax) break;
  }
  const double phi = 2.0 * kPi * u.draw();
  delta_ray(f, T, eps * T, phi);
  return true;
}

/* P6 Bhabha */
bool bhabha(Final& f, Stream& u) {
  const double T = f.out->post.ekin, Tc = scalar(f.c, f.material, S_TCUT);
  if (!(T > Tc)) return false;
  const double g = 1.0 + T / kMe;
  const double beta2 = 1.0 - 1.0 / (g * g);
  const double y = 1.0 / (g + 1.0), w = 1.0 - 2.0 * y;
  const double B1 = 2.0 - y * y, B2 = w * (3.0 + y * y), B3 = w * w + w * w * w, B4 = w * w * w;
  const double x = Tc / T;
  double eps = x;
  for (int it = 0; it < 1000; ++it) {
    const double r1 = u.draw(), r2 = u.draw();
    eps = x / (1.0 - r1 * (1.0 - x));
    const double h = 1.0 - beta2 * eps * (B1 - B2 * eps + B3 * eps * eps - B4 * eps * eps * eps);
    if (h >= r2) break;
  }
  eps = std::min(eps, 1.0);
  const double phi = 2.0 * kPi * u.draw();
  delta_ray(f, T, eps * T, phi);
  return true;
}

/* P8 annihilation in flight (Heitler) */
void annihilate(Final& f, Stream& u) {
  orc_track& e = f.out->post;
  const double T = e.ekin, g = 1.0 + T / kMe;
  const double root = std::sqrt((g - 1.0) / (g + 1.0));
  const double emin = 0.5 - 0.5 * root, emax = 0.5 + 0.5 * root;
  const double lr = std::log(emax / emin), gp1sq = (g + 1.0) * (g + 1.0);
  double eps = 0.5;
  for (int it = 0; it < 1000; ++it) {
    const double r1 = u.draw(), r2 = u.draw();
    eps = emin * std::exp(r1 * lr);
    if (1.0 - eps + (2.0 * g * eps - 1.0) / (eps * gp1sq) >= r2) break;
  }
  const double phi = 2.0 * kPi * u.draw();
  const double Etot = T + 2.0 * kMe;
  const double k1 = eps * Etot, k2 = Etot - k1;
  double cos_t = (eps * (g + 1.0) - 1.0) / (eps * std::sqrt(g * g - 1.0));
  cos_t = std::min(1.0, std::max(-1.0, cos_t));
  const double sin_t = std::sqrt(std::max(0.0, 1.0 - cos_t * cos_t));
  double d1[3];
  orc_rotate(e.dir, cos_t, sin_t, phi, d1);
  const double p = pmom(T);
  double d2[3] = {p * e.dir[0] - k1 * d1[0], p * e.dir[1] - k1 * d1[1], p * e.dir[2] - k1 * d1[2]};
  normalise(d2);
  f.emit(ORC_GAMMA, d1, k1, 0);
  f.emit(ORC_GAMMA, d2, k2, 1);
  f.out->alive = 0;
}

}  // namespace

/* Runs `process` (ORC_OUT_COMPTON .. ORC_OUT_ANNI) on the state already stored in out->post, with
   uniforms U8.. of the parent's (event, id, step) stream (R3).  Sets out->outcome. */
void orc_run_process(const orc_ctx* c, int process, const orc_track* parent, int material,
                     orc_step_result* out, orc_track* sec) {
  Final f{c, parent, material, out, sec};
  Stream u{parent->event, c->cfg.seed, parent->step, parent->id, 8};
  bool open = true;
  switch (process) {
    case ORC_OUT_COMPTON: compton(f, u); break;
    case ORC_OUT_PAIR: pair(f, u); break;
    case ORC_OUT_PHOTO: photo(f, u); break;
    case ORC_OUT_BREM: open = brem(f, u); break;
    case ORC_OUT_IONI: open = parent->species == ORC_ELECTRON ? moller(f, u) : bhabha(f, u); break;
    case ORC_OUT_ANNI: annihilate(f, u); break;
    default: open = false;
  }
  out->outcome = open ? process : ORC_OUT_CLOSED;
}

/* P8 at rest: two photons of energy m back to back, cos(theta) = 2 U4 - 1, phi = 2 pi U5 */
void orc_annihilate_at_rest(const orc_ctx* c, const orc_track* parent, int material, orc_step_result* out,
                            orc_track* sec) {
  Final f{c, parent, material, out, sec};
  const double u4 = orc_uniform(parent->event, c->cfg.seed, parent->id, parent->step, 4);
  const double u5 = orc_uniform(parent->event, c->cfg.seed, parent->id, parent->step, 5);
  const double cos_t = 2.0 * u4 - 1.0, sin_t = std::sqrt(std::max(0.0, 1.0 - cos_t * cos_t));
  const double phi = 2.0 * kPi * u5;
  const double d1[3] = {sin_t * std::cos(phi), sin_t * std::sin(phi), cos_t};
  const double d2[3] = {-d1[0], -d1[1], -d1[2]};
  f.emit(ORC_GAMMA, d1, kMe, 0);
  f.emit(ORC_GAMMA, d2, kMe, 1);
}

extern "C" void orc_interact(const orc_ctx* c, int process, const orc_track* t, int material,
                             orc_step_result* out, orc_track sec[2]) {
  *out = orc_step_result{};
  out->post = *t;
  out->alive = 1;
  orc_run_process(c, process, t, material, out, sec);
  if (out->alive) out->post.step = t->step + 1;
}
