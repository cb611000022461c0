/* ORACLE -- TEST INFRASTRUCTURE ONLY (see oracle.h).
 *
 * M1-M6 and the total cross sections / stopping powers of P1-P8, evaluated in
 * long double on the 2048-point ln T grid (BASELINE.json:north_star: "tabulated on a 2048-point
 * log-energy grid from 1 keV to 100 TeV").  The product's own builder is
 * paper_2209_15445_b200/inputs/materials.py; the two are compared in tests/test_tables.py.
 * Pinned by tests/test_oracle_tables.py: each closed-form total against numerical quadrature of
 * its differential cross section, the Thomson limit, S_coll(T;T2) - S_coll(T;T1) against the first
 * moment of the Moller/Bhabha differential, textbook radiation lengths, S_rad -> T/X0.
 */
#include <cmath>

#include "internal.h"

namespace {

typedef long double ld;
const ld M = 0.51099895L, RE = 2.8179403262e-13L, ALPHA = 1.0L / 137.035999084L, NA = 6.02214076e23L;
const ld PI = 3.141592653589793238462643383279502884L;

/* A material: one element (M1-M3) or a compound of up to 4 (C1-C3):
   C1  nu_i atoms of element i per formula unit, molar mass A_mol = sum nu_i A_i; number densities
       n_i = N_A rho nu_i / A_mol, n_at = sum n_i, n_el = sum n_i Z_i;
   C2  1/X0 = sum_i 4 alpha r_e^2 n_i [Z_i^2 (L_rad,i - f_c,i) + Z_i L'_rad,i]   (Tsai, additive in the atoms);
   C3  ln I = sum_i n_i Z_i ln I_i / n_el  (Bragg additivity of the stopping number), plasma energy from the
       total electron density: hbar omega_p = 28.816 eV sqrt(rho sum nu_i Z_i / A_mol). */
struct Mat {
  int n;
  ld Z[4], A[4], n_i[4], BKi[4];
  ld rho, n_at, n_el, X0, I, hwp, BK;
};

ld tsai_per_atom(ld Z) { /* Z^2 (L_rad - f_c) + Z L'_rad */
  const ld a = ALPHA * Z, a2 = a * a;
  const ld fc = a2 * (1.0L / (1.0L + a2) + 0.20206L - 0.0369L * a2 + 0.0083L * a2 * a2 - 0.002L * a2 * a2 * a2);
  const ld lrad = logl(184.15L * powl(Z, -1.0L / 3.0L));
  const ld lprad = logl(1194.0L * powl(Z, -2.0L / 3.0L));
  return Z * Z * (lrad - fc) + Z * lprad;
}
ld mean_excitation(ld Z) { /* M3, MeV */
  const ld i_ev = Z < 13.0L ? Z * (12.0L + 7.0L / Z) : Z * (9.76L + 58.8L * powl(Z, -1.19L));
  return i_ev * 1.0e-6L;
}

Mat make_compound(int n, const ld* Z, const ld* A, const ld* nu, ld rho) {
  Mat m{};
  m.n = n; m.rho = rho;
  ld a_mol = 0.0L, z_mol = 0.0L;
  for (int i = 0; i < n; ++i) { a_mol += nu[i] * A[i]; z_mol += nu[i] * Z[i]; }
  ld inv_x0 = 0.0L, lnI = 0.0L;
  for (int i = 0; i < n; ++i) {
    m.Z[i] = Z[i]; m.A[i] = A[i];
    m.n_i[i] = NA * rho * nu[i] / a_mol;
    m.n_at += m.n_i[i];
    m.n_el += m.n_i[i] * Z[i];
    inv_x0 += 4.0L * ALPHA * RE * RE * m.n_i[i] * tsai_per_atom(Z[i]);
    lnI += m.n_i[i] * Z[i] * logl(mean_excitation(Z[i]));
    m.BKi[i] = 13.605693e-6L * (Z[i] - 1.0L) * (Z[i] - 1.0L); /* P3 */
  }
  m.X0 = 1.0L / inv_x0;
  m.I = n == 1 ? mean_excitation(Z[0]) : expl(lnI / m.n_el);
  m.hwp = 28.816e-6L * sqrtl(rho * z_mol / a_mol);
  m.BK = m.BKi[0];
  return m;
}

Mat make(ld Z, ld A, ld rho) {
  const ld one = 1.0L;
  return make_compound(1, &Z, &A, &one, rho);
}

/* P1: Klein-Nishina per electron */
ld sigma_kn(ld k) {
  const ld kap = k / M;
  if (kap < 2.0e-3L) {
    const ld st = 8.0L * PI * RE * RE / 3.0L;
    return st * (1.0L - 2.0L * kap + 26.0L * kap * kap / 5.0L - 133.0L * kap * kap * kap / 10.0L +
                 1144.0L * powl(kap, 4) / 35.0L - 544.0L * powl(kap, 5) / 7.0L);
  }
  const ld l = log1pl(2.0L * kap);
  return 2.0L * PI * RE * RE * ((1.0L + kap) / (kap * kap) * (2.0L * (1.0L + kap) / (1.0L + 2.0L * kap) - l / kap) +
                                l / (2.0L * kap) - (1.0L + 3.0L * kap) / ((1.0L + 2.0L * kap) * (1.0L + 2.0L * kap)));
}

/* P2: X0 * Sigma_pair */
ld pair_shape(ld k) {
  if (!(k > 2.0L * M)) return 0.0L;
  const ld a = M / k;
  return 7.0L / 9.0L - 2.0L * a + 4.0L * a * a / 3.0L - 8.0L * a * a * a / 9.0L;
}

/* P3: per atom */
ld sigma_pe(ld k, ld Z) {
  const ld st = 8.0L * PI * RE * RE / 3.0L;
  return 1.25L * 4.0L * sqrtl(2.0L) * powl(ALPHA, 4) * powl(Z, 5) * st * powl(M / k, 3.5L);
}

/* macroscopic photoelectric cross section: sum over the elements */
ld Sigma_pe(const Mat& m, ld k) {
  ld s = 0.0L;
  for (int i = 0; i < m.n; ++i) s += m.n_i[i] * sigma_pe(k, m.Z[i]);
  return s;
}

/* P4: X0 * Sigma_brem and X0 * S_rad */
ld brem_shape(ld T, ld kc) {
  if (!(T > kc)) return 0.0L;
  const ld E = T + M;
  return (4.0L / 3.0L) * logl(T / kc) - (4.0L / 3.0L) * (T - kc) / E + (T * T - kc * kc) / (2.0L * E * E);
}
ld srad_shape(ld T, ld kc) {
  const ld E = T + M, ku = kc < T ? kc : T;
  return (4.0L / 3.0L) * ku - (2.0L / 3.0L) * ku * ku / E + ku * ku * ku / (3.0L * E * E);
}

/* P5 */
ld sigma_moller(ld T, ld Tc) {
  if (!(T > 2.0L * Tc)) return 0.0L;
  const ld g = 1.0L + T / M, b2 = 1.0L - 1.0L / (g * g), x = Tc / T;
  return 2.0L * PI * RE * RE / (b2 * (g - 1.0L)) *
         ((g - 1.0L) * (g - 1.0L) / (g * g) * (0.5L - x) + 1.0L / x - 1.0L / (1.0L - x) -
          (2.0L * g - 1.0L) / (g * g) * logl((1.0L - x) / x));
}

/* P6 */
ld sigma_bhabha(ld T, ld Tc) {
  if (!(T > Tc)) return 0.0L;
  const ld g = 1.0L + T / M, b2 = 1.0L - 1.0L / (g * g), x = Tc / T;
  const ld y = 1.0L / (g + 1.0L), w = 1.0L - 2.0L * y;
  const ld B1 = 2.0L - y * y, B2 = w * (3.0L + y * y), B3 = w * w + w * w * w, B4 = w * w * w;
  return 2.0L * PI * RE * RE / (g - 1.0L) *
         ((1.0L / b2) * (1.0L / x - 1.0L) + B1 * logl(x) + B2 * (1.0L - x) - B3 * (1.0L - x * x) / 2.0L +
          B4 * (1.0L - x * x * x) / 3.0L);
}

/* P8 Heitler */
ld sigma_ann(ld T) {
  const ld g = 1.0L + T / M, sq = sqrtl(g * g - 1.0L);
  return PI * RE * RE / (g + 1.0L) * ((g * g + 4.0L * g + 1.0L) / (g * g - 1.0L) * logl(g + sq) - (g + 3.0L) / sq);
}

/* P7 Berger-Seltzer restricted collision stopping power; Tc < 0 means unrestricted */
ld s_coll(ld T, const Mat& m, ld Tc, bool positron) {
  const ld tau = T / M, g = tau + 1.0L, b2 = 1.0L - 1.0L / (g * g);
  const ld tmax = positron ? tau : 0.5L * tau;
  ld tu = tmax;
  if (Tc >= 0.0L && Tc / M < tmax) tu = Tc / M;
  const ld bg = sqrtl(tau * (tau + 2.0L));
  ld delta = 2.0L * (logl(m.hwp / m.I) + logl(bg) - 0.5L);
  if (delta < 0.0L) delta = 0.0L;
  ld F;
  if (positron) {
    const ld y = 1.0L / (g + 1.0L);
    F = logl(tau * tu) - (b2 / tau) * (tau + 2.0L * tu - 1.5L * tu * tu * y - (tu - tu * tu * tu / 3.0L) * y * y -
                                      (tu * tu / 2.0L - tau * tu * tu * tu / 3.0L + powl(tu, 4) / 4.0L) * y * y * y);
  } else {
    F = -1.0L - b2 + logl((tau - tu) * tu) + tau / (tau - tu) +
        (tu * tu / 2.0L + (2.0L * tau + 1.0L) * logl(1.0L - tu / tau)) / (g * g);
  }
  return 2.0L * PI * RE * RE * M * m.n_el / b2 * (logl(2.0L * (g + 1.0L) / ((m.I / M) * (m.I / M))) + F - delta);
}

}  // namespace

/* exported for the pins: individual closed forms (double in/out, long double inside) */
extern "C" double orc_sigma_compton(double k) { return static_cast<double>(sigma_kn(k)); }
extern "C" double orc_pair_shape(double k) { return static_cast<double>(pair_shape(k)); }
extern "C" double orc_sigma_photo(double k, double Z) { return static_cast<double>(sigma_pe(k, Z)); }
extern "C" double orc_brem_shape(double T, double kc) { return static_cast<double>(brem_shape(T, kc)); }
extern "C" double orc_srad_shape(double T, double kc) { return static_cast<double>(srad_shape(T, kc)); }
extern "C" double orc_sigma_moller(double T, double Tc) { return static_cast<double>(sigma_moller(T, Tc)); }
extern "C" double orc_sigma_bhabha(double T, double Tc) { return static_cast<double>(sigma_bhabha(T, Tc)); }
extern "C" double orc_sigma_annihilation(double T) { return static_cast<double>(sigma_ann(T)); }
extern "C" double orc_s_coll(double T, double Z, double A, double rho, double Tc, int positron) {
  return static_cast<double>(s_coll(T, make(Z, A, rho), Tc, positron != 0));
}

namespace {
void build(const Mat* mp, double Zd, double rhod, double* tables, double* scalars);
}

extern "C" void orc_build_material(double Zd, double Ad, double rhod, double* tables, double* scalars) {
  if (!(rhod > 0.0)) { build(nullptr, Zd, rhod, tables, scalars); return; }
  const Mat m = make(Zd, Ad, rhod);
  build(&m, Zd, rhod, tables, scalars);
}

/* C1-C5: compound of n elements; elem_bk[4], pe_cum[2048][4] = cumulative share of elements 0..j in Sigma_photo
   at every grid node (the last used entry is 1; unused entries are 1 as well). */
extern "C" void orc_build_compound(int n, const double* Z, const double* A, const double* nu, double rho, double* tables,
                                   double* scalars, double* elem_bk, double* pe_cum) {
  using namespace orc;
  ld Zl[4], Al[4], nl[4];
  for (int i = 0; i < n; ++i) { Zl[i] = Z[i]; Al[i] = A[i]; nl[i] = nu[i]; }
  const Mat m = make_compound(n, Zl, Al, nl, rho);
  build(&m, static_cast<double>(m.n_el / m.n_at), rho, tables, scalars);
  for (int j = 0; j < 4; ++j) elem_bk[j] = j < n ? static_cast<double>(m.BKi[j]) : 0.0;
  const ld u0 = logl(1.0e-3L), du = (logl(1.0e8L) - logl(1.0e-3L)) / (kNGrid - 1);
  for (int i = 0; i < kNGrid; ++i) {
    const ld k = expl(u0 + du * i);
    const ld tot = Sigma_pe(m, k);
    ld acc = 0.0L;
    for (int j = 0; j < 4; ++j) {
      if (j < n) acc += m.n_i[j] * sigma_pe(k, m.Z[j]);
      pe_cum[4 * i + j] = j < n - 1 ? static_cast<double>(acc / tot) : 1.0;
    }
  }
}

namespace {
void build(const Mat* mp, double Zd, double rhod, double* tables, double* scalars) {
  using namespace orc;
  const int N = kNGrid;
  for (int i = 0; i < N_TAB * N; ++i) tables[i] = 0.0;
  for (int i = 0; i < N_SCAL; ++i) scalars[i] = 0.0;
  scalars[S_Z] = Zd; scalars[S_RHO] = rhod;
  if (!mp) { /* M1 vacuum: all Sigma = 0, dE/dx = 0 */
    for (int i = 0; i < N; ++i) tables[T_EM_RANGE * N + i] = tables[T_EP_RANGE * N + i] = 1.0e99;
    scalars[S_X0] = 1.0e99; scalars[S_VACUUM] = 1.0;
    return;
  }
  const Mat& m = *mp;
  const ld u0 = logl(1.0e-3L), du = (logl(1.0e8L) - logl(1.0e-3L)) / (N - 1);
  std::vector<ld> T(N), f(N), R(N), sig(N);
  for (int i = 0; i < N; ++i) T[i] = expl(u0 + du * i);
  auto range = [&](const std::vector<ld>& S) { /* M6: R_0 = T_0/S_0 + trapezoid in ln T of T/S */
    for (int i = 0; i < N; ++i) f[i] = T[i] / S[i];
    R[0] = f[0];
    for (int i = 1; i < N; ++i) R[i] = R[i - 1] + 0.5L * du * (f[i] + f[i - 1]);
  };
  /* M4 cuts */
  const ld cut = 0.07L;
  std::vector<ld> S(N);
  for (int i = 0; i < N; ++i) S[i] = s_coll(T[i], m, -1.0L, false) + srad_shape(T[i], T[i]) / m.X0;
  range(S);
  ld tc = 1.0e-3L;
  if (R[0] < cut) {
    int j = 0;
    while (j + 1 < N - 1 && R[j + 1] <= cut) ++j;
    tc = expl(u0 + du * j + du * (cut - R[j]) / (R[j + 1] - R[j]));
  }
  for (int i = 0; i < N; ++i) sig[i] = m.n_el * sigma_kn(T[i]) + pair_shape(T[i]) / m.X0 + Sigma_pe(m, T[i]);
  const ld target = 5.0L / cut;
  ld kc = 1.0e-3L;
  if (sig[0] > target) {
    int j = 0;
    while (j + 1 < N - 1 && sig[j + 1] >= target) ++j;
    kc = expl(u0 + du * j + du * (target - sig[j]) / (sig[j + 1] - sig[j]));
  }
  if (tc < 1.0e-3L) tc = 1.0e-3L;
  if (kc < 1.0e-3L) kc = 1.0e-3L;
  /* the product quantises the cuts to double before using them; so does the oracle */
  tc = static_cast<double>(tc); kc = static_cast<double>(kc);
  scalars[S_X0] = static_cast<double>(m.X0); scalars[S_TCUT] = static_cast<double>(tc);
  scalars[S_KCUT] = static_cast<double>(kc); scalars[S_BK] = static_cast<double>(m.BK);
  scalars[S_NEL] = static_cast<double>(m.n_el); scalars[S_VACUUM] = 0.0;
  for (int i = 0; i < N; ++i) {
    tables[T_G_COMPTON * N + i] = static_cast<double>(m.n_el * sigma_kn(T[i]));
    tables[T_G_PAIR * N + i] = static_cast<double>(pair_shape(T[i]) / m.X0);
    tables[T_G_PHOTO * N + i] = static_cast<double>(Sigma_pe(m, T[i]));
    const ld br = brem_shape(T[i], kc) / m.X0, sr = srad_shape(T[i], kc) / m.X0;
    tables[T_EM_BREM * N + i] = tables[T_EP_BREM * N + i] = static_cast<double>(br);
    tables[T_EM_IONI * N + i] = static_cast<double>(m.n_el * sigma_moller(T[i], tc));
    tables[T_EP_IONI * N + i] = static_cast<double>(m.n_el * sigma_bhabha(T[i], tc));
    tables[T_EP_ANNI * N + i] = static_cast<double>(m.n_el * sigma_ann(T[i]));
    S[i] = s_coll(T[i], m, tc, false) + sr;
    tables[T_EM_DEDX * N + i] = static_cast<double>(S[i]);
  }
  range(S);
  for (int i = 0; i < N; ++i) tables[T_EM_RANGE * N + i] = static_cast<double>(R[i]);
  for (int i = 0; i < N; ++i) {
    S[i] = s_coll(T[i], m, tc, true) + srad_shape(T[i], kc) / m.X0;
    tables[T_EP_DEDX * N + i] = static_cast<double>(S[i]);
  }
  range(S);
  for (int i = 0; i < N; ++i) tables[T_EP_RANGE * N + i] = static_cast<double>(R[i]);
}
}  // namespace
