// Table lookup and the discrete-interaction samplers  (§8(c) M7, P1-P10).
// All functions take scalar arguments and keep no thread-local state.
#pragma once
#include "fastmath.cuh"
#include "rng.cuh"
#include "types.cuh"

namespace adept {

__device__ __forceinline__ double mat_scalar(const DevCtx& c, int mat, int s) { return __ldg(c.scal + mat * N_SCAL + s); }

// M7: cell index and fraction of ln T on the grid
struct GridPos { int i; double f; };
__device__ __forceinline__ GridPos grid_pos(const DevCtx& c, double ekin) {
  const double x = (log_pos(ekin) - c.u0) * c.inv_du;
  int i = static_cast<int>(floor(x));
  i = min(max(i, 0), kNGrid - 2);
  return GridPos{i, x - i};
}
// value of column `col` of an interleaved table with `row` doubles per node
__device__ __forceinline__ double interp(const double* __restrict__ tab, int row, int col, GridPos g) {
  const double y0 = __ldg(tab + g.i * row + col), y1 = __ldg(tab + (g.i + 1) * row + col);
  return y0 + g.f * (y1 - y0);
}

// One 32 B table row (4 columns) in two 16 B loads.
struct Row4 { double v[4]; };
__device__ __forceinline__ Row4 load_row4(const double* __restrict__ row) {
  const double2 a = __ldg(reinterpret_cast<const double2*>(row)), b = __ldg(reinterpret_cast<const double2*>(row) + 1);
  return Row4{{a.x, a.y, b.x, b.y}};
}
__device__ __forceinline__ double lerp_col(const Row4& r0, const Row4& r1, int col, double f) {
  return r0.v[col] + f * (r1.v[col] - r0.v[col]);
}

// M7 inverse range: cell j with R_j <= r < R_{j+1}, then ln T linear in r.  Any search returns the same
// j; this one starts from a hint table indexed by the exponent and top 5 mantissa bits of r (a
// monotone pseudo-logarithm, built by adept_init: hint[k] = largest j with R_j <= lower edge of key
// cell k) and walks up, typically 0-2 nodes, instead of ~10 dependent loads of a binary search.
// Returns 0 when r < R_0 (the track stops).
constexpr int kHintN = 2048;           // key cells per table: 64 octaves of range
constexpr int kHintStride = kHintN + 2;  // [0] = key of R_0, [1..kHintN] = hints, [last] pad
__device__ __forceinline__ int range_key(double r) { return __double2hiint(r) >> 15; }

__device__ __forceinline__ double inverse_range(const DevCtx& c, const double* __restrict__ tab, int row, int col,
                                                const int32_t* __restrict__ hint, double r) {
  if (r < __ldg(tab + col)) return 0.0;
  const int k = min(max(range_key(r) - __ldg(hint), 0), kHintN - 1);
  int lo = __ldg(hint + 1 + k);
  double R0 = __ldg(tab + lo * row + col), R1 = __ldg(tab + (lo + 1) * row + col);
  while (R1 <= r && lo < kNGrid - 2) {
    ++lo;
    R0 = R1;
    R1 = __ldg(tab + (lo + 1) * row + col);
  }
  const double lnT = c.u0 + c.du * lo + c.du * (r - R0) / (R1 - R0);
  return exp(lnT);
}

// P10 rotation of d by polar (cos_t, sin_t) and azimuth phi = pi * phi_over_pi (sincospi reduces the
// argument exactly).  One reciprocal each for 1/rho and the renormalisation.
__device__ __forceinline__ void rotate(const double d[3], double cos_t, double sin_t, double phi_over_pi, double out[3]) {
  const double rho2 = d[0] * d[0] + d[1] * d[1];
  double e1[3], e2[3];
  if (rho2 > 0.0) {
    const double ir = rsqrt(rho2);
    e1[0] = d[0] * d[2] * ir; e1[1] = d[1] * d[2] * ir; e1[2] = -rho2 * ir;
    e2[0] = -d[1] * ir; e2[1] = d[0] * ir; e2[2] = 0.0;
  } else {
    e1[0] = d[2] >= 0.0 ? 1.0 : -1.0; e1[1] = 0.0; e1[2] = 0.0;
    e2[0] = 0.0; e2[1] = 1.0; e2[2] = 0.0;
  }
  double sp, cp;
  sincospi(phi_over_pi, &sp, &cp);
  const double a = sin_t * cp, b = sin_t * sp;
  double n = 0.0;
#pragma unroll
  for (int i = 0; i < 3; ++i) { out[i] = a * e1[i] + b * e2[i] + cos_t * d[i]; n += out[i] * out[i]; }
  n = rsqrt(n);
#pragma unroll
  for (int i = 0; i < 3; ++i) out[i] *= n;
}

__device__ __forceinline__ double momentum(double T) { return sqrt(T * (T + 2.0 * kMe)); }

__device__ __forceinline__ void normalise(double v[3]) {
  const double n = rsqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
  v[0] *= n; v[1] *= n; v[2] *= n;
}

// M5: an e- below T_c or a gamma below k_c is not created (energy deposited locally); e+ always are.
// Child k of a process lives in the fixed slot o.sec[k] (species -1 = not created), so that StepOut is
// only ever indexed statically and stays in registers.
template <int CHILD>
__device__ __forceinline__ void emit(const DevCtx& c, int mat, StepOut& o, int species, const double dir[3], double ekin) {
  const double cut = species == ADEPT_GAMMA ? mat_scalar(c, mat, S_KCUT) : mat_scalar(c, mat, S_TCUT);
  if (species != ADEPT_POSITRON && ekin < cut) { o.edep_cut += ekin; return; }
  Secondary& s = o.sec[CHILD];
  s.dx = dir[0]; s.dy = dir[1]; s.dz = dir[2];
  s.ekin = ekin; s.species = species; s.child = CHILD;
  o.n_sec += 1;
}

// C5 element selector: the K-shell binding energy of the element a photon of energy k is absorbed on.
// In a compound that is element j with probability n_j sigma_j(k) / Sigma_photo(k): U6 of the step's stream (a
// spare slot of R3) against the cumulative shares, which are tabulated on the grid and interpolated like every
// table (M7); the first j with U6 < c_j, else the last element.  A single-element material draws nothing.
__device__ __forceinline__ double photo_binding(const DevCtx& c, int mat, double k, uint32_t event, uint64_t id, uint32_t step) {
  const int n = c.n_elem ? __ldg(c.n_elem + mat) : 1;
  if (n <= 1) return mat_scalar(c, mat, S_BK);
  const GridPos gp = grid_pos(c, k);
  const double* tab = c.pe_cum + (static_cast<size_t>(mat) * kNGrid + gp.i) * 4;
  const Row4 r0 = load_row4(tab), r1 = load_row4(tab + 4);
  Stream u;
  u.init(event, c.seed, id, step);
  const double u6 = u.uniform(6);
  int j = n - 1;
#pragma unroll
  for (int e = 2; e >= 0; --e)
    if (e < n - 1 && u6 < lerp_col(r0, r1, e, gp.f)) j = e;
  return __ldg(c.elem_bk + mat * 4 + j);
}

// ---- P1 Klein-Nishina Compton
__device__ __forceinline__ void compton(const DevCtx& c, int mat, StepOut& o, Stream& u) {
  Track& g = o.post;
  const double k = g.ekin, kap = k / kMe;
  const double e0 = 1.0 / (1.0 + 2.0 * kap);
  const double a1 = -log_pos(e0), a2 = 0.5 * (1.0 - e0 * e0);
  double eps = 1.0, t = 0.0, sin2 = 0.0;
  for (int it = 0; it < 1000; ++it) {
    const double r1 = u.draw(), r2 = u.draw(), r3 = u.draw();
    if (r1 * (a1 + a2) < a1) eps = exp(-r2 * a1);
    else eps = sqrt(e0 * e0 + (1.0 - e0 * e0) * r2);
    t = (1.0 - eps) / (kap * eps);
    sin2 = t * (2.0 - t);
    if (1.0 - eps * sin2 / (1.0 + eps * eps) >= r3) break;
  }
  const double phi = 2.0 * u.draw();   // azimuth in units of pi
  const double cos_t = 1.0 - t, sin_t = sqrt(fmax(sin2, 0.0));
  const double d0[3] = {g.dx, g.dy, g.dz};
  double d1[3];
  rotate(d0, cos_t, sin_t, phi, d1);
  const double k1 = eps * k;
  const double Te = k - k1;
  if (Te >= mat_scalar(c, mat, S_TCUT)) {
    double de[3] = {k * d0[0] - k1 * d1[0], k * d0[1] - k1 * d1[1], k * d0[2] - k1 * d1[2]};
    normalise(de);
    emit<0>(c, mat, o, ADEPT_ELECTRON, de, Te);
  } else {
    o.edep_cut += Te;
  }
  g.dx = d1[0]; g.dy = d1[1]; g.dz = d1[2];
  g.ekin = k1;
  if (k1 < kTmin) { o.edep_cut += k1; o.alive = 0; }
}

// ---- P2 Bethe-Heitler pair, complete screening
__device__ __forceinline__ void pair_production(const DevCtx& c, int mat, StepOut& o, Stream& u) {
  Track& g = o.post;
  const double k = g.ekin, a = kMe / k;
  const double fmax_ = 1.0 - (4.0 / 3.0) * a * (1.0 - a);
  double eps = 0.5;
  for (int it = 0; it < 1000; ++it) {
    const double r1 = u.draw(), r2 = u.draw();
    eps = a + (1.0 - 2.0 * a) * r1;
    if (1.0 - (4.0 / 3.0) * eps * (1.0 - eps) >= r2 * fmax_) break;
  }
  const double phi = 2.0 * u.draw();   // azimuth in units of pi
  const double Ep = eps * k, Em = (1.0 - eps) * k;
  const double Tp = fmax(Ep - kMe, 0.0), Tm = fmax(Em - kMe, 0.0);
  const double thm = kMe / Em, thp = kMe / Ep;
  const double d0[3] = {g.dx, g.dy, g.dz};
  double dm[3], dp[3], sn, cs;
  sincos(thm, &sn, &cs);
  rotate(d0, cs, sn, phi, dm);
  sincos(thp, &sn, &cs);
  rotate(d0, cs, sn, phi + 1.0, dp);
  emit<0>(c, mat, o, ADEPT_ELECTRON, dm, Tm);
  emit<1>(c, mat, o, ADEPT_POSITRON, dp, Tp);
  o.alive = 0;
}

// ---- P3 photoelectric, K shell; `step` = the step the absorption happens in (its stream selects the element)
__device__ void photoelectric(const DevCtx& c, int mat, StepOut& o, uint32_t step) {
  Track& g = o.post;
  const double k = g.ekin, BK = photo_binding(c, mat, k, g.event, g.id, step);
  if (k > BK) {
    o.edep_cut += BK;
    const double d0[3] = {g.dx, g.dy, g.dz};
    emit<0>(c, mat, o, ADEPT_ELECTRON, d0, k - BK);
  } else {
    o.edep_cut += k;
  }
  o.alive = 0;
}

// ---- P4 bremsstrahlung; false when kinematically closed
__device__ __forceinline__ bool bremsstrahlung(const DevCtx& c, int mat, StepOut& o, Stream& u) {
  Track& e = o.post;
  const double T = e.ekin, kc = mat_scalar(c, mat, S_KCUT);
  if (!(T > kc)) return false;
  const double E = T + kMe, lr = log_pos(T / kc);
  double k = kc;
  for (int it = 0; it < 1000; ++it) {
    const double r1 = u.draw(), r2 = u.draw();
    k = kc * exp(r1 * lr);
    const double y = k / E;
    if (4.0 / 3.0 - 4.0 * y / 3.0 + y * y >= (4.0 / 3.0) * r2) break;
  }
  k = fmin(k, T);
  const double phi = 2.0 * u.draw();   // azimuth in units of pi
  const double th = kMe / E;
  const double d0[3] = {e.dx, e.dy, e.dz};
  double dg[3], sn, cs;
  sincos(th, &sn, &cs);
  rotate(d0, cs, sn, phi, dg);
  emit<0>(c, mat, o, ADEPT_GAMMA, dg, k);
  e.ekin = T - k;
  return true;
}

// delta-ray kinematics shared by P5 and P6
__device__ __forceinline__ void delta_ray(const DevCtx& c, int mat, StepOut& o, double T, double Td, double phi) {
  Track& e = o.post;
  const double cos_t = fmin(1.0, sqrt(Td * (T + 2.0 * kMe) / (T * (Td + 2.0 * kMe))));
  const double sin_t = sqrt(fmax(0.0, 1.0 - cos_t * cos_t));
  const double d0[3] = {e.dx, e.dy, e.dz};
  double dd[3];
  rotate(d0, cos_t, sin_t, phi, dd);
  const double p = momentum(T), pd = momentum(Td);
  double dn[3] = {p * d0[0] - pd * dd[0], p * d0[1] - pd * dd[1], p * d0[2] - pd * dd[2]};
  normalise(dn);
  emit<0>(c, mat, o, ADEPT_ELECTRON, dd, Td);
  e.dx = dn[0]; e.dy = dn[1]; e.dz = dn[2];
  e.ekin = T - Td;
}

// ---- P5 Moller
__device__ __forceinline__ bool moller(const DevCtx& c, int mat, StepOut& o, Stream& u) {
  const double T = o.post.ekin, Tc = mat_scalar(c, mat, S_TCUT);
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
  const double phi = 2.0 * u.draw();   // azimuth in units of pi
  delta_ray(c, mat, o, T, eps * T, phi);
  return true;
}

// ---- P6 Bhabha
__device__ __forceinline__ bool bhabha(const DevCtx& c, int mat, StepOut& o, Stream& u) {
  const double T = o.post.ekin, Tc = mat_scalar(c, mat, S_TCUT);
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
  eps = fmin(eps, 1.0);
  const double phi = 2.0 * u.draw();   // azimuth in units of pi
  delta_ray(c, mat, o, T, eps * T, phi);
  return true;
}

// ---- P8 annihilation in flight (Heitler)
__device__ __forceinline__ void annihilation(const DevCtx& c, int mat, StepOut& o, Stream& u) {
  Track& e = o.post;
  const double T = e.ekin, g = 1.0 + T / kMe;
  const double root = sqrt((g - 1.0) / (g + 1.0));
  const double emin = 0.5 - 0.5 * root, emax = 0.5 + 0.5 * root;
  const double lr = log_pos(emax / emin), gp1sq = (g + 1.0) * (g + 1.0);
  double eps = 0.5;
  for (int it = 0; it < 1000; ++it) {
    const double r1 = u.draw(), r2 = u.draw();
    eps = emin * exp(r1 * lr);
    if (1.0 - eps + (2.0 * g * eps - 1.0) / (eps * gp1sq) >= r2) break;
  }
  const double phi = 2.0 * u.draw();   // azimuth in units of pi
  const double Etot = T + 2.0 * kMe;
  const double k1 = eps * Etot, k2 = Etot - k1;
  double cos_t = (eps * (g + 1.0) - 1.0) / (eps * sqrt(g * g - 1.0));
  cos_t = fmin(1.0, fmax(-1.0, cos_t));
  const double sin_t = sqrt(fmax(0.0, 1.0 - cos_t * cos_t));
  const double d0[3] = {e.dx, e.dy, e.dz};
  double d1[3];
  rotate(d0, cos_t, sin_t, phi, d1);
  const double p = momentum(T);
  double d2[3] = {p * d0[0] - k1 * d1[0], p * d0[1] - k1 * d1[1], p * d0[2] - k1 * d1[2]};
  normalise(d2);
  emit<0>(c, mat, o, ADEPT_GAMMA, d1, k1);
  emit<1>(c, mat, o, ADEPT_GAMMA, d2, k2);
  o.alive = 0;
}

// ---- P8 at rest: two photons of energy m back to back, cos(theta) = 2 U4 - 1, phi = 2 pi U5
__device__ __forceinline__ void annihilation_at_rest(const DevCtx& c, int mat, StepOut& o, Stream& u) {
  const double u4 = u.uniform(4), u5 = u.uniform(5);
  const double cos_t = 2.0 * u4 - 1.0, sin_t = sqrt(fmax(0.0, 1.0 - cos_t * cos_t));
  double sp, cp;
  sincospi(2.0 * u5, &sp, &cp);
  const double d1[3] = {sin_t * cp, sin_t * sp, cos_t};
  const double d2[3] = {-d1[0], -d1[1], -d1[2]};
  emit<0>(c, mat, o, ADEPT_GAMMA, d1, kMe);
  emit<1>(c, mat, o, ADEPT_GAMMA, d2, kMe);
}

// Runs one discrete process on the state in o.post with uniforms U8.. of the parent's stream.
__device__ __forceinline__ void run_process(const DevCtx& c, int process, int species, int mat, StepOut& o, Stream& u) {
  bool open = true;
  u.next = 8;
  switch (process) {
    case ADEPT_OUT_COMPTON: compton(c, mat, o, u); break;
    case ADEPT_OUT_PAIR: pair_production(c, mat, o, u); break;
    case ADEPT_OUT_PHOTO: photoelectric(c, mat, o, u.c2); break;
    case ADEPT_OUT_BREM: open = bremsstrahlung(c, mat, o, u); break;
    case ADEPT_OUT_IONI: open = species == ADEPT_ELECTRON ? moller(c, mat, o, u) : bhabha(c, mat, o, u); break;
    case ADEPT_OUT_ANNI: annihilation(c, mat, o, u); break;
    default: open = false;
  }
  o.outcome = open ? process : ADEPT_OUT_CLOSED;
}

}  // namespace adept
