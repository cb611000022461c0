/* ORACLE -- TEST INFRASTRUCTURE ONLY (see oracle.h). Internal declarations shared by the oracle sources. */
#ifndef ORACLE_INTERNAL_H
#define ORACLE_INTERNAL_H
#include <cmath>
#include <cstdint>
#include <limits>
#include <vector>

#include "oracle.h"

namespace orc {

constexpr double kMe = 0.51099895;          /* m_e c^2 [MeV] (SURVEY.md §8 header) */
constexpr double kRe = 2.8179403262e-13;    /* cm */
constexpr double kAlpha = 1.0 / 137.035999084;
constexpr double kNa = 6.02214076e23;
constexpr double kCB = 2.99792458;          /* p[MeV/c] = kCB * B[T] * R[cm] */
constexpr double kPi = 3.14159265358979323846;
constexpr int kNGrid = 2048;
constexpr double kTmin = 1.0e-3;            /* 1 keV: lowest tracked energy */
constexpr double kInf = std::numeric_limits<double>::infinity();

/* table indices inside one material block (M6) */
enum { T_G_COMPTON, T_G_PAIR, T_G_PHOTO, T_EM_BREM, T_EM_IONI, T_EM_DEDX, T_EM_RANGE,
       T_EP_BREM, T_EP_IONI, T_EP_ANNI, T_EP_DEDX, T_EP_RANGE, N_TAB };
/* scalar indices */
enum { S_X0, S_TCUT, S_KCUT, S_BK, S_NEL, S_VACUUM, S_Z, S_RHO, N_SCAL };

struct Volume {
  int solid;
  double dims[3];
  int material;
  int mother;
  int dbegin, dcount;
  double R[9];
  double t[3];
};

}  // namespace orc

struct orc_ctx {
  std::vector<orc::Volume> vol;
  int n_mat = 0;
  std::vector<double> tables;   /* [n_mat][12][2048] */
  std::vector<double> scalars;  /* [n_mat][8] */
  std::vector<int32_t> n_elem;  /* [n_mat]; empty = single elements only */
  std::vector<double> elem_bk;  /* [n_mat][4] */
  std::vector<double> pe_cum;   /* [n_mat][2048][4] */
  orc_field field{};
  std::vector<double> bz;
  orc_config cfg{};
  double u0 = 0, du = 0;        /* grid in ln T */
  /* recorder */
  uint32_t rec_mask = 0, rec_stride = 1;
  orc_track* rec_buf = nullptr;
  size_t rec_cap = 0, rec_n = 0;
  uint64_t rec_counter = 0;
};

namespace orc {

inline const double* table(const orc_ctx* c, int mat, int tab) {
  return c->tables.data() + (static_cast<size_t>(mat) * N_TAB + tab) * kNGrid;
}
inline double scalar(const orc_ctx* c, int mat, int s) { return c->scalars[static_cast<size_t>(mat) * N_SCAL + s]; }

/* sequential uniform stream of one (event, id, step) (R2-R3) */
struct Stream {
  uint32_t event, seed, step;
  uint64_t id;
  uint32_t next;
  double draw() { return orc_uniform(event, seed, id, step, next++); }
};

void to_local(const Volume& v, const double g[3], double l[3]);
void dir_to_local(const Volume& v, const double g[3], double l[3]);

}  // namespace orc
#endif
