/* ORACLE -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, single-threaded CPU implementation of the per-step EM-shower transport loop of
 * arXiv 2209.15445 (AdePT), written from PAPER.md and the model definitions of SURVEY.md §8(c).
 * It shares no code with the CUDA path (paper_2209_15445_b200/csrc) and is imported only by
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
 *
 * Parity status of each function is stated in the header of the file that defines it; the
 * readings taken where the paper is silent are listed in DESIGN.md §3.
 *
 * Units: MeV, cm, tesla.  All floating point is IEEE double (tables: long double internally).
 */
#ifndef ORACLE_H
#define ORACLE_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { ORC_ELECTRON = 0, ORC_POSITRON = 1, ORC_GAMMA = 2 };
enum { ORC_BOX = 0, ORC_TUBE = 1 };
enum { ORC_FIELD_NONE = 0, ORC_FIELD_UNIFORM = 1, ORC_FIELD_MAP_RZ = 2 };

/* outcome of one step */
enum {
  ORC_OUT_BOUNDARY = 0,   /* reached a volume boundary, relocated                     */
  ORC_OUT_COMPTON = 1,
  ORC_OUT_PAIR = 2,
  ORC_OUT_PHOTO = 3,
  ORC_OUT_BREM = 4,
  ORC_OUT_IONI = 5,       /* Moller (e-) or Bhabha (e+)                                */
  ORC_OUT_ANNI = 6,       /* annihilation in flight                                    */
  ORC_OUT_STOPPED = 7,    /* T fell below 1 keV / range exhausted (e+: at-rest annih.) */
  ORC_OUT_TRUNCATED = 8,  /* chord budget exhausted (F4)                               */
  ORC_OUT_LOSS = 9,       /* continuous-loss limited step, track goes on               */
  ORC_OUT_ESCAPED = 10,   /* left the world                                            */
  ORC_OUT_KILLED = 11,    /* step cap (S4)                                             */
  ORC_OUT_CLOSED = 12     /* discrete process chosen but kinematically closed          */
};

typedef struct {
  int32_t n_vol;
  const int32_t* solid;          /* [n_vol] */
  const double* dims;            /* [n_vol][3] */
  const int32_t* material;       /* [n_vol] */
  const int32_t* mother;         /* [n_vol] */
  const int32_t* daughter_begin; /* [n_vol] */
  const int32_t* daughter_count; /* [n_vol] */
  const double* rot;             /* [n_vol][9] global, row-major, local = R^T (g - t) */
  const double* trans;           /* [n_vol][3] global */
} orc_geometry;

#define ORC_MAX_ELEMENTS 4
typedef struct {
  int32_t n_mat;
  const double* tables;  /* [n_mat][12][2048] */
  const double* scalars; /* [n_mat][8]: X0, T_c, k_c, B_K, n_el, vacuum flag, Z, rho */
  /* Compound materials ("element selector"; DESIGN.md §3 C1-C5).  All three NULL
     = every material is a single element.  The tables above already hold the sums over the elements. */
  const int32_t* n_elem; /* [n_mat] number of elements, 1..ORC_MAX_ELEMENTS (vacuum: 1)                         */
  const double* elem_bk; /* [n_mat][4] K-shell binding energy of each element [MeV]                            */
  const double* pe_cum;  /* [n_mat][2048][4] cumulative share of elements 0..j in Sigma_photo on the ln T grid */
} orc_materials;

typedef struct {
  int32_t kind;
  double B[3];
  int32_t nr, nz;
  double r0, z0, dr, dz;
  const double* bz; /* [nz][nr] */
} orc_field;

typedef struct {
  double delta_chord; /* F2, 1e-3 cm */
  double eps_push;    /* G5, 1e-7 cm */
  double alpha_R;     /* S2, 0.2     */
  double rho_R;       /* S2, 0.1 cm  */
  int32_t chord_budget; /* F4, 16   */
  uint32_t seed;        /* Philox key word 1 (R1) */
  uint32_t max_steps;   /* S4, 1e6  */
  int32_t reserved;
} orc_config;

typedef struct {
  double pos[3];
  double dir[3];
  double ekin;
  uint64_t id;
  uint32_t event;
  uint32_t step;
  uint32_t volume;
  int32_t species;
} orc_track;

typedef struct {
  orc_track post;   /* state after the step (valid if alive)             */
  int32_t alive;
  int32_t outcome;  /* ORC_OUT_*                                         */
  int32_t n_sec;    /* 0..2 secondaries written                          */
  int32_t chords;   /* chords used by field propagation                  */
  double s;         /* true path length of the step                      */
  double edep_dep;  /* continuous loss, scored in the pre-step volume    */
  double edep_cut;  /* below-cut / binding / stopped, same volume        */
  double escaped;
  double killed;
} orc_step_result;

typedef struct {
  double deposited, below_cut, escaped, killed, primary;
} orc_ledger;

typedef struct {
  uint64_t steps[3];        /* per species                               */
  uint64_t outcomes[13];    /* per ORC_OUT_*                             */
  uint64_t secondaries[3];  /* created, per species                      */
  uint64_t chords;
  uint64_t peak_stack;
  uint64_t iterations;      /* steps of the longest parent->child chain = population-stepping
                               iterations a GPU needs for the same primaries  */
} orc_stats;

typedef struct orc_ctx orc_ctx;

orc_ctx* orc_create(const orc_geometry*, const orc_materials*, const orc_field*, const orc_config*);
void orc_destroy(orc_ctx*);

/* R1-R2 */
void orc_philox(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
double orc_uniform(uint32_t event, uint32_t seed, uint64_t id, uint32_t step, uint32_t n);
uint64_t orc_child_id(uint32_t event, uint32_t seed, uint64_t id, uint32_t step, uint32_t child);

/* M7 */
double orc_lookup(const orc_ctx*, int material, int table, double ekin);
double orc_inverse_range(const orc_ctx*, int material, int range_table, double range);

/* G1-G5 (loop navigator) */
double orc_distance(const orc_ctx*, const double pos[3], const double dir[3], uint32_t volume, double s_max);
int64_t orc_locate(const orc_ctx*, const double pos[3]); /* -1 = outside the world */
int orc_inside(const orc_ctx*, const double pos[3], uint32_t volume);
double orc_solid_entry(int solid, const double dims[3], const double p[3], const double d[3]);
double orc_solid_exit(int solid, const double dims[3], const double p[3], const double d[3]);

/* F1-F4: propagate a charged track for s_phys; returns flag 0 physics / 1 boundary / 2 truncated */
int orc_propagate(const orc_ctx*, int charge, double ekin, double pos[3], double dir[3], uint32_t volume,
                  double s_phys, double* s_done, int* chords, double pushdir[3]);
void orc_helix(const double B[3], int charge, double pmom, double h, const double p[3], const double d[3],
               double p1[3], double d1[3]);
void orc_rk4(const orc_ctx*, int charge, double pmom, double h, const double p[3], const double d[3],
             double p1[3], double d1[3]);
void orc_field_at(const orc_ctx*, const double p[3], double B[3]);

/* P10 */
void orc_rotate(const double d[3], double cos_t, double sin_t, double phi, double out[3]);

/* P1-P8: run one interaction on `t` (uniforms U8.. of its (event,id,step) stream). */
void orc_interact(const orc_ctx*, int process, const orc_track* t, int material, orc_step_result* out,
                  orc_track sec[2]);

/* S1-S2: exactly one step */
void orc_step(const orc_ctx*, const orc_track* in, orc_step_result* out, orc_track sec[2]);

/* place primaries: volume = Locate(p0 + eps d0) (G5); returns -1 if outside */
int64_t orc_place(const orc_ctx*, const double pos[3], const double dir[3]);

/* full transport of n primaries (LIFO stack per primary); edep[n_vol] and ledger are accumulated */
int orc_run(orc_ctx*, size_t n, const orc_track* primaries, double* edep, orc_ledger* ledger,
            orc_stats* stats);

/* record pre-step states during orc_run: every `stride`-th step of the species in `mask`
   (bit s), up to cap entries; pass cap = 0 to switch off */
void orc_set_recorder(orc_ctx*, uint32_t mask, uint32_t stride, orc_track* buf, size_t cap);
size_t orc_recorded(const orc_ctx*);

/* M1-M6: the oracle's own table builder (long double). tables [12][2048], scalars [8]. */
void orc_build_material(double Z, double A, double rho, double* tables, double* scalars);
/* C1-C5: the same for a compound of n <= ORC_MAX_ELEMENTS elements with nu[i] atoms of (Z[i], A[i]) per formula
   unit; also fills elem_bk[4] and pe_cum[2048][4] (scalars: Z = n_el / n_at, B_K = that of element 0). */
void orc_build_compound(int n, const double* Z, const double* A, const double* nu, double rho, double* tables,
                        double* scalars, double* elem_bk, double* pe_cum);
/* the individual closed forms behind the tables (P1-P8), for the pins */
double orc_sigma_compton(double k);               /* per electron [cm^2] */
double orc_pair_shape(double k);                  /* X0 * Sigma_pair     */
double orc_sigma_photo(double k, double Z);       /* per atom [cm^2]     */
double orc_brem_shape(double T, double kc);       /* X0 * Sigma_brem     */
double orc_srad_shape(double T, double kc);       /* X0 * S_rad [MeV]    */
double orc_sigma_moller(double T, double Tc);     /* per electron        */
double orc_sigma_bhabha(double T, double Tc);     /* per electron        */
double orc_sigma_annihilation(double T);          /* per electron        */
double orc_s_coll(double T, double Z, double A, double rho, double Tc, int positron); /* Tc<0: unrestricted */

#ifdef __cplusplus
}
#endif
#endif
