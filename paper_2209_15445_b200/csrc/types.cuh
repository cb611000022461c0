// Device-side data layout of the transport library.  sm_100a only.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/adept.h"

namespace adept {

constexpr double kMe = 0.51099895;   // m_e c^2 [MeV]
constexpr double kCB = 2.99792458;   // p[MeV/c] = kCB * B[T] * R[cm]
constexpr double kPi = 3.14159265358979323846;
constexpr double kTmin = 1.0e-3;     // 1 keV
constexpr int kNGrid = ADEPT_N_GRID;
constexpr unsigned kFull = 0xffffffffu;
constexpr uint32_t kDeadVolume = 0xffffffffu;
constexpr double kIsolationMargin = 4.0e-3;  // [cm] see DevVolume::isolated (twice the single-precision push of the ray-cast and its rounding)
constexpr float kPushF32 = 1.0e-3f;          // [cm] boundary push of the single-precision ray-cast (float spacing at 300 cm is 3e-5 cm)

#define ADEPT_INF (__longlong_as_double(0x7ff0000000000000LL))

// material scalar slots (adept_material as 8 doubles)
enum { S_X0, S_TCUT, S_KCUT, S_BK, S_NEL, S_VACUUM, S_Z, S_RHO, N_SCAL };

// Interleaved table slices (one node = one contiguous row, so a lookup touches 2 adjacent rows):
//   gamma    row = {Compton, pair, photo, pad}            32 B
//   electron row = {brem, Moller, dE/dx, range}           32 B
//   positron row = {brem, Bhabha, annihilation, dE/dx, range, pad, pad, pad} 64 B
constexpr int kRowG = 4, kRowEm = 4, kRowEp = 8;

// Hot part of a touchable (80 B); the 3x3 rotation lives in DevCtx::rot and is only read for rotated
// placements, so the 152 volumes of the calorimeter stay L1-resident (12 KB).
template <typename R>
struct __align__(16) VolT {
  R t[3];
  R dims[3];
  int32_t solid;
  int32_t material;
  int32_t dbegin;
  int32_t dcount;
  int32_t bvh;       // index into DevCtx::bvh, -1 = none (loop over daughters)
  int32_t identity;  // 1 if the rotation is the identity (transform reduces to a subtraction, bit-identical)
  int32_t mother;    // -1 for the world
  int32_t isolated;  // 1: a box with no sibling within kIsolationMargin (adept_init), see nav_relocate
};
using DevVolume = VolT<double>;

// Implicit complete 32-ary BVH over the daughters of one volume, in the world frame.
// Primitives are sorted along a Morton curve; node k of level L covers nodes [32k, 32k+32) of level L-1
// (level 0 covers primitives).  Boxes are stored SoA: lo.x, lo.y, lo.z, hi.x, hi.y, hi.z.
constexpr int kBvhMaxLevels = 5;
template <typename R>
struct BvhT {
  int32_t n_prims;
  int32_t n_levels;                  // number of node levels (>= 1)
  int32_t n_nodes[kBvhMaxLevels];    // nodes per level
  const R* prim_box;                 // [6][n_prims]
  const int32_t* prim_vol;           // [n_prims] touchable id
  const R* node_box[kBvhMaxLevels];  // [6][n_nodes[L]]
  // per-daughter neighbour lists (geom.cuh NavCache): for daughter d (index relative to the volume's first
  // daughter) the touchable ids of the siblings within nbr_reach of its solid, itself included
  const int32_t* nbr;                // [n_prims][kNbrCap]
  const int32_t* nbr_count;          // [n_prims] entries, -1 = the list did not fit
  double nbr_reach;                  // [cm], <= 0: no lists
};
using DevBvh = BvhT<double>;

// One species' track buffer, structure of arrays (76 B per track).
struct TrackSoA {
  double *x, *y, *z, *dx, *dy, *dz, *ekin;
  uint64_t* id;
  uint32_t *event, *step, *vol;
};

// Interaction staging queues (one per process and species, so a queue is species-uniform):
//   0 Compton, 1 pair, 2 photoelectric (gamma); 3 brems, 4 Moller (e-); 5 brems, 6 Bhabha, 7 annihilation (e+)
constexpr int kNumStage = 8;

// Every hot counter sits in its own 128 B line: appends to different queues never serialise on one
// L2 atomic unit (measured: with all counters in one line the append atomics were 24 % of the stall
// samples of the gamma move kernel, profiles/r1_summary.md).
struct alignas(128) PaddedCounter {
  uint32_t v;
  uint32_t pad[31];
};
struct SlotCounters {
  PaddedCounter count[2][3];        // [buffer parity][species] live entries
  PaddedCounter n_stage[kNumStage]; // staged tracks per interaction queue
  PaddedCounter n_leaked;
  PaddedCounter overflow;           // set when any queue overflowed
  PaddedCounter live;               // population after the last finished iteration
  PaddedCounter ticket;             // blocks of the interaction kernel that have finished (last one ends the step)
};

struct DevStats {
  unsigned long long steps[3];
  unsigned long long outcomes[ADEPT_N_OUTCOMES];
  unsigned long long secondaries[3];
  unsigned long long chords;
  unsigned long long iterations;
  unsigned long long peak_population;
};

struct DevSlot {
  TrackSoA buf[2][3];       // [parity][species]
  SlotCounters* counters;
  double* edep;             // [edep_replicas][edep_stride]: replicated per-volume deposits, folded by adept_read_scoring
  uint32_t edep_stride;     // doubles per replica (n_volumes rounded up to a 128 B multiple)
  uint32_t edep_mask;       // replicas - 1 (power of two)
  double* ledger;           // [5]: deposited, below_cut, escaped, killed, primary
  DevStats* stats;
  adept_track* leaked;      // [leak_capacity]
  adept_track* pending;         // [pending_capacity] located primaries waiting for injection (inject_chunk > 0)
  unsigned long long* trace_t;  // [ADEPT_TRACE_CAPACITY] %globaltimer at the end of each population step
  uint32_t* trace_pop;          // [ADEPT_TRACE_CAPACITY][3] e-, e+, gamma tracks that entered it
  uint32_t* trace_n;            // entries written since adept_get_iteration_trace
  TrackSoA stage[kNumStage];  // tracks waiting for their discrete interaction (stage_capacity entries each)
};

struct DevCtx {
  const DevVolume* vol;
  const double* rot;        // [n_vol][9]
  const int32_t* nbr;       // [n_vol][6] relocation hints: volume beyond each box face, -1 = none (geom.cuh nav_relocate)
  int32_t n_vol;
  const DevBvh* bvh;
  // the same geometry in single precision (the ray-cast validator's ADEPT_NAV_*_F32 modes): boxes of
  // the BVH rounded outwards
  const VolT<float>* vol32;
  const float* rot32;
  const BvhT<float>* bvh32;
  int32_t navigator;
  const double* tab_g;      // [n_mat][2048][kRowG]
  const double* tab_em;     // [n_mat][2048][kRowEm]
  const double* tab_ep;     // [n_mat][2048][kRowEp]
  const double* scal;       // [n_mat][N_SCAL]
  const int32_t* rhint;     // [n_mat][2 (e-, e+)][kHintStride] inverse-range search hints (physics.cuh)
  const int32_t* n_elem;    // [n_mat] elements per material, nullptr = single elements only (physics.cuh photo_binding)
  const double* elem_bk;    // [n_mat][4] K-shell binding energy per element
  const double* pe_cum;     // [n_mat][2048][4] cumulative shares of the elements in the photoelectric cross section
  int32_t n_mat;
  int32_t field_kind;
  double B[3];
  double Bn, bhat[3];       // |B| and B / |B| of a uniform field (adept_init)
  int32_t nr, nz;
  double r0, z0, dr, dz, inv_dr, inv_dz, fr_max, fz_max;   // (fr_max = nr - 1, fz_max = nz - 1 as doubles)
  const double* bz;
  double u0, inv_du, du;
  double delta_chord, eps_push, alpha_R, rho_R;
  int32_t chord_budget;
  uint32_t seed, max_steps;
  int32_t steps_per_launch; // adept_config::steps_per_launch (0 = automatic, kernels.cuh inner_steps)
  int32_t sparse_waves;     // charged.cuh: waves of sparse tiles a BVH field kernel may take (1, or more when the slot has the GPU to itself)
  int32_t transit;          // 1: BVH volumes have per-daughter neighbour lists: a track that leaves a daughter into such a
                            // (vacuum) mother takes the step across the gap in the same launch, whatever the population
  uint32_t capacity;        // per species per buffer
  uint32_t stage_capacity;  // per interaction queue
  uint32_t leak_capacity;
};

// Register-resident track and step result.
struct Track {
  double x, y, z, dx, dy, dz, ekin;
  uint64_t id;
  uint32_t event, step, vol;
  int species;
};

struct Secondary {
  double dx, dy, dz, ekin;
  int species;     // -1 = none
  uint32_t child;  // child index (R3)
};

struct StepOut {
  Track post;
  int alive, outcome, chords;
  double s, edep_dep, edep_cut, escaped, killed;
  Secondary sec[2];
  int n_sec;
};

}  // namespace adept
