/* adept.h -- C ABI of the B200-native EM-shower transport library (libadept_b200.so).
 *
 * The boundary follows the paper's problem statement: the library "takes particles ... as input and
 * gives back the energy depositions and any 'outgoing' particles", processes a buffered
 * batch and returns hits "in arrays transferred back from the device to the host at the
 * end of each event".  Entry-point names are those of BASELINE.json:north_star /
 * SURVEY.md §8(b).
 *
 * Conventions
 *  - Units: MeV, cm, tesla.  All physics state is IEEE double.
 *  - Every pointer argument is a HOST pointer unless its name starts with d_ (device pointer).
 *  - Inputs are caller-owned and copied during the call; outputs are caller-owned buffers.
 *  - The only device memory the library uses for transport is the caller's workspace (allocated by
 *    the caller, e.g. with PyTorch); the library owns nothing after adept_shutdown.
 *  - Every call returns an int status: ADEPT_OK or a negative error.  No call throws or aborts;
 *    adept_last_error() returns a static, thread-local description of the last failure.
 *  - `cuda_stream` arguments are cudaStream_t values passed as void* (NULL = the legacy default stream).
 *  - Species codes: 0 = e-, 1 = e+, 2 = gamma.
 */
#ifndef ADEPT_H
#define ADEPT_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
  ADEPT_OK = 0,
  ADEPT_EINVAL = -1,    /* bad argument (null pointer, index out of range, malformed geometry)      */
  ADEPT_ENOMEM = -2,    /* workspace too small / host allocation failed                            */
  ADEPT_EOVERFLOW = -3, /* a track queue of the slot overflowed: the slot's results are invalid and
                           the slot has been reset (empty, scoring zeroed), ready for reuse        */
  ADEPT_ECUDA = -4,     /* a CUDA runtime call failed                                              */
  ADEPT_ESTATE = -5     /* call not valid in this state (e.g. slot still holds live tracks)        */
};

enum { ADEPT_ELECTRON = 0, ADEPT_POSITRON = 1, ADEPT_GAMMA = 2 };
enum { ADEPT_BOX = 0, ADEPT_TUBE = 1 };
enum { ADEPT_FIELD_NONE = 0, ADEPT_FIELD_UNIFORM = 1, ADEPT_FIELD_MAP_RZ = 2 };
enum { ADEPT_NAV_LOOP = 0, ADEPT_NAV_BVH = 1,
       /* single-precision geometry: solids, transforms and BVH boxes in fp32; ray-cast validator only */
       ADEPT_NAV_LOOP_F32 = 2, ADEPT_NAV_BVH_F32 = 3 };

/* Outcome of one step. */
enum {
  ADEPT_OUT_BOUNDARY = 0, ADEPT_OUT_COMPTON = 1, ADEPT_OUT_PAIR = 2, ADEPT_OUT_PHOTO = 3,
  ADEPT_OUT_BREM = 4, ADEPT_OUT_IONI = 5, ADEPT_OUT_ANNI = 6, ADEPT_OUT_STOPPED = 7,
  ADEPT_OUT_TRUNCATED = 8, ADEPT_OUT_LOSS = 9, ADEPT_OUT_ESCAPED = 10, ADEPT_OUT_KILLED = 11,
  ADEPT_OUT_CLOSED = 12, ADEPT_N_OUTCOMES = 13
};

/* Geometry: a tree of placed solids, every logical volume placed once, so
 * the index into these arrays (the touchable id) is the whole navigation state.
 * Volume 0 is the world.  The daughters of a volume are contiguous, in index order, and lie fully
 * inside it; siblings are disjoint.  rot/trans are the GLOBAL transform of the touchable:
 * local = rot^T (global - trans), rot row-major with the local axes as columns. */
typedef struct {
  int32_t n_volumes;
  const int32_t* solid;          /* [n]    ADEPT_BOX | ADEPT_TUBE                                  */
  const double* dims;            /* [n][3] box: half lengths; tube: rmin, rmax, half length z      */
  const int32_t* material;       /* [n]    index into the material arrays                          */
  const int32_t* mother;         /* [n]    -1 for the world                                        */
  const int32_t* daughter_begin; /* [n]                                                            */
  const int32_t* daughter_count; /* [n]                                                            */
  const double* rot;             /* [n][9]                                                         */
  const double* trans;           /* [n][3]                                                         */
} adept_geometry;

/* Per-material scalars. */
typedef struct {
  double X0;      /* radiation length [cm]                       */
  double e_cut;   /* T_c: e-/e+ production cut [MeV]             */
  double g_cut;   /* k_c: gamma production cut [MeV]             */
  double B_K;     /* K-shell binding energy [MeV]                */
  double n_el;    /* electron density [1/cm^3]                   */
  double vacuum;  /* 1.0 for vacuum (no physics), else 0.0       */
  double Z;
  double rho;
} adept_material;

/* The 12 tables of every material on the 2048-point grid uniform in ln T from 1 keV to 100 TeV
 * (SURVEY.md §8(c) M6): gamma {Compton, pair, photoelectric}; e- {brem, Moller, dE/dx, range};
 * e+ {brem, Bhabha, annihilation, dE/dx, range}.  Macroscopic cross sections in 1/cm. */
#define ADEPT_N_TABLES 12
#define ADEPT_N_GRID 2048
#define ADEPT_MAX_ELEMENTS 4
typedef struct {
  const double* data; /* [n_materials][12][2048] */
  /* Compound materials ("element selector"; DESIGN.md §3 C1-C5).  The tables above
   * hold the sums over the elements of each material.  Where the final state depends on the target element -- the
   * K-shell binding energy of a photoelectric absorption -- the element is sampled with uniform U6 of the step
   * against the cumulative shares below, interpolated in ln T like every table.  All three NULL: every material
   * is a single element (the binding energy is adept_material::B_K, nothing is drawn). */
  const int32_t* n_elem; /* [n_materials]          elements of the material, 1..ADEPT_MAX_ELEMENTS              */
  const double* elem_bk; /* [n_materials][4]       K-shell binding energy of each element [MeV]                 */
  const double* pe_cum;  /* [n_materials][2048][4] share of elements 0..j in Sigma_photo at each grid node      */
} adept_tables;

/* Magnetic field.  MAP_RZ: B = (0, 0, bz(r, z)), bilinear, clamped outside. */
typedef struct {
  int32_t kind;
  double B[3];       /* ADEPT_FIELD_UNIFORM */
  int32_t nr, nz;    /* ADEPT_FIELD_MAP_RZ  */
  double r0, z0, dr, dz;
  const double* bz;  /* [nz][nr] */
} adept_field;

typedef struct {
  double delta_chord;      /* max sagitta of a chord [cm], default 1e-3               */
  double eps_push;         /* boundary push [cm], default 1e-7                       */
  double alpha_R, rho_R;   /* continuous-loss step function, 0.2 and 0.1 cm          */
  int32_t chord_budget;    /* chords per step before truncation, 16     */
  uint32_t seed;           /* Philox key word 1                                      */
  uint32_t max_steps;      /* a track is killed after this many steps, 1e6           */
  int32_t navigator;       /* ADEPT_NAV_LOOP | ADEPT_NAV_BVH                                        */
  int32_t n_event_slots;   /* independent transport contexts (config 5)                */
  int32_t sync_interval;   /* population-step iterations launched between host checks, default 16    */
  uint64_t track_capacity; /* per slot, per species: entries of each of the two track buffers       */
  uint64_t leak_capacity;  /* per slot: tracks that left the world kept for adept_read_leaked       */
  uint64_t stage_capacity; /* per slot, per interaction queue: tracks staged for their discrete
                              interaction in one population step (0 = track_capacity)               */
  int32_t time_kernels;    /* 1: bracket every step-kernel launch with CUDA events (adept_get_kernel_times);
                              the events cost ~5 us of stream time per launch, so timed passes are slower */
  uint64_t inject_chunk;   /* staggered injection: 0 (default) = every enqueued primary
                              enters the first population step; n > 0 = enqueued primaries wait in a per-slot
                              pending store and at most n of them enter each population step, in enqueue order,
                              so that showers overlap at a lower peak population                            */
  uint64_t pending_capacity; /* per slot: primaries the pending store holds (0 = track_capacity); used only
                              when inject_chunk > 0                                                          */
  int32_t concurrent_species; /* 1 (default): gamma and charged move kernels on two streams;
                              0: all kernels of a slot on the caller's stream, one after the other          */
  int32_t steps_per_launch; /* steps a lane may take of its own track inside one move-kernel launch while the outcome
                              keeps the track in its species buffer (boundary, continuous-loss limit, chord budget):
                              0 (default) = chosen per launch from the population (1 for a full GPU, more for the
                              tails), n > 0 = at most n.  Random numbers are keyed by (event, track, step), so the
                              showers are identical whatever the value                                          */
  int32_t use_graphs;      /* 1 (default): a host round of sync_interval population steps is replayed as one CUDA
                              graph per slot (needs an even sync_interval; off while per-launch timing is on or
                              primaries wait for injection); 0: every kernel is launched individually           */
  int32_t low_occupancy_below; /* BVH geometry in a field only: the e+- move kernel exists in two builds of the same
                              source, for three resident blocks per SM and for two (255 registers, no spills: faster
                              where a launch lasts as long as its longest chain of chords and traversals).  A host round
                              whose population, as the host last saw it, is below this number of tracks launches the
                              second: 0 (default) = 262 144, < 0 = never.  The two builds agree to rounding, not bit
                              for bit (the compiler contracts them differently)                                   */
} adept_config;

typedef struct {
  double pos[3];
  double dir[3];
  double ekin;
  uint64_t id;
  uint32_t event;
  uint32_t step;
  uint32_t volume;
  int32_t species;
} adept_track;

typedef struct {
  adept_track post; /* state after the step (meaningful if alive)                        */
  int32_t alive;
  int32_t outcome;  /* ADEPT_OUT_*                                                       */
  int32_t n_sec;    /* secondaries created (0..2)                                        */
  int32_t chords;
  double s;         /* path length of the step                                           */
  double edep_dep;  /* continuous loss scored in the pre-step volume                     */
  double edep_cut;  /* below-cut / binding / stopped energy scored in the same volume    */
  double escaped;
  double killed;
} adept_step_result;

typedef struct {
  double deposited, below_cut, escaped, killed, primary;
} adept_ledger;

typedef struct {
  uint64_t steps[3];                    /* per species                                    */
  uint64_t outcomes[ADEPT_N_OUTCOMES];
  uint64_t secondaries[3];              /* created, per species                           */
  uint64_t chords;
  uint64_t iterations;                  /* population steps executed                      */
  uint64_t peak_population;             /* max live tracks over iterations                */
  uint64_t launches;                    /* kernels launched by adept_transport            */
} adept_stats;

typedef struct adept_ctx adept_ctx;

const char* adept_last_error(void);

/* Fills *cfg with the defaults listed above (n_event_slots 1, BVH navigator, capacity 1<<20). */
void adept_default_config(adept_config* cfg);

/* Bytes of device workspace adept_init needs for this configuration (0 on invalid input). */
size_t adept_workspace_bytes(const adept_config*, const adept_geometry*, int n_materials, const adept_field*);

/* Builds the device image (volumes, per-volume BVHs, interleaved table slices, field map)
 * inside d_workspace and returns a context.  ADEPT_EINVAL on malformed geometry, ADEPT_ENOMEM if
 * workspace_bytes < adept_workspace_bytes(...). */
int adept_init(adept_ctx** out, const adept_geometry*, const adept_material* mats, int n_mats,
               const adept_tables*, const adept_field*, const adept_config*, void* d_workspace,
               size_t workspace_bytes);

/* Appends n primaries of one event to a slot; track ids are 0..n-1 (call once per event).  Primaries
 * are placed at Locate(pos + eps_push dir); one outside the world is ADEPT_EINVAL.
 * pos3/dir3 are [n][3]. Synchronous with respect to the host buffers. */
int adept_enqueue_primaries(adept_ctx*, int event_slot, uint32_t event_id, int n, const int8_t* species,
                            const double* pos3, const double* dir3, const double* ekin);

/* Same, for primaries of many events in one call: event_ids[n], track_ids[n]. */
int adept_enqueue_batch(adept_ctx*, int event_slot, int n, const uint32_t* event_ids, const uint64_t* track_ids,
                        const int8_t* species, const double* pos3, const double* dir3, const double* ekin);

/* Steps the slot's whole population until its queues are empty.  Kernels run on
 * cuda_stream (plus library-owned helper streams ordered after it); returns when the slot is empty.
 * ADEPT_EOVERFLOW: a queue of the slot was too small (track_capacity / stage_capacity); the pass is
 * abandoned and the slot reset as by adept_reset_slot, so the caller may enqueue a smaller batch. */
int adept_transport(adept_ctx*, int event_slot, void* cuda_stream);

/* Transports several slots concurrently, slot i on streams[i] (config 5).  A slot listed
 * twice, or one already in transport, is ADEPT_EINVAL.  On any error no listed slot stays marked live. */
int adept_transport_many(adept_ctx*, int n_slots, const int* event_slots, void* const* cuda_streams);

/* Empties a slot: drops its tracks, pending primaries and leaked tracks and zeroes its scoring arrays,
 * ledger and iteration trace (the cumulative counters of adept_get_stats stay).  Synchronous. */
int adept_reset_slot(adept_ctx*, int event_slot);

/* Copies the slot's per-volume energy deposit (n_volumes doubles, indexed by touchable id) and its
 * ledger to the host, then zeroes them on the device. */
int adept_read_scoring(adept_ctx*, int event_slot, double* edep_per_volume, size_t n_volumes,
                       adept_ledger* ledger, void* cuda_stream);

/* Tracks that left the world ("outgoing particles"): up to cap of them; *n = number
 * that leaked (may exceed cap).  Resets the slot's leak buffer. */
int adept_read_leaked(adept_ctx*, int event_slot, adept_track* out, size_t cap, size_t* n);

int adept_get_stats(adept_ctx*, int event_slot, adept_stats* out);

/* With config.time_kernels: device time [ms] and launch count of the gamma move kernel [0], the
 * charged move kernel [1] and the interaction kernel [2] of this slot, accumulated since the last call
 * (CUDA events recorded on the stream the kernels are launched on).  While timing is on, the kernels of
 * a population step run one after the other on the caller's stream, so every event pair brackets one
 * kernel alone; the events themselves cost ~5 us of stream time per launch.  adept_set_kernel_timing
 * switches the events off (0) and on (1) between passes of a context created with time_kernels = 1, so
 * that a benchmark can time untimed passes and instrumented passes of the same context.
 * A context without a field and without a BVH volume (and with config.concurrent_species != 0) runs the gamma and
 * the charged move kernel as the blocks of ONE launch; [0] is then that merged kernel and [1] stays empty (0 ms, 0
 * launches): create the context with concurrent_species = 0 to time the two kernels by themselves. */
int adept_set_kernel_timing(adept_ctx*, int on);
#define ADEPT_N_TIMED_KERNELS 3
int adept_get_kernel_times(adept_ctx*, int event_slot, double ms[ADEPT_N_TIMED_KERNELS],
                           uint64_t launches[ADEPT_N_TIMED_KERNELS]);

/* Trace of the slot's population steps since the previous call (at most ADEPT_TRACE_CAPACITY of them):
 * t_ns[i] = device %globaltimer [ns] when population step i finished, population[3 * i + s] = tracks of
 * species s (0 e-, 1 e+, 2 gamma) that entered it.  Written by the kernel that ends a population step, so
 * recording costs no stream time.  *n = steps copied (<= cap; population holds 3 * cap entries).  The
 * slot must not be in transport. */
#define ADEPT_TRACE_CAPACITY 4096
int adept_get_iteration_trace(adept_ctx*, int event_slot, uint64_t* t_ns, uint32_t* population, size_t cap, size_t* n);

/* Ray-cast validator of the navigator (PAPER.md:49 and Fig. 1): ray i from pos3[i] along the unit
 * vector dir3[i] is marched boundary by boundary -- distance to boundary, push, relocation: the calls of a photon
 * step -- until it leaves the world or has crossed max_crossings boundaries.  column[i] = sum of path length x
 * density [g/cm^2], crossings[i] = boundaries crossed (-1 if the ray starts outside the world).  Host arrays in
 * and out; *device_ms (may be NULL) = CUDA-event time of the kernel.  The navigator is chosen here.
 * ADEPT_NAV_LOOP_F32 / ADEPT_NAV_BVH_F32 march the same rays through the single-precision copy of the geometry
 * (all geometry types in fp32; validated by comparing the pictures): positions,
 * distances and the column density are fp32, the boundary push is 1e-3 cm (float spacing at 300 cm is 3e-5 cm). */
int adept_raycast_batch(adept_ctx*, int navigator, int n, const double* pos3, const double* dir3, int max_crossings,
                        double* column, int32_t* crossings, double* device_ms, void* cuda_stream);

/* adept_raycast_batch for callers that must not allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same kernel, the same arguments but device_ms (timing it would take two
 * events created per call), the same results bit for bit.  The device copies of the rays and of the results live
 * in one file-scope `static __device__` array of ADEPT_STATIC_MAX_RAYS x 60 B = 3.75 MiB instead of cudaMalloc'ed
 * buffers; every GPU that loads the library holds that array until the process exits.  The call makes no
 * cudaMalloc, cudaFree, event or stream creation, or other allocating runtime call: two memsets (the results
 * start at zero: the array keeps what the previous call left in it), two uploads, the kernel, two downloads and a
 * synchronisation of cuda_stream.  The array's device address is asked of the runtime once per device
 * (cudaGetSymbolAddress, with the context's device current), on that device's first call.
 * n > ADEPT_STATIC_MAX_RAYS: ADEPT_EINVAL, nothing is launched (split the batch, or call adept_raycast_batch).
 * All calls on a device share the one array, whatever their context or stream: calls that overlap on the GPU
 * (two host threads, or two contexts on two streams) race on it and return garbage; the caller serialises them.
 * Calls one after the other on one host thread are safe (each ends with cuda_stream synchronised). */
#define ADEPT_STATIC_MAX_RAYS 65536
int adept_raycast_batch_static(adept_ctx*, int navigator, int n, const double* pos3, const double* dir3, int max_crossings,
                               double* column, int32_t* crossings, void* cuda_stream);

/* ---- Hybrid-workflow boundary.  The host simulation hands over, one at
 * a time, the tracks that enter the GPU region; they are buffered on the host until `threshold` of them
 * trigger synchronous transport of the batch in `event_slot` on `cuda_stream`; adept_buffer_flush transports
 * what is left (the paper's Flush, called when the host's own stack is empty).  Deposits of all batches
 * accumulate per volume; tracks that left the world ("outgoing particles") are collected for the caller to
 * put back on its stack.  The buffer owns host memory only and must be destroyed before adept_shutdown.
 * adept_buffer_add / _flush return 1 when a batch was transported, 0 when not, < 0 on error.
 * adept_buffer_take copies and clears what has accumulated (any of edep / ledger / outgoing may be NULL;
 * outgoing needs room for *n_outgoing tracks: ask adept_buffer_pending first). */
typedef struct adept_buffer adept_buffer;
int adept_buffer_create(adept_buffer** out, adept_ctx*, int event_slot, size_t threshold, void* cuda_stream);
int adept_buffer_add(adept_buffer*, uint32_t event_id, uint64_t track_id, int species, const double pos[3],
                     const double dir[3], double ekin);
int adept_buffer_flush(adept_buffer*);
int adept_buffer_pending(const adept_buffer*, size_t* n_buffered, size_t* n_outgoing, uint64_t* n_batches);
int adept_buffer_take(adept_buffer*, double* edep_per_volume, size_t n_volumes, adept_ledger* ledger,
                      adept_track* outgoing, size_t cap, size_t* n_outgoing);
int adept_buffer_destroy(adept_buffer*);

/* Test hook for the kernels adept_transport runs.  Loads n tracks -- any species, step, id and volume, taken
 * as given (no Locate, steps not reset) -- into the EMPTY slot, runs EXACTLY ONE population step
 * with the very kernels and launch configuration of adept_transport (gamma move, charged move, interaction;
 * one step per track whatever config.steps_per_launch says) and copies the tracks of the next population --
 * survivors and secondaries of all species, in no particular order -- to out[0 .. *n_out) (*n_out may exceed
 * out_cap; only out_cap are copied).  The slot is empty again afterwards; deposits, the ledger (primary = energy
 * carried by the n tracks), leaked tracks and the counters are read with the usual calls.  Allocates its
 * transfer buffers with cudaMalloc, outside the workspace (test hooks do; transport never does). */
int adept_step_population(adept_ctx*, int event_slot, int n, const adept_track* in, adept_track* out, size_t out_cap,
                          size_t* n_out, void* cuda_stream);

/* Test hook of the generic per-lane step (csrc/step.cuh: move and interaction chained in one lane, any species): exactly
 * one step for each of n tracks, results in input order; secondaries[2*i + k].  Transport does not run this form; it is
 * kept as a second, structurally different arm of the frozen-step parity tests (the first is adept_step_population). */
int adept_step_frozen(adept_ctx*, int n, const adept_track* in, adept_step_result* out,
                      adept_track* secondaries, void* cuda_stream);

/* Test hooks for navigation: distance to boundary and Locate for n rays/points,
 * with the navigator chosen here regardless of the configuration. */
int adept_distance_batch(adept_ctx*, int navigator, int n, const double* pos3, const double* dir3,
                         const uint32_t* volume, const double* s_max, double* out, void* cuda_stream);
int adept_locate_batch(adept_ctx*, int navigator, int n, const double* pos3, int64_t* out, void* cuda_stream);
/* Relocation as the move kernel does it after a boundary (the hinted neighbour beyond exit face face[i]
 * of box volume from[i] first -- face = 2 * axis + (direction > 0) in the volume's frame, -1 or a null
 * array = no hint -- else climb from from[i] until the point is inside, then descend): must equal
 * adept_locate_batch for every starting volume and every face, right or wrong. */
int adept_relocate_batch(adept_ctx*, int navigator, int n, const double* pos3, const uint32_t* from,
                         const int32_t* face, int64_t* out, void* cuda_stream);

int adept_shutdown(adept_ctx*);

#ifdef __cplusplus
}
#endif
#endif
