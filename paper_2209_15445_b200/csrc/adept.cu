// Host side of the C ABI (include/adept.h): workspace carving, device image (volumes, per-volume BVH,
// interleaved table slices, field map), primaries, the transport loop and readback.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <numeric>
#include <thread>
#include <vector>

#include "kernels.cuh"
#include "gamma.cuh"
#include "charged.cuh"

using namespace adept;

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}

#define ADEPT_ON_DEVICE(ctx)                                                         \
  DeviceGuard device_guard_((ctx)->device);                                          \
  if (!device_guard_.ok) return fail(ADEPT_ECUDA, "cannot make device %d current", (ctx)->device)

#define CUDA_TRY(expr)                                                                         \
  do {                                                                                         \
    cudaError_t e_ = (expr);                                                                   \
    if (e_ != cudaSuccess) return fail(ADEPT_ECUDA, "%s: %s", #expr, cudaGetErrorString(e_));  \
  } while (0)

// Makes the context's device current for the duration of an ABI call and restores the caller's.
struct DeviceGuard {
  int prev = -1;
  bool ok = true;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
    if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
    if (prev == dev) prev = -1;
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// Device scratch of the test hooks (they allocate outside the caller's workspace; transport never does):
// freed on every exit path.
template <typename T>
struct DevBuf {
  T* p = nullptr;
  ~DevBuf() { if (p) cudaFree(p); }
  cudaError_t alloc(size_t n) { return cudaMalloc(&p, std::max<size_t>(n, 1) * sizeof(T)); }
  operator T*() const { return p; }
};

constexpr int kBvhMinDaughters = 65;  // below this a per-lane loop over the daughters is cheaper

// Bump allocator over the caller's workspace; with base == nullptr it only measures.
struct Carver {
  char* base;
  size_t off = 0;
  explicit Carver(void* b) : base(static_cast<char*>(b)) {}
  template <typename T>
  T* take(size_t n) {
    off = (off + 255) & ~static_cast<size_t>(255);
    T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
    off += n * sizeof(T);
    return p;
  }
};

struct HostBvh {
  int volume;
  std::vector<int32_t> prim_vol;
  std::vector<double> prim_box;                // [6][n]
  std::vector<std::vector<double>> node_box;   // per level [6][n_nodes]
  std::vector<int> n_nodes;
  std::vector<int32_t> nbr, nbr_count;         // [n][kNbrCap], [n]: per-daughter neighbour lists (geom.cuh NavCache)
  double nbr_reach = 0.0;
};

// World-frame AABB of a placed solid, padded so that rounding can never make it miss a true hit.
void world_aabb(const adept_geometry* g, int v, double lo[3], double hi[3]) {
  const double* R = g->rot + 9 * v;
  const double* t = g->trans + 3 * v;
  const double* d = g->dims + 3 * v;
  const double h[3] = {g->solid[v] == ADEPT_BOX ? d[0] : d[1], g->solid[v] == ADEPT_BOX ? d[1] : d[1], d[2]};
  for (int i = 0; i < 3; ++i) {
    const double e = std::fabs(R[3 * i + 0]) * h[0] + std::fabs(R[3 * i + 1]) * h[1] + std::fabs(R[3 * i + 2]) * h[2];
    const double pad = 1e-9 + 1e-12 * (std::fabs(t[i]) + e);
    lo[i] = t[i] - e - pad;
    hi[i] = t[i] + e + pad;
  }
}

// True if the placed boxes a and b are farther apart than `margin` (separating-axis test on the 15 axes of
// two oriented boxes; conservative: false when in doubt).  Columns of R are the local axes in the world frame.
bool boxes_apart(const adept_geometry* g, int a, int b, double margin) {
  const double *Ra = g->rot + 9 * a, *Rb = g->rot + 9 * b, *ha = g->dims + 3 * a, *hb = g->dims + 3 * b;
  const double T[3] = {g->trans[3 * b] - g->trans[3 * a], g->trans[3 * b + 1] - g->trans[3 * a + 1], g->trans[3 * b + 2] - g->trans[3 * a + 2]};
  double A[3][3], B[3][3];
  for (int j = 0; j < 3; ++j) for (int i = 0; i < 3; ++i) { A[j][i] = Ra[3 * i + j]; B[j][i] = Rb[3 * i + j]; }
  auto apart_on = [&](const double L[3]) {
    const double n = std::sqrt(L[0] * L[0] + L[1] * L[1] + L[2] * L[2]);
    if (n < 1e-9) return false;
    double ra = 0.0, rb = 0.0;
    for (int j = 0; j < 3; ++j) {
      ra += ha[j] * std::fabs(A[j][0] * L[0] + A[j][1] * L[1] + A[j][2] * L[2]);
      rb += hb[j] * std::fabs(B[j][0] * L[0] + B[j][1] * L[1] + B[j][2] * L[2]);
    }
    return std::fabs(T[0] * L[0] + T[1] * L[1] + T[2] * L[2]) > ra + rb + (margin + 1e-9) * n;
  };
  for (int j = 0; j < 3; ++j) if (apart_on(A[j]) || apart_on(B[j])) return true;
  for (int j = 0; j < 3; ++j)
    for (int k = 0; k < 3; ++k) {
      const double L[3] = {A[j][1] * B[k][2] - A[j][2] * B[k][1], A[j][2] * B[k][0] - A[j][0] * B[k][2], A[j][0] * B[k][1] - A[j][1] * B[k][0]};
      if (apart_on(L)) return true;
    }
  return false;
}

// DevVolume::isolated for the daughters of volume m: a box daughter is isolated when every sibling is
// farther than `margin` from it.  Sweep along the axis on which the daughters spread most; pairs whose
// padded world boxes overlap are decided by boxes_apart (a tube sibling counts as near).
void mark_isolated(const adept_geometry* g, int m, double margin, std::vector<int32_t>& isolated) {
  const int b0 = g->daughter_begin[m], n = g->daughter_count[m];
  std::vector<double> lo(3 * static_cast<size_t>(n)), hi(3 * static_cast<size_t>(n));
  double span[3] = {0, 0, 0}, mn[3] = {1e300, 1e300, 1e300}, mx[3] = {-1e300, -1e300, -1e300};
  for (int k = 0; k < n; ++k) {
    world_aabb(g, b0 + k, &lo[3 * k], &hi[3 * k]);
    for (int i = 0; i < 3; ++i) { mn[i] = std::min(mn[i], lo[3 * k + i]); mx[i] = std::max(mx[i], hi[3 * k + i]); }
    isolated[b0 + k] = g->solid[b0 + k] == ADEPT_BOX ? 1 : 0;
  }
  for (int i = 0; i < 3; ++i) span[i] = mx[i] - mn[i];
  const int ax = span[0] >= span[1] && span[0] >= span[2] ? 0 : (span[1] >= span[2] ? 1 : 2);
  const int a1 = (ax + 1) % 3, a2 = (ax + 2) % 3;
  std::vector<int> order(n);
  std::iota(order.begin(), order.end(), 0);
  std::sort(order.begin(), order.end(), [&](int p, int q) { return lo[3 * p + ax] < lo[3 * q + ax]; });
  for (int ii = 0; ii < n; ++ii) {
    const int p = order[ii];
    for (int jj = ii + 1; jj < n; ++jj) {
      const int q = order[jj];
      if (lo[3 * q + ax] > hi[3 * p + ax] + margin) break;
      if (lo[3 * q + a1] > hi[3 * p + a1] + margin || lo[3 * p + a1] > hi[3 * q + a1] + margin) continue;
      if (lo[3 * q + a2] > hi[3 * p + a2] + margin || lo[3 * p + a2] > hi[3 * q + a2] + margin) continue;
      if (!isolated[b0 + p] && !isolated[b0 + q]) continue;
      const bool both_boxes = g->solid[b0 + p] == ADEPT_BOX && g->solid[b0 + q] == ADEPT_BOX;
      if (both_boxes && boxes_apart(g, b0 + p, b0 + q, margin)) continue;
      isolated[b0 + p] = 0; isolated[b0 + q] = 0;
    }
  }
}

// Per-daughter neighbour lists of volume m (geom.cuh NavCache): for daughter k the siblings that come within `reach`
// of its solid, itself first.  Conservative: a pair is left out only when the separating-axis test proves two boxes
// farther apart than `reach`, or the padded world boxes of any two solids are.  Returns the share of daughters
// whose list fits kNbrCap (the others get count -1).
double neighbour_lists(const adept_geometry* g, int m, double reach, std::vector<int32_t>& nbr, std::vector<int32_t>& count) {
  const int b0 = g->daughter_begin[m], n = g->daughter_count[m];
  std::vector<double> lo(3 * static_cast<size_t>(n)), hi(3 * static_cast<size_t>(n));
  double mn[3] = {1e300, 1e300, 1e300}, mx[3] = {-1e300, -1e300, -1e300};
  for (int k = 0; k < n; ++k) {
    world_aabb(g, b0 + k, &lo[3 * k], &hi[3 * k]);
    for (int i = 0; i < 3; ++i) { mn[i] = std::min(mn[i], lo[3 * k + i]); mx[i] = std::max(mx[i], hi[3 * k + i]); }
  }
  const int ax = (mx[0] - mn[0] >= mx[1] - mn[1] && mx[0] - mn[0] >= mx[2] - mn[2]) ? 0 : (mx[1] - mn[1] >= mx[2] - mn[2] ? 1 : 2);
  const int a1 = (ax + 1) % 3, a2 = (ax + 2) % 3;
  std::vector<int> order(n);
  std::iota(order.begin(), order.end(), 0);
  std::sort(order.begin(), order.end(), [&](int p, int q) { return lo[3 * p + ax] < lo[3 * q + ax]; });
  std::vector<std::vector<int32_t>> lists(n);
  for (int k = 0; k < n; ++k) lists[k].push_back(b0 + k);
  for (int ii = 0; ii < n; ++ii) {
    const int p = order[ii];
    for (int jj = ii + 1; jj < n; ++jj) {
      const int q = order[jj];
      if (lo[3 * q + ax] > hi[3 * p + ax] + reach) break;
      if (lo[3 * q + a1] > hi[3 * p + a1] + reach || lo[3 * p + a1] > hi[3 * q + a1] + reach) continue;
      if (lo[3 * q + a2] > hi[3 * p + a2] + reach || lo[3 * p + a2] > hi[3 * q + a2] + reach) continue;
      const bool both_boxes = g->solid[b0 + p] == ADEPT_BOX && g->solid[b0 + q] == ADEPT_BOX;
      if (both_boxes && boxes_apart(g, b0 + p, b0 + q, reach)) continue;
      lists[p].push_back(b0 + q);
      lists[q].push_back(b0 + p);
    }
  }
  nbr.assign(static_cast<size_t>(n) * kNbrCap, -1);
  count.assign(n, -1);
  int fit = 0;
  for (int k = 0; k < n; ++k) {
    if (static_cast<int>(lists[k].size()) > kNbrCap) continue;
    std::sort(lists[k].begin() + 1, lists[k].end());
    std::copy(lists[k].begin(), lists[k].end(), nbr.begin() + static_cast<size_t>(k) * kNbrCap);
    count[k] = static_cast<int32_t>(lists[k].size());
    ++fit;
  }
  return n ? static_cast<double>(fit) / n : 0.0;
}

HostBvh build_bvh(const adept_geometry* g, int v) {
  HostBvh b;
  b.volume = v;
  const int n = g->daughter_count[v], first = g->daughter_begin[v];
  std::vector<double> lo(3 * n), hi(3 * n);
  for (int k = 0; k < n; ++k) world_aabb(g, first + k, &lo[3 * k], &hi[3 * k]);
  // Order of the primitives: recursive bisection of the centres along the longest axis of their bounding box,
  // the cut placed at a multiple of the largest power of 32 below the range, so that every aligned run of 32,
  // 1024, ... consecutive primitives -- the implicit nodes of the tree -- is a compact group.  (Sorting along a
  // Morton curve of the 3-D centres, as round 1 did, tears the thin shell of a barrel apart: a point in a gap
  // between crystals lay in 6.1 leaf boxes, with this order in 2.4.)
  std::vector<int> order(n);
  std::iota(order.begin(), order.end(), 0);
  std::vector<double> cen(3 * static_cast<size_t>(n));
  for (int k = 0; k < n; ++k)
    for (int i = 0; i < 3; ++i) cen[3 * k + i] = 0.5 * (lo[3 * k + i] + hi[3 * k + i]);
  struct Range { int begin, end; };
  std::vector<Range> todo{{0, n}};
  while (!todo.empty()) {
    const Range r = todo.back();
    todo.pop_back();
    const int m = r.end - r.begin;
    if (m <= 32) continue;
    int block = 32;
    while (static_cast<long long>(block) * 32 < m) block *= 32;
    const int n_blocks = (m + block - 1) / block;
    const int left = (n_blocks + 1) / 2 * block;            // left half in whole blocks
    double mn[3] = {1e300, 1e300, 1e300}, mx[3] = {-1e300, -1e300, -1e300};
    for (int k = r.begin; k < r.end; ++k)
      for (int i = 0; i < 3; ++i) { mn[i] = std::min(mn[i], cen[3 * order[k] + i]); mx[i] = std::max(mx[i], cen[3 * order[k] + i]); }
    const int ax = (mx[0] - mn[0] >= mx[1] - mn[1] && mx[0] - mn[0] >= mx[2] - mn[2]) ? 0 : (mx[1] - mn[1] >= mx[2] - mn[2] ? 1 : 2);
    std::nth_element(order.begin() + r.begin, order.begin() + r.begin + left, order.begin() + r.end,
                     [&](int p, int q) { return cen[3 * p + ax] < cen[3 * q + ax] || (cen[3 * p + ax] == cen[3 * q + ax] && p < q); });
    todo.push_back({r.begin, r.begin + left});
    todo.push_back({r.begin + left, r.end});
  }
  b.prim_vol.resize(n);
  b.prim_box.resize(6 * static_cast<size_t>(n));
  for (int k = 0; k < n; ++k) {
    const int src = order[k];
    b.prim_vol[k] = first + src;
    for (int i = 0; i < 3; ++i) {
      b.prim_box[static_cast<size_t>(i) * n + k] = lo[3 * src + i];
      b.prim_box[static_cast<size_t>(3 + i) * n + k] = hi[3 * src + i];
    }
  }
  // levels: node k of level L = union of children [32k, 32k+32) of level L-1
  const std::vector<double>* child = &b.prim_box;
  int n_child = n;
  for (;;) {
    const int nn = (n_child + 31) / 32;
    std::vector<double> box(6 * static_cast<size_t>(nn));
    for (int k = 0; k < nn; ++k) {
      for (int i = 0; i < 3; ++i) {
        double l = 1e300, h = -1e300;
        for (int j = 32 * k; j < std::min(32 * k + 32, n_child); ++j) {
          l = std::min(l, (*child)[static_cast<size_t>(i) * n_child + j]);
          h = std::max(h, (*child)[static_cast<size_t>(3 + i) * n_child + j]);
        }
        box[static_cast<size_t>(i) * nn + k] = l;
        box[static_cast<size_t>(3 + i) * nn + k] = h;
      }
    }
    b.node_box.push_back(std::move(box));
    b.n_nodes.push_back(nn);
    if (nn <= 32) break;
    child = &b.node_box.back();
    n_child = nn;
  }
  // neighbour lists: the largest reach for which (nearly) every daughter's list fits
  for (double reach : {1.0, 0.5, 0.25, 0.125, 0.0625}) {
    if (neighbour_lists(g, v, reach, b.nbr, b.nbr_count) >= 0.95) { b.nbr_reach = reach; break; }
  }
  if (b.nbr_reach == 0.0) { b.nbr.assign(static_cast<size_t>(n) * kNbrCap, -1); b.nbr_count.assign(n, -1); }
  return b;
}

}  // namespace

struct SlotHost {
  DevSlot dev{};
  cudaStream_t helper = nullptr;     // charged-species kernel runs here, forked from the caller's stream
  cudaEvent_t fork = nullptr, join = nullptr;
  SlotCounters* pinned = nullptr;    // host mirror of the counters
  unsigned long long launches = 0;
  bool live = false;
  size_t n_pending = 0, n_injected = 0;   // staggered injection: primaries in the pending store / already injected
  size_t population = 0;                  // live tracks as last seen by the host (enqueue, end of a round)
  // CUDA graphs of one host round (sync_interval population steps) with the lean [0] and the multi-step [1]
  // move kernels, captured once on `cap` and replayed
  cudaStream_t cap = nullptr;
  cudaGraphExec_t gexec[6] = {};   // per kernel variant (round_variant)
  bool graph_failed[6] = {};
  // optional per-launch timing (config.time_kernels)
  std::vector<cudaEvent_t> tev;      // [sync_interval][kTimed kernels][start, stop]
  int tev_used = 0;
  double kernel_ms[ADEPT_N_TIMED_KERNELS] = {};
  unsigned long long kernel_launches[ADEPT_N_TIMED_KERNELS] = {};
};

struct adept_ctx {
  adept_config cfg{};
  DevCtx dev{};
  int device = 0;                    // CUDA device of the workspace: made current at every ABI entry
  int n_vol = 0, n_mat = 0;
  std::vector<SlotHost> slots;
  adept_track* d_stage = nullptr;    // staging area for primaries (inside the workspace)
  uint32_t* d_bad = nullptr;
  size_t stage_cap = 0;
  int grid_gamma = 0, grid_charged = 0, grid_charged_low = 0, grid_inter = 0;
  // move kernels specialised for this context's field kind and for geometries without BVH volumes; [1] = the
  // variants in which a lane takes several steps of its own track per launch (small populations); [2] = [1] with
  // the e+- kernel compiled for two resident blocks per SM (BVH geometry in a field only, else null: charged.cuh)
  using Kernel = void (*)(DevCtx, DevSlot, int);
  Kernel k_move_gamma[3] = {nullptr, nullptr, nullptr}, k_move_charged[3] = {nullptr, nullptr, nullptr};
  Kernel k_move_merged[3] = {nullptr, nullptr, nullptr};   // one launch for all three species (charged.cuh move_kernel), or null
  bool timing_on = false;            // per-launch CUDA events active (adept_set_kernel_timing)
};

namespace {
void destroy_ctx(adept_ctx* ctx) {
  for (SlotHost& sh : ctx->slots) {
    for (cudaGraphExec_t ge : sh.gexec) if (ge) cudaGraphExecDestroy(ge);
    if (sh.cap) cudaStreamDestroy(sh.cap);
    if (sh.helper) cudaStreamDestroy(sh.helper);
    if (sh.fork) cudaEventDestroy(sh.fork);
    if (sh.join) cudaEventDestroy(sh.join);
    if (sh.pinned) cudaFreeHost(sh.pinned);
    for (cudaEvent_t e : sh.tev) if (e) cudaEventDestroy(e);
  }
  delete ctx;
}
}  // namespace

extern "C" const char* adept_last_error(void) { return g_err; }

extern "C" void adept_default_config(adept_config* c) {
  if (!c) return;
  std::memset(c, 0, sizeof(*c));
  c->delta_chord = 1e-3; c->eps_push = 1e-7; c->alpha_R = 0.2; c->rho_R = 0.1;
  c->chord_budget = 16; c->seed = 1; c->max_steps = 1000000;
  c->navigator = ADEPT_NAV_BVH; c->n_event_slots = 1; c->sync_interval = 16;
  c->track_capacity = 1u << 20; c->leak_capacity = 1u << 16; c->stage_capacity = 0;
  c->concurrent_species = 1;
  c->steps_per_launch = 0;
  c->use_graphs = 1;
  c->low_occupancy_below = 0;
}

namespace {

int validate(const adept_config* cfg, const adept_geometry* g, int n_mats, const adept_field* f) {
  if (!cfg || !g || !f) return fail(ADEPT_EINVAL, "null argument");
  if (g->n_volumes < 1 || n_mats < 1) return fail(ADEPT_EINVAL, "empty geometry or material list");
  if (!g->solid || !g->dims || !g->material || !g->mother || !g->daughter_begin || !g->daughter_count || !g->rot || !g->trans)
    return fail(ADEPT_EINVAL, "null geometry array");
  if (cfg->n_event_slots < 1 || cfg->n_event_slots > 1024) return fail(ADEPT_EINVAL, "n_event_slots out of range");
  if (cfg->track_capacity < 32 || cfg->track_capacity > 0x3fffffffu) return fail(ADEPT_EINVAL, "track_capacity out of range");
  if (cfg->stage_capacity != 0 && (cfg->stage_capacity < 32 || cfg->stage_capacity > 0x3fffffffu)) return fail(ADEPT_EINVAL, "stage_capacity out of range");
  if (cfg->chord_budget < 1 || cfg->sync_interval < 1) return fail(ADEPT_EINVAL, "chord_budget / sync_interval must be >= 1");
  if (cfg->navigator != ADEPT_NAV_LOOP && cfg->navigator != ADEPT_NAV_BVH)
    return fail(ADEPT_EINVAL, "transport runs on the fp64 navigators (ADEPT_NAV_LOOP or ADEPT_NAV_BVH)");
  if (cfg->steps_per_launch < 0 || cfg->steps_per_launch > 4096) return fail(ADEPT_EINVAL, "steps_per_launch out of range");
  if (g->mother[0] != -1) return fail(ADEPT_EINVAL, "volume 0 must be the world");
  for (int v = 0; v < g->n_volumes; ++v) {
    if (g->solid[v] != ADEPT_BOX && g->solid[v] != ADEPT_TUBE) return fail(ADEPT_EINVAL, "volume %d: unknown solid", v);
    if (g->material[v] < 0 || g->material[v] >= n_mats) return fail(ADEPT_EINVAL, "volume %d: material out of range", v);
    const int b = g->daughter_begin[v], n = g->daughter_count[v];
    if (n < 0 || (n > 0 && (b <= v || b + n > g->n_volumes))) return fail(ADEPT_EINVAL, "volume %d: bad daughter range", v);
    for (int k = 0; k < n; ++k)
      if (g->mother[b + k] != v) return fail(ADEPT_EINVAL, "volume %d: daughter %d has another mother", v, b + k);
    if (v > 0 && (g->mother[v] < 0 || g->mother[v] >= v)) return fail(ADEPT_EINVAL, "volume %d: bad mother", v);
  }
  if (f->kind == ADEPT_FIELD_MAP_RZ && (f->nr < 2 || f->nz < 2 || !f->bz || !(f->dr > 0) || !(f->dz > 0)))
    return fail(ADEPT_EINVAL, "malformed field map");
  if (f->kind < ADEPT_FIELD_NONE || f->kind > ADEPT_FIELD_MAP_RZ) return fail(ADEPT_EINVAL, "unknown field kind");
  return ADEPT_OK;
}

struct Layout {
  DevVolume* vol; double* rot; int32_t* nbr; int32_t* rhint; DevBvh* bvh; double *tab_g, *tab_em, *tab_ep, *scal, *bz;
  int32_t* n_elem; double *elem_bk, *pe_cum;
  VolT<float>* vol32; float* rot32; BvhT<float>* bvh32; std::vector<float*> bvh32_prim_box; std::vector<std::vector<float*>> bvh32_node_box;
  std::vector<double*> bvh_prim_box; std::vector<int32_t*> bvh_prim_vol; std::vector<std::vector<double*>> bvh_node_box;
  std::vector<int32_t*> bvh_nbr, bvh_nbr_count;
  adept_track* stage; uint32_t* bad; size_t stage_cap;
  std::vector<DevSlot> slots;
};

// Carves (or, with base == nullptr, measures) the whole workspace.
size_t carve(void* base, const adept_config* cfg, const adept_geometry* g, int n_mats, const adept_field* f,
             const std::vector<HostBvh>* bvhs, Layout* out) {
  Carver cv(base);
  Layout L{};
  L.vol = cv.take<DevVolume>(g->n_volumes);
  L.rot = cv.take<double>(9 * static_cast<size_t>(g->n_volumes));
  L.nbr = cv.take<int32_t>(6 * static_cast<size_t>(g->n_volumes));
  std::vector<int> bvh_vols;
  for (int v = 0; v < g->n_volumes; ++v) if (g->daughter_count[v] >= kBvhMinDaughters) bvh_vols.push_back(v);
  L.bvh = cv.take<DevBvh>(std::max<size_t>(bvh_vols.size(), 1));
  L.vol32 = cv.take<VolT<float>>(g->n_volumes);
  L.rot32 = cv.take<float>(9 * static_cast<size_t>(g->n_volumes));
  L.bvh32 = cv.take<BvhT<float>>(std::max<size_t>(bvh_vols.size(), 1));
  for (size_t k = 0; k < bvh_vols.size(); ++k) {
    const int n = g->daughter_count[bvh_vols[k]];
    L.bvh_prim_box.push_back(cv.take<double>(6 * static_cast<size_t>(n)));
    L.bvh_prim_vol.push_back(cv.take<int32_t>(n));
    L.bvh_nbr.push_back(cv.take<int32_t>(static_cast<size_t>(n) * kNbrCap));
    L.bvh_nbr_count.push_back(cv.take<int32_t>(n));
    std::vector<double*> lv;
    std::vector<float*> lv32;
    L.bvh32_prim_box.push_back(cv.take<float>(6 * static_cast<size_t>(n)));
    int nn = n;
    do {
      nn = (nn + 31) / 32;
      lv.push_back(cv.take<double>(6 * static_cast<size_t>(nn)));
      lv32.push_back(cv.take<float>(6 * static_cast<size_t>(nn)));
    } while (nn > 32);
    L.bvh_node_box.push_back(lv);
    L.bvh32_node_box.push_back(lv32);
  }
  (void)bvhs;
  L.tab_g = cv.take<double>(static_cast<size_t>(n_mats) * kNGrid * kRowG);
  L.tab_em = cv.take<double>(static_cast<size_t>(n_mats) * kNGrid * kRowEm);
  L.tab_ep = cv.take<double>(static_cast<size_t>(n_mats) * kNGrid * kRowEp);
  L.scal = cv.take<double>(static_cast<size_t>(n_mats) * N_SCAL);
  L.rhint = cv.take<int32_t>(static_cast<size_t>(n_mats) * 2 * kHintStride);
  L.n_elem = cv.take<int32_t>(n_mats);
  L.elem_bk = cv.take<double>(static_cast<size_t>(n_mats) * ADEPT_MAX_ELEMENTS);
  L.pe_cum = cv.take<double>(static_cast<size_t>(n_mats) * kNGrid * ADEPT_MAX_ELEMENTS);
  L.bz = cv.take<double>(f->kind == ADEPT_FIELD_MAP_RZ ? static_cast<size_t>(f->nr) * f->nz : 1);
  L.stage_cap = std::min<size_t>(cfg->track_capacity, 1u << 20);
  L.stage = cv.take<adept_track>(L.stage_cap);
  L.bad = cv.take<uint32_t>(1);
  const size_t cap = cfg->track_capacity;
  const size_t scap = cfg->stage_capacity ? cfg->stage_capacity : cap;
  auto take_soa = [&cv](TrackSoA& b, size_t n) {
    n = (n + kBlock - 1) / kBlock * kBlock;   // whole tiles: the kernels fetch a buffer tile by tile (TMA bulk copies)
    b.x = cv.take<double>(n); b.y = cv.take<double>(n); b.z = cv.take<double>(n);
    b.dx = cv.take<double>(n); b.dy = cv.take<double>(n); b.dz = cv.take<double>(n);
    b.ekin = cv.take<double>(n); b.id = cv.take<uint64_t>(n);
    b.event = cv.take<uint32_t>(n); b.step = cv.take<uint32_t>(n); b.vol = cv.take<uint32_t>(n);
  };
  for (int s = 0; s < cfg->n_event_slots; ++s) {
    DevSlot d{};
    for (int p = 0; p < 2; ++p)
      for (int sp = 0; sp < 3; ++sp) take_soa(d.buf[p][sp], cap);
    for (int q = 0; q < kNumStage; ++q) take_soa(d.stage[q], scap);
    d.counters = cv.take<SlotCounters>(1);
    {  // replicated scoring arrays (kernels.cuh: score): up to 64 replicas within 2 MiB per slot
      const uint32_t stride = (static_cast<uint32_t>(g->n_volumes) + 15u) & ~15u;
      uint32_t rep = 64;
      while (rep > 1 && static_cast<size_t>(rep) * stride * sizeof(double) > (2u << 20)) rep >>= 1;
      d.edep = cv.take<double>(static_cast<size_t>(rep) * stride);
      d.edep_stride = stride;
      d.edep_mask = rep - 1;
    }
    d.ledger = cv.take<double>(8);
    d.stats = cv.take<DevStats>(1);
    d.leaked = cv.take<adept_track>(std::max<size_t>(cfg->leak_capacity, 1));
    d.pending = cfg->inject_chunk ? cv.take<adept_track>(cfg->pending_capacity ? cfg->pending_capacity : cap) : nullptr;
    d.trace_t = cv.take<unsigned long long>(ADEPT_TRACE_CAPACITY);
    d.trace_pop = cv.take<uint32_t>(3 * ADEPT_TRACE_CAPACITY);
    d.trace_n = cv.take<uint32_t>(1);
    L.slots.push_back(d);
  }
  if (out) *out = std::move(L);
  return (cv.off + 255) & ~static_cast<size_t>(255);
}

}  // namespace

extern "C" size_t adept_workspace_bytes(const adept_config* cfg, const adept_geometry* g, int n_mats, const adept_field* f) {
  if (validate(cfg, g, n_mats, f) != ADEPT_OK) return 0;
  return carve(nullptr, cfg, g, n_mats, f, nullptr, nullptr);
}

extern "C" int adept_init(adept_ctx** out, const adept_geometry* g, const adept_material* mats, int n_mats,
                          const adept_tables* tables, const adept_field* f, const adept_config* cfg, void* d_workspace,
                          size_t workspace_bytes) {
  if (!out || !mats || !tables || !tables->data || !d_workspace) return fail(ADEPT_EINVAL, "null argument");
  const int rc = validate(cfg, g, n_mats, f);
  if (rc != ADEPT_OK) return rc;
  Layout L;
  const size_t need = carve(d_workspace, cfg, g, n_mats, f, nullptr, &L);
  if (workspace_bytes < need) return fail(ADEPT_ENOMEM, "workspace has %zu bytes, %zu needed", workspace_bytes, need);
  // the context lives on the device that owns the workspace, whatever device is current in later calls
  cudaPointerAttributes attr{};
  if (cudaPointerGetAttributes(&attr, d_workspace) != cudaSuccess || attr.type != cudaMemoryTypeDevice) {
    cudaGetLastError();
    return fail(ADEPT_EINVAL, "d_workspace is not device memory");
  }
  DeviceGuard device_guard_(attr.device);
  if (!device_guard_.ok) return fail(ADEPT_ECUDA, "cannot make device %d current", attr.device);
  CUDA_TRY(cudaMemset(d_workspace, 0, need));

  // ---- volumes + BVHs
  const int nv = g->n_volumes;
  std::vector<DevVolume> hv(nv);
  std::vector<DevBvh> hb;
  std::vector<BvhT<float>> hb32;
  std::vector<int32_t> isolated(nv, 0);
  bool any_lists = false;
  for (int v = 0; v < nv; ++v)
    if (g->daughter_count[v] >= kBvhMinDaughters) {
      mark_isolated(g, v, kIsolationMargin, isolated);
      if (std::getenv("ADEPT_VERBOSE")) {
        const int b0 = g->daughter_begin[v], n = g->daughter_count[v];
        std::fprintf(stderr, "adept_init: volume %d: %d of %d daughters isolated (margin %g cm)\n", v,
                     static_cast<int>(std::count(isolated.begin() + b0, isolated.begin() + b0 + n, 1)), n, kIsolationMargin);
      }
    }
  for (int v = 0; v < nv; ++v) {
    DevVolume& d = hv[v];
    for (int k = 0; k < 3; ++k) { d.t[k] = g->trans[3 * v + k]; d.dims[k] = g->dims[3 * v + k]; }
    bool ident = true;
    for (int k = 0; k < 9; ++k) ident = ident && g->rot[9 * v + k] == ((k % 4 == 0) ? 1.0 : 0.0);
    d.solid = g->solid[v]; d.material = g->material[v];
    d.dbegin = g->daughter_begin[v]; d.dcount = g->daughter_count[v];
    d.identity = ident ? 1 : 0;
    d.mother = g->mother[v]; d.isolated = isolated[v];
    d.bvh = -1;
    if (d.dcount >= kBvhMinDaughters) {
      const HostBvh b = build_bvh(g, v);
      const size_t k = hb.size();
      if (static_cast<int>(b.n_nodes.size()) > kBvhMaxLevels) return fail(ADEPT_EINVAL, "volume %d: too many daughters", v);
      DevBvh db{};
      db.n_prims = d.dcount;
      db.n_levels = static_cast<int>(b.n_nodes.size());
      db.prim_box = L.bvh_prim_box[k];
      db.prim_vol = L.bvh_prim_vol[k];
      CUDA_TRY(cudaMemcpy(L.bvh_prim_box[k], b.prim_box.data(), b.prim_box.size() * sizeof(double), cudaMemcpyHostToDevice));
      CUDA_TRY(cudaMemcpy(L.bvh_prim_vol[k], b.prim_vol.data(), b.prim_vol.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
      db.nbr = L.bvh_nbr[k]; db.nbr_count = L.bvh_nbr_count[k]; db.nbr_reach = b.nbr_reach;
      CUDA_TRY(cudaMemcpy(L.bvh_nbr[k], b.nbr.data(), b.nbr.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
      CUDA_TRY(cudaMemcpy(L.bvh_nbr_count[k], b.nbr_count.data(), b.nbr_count.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
      if (std::getenv("ADEPT_VERBOSE"))
        std::fprintf(stderr, "adept_init: volume %d: neighbour lists with reach %g cm, %d of %d daughters listed\n", v, b.nbr_reach,
                     static_cast<int>(std::count_if(b.nbr_count.begin(), b.nbr_count.end(), [](int32_t x) { return x >= 0; })), d.dcount);
      if (b.nbr_reach > 0.0) any_lists = true;
      for (int l = 0; l < db.n_levels; ++l) {
        db.n_nodes[l] = b.n_nodes[l];
        db.node_box[l] = L.bvh_node_box[k][l];
        CUDA_TRY(cudaMemcpy(L.bvh_node_box[k][l], b.node_box[l].data(), b.node_box[l].size() * sizeof(double), cudaMemcpyHostToDevice));
      }
      // single-precision copy: boxes rounded outwards (a float box must not be smaller than the fp32 solid inside it)
      auto outward = [](const std::vector<double>& box) {
        std::vector<float> f(box.size());
        const size_t third = box.size() / 2;      // [lo.xyz | hi.xyz]
        for (size_t i = 0; i < box.size(); ++i) {
          const double pad = 1.0e-4 + 4.0e-7 * std::fabs(box[i]);
          f[i] = static_cast<float>(i < third ? box[i] - pad : box[i] + pad);
        }
        return f;
      };
      BvhT<float> db32{};
      db32.n_prims = db.n_prims; db32.n_levels = db.n_levels; db32.prim_vol = db.prim_vol;
      db32.nbr = db.nbr; db32.nbr_count = db.nbr_count; db32.nbr_reach = 0.0;
      db32.prim_box = L.bvh32_prim_box[k];
      {
        const std::vector<float> f = outward(b.prim_box);
        CUDA_TRY(cudaMemcpy(L.bvh32_prim_box[k], f.data(), f.size() * sizeof(float), cudaMemcpyHostToDevice));
      }
      for (int l = 0; l < db.n_levels; ++l) {
        db32.n_nodes[l] = b.n_nodes[l];
        db32.node_box[l] = L.bvh32_node_box[k][l];
        const std::vector<float> f = outward(b.node_box[l]);
        CUDA_TRY(cudaMemcpy(L.bvh32_node_box[k][l], f.data(), f.size() * sizeof(float), cudaMemcpyHostToDevice));
      }
      hb32.push_back(db32);
      d.bvh = static_cast<int>(k);
      hb.push_back(db);
    }
  }
  CUDA_TRY(cudaMemcpy(L.vol, hv.data(), hv.size() * sizeof(DevVolume), cudaMemcpyHostToDevice));
  CUDA_TRY(cudaMemcpy(L.rot, g->rot, 9 * static_cast<size_t>(nv) * sizeof(double), cudaMemcpyHostToDevice));
  if (!hb.empty()) CUDA_TRY(cudaMemcpy(L.bvh, hb.data(), hb.size() * sizeof(DevBvh), cudaMemcpyHostToDevice));
  {  // the geometry in single precision
    std::vector<VolT<float>> hv32(nv);
    std::vector<float> rot32(9 * static_cast<size_t>(nv));
    for (int v = 0; v < nv; ++v) {
      VolT<float>& f = hv32[v];
      for (int k = 0; k < 3; ++k) { f.t[k] = static_cast<float>(hv[v].t[k]); f.dims[k] = static_cast<float>(hv[v].dims[k]); }
      f.solid = hv[v].solid; f.material = hv[v].material; f.dbegin = hv[v].dbegin; f.dcount = hv[v].dcount;
      f.bvh = hv[v].bvh; f.identity = hv[v].identity; f.mother = hv[v].mother; f.isolated = hv[v].isolated;
      for (int k = 0; k < 9; ++k) rot32[9 * static_cast<size_t>(v) + k] = static_cast<float>(g->rot[9 * static_cast<size_t>(v) + k]);
    }
    CUDA_TRY(cudaMemcpy(L.vol32, hv32.data(), hv32.size() * sizeof(VolT<float>), cudaMemcpyHostToDevice));
    CUDA_TRY(cudaMemcpy(L.rot32, rot32.data(), rot32.size() * sizeof(float), cudaMemcpyHostToDevice));
    if (!hb32.empty()) CUDA_TRY(cudaMemcpy(L.bvh32, hb32.data(), hb32.size() * sizeof(BvhT<float>), cudaMemcpyHostToDevice));
  }

  // ---- interleaved table slices (one node = one row)
  {
    const size_t N = kNGrid;
    std::vector<double> tg(n_mats * N * kRowG, 0.0), te(n_mats * N * kRowEm, 0.0), tp(n_mats * N * kRowEp, 0.0);
    for (int m = 0; m < n_mats; ++m) {
      const double* src = tables->data + static_cast<size_t>(m) * ADEPT_N_TABLES * N;
      if (mats[m].vacuum != 0.0) continue;   // a vacuum has no physics: its rows stay zero (the gamma kernel relies on it)
      for (size_t i = 0; i < N; ++i) {
        for (int k = 0; k < 3; ++k) tg[(m * N + i) * kRowG + k] = src[k * N + i];
        for (int k = 0; k < 4; ++k) te[(m * N + i) * kRowEm + k] = src[(3 + k) * N + i];
        for (int k = 0; k < 5; ++k) tp[(m * N + i) * kRowEp + k] = src[(7 + k) * N + i];
      }
    }
    CUDA_TRY(cudaMemcpy(L.tab_g, tg.data(), tg.size() * sizeof(double), cudaMemcpyHostToDevice));
    CUDA_TRY(cudaMemcpy(L.tab_em, te.data(), te.size() * sizeof(double), cudaMemcpyHostToDevice));
    CUDA_TRY(cudaMemcpy(L.tab_ep, tp.data(), tp.size() * sizeof(double), cudaMemcpyHostToDevice));
    // inverse-range search hints (physics.cuh inverse_range): for key cell k, the largest node j whose
    // range R_j does not exceed the smallest r of the cell
    std::vector<int32_t> hint(static_cast<size_t>(n_mats) * 2 * kHintStride, 0);
    for (int m = 0; m < n_mats; ++m)
      for (int sp = 0; sp < 2; ++sp) {
        const double* R = tables->data + (static_cast<size_t>(m) * ADEPT_N_TABLES + (sp == 0 ? 6 : 11)) * N;
        int32_t* h = hint.data() + (static_cast<size_t>(m) * 2 + sp) * kHintStride;
        auto key = [](double r) { int64_t b; std::memcpy(&b, &r, 8); return static_cast<int32_t>(b >> 47); };
        const int32_t key0 = R[0] > 0.0 ? key(R[0]) : 0;
        h[0] = key0;
        size_t j = 0;
        for (int k = 0; k < kHintN; ++k) {
          const int64_t bits = static_cast<int64_t>(key0 + k) << 47;   // smallest double of the key cell
          double r_lo;
          std::memcpy(&r_lo, &bits, 8);
          while (j + 2 < N && R[j + 1] <= r_lo) ++j;
          h[1 + k] = static_cast<int32_t>(j);
        }
      }
    CUDA_TRY(cudaMemcpy(L.rhint, hint.data(), hint.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
    static_assert(sizeof(adept_material) == N_SCAL * sizeof(double), "adept_material layout");
    CUDA_TRY(cudaMemcpy(L.scal, mats, static_cast<size_t>(n_mats) * sizeof(adept_material), cudaMemcpyHostToDevice));
  }
  if (f->kind == ADEPT_FIELD_MAP_RZ)
    CUDA_TRY(cudaMemcpy(L.bz, f->bz, static_cast<size_t>(f->nr) * f->nz * sizeof(double), cudaMemcpyHostToDevice));
  // element selector of compound materials (all three arrays or none)
  const bool compounds = tables->n_elem && tables->elem_bk && tables->pe_cum;
  if (!compounds && (tables->n_elem || tables->elem_bk || tables->pe_cum))
    return fail(ADEPT_EINVAL, "adept_tables: n_elem, elem_bk and pe_cum must be given together");
  if (compounds) {
    for (int m = 0; m < n_mats; ++m)
      if (tables->n_elem[m] < 1 || tables->n_elem[m] > ADEPT_MAX_ELEMENTS) return fail(ADEPT_EINVAL, "material %d: n_elem out of range", m);
    CUDA_TRY(cudaMemcpy(L.n_elem, tables->n_elem, static_cast<size_t>(n_mats) * sizeof(int32_t), cudaMemcpyHostToDevice));
    CUDA_TRY(cudaMemcpy(L.elem_bk, tables->elem_bk, static_cast<size_t>(n_mats) * ADEPT_MAX_ELEMENTS * sizeof(double), cudaMemcpyHostToDevice));
    CUDA_TRY(cudaMemcpy(L.pe_cum, tables->pe_cum, static_cast<size_t>(n_mats) * kNGrid * ADEPT_MAX_ELEMENTS * sizeof(double), cudaMemcpyHostToDevice));
  }

  adept_ctx* ctx = new (std::nothrow) adept_ctx;
  if (!ctx) return fail(ADEPT_ENOMEM, "host allocation failed");
  struct Holder { adept_ctx* c; ~Holder() { if (c) destroy_ctx(c); } } holder{ctx};   // freed on every error return below
  ctx->cfg = *cfg;
  ctx->device = attr.device;
  ctx->n_vol = nv; ctx->n_mat = n_mats;
  DevCtx& d = ctx->dev;
  d.vol = L.vol; d.rot = L.rot; d.nbr = L.nbr; d.n_vol = nv; d.bvh = L.bvh; d.navigator = cfg->navigator;
  d.vol32 = L.vol32; d.rot32 = L.rot32; d.bvh32 = L.bvh32;
  d.tab_g = L.tab_g; d.tab_em = L.tab_em; d.tab_ep = L.tab_ep; d.scal = L.scal; d.rhint = L.rhint; d.n_mat = n_mats;
  d.n_elem = compounds ? L.n_elem : nullptr; d.elem_bk = L.elem_bk; d.pe_cum = L.pe_cum;
  d.field_kind = f->kind;
  for (int k = 0; k < 3; ++k) d.B[k] = f->B[k];
  d.Bn = std::sqrt(f->B[0] * f->B[0] + f->B[1] * f->B[1] + f->B[2] * f->B[2]);
  for (int k = 0; k < 3; ++k) d.bhat[k] = d.Bn > 0.0 ? f->B[k] / d.Bn : 0.0;
  d.nr = f->nr; d.nz = f->nz; d.r0 = f->r0; d.z0 = f->z0; d.dr = f->dr; d.dz = f->dz; d.bz = L.bz;
  d.inv_dr = f->dr > 0.0 ? 1.0 / f->dr : 0.0; d.inv_dz = f->dz > 0.0 ? 1.0 / f->dz : 0.0;
  d.fr_max = f->nr - 1; d.fz_max = f->nz - 1;
  d.u0 = std::log(1.0e-3);
  d.du = (std::log(1.0e8) - std::log(1.0e-3)) / (kNGrid - 1);
  d.inv_du = 1.0 / d.du;
  d.delta_chord = cfg->delta_chord; d.eps_push = cfg->eps_push; d.alpha_R = cfg->alpha_R; d.rho_R = cfg->rho_R;
  d.chord_budget = cfg->chord_budget; d.seed = cfg->seed; d.max_steps = cfg->max_steps;
  d.steps_per_launch = cfg->steps_per_launch;
  d.transit = (any_lists && cfg->navigator == ADEPT_NAV_BVH && cfg->steps_per_launch != 1) ? 1 : 0;
  d.capacity = static_cast<uint32_t>(cfg->track_capacity);
  d.stage_capacity = static_cast<uint32_t>(cfg->stage_capacity ? cfg->stage_capacity : cfg->track_capacity);
  d.leak_capacity = static_cast<uint32_t>(cfg->leak_capacity);
  ctx->d_stage = L.stage; ctx->d_bad = L.bad; ctx->stage_cap = L.stage_cap;

  // ---- relocation hints: the volume beyond each face of each box (kernels.cuh hint_kernel)
  hint_kernel<<<std::min((6 * nv + kBlock - 1) / kBlock, 4096), kBlock>>>(d, L.nbr);
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaDeviceSynchronize());

  int sms = 0, occ_g = 1, occ_c = 1, occ_i = 1;
  CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, ctx->device));
  {
    const bool bvh = cfg->navigator == ADEPT_NAV_BVH && !hb.empty();
    ctx->k_move_gamma[0] = bvh ? gamma_move_kernel<true, false> : gamma_move_kernel<false, false>;
    ctx->k_move_gamma[1] = bvh ? gamma_move_kernel<true, true> : gamma_move_kernel<false, true>;
#define ADEPT_CHARGED_KERNELS(F)                                                                                   \
  ctx->k_move_charged[0] = bvh ? charged_move_kernel<F, true, false> : charged_move_kernel<F, false, false>;        \
  ctx->k_move_charged[1] = bvh ? charged_move_kernel<F, true, true> : charged_move_kernel<F, false, true>
    switch (f->kind) {
      case ADEPT_FIELD_NONE: ADEPT_CHARGED_KERNELS(ADEPT_FIELD_NONE); break;
      case ADEPT_FIELD_UNIFORM:
        ADEPT_CHARGED_KERNELS(ADEPT_FIELD_UNIFORM);
        if (bvh) ctx->k_move_charged[2] = charged_move_kernel<ADEPT_FIELD_UNIFORM, true, true, true>;
        break;
      default:
        ADEPT_CHARGED_KERNELS(ADEPT_FIELD_MAP_RZ);
        if (bvh) ctx->k_move_charged[2] = charged_move_kernel<ADEPT_FIELD_MAP_RZ, true, true, true>;
        break;
    }
#undef ADEPT_CHARGED_KERNELS
    if (ctx->k_move_charged[2]) {
      int occ_low = 1;
      ctx->k_move_gamma[2] = ctx->k_move_gamma[1];
      CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_low, ctx->k_move_charged[2], kBlock, 0));
      ctx->grid_charged_low = sms * std::max(occ_low, 1);
    }
    // one grid for both variants of a kernel (the lean one sets it: it is the one that fills the GPU)
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_g, ctx->k_move_gamma[0], kBlock, 0));
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_c, ctx->k_move_charged[0], kBlock, 0));
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_i, interact_kernel, kBlock, 0));
  }
  ctx->grid_gamma = sms * std::max(occ_g, 1);
  ctx->grid_charged = sms * std::max(occ_c, 1);
  if (f->kind == ADEPT_FIELD_NONE && !(cfg->navigator == ADEPT_NAV_BVH && !hb.empty()) && cfg->concurrent_species != 0 &&
      ctx->grid_gamma == ctx->grid_charged) {
    ctx->k_move_merged[0] = move_kernel<false>;
    ctx->k_move_merged[1] = move_kernel<true>;
  }
  ctx->grid_inter = sms * std::max(occ_i, 1);

  ctx->slots.resize(cfg->n_event_slots);
  for (int s = 0; s < cfg->n_event_slots; ++s) {
    SlotHost& sh = ctx->slots[s];
    sh.dev = L.slots[s];
    CUDA_TRY(cudaStreamCreateWithFlags(&sh.helper, cudaStreamNonBlocking));
    CUDA_TRY(cudaEventCreateWithFlags(&sh.fork, cudaEventDisableTiming));
    CUDA_TRY(cudaEventCreateWithFlags(&sh.join, cudaEventDisableTiming));
    CUDA_TRY(cudaMallocHost(&sh.pinned, sizeof(SlotCounters)));
    std::memset(sh.pinned, 0, sizeof(SlotCounters));
    if (cfg->time_kernels) {
      sh.tev.resize(static_cast<size_t>(cfg->sync_interval) * 2 * ADEPT_N_TIMED_KERNELS);
      for (cudaEvent_t& e : sh.tev) CUDA_TRY(cudaEventCreate(&e));
    }
  }
  ctx->timing_on = cfg->time_kernels != 0;
  holder.c = nullptr;
  *out = ctx;
  return ADEPT_OK;
}

extern "C" int adept_set_kernel_timing(adept_ctx* ctx, int on) {
  if (!ctx) return fail(ADEPT_EINVAL, "null context");
  ADEPT_ON_DEVICE(ctx);
  if (on && !ctx->cfg.time_kernels) return fail(ADEPT_ESTATE, "context was not created with time_kernels");
  for (const SlotHost& sh : ctx->slots) if (sh.live) return fail(ADEPT_ESTATE, "a slot is being transported");
  ctx->timing_on = on != 0;
  return ADEPT_OK;
}

extern "C" int adept_shutdown(adept_ctx* ctx) {
  if (!ctx) return fail(ADEPT_EINVAL, "null context");
  ADEPT_ON_DEVICE(ctx);
  destroy_ctx(ctx);
  return ADEPT_OK;
}

namespace {
int check_slot(adept_ctx* ctx, int slot) {
  if (!ctx) return fail(ADEPT_EINVAL, "null context");
  if (slot < 0 || slot >= static_cast<int>(ctx->slots.size())) return fail(ADEPT_EINVAL, "event slot %d out of range", slot);
  return ADEPT_OK;
}

// Empties a slot on `st`: counters (populations, staging queues, leaked tracks, overflow flag), every replica
// of the scoring array, the ledger and the iteration trace.  The cumulative DevStats stay.
int reset_slot_async(adept_ctx* ctx, SlotHost& sh, cudaStream_t st) {
  CUDA_TRY(cudaMemsetAsync(sh.dev.counters, 0, sizeof(SlotCounters), st));
  CUDA_TRY(cudaMemsetAsync(sh.dev.edep, 0, static_cast<size_t>(sh.dev.edep_mask + 1) * sh.dev.edep_stride * sizeof(double), st));
  CUDA_TRY(cudaMemsetAsync(sh.dev.ledger, 0, 8 * sizeof(double), st));
  CUDA_TRY(cudaMemsetAsync(sh.dev.trace_n, 0, sizeof(uint32_t), st));
  sh.n_pending = sh.n_injected = 0;
  sh.population = 0;
  (void)ctx;
  return ADEPT_OK;
}
}  // namespace

extern "C" int adept_reset_slot(adept_ctx* ctx, int slot) {
  const int rc = check_slot(ctx, slot);
  if (rc != ADEPT_OK) return rc;
  ADEPT_ON_DEVICE(ctx);
  SlotHost& sh = ctx->slots[slot];
  if (sh.live) return fail(ADEPT_ESTATE, "slot %d is being transported", slot);
  CUDA_TRY(cudaDeviceSynchronize());
  const int r2 = reset_slot_async(ctx, sh, nullptr);
  if (r2 != ADEPT_OK) return r2;
  CUDA_TRY(cudaDeviceSynchronize());
  return ADEPT_OK;
}

extern "C" int adept_enqueue_batch(adept_ctx* ctx, int slot, int n, const uint32_t* event_ids, const uint64_t* track_ids,
                                   const int8_t* species, const double* pos3, const double* dir3, const double* ekin) {
  int rc = check_slot(ctx, slot);
  if (rc != ADEPT_OK) return rc;
  if (n < 0 || (n > 0 && (!event_ids || !track_ids || !species || !pos3 || !dir3 || !ekin))) return fail(ADEPT_EINVAL, "null argument");
  ADEPT_ON_DEVICE(ctx);
  // Runs on the legacy default stream and ends with a blocking copy of the error counter: the primaries are in
  // the slot when the call returns, whatever stream the transport then uses.
  SlotHost& sh = ctx->slots[slot];
  if (sh.live) return fail(ADEPT_ESTATE, "slot %d is being transported", slot);
  const bool stagger = ctx->cfg.inject_chunk != 0;
  const size_t pcap = ctx->cfg.pending_capacity ? ctx->cfg.pending_capacity : ctx->cfg.track_capacity;
  if (stagger && sh.n_pending + static_cast<size_t>(n) > pcap)
    return fail(ADEPT_EOVERFLOW, "slot %d: pending store full (%zu + %d > %zu primaries)", slot, sh.n_pending, n, pcap);
  std::vector<adept_track> host(std::min<size_t>(n, ctx->stage_cap));
  for (size_t done = 0; done < static_cast<size_t>(n);) {
    const size_t m = std::min(ctx->stage_cap, static_cast<size_t>(n) - done);
    for (size_t i = 0; i < m; ++i) {
      adept_track& t = host[i];
      const size_t k = done + i;
      for (int a = 0; a < 3; ++a) { t.pos[a] = pos3[3 * k + a]; t.dir[a] = dir3[3 * k + a]; }
      t.ekin = ekin[k]; t.id = track_ids[k]; t.event = event_ids[k]; t.step = 0; t.volume = 0; t.species = species[k];
      if (!(t.ekin >= 0.0)) return fail(ADEPT_EINVAL, "primary %zu: negative or NaN energy", k);
    }
    CUDA_TRY(cudaMemcpy(ctx->d_stage, host.data(), m * sizeof(adept_track), cudaMemcpyHostToDevice));
    CUDA_TRY(cudaMemset(ctx->d_bad, 0, sizeof(uint32_t)));
    const int grid = static_cast<int>(std::min<size_t>((m + kBlock - 1) / kBlock, 4096));
    enqueue_kernel<<<grid, kBlock>>>(ctx->dev, sh.dev, ctx->d_stage, static_cast<int>(m), ctx->d_bad,
                                     stagger ? sh.dev.pending + sh.n_pending : nullptr);
    CUDA_TRY(cudaGetLastError());
    uint32_t bad = 0;
    CUDA_TRY(cudaMemcpy(&bad, ctx->d_bad, sizeof(uint32_t), cudaMemcpyDeviceToHost));
    if (bad) return fail(ADEPT_EINVAL, "%u primaries lie outside the world or have an unknown species", bad);
    if (stagger) sh.n_pending += m; else sh.population += m;
    done += m;
  }
  return ADEPT_OK;
}

extern "C" int adept_enqueue_primaries(adept_ctx* ctx, int slot, uint32_t event_id, int n, const int8_t* species,
                                       const double* pos3, const double* dir3, const double* ekin) {
  if (n < 0) return fail(ADEPT_EINVAL, "negative count");
  std::vector<uint32_t> ev(n, event_id);
  std::vector<uint64_t> id(n);
  std::iota(id.begin(), id.end(), 0ull);
  return adept_enqueue_batch(ctx, slot, n, ev.data(), id.data(), species, pos3, dir3, ekin);
}

namespace {

// waves of sparse tiles of a BVH field kernel whose slot has the GPU to itself (round_variant)
#ifndef ADEPT_SPARSE_WAVES_ALONE
#define ADEPT_SPARSE_WAVES_ALONE 4
#endif

// One population step of a slot: gamma move kernel on the caller's stream, charged move kernel on the
// helper stream (species kernels on different streams, synchronised with events), then the
// interaction kernel over what they staged and the buffer swap.
int launch_iteration(adept_ctx* ctx, SlotHost& sh, cudaStream_t st, int parity, const DevCtx& dc_in, int variant) {
  const int multi = variant % 3;   // kernels; variant >= 3: the slot has the GPU to itself (round_variant)
  DevCtx dc = dc_in;
  dc.sparse_waves = variant >= 3 ? ADEPT_SPARSE_WAVES_ALONE : 1;
  constexpr int kEv = 2 * ADEPT_N_TIMED_KERNELS;
  if (sh.n_injected < sh.n_pending) {   // staggered injection: the next chunk joins the population of this step
    const size_t m = std::min<size_t>(ctx->cfg.inject_chunk, sh.n_pending - sh.n_injected);
    inject_kernel<<<static_cast<int>(std::min<size_t>((m + kBlock - 1) / kBlock, 1024)), kBlock, 0, st>>>(
        dc, sh.dev, parity, static_cast<uint32_t>(sh.n_injected), static_cast<uint32_t>(m));
    sh.n_injected += m;
    sh.launches += 1;
  }
  const bool timed = ctx->timing_on && !sh.tev.empty() && sh.tev_used + kEv <= static_cast<int>(sh.tev.size());
  // a timed pass runs the kernels one after the other, so that an event pair brackets one kernel alone
  if (ctx->k_move_merged[multi]) {   // all three species in one launch (timed as kernel [0]; [1] stays empty)
    cudaEvent_t* ev = timed ? &sh.tev[sh.tev_used] : nullptr;
    if (timed) CUDA_TRY(cudaEventRecord(ev[0], st));
    ctx->k_move_merged[multi]<<<dim3(ctx->grid_gamma, 3), kBlock, 0, st>>>(dc, sh.dev, parity);
    if (timed) { CUDA_TRY(cudaEventRecord(ev[1], st)); CUDA_TRY(cudaEventRecord(ev[4], st)); }
    interact_kernel<<<ctx->grid_inter, kBlock, 0, st>>>(dc, sh.dev, parity);
    if (timed) { CUDA_TRY(cudaEventRecord(ev[5], st)); sh.tev_used += kEv; }
    sh.launches += 2;
    return ADEPT_OK;
  }
  const bool fork = ctx->cfg.concurrent_species != 0 && !ctx->timing_on;
  cudaStream_t sc = fork ? sh.helper : st;   // stream of the charged move kernel
  if (fork) {
    CUDA_TRY(cudaEventRecord(sh.fork, st));
    CUDA_TRY(cudaStreamWaitEvent(sh.helper, sh.fork, 0));
  }
  cudaEvent_t* ev = timed ? &sh.tev[sh.tev_used] : nullptr;
  if (timed) CUDA_TRY(cudaEventRecord(ev[0], st));
  ctx->k_move_gamma[multi]<<<dim3(ctx->grid_gamma, 1), kBlock, 0, st>>>(dc, sh.dev, parity);
  if (timed) CUDA_TRY(cudaEventRecord(ev[1], st));
  if (timed) CUDA_TRY(cudaEventRecord(ev[2], sc));
  ctx->k_move_charged[multi]<<<dim3(multi == 2 ? ctx->grid_charged_low : ctx->grid_charged, 2), kBlock, 0, sc>>>(dc, sh.dev, parity);
  if (timed) CUDA_TRY(cudaEventRecord(ev[3], sc));
  if (fork) {
    CUDA_TRY(cudaEventRecord(sh.join, sh.helper));
    CUDA_TRY(cudaStreamWaitEvent(st, sh.join, 0));
  }
  if (timed) CUDA_TRY(cudaEventRecord(ev[4], st));
  interact_kernel<<<ctx->grid_inter, kBlock, 0, st>>>(dc, sh.dev, parity);
  if (timed) { CUDA_TRY(cudaEventRecord(ev[5], st)); sh.tev_used += kEv; }
  sh.launches += 3;
  return ADEPT_OK;
}

// One host round -- sync_interval population steps, starting at parity 0 -- as a CUDA graph: the slot's
// kernels, forks and joins are captured once on a library-owned stream and replayed with one launch per
// round.  A small event (config 5: 200 primaries, thousands of nearly empty population steps on each of 16
// streams) is otherwise bound by the host issuing ~10 API calls per step.  Needs an even sync_interval (every
// round then starts at parity 0), no per-launch timing and no pending injection; returns false to fall back.
bool round_graph(adept_ctx* ctx, SlotHost& sh, int multi /* variant index 0..5 */) {
  if (sh.gexec[multi]) return true;
  if (sh.graph_failed[multi] || !ctx->cfg.use_graphs || (ctx->cfg.sync_interval & 1)) return false;
  if (!sh.cap && cudaStreamCreateWithFlags(&sh.cap, cudaStreamNonBlocking) != cudaSuccess) { sh.graph_failed[multi] = true; return false; }
  const unsigned long long launches = sh.launches;
  cudaGraph_t graph = nullptr;
  bool ok = cudaStreamBeginCapture(sh.cap, cudaStreamCaptureModeRelaxed) == cudaSuccess;
  if (ok) {
    for (int it = 0; it < ctx->cfg.sync_interval && ok; ++it) ok = launch_iteration(ctx, sh, sh.cap, it & 1, ctx->dev, multi) == ADEPT_OK;
    ok = (cudaStreamEndCapture(sh.cap, &graph) == cudaSuccess) && ok && graph;
  }
  if (ok) ok = cudaGraphInstantiate(&sh.gexec[multi], graph, 0) == cudaSuccess;
  if (graph) cudaGraphDestroy(graph);
  sh.launches = launches;
  if (!ok) { cudaGetLastError(); sh.gexec[multi] = nullptr; sh.graph_failed[multi] = true; }
  return ok;
}

// Which move kernels the next host round of a slot runs: the multi-step variants once the population the host
// last saw no longer fills the GPU (their lanes go on stepping their own tracks, kernels.cuh inner_steps).
// The showers do not depend on the choice; a stale population costs speed only.
constexpr size_t kMultiBelow = 65536;
// BVH geometry in a field: below this population a launch lasts as long as its longest chain of chords and traversals,
// and the e+- kernel without register spills (two resident blocks per SM) is the faster one (charged.cuh)
#ifndef ADEPT_LOWOCC_BELOW
#define ADEPT_LOWOCC_BELOW 262144
#endif
// + 3 (`alone`): the call transports one or two slots, so this slot's kernels have the GPU (nearly) to themselves: a BVH
// field kernel may then spread a small e+- population over several waves of sparse tiles and still take the chord loop
// with several lanes per track (charged.cuh; config 4 863 -> 820 ms per pass with 4 waves, 832 with 2; with sixteen slots
// side by side it costs: config 5 33.0 -> 27.5 events/s, which is why it hangs on the number of slots)
int round_variant(const adept_ctx* ctx, const SlotHost& sh, bool alone = false) {
  if (alone && ctx->k_move_charged[2]) return 3 + round_variant(ctx, sh, false);
  if (ctx->cfg.steps_per_launch == 1) return 0;
  const size_t population = sh.population + (sh.n_pending - sh.n_injected);
  const int below = ctx->cfg.low_occupancy_below == 0 ? ADEPT_LOWOCC_BELOW : ctx->cfg.low_occupancy_below;
  if (ctx->k_move_charged[2] && below > 0 && population < static_cast<size_t>(below)) return 2;
  if (ctx->dev.transit) return 1;   // the multi-step variants also take the passage through a vacuum gap in the same launch
  return population < kMultiBelow ? 1 : 0;
}

}  // namespace

extern "C" int adept_transport_many(adept_ctx* ctx, int n_slots, const int* slots, void* const* streams) {
  if (!ctx || n_slots < 0 || (n_slots > 0 && (!slots || !streams))) return fail(ADEPT_EINVAL, "null argument");
  ADEPT_ON_DEVICE(ctx);
  for (int k = 0; k < n_slots; ++k) {
    const int rc = check_slot(ctx, slots[k]);
    if (rc != ADEPT_OK) return rc;
  }
  // Marks the listed slots live; whatever way this call ends, none of them stays marked.
  struct LiveMarks {
    adept_ctx* ctx; const int* slots; int n = 0;
    ~LiveMarks() { for (int k = 0; k < n; ++k) ctx->slots[slots[k]].live = false; }
  } marks{ctx, slots};
  for (int k = 0; k < n_slots; ++k) {
    SlotHost& sh = ctx->slots[slots[k]];
    if (sh.live) return fail(ADEPT_EINVAL, "event slot %d is listed twice or already in transport", slots[k]);
    sh.live = true;
    marks.n = k + 1;
  }
  std::vector<int> parity(n_slots, 0);
  int n_live = n_slots, rc_final = ADEPT_OK;
  // One host round of slot k: sync_interval population steps (one graph launch where possible) and the copy of its
  // counters, all on the slot's stream.
  const auto issue_round = [&](int k) -> int {
    SlotHost& sh = ctx->slots[slots[k]];
    cudaStream_t st = static_cast<cudaStream_t>(streams[k]);
    const int variant = round_variant(ctx, sh, n_slots <= 2);
    if (parity[k] == 0 && !ctx->timing_on && sh.n_injected == sh.n_pending && round_graph(ctx, sh, variant)) {
      CUDA_TRY(cudaGraphLaunch(sh.gexec[variant], st));
      sh.launches += (ctx->k_move_merged[variant % 3] ? 2ull : 3ull) * ctx->cfg.sync_interval;   // kernels of the replayed round
    } else {
      for (int it = 0; it < ctx->cfg.sync_interval; ++it) {
        const int rc = launch_iteration(ctx, sh, st, parity[k], ctx->dev, variant);
        if (rc != ADEPT_OK) return rc;
        parity[k] ^= 1;
      }
    }
    CUDA_TRY(cudaMemcpyAsync(sh.pinned, sh.dev.counters, sizeof(SlotCounters), cudaMemcpyDeviceToHost, st));
    return ADEPT_OK;
  };
  // What the round of slot k left behind (its stream is idle): kernel times, overflow, population; *done = the slot is empty.
  const auto finish_round = [&](int k, bool* done) -> int {
    SlotHost& sh = ctx->slots[slots[k]];
    cudaStream_t st = static_cast<cudaStream_t>(streams[k]);
    for (int e = 0; e + 2 * ADEPT_N_TIMED_KERNELS <= sh.tev_used; e += 2 * ADEPT_N_TIMED_KERNELS)
      for (int kk = 0; kk < ADEPT_N_TIMED_KERNELS; ++kk) {
        if (kk == 1 && ctx->k_move_merged[0]) continue;   // the merged move kernel is kernel [0]
        float ms = 0.f;
        CUDA_TRY(cudaEventElapsedTime(&ms, sh.tev[e + 2 * kk], sh.tev[e + 2 * kk + 1]));
        sh.kernel_ms[kk] += ms;
        sh.kernel_launches[kk] += 1;
      }
    sh.tev_used = 0;
    const bool overflow = sh.pinned->overflow.v != 0;
    sh.population = sh.pinned->live.v;
    if (overflow) {
      // The pass is abandoned: the slot is emptied (tracks, staging queues, scoring, ledger, leaked tracks) so
      // that the caller can enqueue a smaller batch into it.
      rc_final = fail(ADEPT_EOVERFLOW, "slot %d: track queue overflow (capacity %llu per species, %llu per staging queue); slot reset",
                      slots[k], static_cast<unsigned long long>(ctx->dev.capacity), static_cast<unsigned long long>(ctx->dev.stage_capacity));
      const int rr = reset_slot_async(ctx, sh, st);
      if (rr != ADEPT_OK) return rr;
      CUDA_TRY(cudaStreamSynchronize(st));
    }
    *done = (sh.pinned->live.v == 0 && sh.n_injected == sh.n_pending) || overflow;
    if (*done) {
      sh.n_pending = sh.n_injected = 0;
      sh.population = 0;
      sh.live = false;
      --n_live;
      // counts are all zero: the (empty) slot is at parity 0 for the next enqueue whatever parity[k] is
    }
    return ADEPT_OK;
  };
  // Every slot advances at its own pace: its next round is issued as soon as its own round has finished, not when the
  // slowest slot's has (config 5: the rounds of 16 events last from a fraction of a millisecond to tens of them).
  for (int k = 0; k < n_slots; ++k) {
    const int rc = issue_round(k);
    if (rc != ADEPT_OK) return rc;
  }
  while (n_live > 0) {
    bool progressed = false;
    for (int k = 0; k < n_slots; ++k) {
      SlotHost& sh = ctx->slots[slots[k]];
      if (!sh.live) continue;
      cudaStream_t st = static_cast<cudaStream_t>(streams[k]);
      if (n_live == 1) {
        CUDA_TRY(cudaStreamSynchronize(st));      // a single slot left: wait for it, no polling
      } else {
        const cudaError_t q = cudaStreamQuery(st);
        if (q == cudaErrorNotReady) continue;
        CUDA_TRY(q);
      }
      bool done = false;
      int rc = finish_round(k, &done);
      if (rc != ADEPT_OK) return rc;
      if (!done) {
        rc = issue_round(k);
        if (rc != ADEPT_OK) return rc;
      }
      progressed = true;
    }
    if (!progressed) std::this_thread::yield();
  }
  CUDA_TRY(cudaGetLastError());
  if (rc_final != ADEPT_OK) fail(rc_final, "a slot's track queue overflowed (track_capacity %llu, stage_capacity %llu); the slot was reset",
                                 static_cast<unsigned long long>(ctx->dev.capacity), static_cast<unsigned long long>(ctx->dev.stage_capacity));
  return rc_final;
}

extern "C" int adept_transport(adept_ctx* ctx, int slot, void* stream) {
  return adept_transport_many(ctx, 1, &slot, &stream);
}

extern "C" int adept_read_scoring(adept_ctx* ctx, int slot, double* edep, size_t n_volumes, adept_ledger* ledger, void* stream) {
  const int rc = check_slot(ctx, slot);
  if (rc != ADEPT_OK) return rc;
  ADEPT_ON_DEVICE(ctx);
  if (edep && n_volumes != static_cast<size_t>(ctx->n_vol)) return fail(ADEPT_EINVAL, "n_volumes is %zu, geometry has %d", n_volumes, ctx->n_vol);
  SlotHost& sh = ctx->slots[slot];
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  fold_edep_kernel<<<(ctx->n_vol + 255) / 256, 256, 0, st>>>(sh.dev, ctx->n_vol);
  if (edep) CUDA_TRY(cudaMemcpyAsync(edep, sh.dev.edep, n_volumes * sizeof(double), cudaMemcpyDeviceToHost, st));
  double led[5];
  CUDA_TRY(cudaMemcpyAsync(led, sh.dev.ledger, sizeof(led), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaMemsetAsync(sh.dev.edep, 0, static_cast<size_t>(ctx->n_vol) * sizeof(double), st));
  CUDA_TRY(cudaMemsetAsync(sh.dev.ledger, 0, 8 * sizeof(double), st));
  CUDA_TRY(cudaStreamSynchronize(st));
  if (ledger) { ledger->deposited = led[0]; ledger->below_cut = led[1]; ledger->escaped = led[2]; ledger->killed = led[3]; ledger->primary = led[4]; }
  return ADEPT_OK;
}

extern "C" int adept_read_leaked(adept_ctx* ctx, int slot, adept_track* out, size_t cap, size_t* n) {
  const int rc = check_slot(ctx, slot);
  if (rc != ADEPT_OK) return rc;
  ADEPT_ON_DEVICE(ctx);
  if (!n) return fail(ADEPT_EINVAL, "null argument");
  SlotHost& sh = ctx->slots[slot];
  uint32_t n_leaked = 0;
  CUDA_TRY(cudaMemcpy(&n_leaked, &sh.dev.counters->n_leaked.v, sizeof(uint32_t), cudaMemcpyDeviceToHost));
  *n = n_leaked;
  const size_t m = std::min<size_t>(std::min<size_t>(n_leaked, cap), ctx->cfg.leak_capacity);
  if (m && out) CUDA_TRY(cudaMemcpy(out, sh.dev.leaked, m * sizeof(adept_track), cudaMemcpyDeviceToHost));
  CUDA_TRY(cudaMemset(&sh.dev.counters->n_leaked.v, 0, sizeof(uint32_t)));
  return ADEPT_OK;
}

extern "C" int adept_get_stats(adept_ctx* ctx, int slot, adept_stats* out) {
  const int rc = check_slot(ctx, slot);
  if (rc != ADEPT_OK) return rc;
  ADEPT_ON_DEVICE(ctx);
  if (!out) return fail(ADEPT_EINVAL, "null argument");
  DevStats s;
  CUDA_TRY(cudaMemcpy(&s, ctx->slots[slot].dev.stats, sizeof(s), cudaMemcpyDeviceToHost));
  for (int k = 0; k < 3; ++k) { out->steps[k] = s.steps[k]; out->secondaries[k] = s.secondaries[k]; }
  for (int k = 0; k < ADEPT_N_OUTCOMES; ++k) out->outcomes[k] = s.outcomes[k];
  out->chords = s.chords; out->iterations = s.iterations; out->peak_population = s.peak_population;
  out->launches = ctx->slots[slot].launches;
  return ADEPT_OK;
}

extern "C" int adept_get_iteration_trace(adept_ctx* ctx, int slot, uint64_t* t_ns, uint32_t* population, size_t cap, size_t* n) {
  const int rc = check_slot(ctx, slot);
  if (rc != ADEPT_OK) return rc;
  ADEPT_ON_DEVICE(ctx);
  if (!n) return fail(ADEPT_EINVAL, "null argument");
  SlotHost& sh = ctx->slots[slot];
  if (sh.live) return fail(ADEPT_ESTATE, "slot %d is being transported", slot);
  uint32_t m = 0;
  CUDA_TRY(cudaMemcpy(&m, sh.dev.trace_n, sizeof(uint32_t), cudaMemcpyDeviceToHost));
  const size_t k = std::min<size_t>(std::min<size_t>(m, cap), ADEPT_TRACE_CAPACITY);
  if (k && t_ns) CUDA_TRY(cudaMemcpy(t_ns, sh.dev.trace_t, k * sizeof(uint64_t), cudaMemcpyDeviceToHost));
  if (k && population) CUDA_TRY(cudaMemcpy(population, sh.dev.trace_pop, 3 * k * sizeof(uint32_t), cudaMemcpyDeviceToHost));
  CUDA_TRY(cudaMemset(sh.dev.trace_n, 0, sizeof(uint32_t)));
  *n = k;
  return ADEPT_OK;
}

extern "C" int adept_get_kernel_times(adept_ctx* ctx, int slot, double ms[ADEPT_N_TIMED_KERNELS],
                                      uint64_t launches[ADEPT_N_TIMED_KERNELS]) {
  const int rc = check_slot(ctx, slot);
  if (rc != ADEPT_OK) return rc;
  if (!ms || !launches) return fail(ADEPT_EINVAL, "null argument");
  SlotHost& sh = ctx->slots[slot];
  if (sh.tev.empty()) return fail(ADEPT_ESTATE, "context was not created with time_kernels");
  for (int k = 0; k < ADEPT_N_TIMED_KERNELS; ++k) { ms[k] = sh.kernel_ms[k]; launches[k] = sh.kernel_launches[k]; sh.kernel_ms[k] = 0.0; sh.kernel_launches[k] = 0; }
  return ADEPT_OK;
}

extern "C" int adept_step_frozen(adept_ctx* ctx, int n, const adept_track* in, adept_step_result* out, adept_track* sec, void* stream) {
  if (!ctx || n < 0 || (n > 0 && (!in || !out || !sec))) return fail(ADEPT_EINVAL, "null argument");
  if (n == 0) return ADEPT_OK;
  for (int i = 0; i < n; ++i)
    if (in[i].volume >= static_cast<uint32_t>(ctx->n_vol) || in[i].species < 0 || in[i].species > 2)
      return fail(ADEPT_EINVAL, "track %d: volume or species out of range", i);
  ADEPT_ON_DEVICE(ctx);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  DevBuf<adept_track> d_in, d_sec;
  DevBuf<adept_step_result> d_out;
  CUDA_TRY(d_in.alloc(n)); CUDA_TRY(d_out.alloc(n)); CUDA_TRY(d_sec.alloc(2 * static_cast<size_t>(n)));
  CUDA_TRY(cudaMemcpyAsync(d_in, in, n * sizeof(adept_track), cudaMemcpyHostToDevice, st));
  const int grid = std::min((n + kBlock - 1) / kBlock, 65535);
  frozen_kernel<<<grid, kBlock, 0, st>>>(ctx->dev, d_in, d_out, d_sec, n);
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaMemcpyAsync(out, d_out, n * sizeof(adept_step_result), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaMemcpyAsync(sec, d_sec, 2 * static_cast<size_t>(n) * sizeof(adept_track), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  return ADEPT_OK;
}

extern "C" int adept_step_population(adept_ctx* ctx, int slot, int n, const adept_track* in, adept_track* out, size_t out_cap,
                                     size_t* n_out, void* stream) {
  const int rc = check_slot(ctx, slot);
  if (rc != ADEPT_OK) return rc;
  if (n < 0 || !n_out || (n > 0 && !in) || (out_cap > 0 && !out)) return fail(ADEPT_EINVAL, "null argument");
  *n_out = 0;
  for (int i = 0; i < n; ++i)
    if (in[i].volume >= static_cast<uint32_t>(ctx->n_vol) || in[i].species < 0 || in[i].species > 2 || !(in[i].ekin >= 0.0))
      return fail(ADEPT_EINVAL, "track %d: volume, species or energy out of range", i);
  ADEPT_ON_DEVICE(ctx);
  SlotHost& sh = ctx->slots[slot];
  if (sh.live || sh.n_pending != sh.n_injected) return fail(ADEPT_ESTATE, "slot %d is not empty", slot);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  CUDA_TRY(cudaMemcpyAsync(sh.pinned, sh.dev.counters, sizeof(SlotCounters), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  if (sh.pinned->live.v != 0) return fail(ADEPT_ESTATE, "slot %d holds %u live tracks", slot, sh.pinned->live.v);
  if (n == 0) return ADEPT_OK;
  DevBuf<adept_track> d_in, d_out;
  CUDA_TRY(d_in.alloc(n));
  CUDA_TRY(cudaMemcpyAsync(d_in, in, static_cast<size_t>(n) * sizeof(adept_track), cudaMemcpyHostToDevice, st));
  load_tracks_kernel<<<std::min((n + kBlock - 1) / kBlock, 4096), kBlock, 0, st>>>(ctx->dev, sh.dev, d_in, n);
  CUDA_TRY(cudaGetLastError());
  // exactly one population step: the kernels and grids of adept_transport, one step per track and launch
  // (the variant of the move kernels adept_transport would pick for a population of n, held to one step per track)
  DevCtx one = ctx->dev;
  one.steps_per_launch = 1;
  one.transit = 0;
  sh.population = static_cast<size_t>(n);
  const int variant = round_variant(ctx, sh);
  sh.population = 0;
  const bool timing = ctx->timing_on;
  ctx->timing_on = false;
  const int rl = launch_iteration(ctx, sh, st, 0, one, variant);
  ctx->timing_on = timing;
  if (rl != ADEPT_OK) return rl;
  CUDA_TRY(cudaMemcpyAsync(sh.pinned, sh.dev.counters, sizeof(SlotCounters), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  if (sh.pinned->overflow.v) {
    const int rr = reset_slot_async(ctx, sh, st);
    if (rr != ADEPT_OK) return rr;
    CUDA_TRY(cudaStreamSynchronize(st));
    return fail(ADEPT_EOVERFLOW, "slot %d: track queue overflow in the population step; slot reset", slot);
  }
  uint32_t cnt[3];
  size_t total = 0;
  for (int sp = 0; sp < 3; ++sp) { cnt[sp] = sh.pinned->count[1][sp].v; total += cnt[sp]; }
  *n_out = total;
  if (total > 0) {
    CUDA_TRY(d_out.alloc(total));
    gather_tracks_kernel<<<static_cast<int>(std::min<size_t>((total + kBlock - 1) / kBlock, 4096)), kBlock, 0, st>>>(
        sh.dev, 1, cnt[0], cnt[1], cnt[2], d_out);
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaMemcpyAsync(out, d_out, std::min(total, out_cap) * sizeof(adept_track), cudaMemcpyDeviceToHost, st));
  }
  // the slot is empty again: the next population is dropped
  for (int sp = 0; sp < 3; ++sp) CUDA_TRY(cudaMemsetAsync(&sh.dev.counters->count[1][sp].v, 0, sizeof(uint32_t), st));
  CUDA_TRY(cudaMemsetAsync(&sh.dev.counters->live.v, 0, sizeof(uint32_t), st));
  CUDA_TRY(cudaStreamSynchronize(st));
  return ADEPT_OK;
}

extern "C" int adept_distance_batch(adept_ctx* ctx, int nav, int n, const double* pos3, const double* dir3, const uint32_t* volume,
                                    const double* s_max, double* out, void* stream) {
  if (!ctx || n < 0 || (n > 0 && (!pos3 || !dir3 || !volume || !s_max || !out))) return fail(ADEPT_EINVAL, "null argument");
  if (n == 0) return ADEPT_OK;
  for (int i = 0; i < n; ++i) if (volume[i] >= static_cast<uint32_t>(ctx->n_vol)) return fail(ADEPT_EINVAL, "ray %d: volume out of range", i);
  ADEPT_ON_DEVICE(ctx);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  DevBuf<double> d_pos, d_dir, d_smax, d_out;
  DevBuf<uint32_t> d_vol;
  CUDA_TRY(d_pos.alloc(3 * static_cast<size_t>(n))); CUDA_TRY(d_dir.alloc(3 * static_cast<size_t>(n)));
  CUDA_TRY(d_smax.alloc(n)); CUDA_TRY(d_out.alloc(n)); CUDA_TRY(d_vol.alloc(n));
  CUDA_TRY(cudaMemcpyAsync(d_pos, pos3, 3 * n * sizeof(double), cudaMemcpyHostToDevice, st));
  CUDA_TRY(cudaMemcpyAsync(d_dir, dir3, 3 * n * sizeof(double), cudaMemcpyHostToDevice, st));
  CUDA_TRY(cudaMemcpyAsync(d_smax, s_max, n * sizeof(double), cudaMemcpyHostToDevice, st));
  CUDA_TRY(cudaMemcpyAsync(d_vol, volume, n * sizeof(uint32_t), cudaMemcpyHostToDevice, st));
  distance_kernel<<<std::min((n + kBlock - 1) / kBlock, 65535), kBlock, 0, st>>>(ctx->dev, nav, n, d_pos, d_dir, d_vol, d_smax, d_out);
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaMemcpyAsync(out, d_out, n * sizeof(double), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  return ADEPT_OK;
}

extern "C" int adept_raycast_batch(adept_ctx* ctx, int nav, int n, const double* pos3, const double* dir3, int max_crossings,
                                   double* column, int32_t* crossings, double* device_ms, void* stream) {
  if (!ctx || n < 0 || (n > 0 && (!pos3 || !dir3 || !column || !crossings))) return fail(ADEPT_EINVAL, "null argument");
  if (nav < ADEPT_NAV_LOOP || nav > ADEPT_NAV_BVH_F32) return fail(ADEPT_EINVAL, "unknown navigator");
  if (max_crossings < 1) return fail(ADEPT_EINVAL, "max_crossings must be >= 1");
  if (n == 0) return ADEPT_OK;
  ADEPT_ON_DEVICE(ctx);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  double *d_pos = nullptr, *d_dir = nullptr, *d_col = nullptr;
  int32_t* d_nx = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  int rc = ADEPT_OK;
  const size_t nb = static_cast<size_t>(n) * 3 * sizeof(double);
  do {
    if (cudaMalloc(&d_pos, nb) != cudaSuccess || cudaMalloc(&d_dir, nb) != cudaSuccess ||
        cudaMalloc(&d_col, static_cast<size_t>(n) * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&d_nx, static_cast<size_t>(n) * sizeof(int32_t)) != cudaSuccess ||
        cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) { rc = fail(ADEPT_ENOMEM, "ray-cast buffers"); break; }
    if (cudaMemcpyAsync(d_pos, pos3, nb, cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(d_dir, dir3, nb, cudaMemcpyHostToDevice, st) != cudaSuccess) { rc = fail(ADEPT_ECUDA, "ray-cast upload"); break; }
    cudaEventRecord(e0, st);
    const int grid = std::min((n + kBlock - 1) / kBlock, 65535);
    if (nav >= ADEPT_NAV_LOOP_F32)   // ADEPT_NAV_LOOP_F32 -> loop, ADEPT_NAV_BVH_F32 -> BVH, on the fp32 geometry
      raycast_kernel<float><<<grid, kBlock, 0, st>>>(ctx->dev, nav - ADEPT_NAV_LOOP_F32, n, d_pos, d_dir, max_crossings, d_col, d_nx);
    else
      raycast_kernel<double><<<grid, kBlock, 0, st>>>(ctx->dev, nav, n, d_pos, d_dir, max_crossings, d_col, d_nx);
    cudaEventRecord(e1, st);
    if (cudaMemcpyAsync(column, d_col, static_cast<size_t>(n) * sizeof(double), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaMemcpyAsync(crossings, d_nx, static_cast<size_t>(n) * sizeof(int32_t), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) { rc = fail(ADEPT_ECUDA, "ray-cast kernel"); break; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (device_ms) *device_ms = ms;
  } while (false);
  cudaFree(d_pos); cudaFree(d_dir); cudaFree(d_col); cudaFree(d_nx);
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  return rc;
}

// ---- adept_raycast_batch without an allocation (include/adept.h adept_raycast_batch_static) ----
// The ray-cast kernel reads ray origins and directions and writes column densities and crossing counts in device
// memory; adept_raycast_batch takes those four buffers from cudaMalloc, this variant from one file-scope array.
// Every GPU that loads the library holds the array (3.75 MiB) until the process exits.  In host code the name
// g_static_scratch is a stand-in for the symbol, not a device address: kernels are given what
// cudaGetSymbolAddress returned on their device.
constexpr size_t kStaticMaxRays = ADEPT_STATIC_MAX_RAYS;
constexpr size_t kStaticPos = 0;                                                // [n][3] doubles
constexpr size_t kStaticDir = kStaticPos + kStaticMaxRays * 3 * sizeof(double); // [n][3] doubles
constexpr size_t kStaticCol = kStaticDir + kStaticMaxRays * 3 * sizeof(double); // [n] doubles
constexpr size_t kStaticNx = kStaticCol + kStaticMaxRays * sizeof(double);      // [n] int32
constexpr size_t kStaticBytes = kStaticNx + kStaticMaxRays * sizeof(int32_t);
static_assert(kStaticDir % 256 == 0 && kStaticCol % 256 == 0 && kStaticNx % 256 == 0, "sub-buffers keep the array's alignment");
static __device__ __align__(256) unsigned char g_static_scratch[kStaticBytes];

namespace {

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mutex;
unsigned char* g_static_addr[kStaticMaxDevices] = {};  // device address of g_static_scratch, per device ordinal

// Address of g_static_scratch on `device`, which the caller has made current: asked of the runtime once per device.
int static_scratch(int device, unsigned char** out) {
  if (device < 0 || device >= kStaticMaxDevices) return fail(ADEPT_EINVAL, "device %d: the static scratch serves devices 0..%d", device, kStaticMaxDevices - 1);
  std::lock_guard<std::mutex> lock(g_static_mutex);
  if (!g_static_addr[device]) {
    unsigned char* ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g_static_scratch);
    if (e != cudaSuccess || !ptr) return fail(ADEPT_ECUDA, "cudaGetSymbolAddress(g_static_scratch) on device %d: %s", device, cudaGetErrorString(e));
    g_static_addr[device] = ptr;
  }
  *out = g_static_addr[device];
  return ADEPT_OK;
}

}  // namespace

extern "C" int adept_raycast_batch_static(adept_ctx* ctx, int nav, int n, const double* pos3, const double* dir3, int max_crossings,
                                          double* column, int32_t* crossings, void* stream) {
  if (!ctx || n < 0 || (n > 0 && (!pos3 || !dir3 || !column || !crossings))) return fail(ADEPT_EINVAL, "null argument");
  if (nav < ADEPT_NAV_LOOP || nav > ADEPT_NAV_BVH_F32) return fail(ADEPT_EINVAL, "unknown navigator");
  if (max_crossings < 1) return fail(ADEPT_EINVAL, "max_crossings must be >= 1");
  if (static_cast<size_t>(n) > kStaticMaxRays)
    return fail(ADEPT_EINVAL, "adept_raycast_batch_static: %d rays exceed ADEPT_STATIC_MAX_RAYS = %d (the static scratch array); "
                "split the batch or call adept_raycast_batch", n, ADEPT_STATIC_MAX_RAYS);
  if (n == 0) return ADEPT_OK;
  ADEPT_ON_DEVICE(ctx);
  unsigned char* base = nullptr;
  const int rc = static_scratch(ctx->device, &base);
  if (rc != ADEPT_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  double* d_pos = reinterpret_cast<double*>(base + kStaticPos);
  double* d_dir = reinterpret_cast<double*>(base + kStaticDir);
  double* d_col = reinterpret_cast<double*>(base + kStaticCol);
  int32_t* d_nx = reinterpret_cast<int32_t*>(base + kStaticNx);
  const size_t nb = static_cast<size_t>(n) * 3 * sizeof(double);
  // the array keeps the last call's contents: the results start at zero, the inputs are overwritten
  CUDA_TRY(cudaMemsetAsync(d_col, 0, static_cast<size_t>(n) * sizeof(double), st));
  CUDA_TRY(cudaMemsetAsync(d_nx, 0, static_cast<size_t>(n) * sizeof(int32_t), st));
  CUDA_TRY(cudaMemcpyAsync(d_pos, pos3, nb, cudaMemcpyHostToDevice, st));
  CUDA_TRY(cudaMemcpyAsync(d_dir, dir3, nb, cudaMemcpyHostToDevice, st));
  const int grid = std::min((n + kBlock - 1) / kBlock, 65535);
  if (nav >= ADEPT_NAV_LOOP_F32)
    raycast_kernel<float><<<grid, kBlock, 0, st>>>(ctx->dev, nav - ADEPT_NAV_LOOP_F32, n, d_pos, d_dir, max_crossings, d_col, d_nx);
  else
    raycast_kernel<double><<<grid, kBlock, 0, st>>>(ctx->dev, nav, n, d_pos, d_dir, max_crossings, d_col, d_nx);
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaMemcpyAsync(column, d_col, static_cast<size_t>(n) * sizeof(double), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaMemcpyAsync(crossings, d_nx, static_cast<size_t>(n) * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  return ADEPT_OK;
}

extern "C" int adept_locate_batch(adept_ctx* ctx, int nav, int n, const double* pos3, int64_t* out, void* stream) {
  if (!ctx || n < 0 || (n > 0 && (!pos3 || !out))) return fail(ADEPT_EINVAL, "null argument");
  if (n == 0) return ADEPT_OK;
  ADEPT_ON_DEVICE(ctx);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  DevBuf<double> d_pos;
  DevBuf<long long> d_out;
  CUDA_TRY(d_pos.alloc(3 * static_cast<size_t>(n))); CUDA_TRY(d_out.alloc(n));
  CUDA_TRY(cudaMemcpyAsync(d_pos, pos3, 3 * n * sizeof(double), cudaMemcpyHostToDevice, st));
  locate_kernel<<<std::min((n + kBlock - 1) / kBlock, 65535), kBlock, 0, st>>>(ctx->dev, nav, n, d_pos, d_out);
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaMemcpyAsync(out, d_out, n * sizeof(long long), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  return ADEPT_OK;
}

extern "C" int adept_relocate_batch(adept_ctx* ctx, int nav, int n, const double* pos3, const uint32_t* from, const int32_t* face,
                                    int64_t* out, void* stream) {
  if (!ctx || n < 0 || (n > 0 && (!pos3 || !from || !out))) return fail(ADEPT_EINVAL, "null argument");
  if (n == 0) return ADEPT_OK;
  for (int i = 0; i < n; ++i) {
    if (from[i] >= static_cast<uint32_t>(ctx->n_vol)) return fail(ADEPT_EINVAL, "point %d: volume out of range", i);
    if (face && (face[i] < -1 || face[i] > 5)) return fail(ADEPT_EINVAL, "point %d: face out of range", i);
  }
  ADEPT_ON_DEVICE(ctx);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  DevBuf<double> d_pos;
  DevBuf<uint32_t> d_from;
  DevBuf<int32_t> d_face;
  DevBuf<long long> d_out;
  CUDA_TRY(d_pos.alloc(3 * static_cast<size_t>(n))); CUDA_TRY(d_from.alloc(n)); CUDA_TRY(d_out.alloc(n));
  CUDA_TRY(cudaMemcpyAsync(d_pos, pos3, 3 * n * sizeof(double), cudaMemcpyHostToDevice, st));
  CUDA_TRY(cudaMemcpyAsync(d_from, from, n * sizeof(uint32_t), cudaMemcpyHostToDevice, st));
  if (face) {
    CUDA_TRY(d_face.alloc(n));
    CUDA_TRY(cudaMemcpyAsync(d_face, face, n * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  }
  relocate_kernel<<<std::min((n + kBlock - 1) / kBlock, 65535), kBlock, 0, st>>>(ctx->dev, nav, n, d_pos, d_from,
                                                                                 face ? d_face.p : nullptr, d_out);
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaMemcpyAsync(out, d_out, n * sizeof(long long), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  return ADEPT_OK;
}

// ------------------------------------------------------------------------------------------------
// Hybrid-workflow boundary: the host simulation hands tracks over one at
// a time; they are buffered until a threshold triggers synchronous transport of the batch; Flush
// transports what is left; deposits accumulate per volume and the tracks that left the world ("outgoing
// particles") are kept for the caller to put back on its own stack.
struct adept_buffer {
  adept_ctx* ctx = nullptr;
  int slot = 0;
  size_t threshold = 0;
  cudaStream_t stream = nullptr;
  std::vector<uint32_t> event;
  std::vector<uint64_t> id;
  std::vector<int8_t> species;
  std::vector<double> pos, dir, ekin;
  std::vector<double> edep, scratch;       // accumulated per-volume deposits; one batch
  adept_ledger ledger{};
  std::vector<adept_track> outgoing;
  uint64_t batches = 0, tracks_in = 0;
};

extern "C" int adept_buffer_create(adept_buffer** out, adept_ctx* ctx, int slot, size_t threshold, void* stream) {
  if (!out) return fail(ADEPT_EINVAL, "null argument");
  *out = nullptr;
  const int rc = check_slot(ctx, slot);
  if (rc != ADEPT_OK) return rc;
  if (threshold < 1 || threshold > ctx->cfg.track_capacity) return fail(ADEPT_EINVAL, "threshold must be in [1, track_capacity]");
  adept_buffer* b = new adept_buffer;
  b->ctx = ctx; b->slot = slot; b->threshold = threshold; b->stream = static_cast<cudaStream_t>(stream);
  b->edep.assign(ctx->n_vol, 0.0);
  b->scratch.assign(ctx->n_vol, 0.0);
  *out = b;
  return ADEPT_OK;
}

extern "C" int adept_buffer_flush(adept_buffer* b) {
  if (!b) return fail(ADEPT_EINVAL, "null buffer");
  const int n = static_cast<int>(b->ekin.size());
  if (n == 0) return 0;
  int rc = adept_enqueue_batch(b->ctx, b->slot, n, b->event.data(), b->id.data(), b->species.data(), b->pos.data(),
                               b->dir.data(), b->ekin.data());
  if (rc != ADEPT_OK) return rc;
  b->event.clear(); b->id.clear(); b->species.clear(); b->pos.clear(); b->dir.clear(); b->ekin.clear();
  rc = adept_transport(b->ctx, b->slot, b->stream);
  if (rc != ADEPT_OK) return rc;
  adept_ledger led{};
  rc = adept_read_scoring(b->ctx, b->slot, b->scratch.data(), b->scratch.size(), &led, b->stream);
  if (rc != ADEPT_OK) return rc;
  for (size_t v = 0; v < b->edep.size(); ++v) b->edep[v] += b->scratch[v];
  b->ledger.deposited += led.deposited; b->ledger.below_cut += led.below_cut; b->ledger.escaped += led.escaped;
  b->ledger.killed += led.killed; b->ledger.primary += led.primary;
  size_t n_leaked = 0;
  const size_t old = b->outgoing.size();
  b->outgoing.resize(old + b->ctx->cfg.leak_capacity);
  rc = adept_read_leaked(b->ctx, b->slot, b->outgoing.data() + old, b->ctx->cfg.leak_capacity, &n_leaked);
  if (rc != ADEPT_OK) { b->outgoing.resize(old); return rc; }
  b->outgoing.resize(old + std::min<size_t>(n_leaked, b->ctx->cfg.leak_capacity));
  if (n_leaked > b->ctx->cfg.leak_capacity) return fail(ADEPT_EOVERFLOW, "%zu outgoing tracks, leak_capacity is %llu", n_leaked,
                                                        static_cast<unsigned long long>(b->ctx->cfg.leak_capacity));
  b->batches += 1;
  return 1;
}

extern "C" int adept_buffer_add(adept_buffer* b, uint32_t event_id, uint64_t track_id, int species, const double pos[3],
                                const double dir[3], double ekin) {
  if (!b || !pos || !dir) return fail(ADEPT_EINVAL, "null argument");
  if (species < 0 || species > 2) return fail(ADEPT_EINVAL, "unknown species %d", species);
  if (!(ekin >= 0.0)) return fail(ADEPT_EINVAL, "negative or NaN energy");
  b->event.push_back(event_id); b->id.push_back(track_id); b->species.push_back(static_cast<int8_t>(species));
  for (int a = 0; a < 3; ++a) { b->pos.push_back(pos[a]); b->dir.push_back(dir[a]); }
  b->ekin.push_back(ekin);
  b->tracks_in += 1;
  if (b->ekin.size() >= b->threshold) return adept_buffer_flush(b);
  return 0;
}

extern "C" int adept_buffer_pending(const adept_buffer* b, size_t* n_buffered, size_t* n_outgoing, uint64_t* n_batches) {
  if (!b) return fail(ADEPT_EINVAL, "null buffer");
  if (n_buffered) *n_buffered = b->ekin.size();
  if (n_outgoing) *n_outgoing = b->outgoing.size();
  if (n_batches) *n_batches = b->batches;
  return ADEPT_OK;
}

extern "C" int adept_buffer_take(adept_buffer* b, double* edep, size_t n_volumes, adept_ledger* ledger, adept_track* outgoing,
                                 size_t cap, size_t* n_outgoing) {
  if (!b) return fail(ADEPT_EINVAL, "null buffer");
  if (edep && n_volumes != b->edep.size()) return fail(ADEPT_EINVAL, "n_volumes is %zu, geometry has %zu", n_volumes, b->edep.size());
  if (outgoing && b->outgoing.size() > cap) return fail(ADEPT_EINVAL, "%zu outgoing tracks do not fit %zu", b->outgoing.size(), cap);
  if (edep) { std::memcpy(edep, b->edep.data(), n_volumes * sizeof(double)); std::fill(b->edep.begin(), b->edep.end(), 0.0); }
  if (ledger) { *ledger = b->ledger; b->ledger = adept_ledger{}; }
  if (n_outgoing) *n_outgoing = b->outgoing.size();
  if (outgoing) { std::memcpy(outgoing, b->outgoing.data(), b->outgoing.size() * sizeof(adept_track)); b->outgoing.clear(); }
  return ADEPT_OK;
}

extern "C" int adept_buffer_destroy(adept_buffer* b) {
  delete b;
  return ADEPT_OK;
}
