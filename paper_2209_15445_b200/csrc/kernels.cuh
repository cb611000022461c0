// Transport kernels: population stepping over per-species SoA track buffers  (SURVEY.md §8 rows A0,
// A9, A10).  Differences from the paper's design: the per-species
// "current/next" arrays hold the track records themselves (SoA, ping-pong) instead of indices into
// an append-only store, so every read and write of track state is coalesced and finished slots are
// reclaimed every step; survivors and secondaries are appended with warp-aggregated atomics.
#pragma once
#include "step.cuh"

namespace adept {

constexpr int kBlock = 128;
// minimum resident blocks per SM asked of the compiler (register caps chosen from measurement)
#ifndef ADEPT_MINB_G
#define ADEPT_MINB_G 4
#endif
#ifndef ADEPT_MINB_C
#define ADEPT_MINB_C 3
#endif
#ifndef ADEPT_MINB_I
#define ADEPT_MINB_I 6
#endif

__device__ __forceinline__ Track load_track(const TrackSoA& b, uint32_t i, int species) {
  Track t;
  t.x = b.x[i]; t.y = b.y[i]; t.z = b.z[i];
  t.dx = b.dx[i]; t.dy = b.dy[i]; t.dz = b.dz[i];
  t.ekin = b.ekin[i]; t.id = b.id[i];
  t.event = b.event[i]; t.step = b.step[i]; t.vol = b.vol[i];
  t.species = species;
  return t;
}

__device__ __forceinline__ void store_track(const TrackSoA& b, uint32_t i, const Track& t) {
  b.x[i] = t.x; b.y[i] = t.y; b.z[i] = t.z;
  b.dx[i] = t.dx; b.dy[i] = t.dy; b.dz[i] = t.dz;
  b.ekin[i] = t.ekin; b.id[i] = t.id;
  b.event[i] = t.event; b.step[i] = t.step; b.vol[i] = t.vol;
}

// Warp-aggregated append (A0): lanes with `want` get consecutive slots of `counter`; one atomic per warp.
__device__ __forceinline__ uint32_t warp_append(uint32_t* counter, bool want) {
  const unsigned m = __ballot_sync(kFull, want);
  if (m == 0) return 0;
  const int lane = threadIdx.x & 31;
  const int leader = __ffs(m) - 1;
  uint32_t base = 0;
  if (lane == leader) base = atomicAdd(counter, __popc(m));
  base = __shfl_sync(kFull, base, leader);
  return base + __popc(m & ((1u << lane) - 1u));
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
  return v;
}

// A9: warp-reduced scoring.  Lanes depositing into the same volume are combined (match_any) and the
// group leader issues one fp64 atomic; with 100 scoring slabs most warps issue 1-3 atomics.
__device__ __forceinline__ void score(double* edep, uint32_t vol, double e, bool active) {
  const bool has = active && e != 0.0;
  const unsigned hm = __ballot_sync(kFull, has);
  if (hm == 0 || !has) return;                      // lanes without a deposit take no part
  const unsigned peers = __match_any_sync(hm, vol);
  const int lane = threadIdx.x & 31;
  double sum = 0.0;
  unsigned m = peers;
  while (m) {  // sum over the group (groups are disjoint; every lane walks its own peer mask)
    const int src = __ffs(m) - 1;
    m &= m - 1;
    sum += __shfl_sync(peers, e, src);
  }
  if (lane == __ffs(peers) - 1) atomicAdd(edep + vol, sum);
}

struct BlockTally {
  double ledger[4];                       // deposited, below_cut, escaped, killed
  unsigned long long steps, chords;
  unsigned long long outcomes[ADEPT_N_OUTCOMES];
  unsigned long long secondaries[3];
  unsigned int touched;
};

// per-thread partial sums, folded into the block tally at the end of the kernel
struct LaneTally {
  double dep = 0.0, cut = 0.0, esc = 0.0, kill = 0.0;
  unsigned steps = 0, chords = 0;
};

__device__ __forceinline__ void flush_tally(BlockTally& tally, const LaneTally& l, const DevSlot& slot, int species) {
  const int lane = threadIdx.x & 31;
  const double dep = warp_sum(l.dep), cut = warp_sum(l.cut), esc = warp_sum(l.esc), kill = warp_sum(l.kill);
  if (lane == 0) {
    if (dep != 0.0) atomicAdd(&tally.ledger[0], dep);
    if (cut != 0.0) atomicAdd(&tally.ledger[1], cut);
    if (esc != 0.0) atomicAdd(&tally.ledger[2], esc);
    if (kill != 0.0) atomicAdd(&tally.ledger[3], kill);
  }
  if (l.steps) {
    atomicAdd(&tally.steps, static_cast<unsigned long long>(l.steps));
    atomicAdd(&tally.chords, static_cast<unsigned long long>(l.chords));
  }
  __syncthreads();
  if (threadIdx.x == 0 && tally.touched) {
    for (int k = 0; k < 4; ++k) if (tally.ledger[k] != 0.0) atomicAdd(slot.ledger + k, tally.ledger[k]);
    if (tally.steps) atomicAdd(&slot.stats->steps[species], tally.steps);
    if (tally.chords) atomicAdd(&slot.stats->chords, tally.chords);
    for (int k = 0; k < ADEPT_N_OUTCOMES; ++k) if (tally.outcomes[k]) atomicAdd(&slot.stats->outcomes[k], tally.outcomes[k]);
    for (int k = 0; k < 3; ++k) if (tally.secondaries[k]) atomicAdd(&slot.stats->secondaries[k], tally.secondaries[k]);
  }
}

// Appends the secondaries of a step to the next buffers.  All six (k, species) groups of the warp are
// reserved in ONE round of atomics (lane sp adds the warp's total for species sp), so a warp waits for
// a single atomic latency.  Warp-convergent.  `u` is the parent's stream (child ids, R3).
__device__ __forceinline__ void append_secondaries(const DevCtx& c, const DevSlot& slot, int parity, bool active,
                                                   uint32_t event, const Stream& u, const StepOut& o, BlockTally& tally) {
  SlotCounters* cnt = slot.counters;
  const int s0 = (active && o.n_sec > 0) ? o.sec[0].species : -1;
  const int s1 = (active && o.n_sec > 1) ? o.sec[1].species : -1;
  if (__ballot_sync(kFull, s0 >= 0) == 0) return;        // sec[1] exists only with sec[0]
  const int lane = threadIdx.x & 31;
  const unsigned lt = (1u << lane) - 1u;
  unsigned m0[3], m1[3];
#pragma unroll
  for (int sp = 0; sp < 3; ++sp) { m0[sp] = __ballot_sync(kFull, s0 == sp); m1[sp] = __ballot_sync(kFull, s1 == sp); }
  uint32_t mine = 0;
  if (lane < 3) {
    const unsigned n = __popc(lane == 0 ? m0[0] : lane == 1 ? m0[1] : m0[2]) + __popc(lane == 0 ? m1[0] : lane == 1 ? m1[1] : m1[2]);
    if (n) { mine = atomicAdd(&cnt->count[parity ^ 1][lane], n); atomicAdd(&tally.secondaries[lane], static_cast<unsigned long long>(n)); }
  }
  uint32_t base[3];
#pragma unroll
  for (int sp = 0; sp < 3; ++sp) base[sp] = __shfl_sync(kFull, mine, sp);
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    const int ss = k == 0 ? s0 : s1;
    if (ss < 0) continue;
    const uint32_t j = k == 0 ? base[ss] + __popc(m0[ss] & lt) : base[ss] + __popc(m0[ss]) + __popc(m1[ss] & lt);
    if (j < c.capacity) {
      Track s;
      s.x = o.post.x; s.y = o.post.y; s.z = o.post.z;
      s.dx = o.sec[k].dx; s.dy = o.sec[k].dy; s.dz = o.sec[k].dz;
      s.ekin = o.sec[k].ekin; s.id = u.child_id(o.sec[k].child); s.event = event; s.step = 0; s.vol = o.post.vol; s.species = ss;
      store_track(slot.buf[parity ^ 1][ss], j, s);
    } else {
      cnt->overflow = 1;
    }
  }
}

__device__ __forceinline__ void record_leak(const DevCtx& c, const DevSlot& slot, const Track& t, int species) {
  const uint32_t j = atomicAdd(&slot.counters->n_leaked, 1u);
  if (j < c.leak_capacity) {
    adept_track& L = slot.leaked[j];
    L.pos[0] = t.x; L.pos[1] = t.y; L.pos[2] = t.z;
    L.dir[0] = t.dx; L.dir[1] = t.dy; L.dir[2] = t.dz;
    L.ekin = t.ekin; L.id = t.id; L.event = t.event; L.step = t.step; L.volume = kDeadVolume;
    L.species = species;
  }
}

// ------------------------------------------------------------------------------------------------
// Fused mode: one kernel per species group does the whole step.  grid.y = species of a charged launch.
template <int MODE>
__global__ void __launch_bounds__(kBlock) step_kernel(const __grid_constant__ DevCtx c, const __grid_constant__ DevSlot slot,
                                                      int parity) {
  const int species = MODE == MODE_GAMMA ? ADEPT_GAMMA : static_cast<int>(blockIdx.y);
  const TrackSoA& cur = slot.buf[parity][species];
  SlotCounters* cnt = slot.counters;
  const uint32_t n = cnt->count[parity][species];

  __shared__ BlockTally tally;
  if (threadIdx.x == 0) tally = BlockTally{};
  __syncthreads();
  LaneTally lt;

  const uint32_t n_round = (n + 31u) & ~31u;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_round; i += gridDim.x * blockDim.x) {
    bool active = i < n;
    Track in{};
    if (active) in = load_track(cur, i, species);
    in.species = species;
    active = active && in.vol != kDeadVolume;
    StepOut o;
    step_track<MODE>(c, c.navigator, active, in, o);

    score(slot.edep, in.vol, o.edep_dep + o.edep_cut, active);
    if (active) {
      lt.dep += o.edep_dep; lt.cut += o.edep_cut; lt.esc += o.escaped; lt.kill += o.killed;
      ++lt.steps; lt.chords += o.chords;
      atomicAdd(&tally.outcomes[o.outcome], 1ull);
      tally.touched = 1;
    }
    const bool live = active && o.alive;
    const uint32_t j = warp_append(&cnt->count[parity ^ 1][species], live);
    if (live) {
      if (j < c.capacity) store_track(slot.buf[parity ^ 1][species], j, o.post);
      else cnt->overflow = 1;
    }
    Stream u;
    u.init(in.event, c.seed, in.id, in.step);
    append_secondaries(c, slot, parity, active, in.event, u, o, tally);
    if (active && o.outcome == ADEPT_OUT_ESCAPED) { o.post.step = in.step + 1; record_leak(c, slot, o.post, species); }
  }
  flush_tally(tally, lt, slot, species);
}

// ------------------------------------------------------------------------------------------------
// Split mode: move kernels leave relocation and interactions to their own kernels.
//   reloc_queue entry: species << 30 | index into the next buffer of that species
//   inter_queue[q][k]: same encoding, q = 0 Compton, 1 pair, 2 photoelectric, 3 brems, 4 Moller, 5 annihilation, 6 Bhabha
constexpr int kNumInterQueues = 7;

__device__ __forceinline__ int inter_queue_index(int process, int species) {
  return (process == ADEPT_OUT_IONI && species == ADEPT_POSITRON) ? 6 : process - 1;
}
__device__ __forceinline__ int inter_queue_process(int q) { return q == 6 ? ADEPT_OUT_IONI : q + 1; }

template <int MODE, int FIELD, bool BVH>
__global__ void __launch_bounds__(kBlock, MODE == MODE_GAMMA ? ADEPT_MINB_G : ADEPT_MINB_C) move_kernel(const __grid_constant__ DevCtx c, const __grid_constant__ DevSlot slot,
                                                      int parity) {
  const int species = MODE == MODE_GAMMA ? ADEPT_GAMMA : static_cast<int>(blockIdx.y);
  const TrackSoA& cur = slot.buf[parity][species];
  SlotCounters* cnt = slot.counters;
  const uint32_t n = cnt->count[parity][species];

  __shared__ BlockTally tally;
  if (threadIdx.x == 0) tally = BlockTally{};
  __syncthreads();
  LaneTally lt;

  const uint32_t n_round = (n + 31u) & ~31u;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_round; i += gridDim.x * blockDim.x) {
    bool active = i < n;
    Track in{};
    if (active) in = load_track(cur, i, species);
    in.species = species;
    active = active && in.vol != kDeadVolume;
    StepOut o;
    Stream u;
    int process, mat;
    const int next = step_move<MODE, FIELD, BVH>(c, c.navigator, active, in, o, u, process, mat);

    score(slot.edep, in.vol, o.edep_dep + o.edep_cut, active);
    if (active) {
      lt.dep += o.edep_dep; lt.cut += o.edep_cut; lt.kill += o.killed;
      ++lt.steps; lt.chords += o.chords;
      if (next == NEXT_NONE) atomicAdd(&tally.outcomes[o.outcome], 1ull);
      tally.touched = 1;
    }
    // One round of atomics reserves everything this warp appends: lane 0 the survivor slots, lane 1 the
    // relocation-queue entries, lanes 2.. the entries of the process queues this kernel feeds.
    const bool live = active && o.alive;
    constexpr int kQ0 = MODE == MODE_GAMMA ? 0 : 3, kNQ = MODE == MODE_GAMMA ? 3 : 4;
    const int q = (live && next == NEXT_INTERACT) ? inter_queue_index(process, species) - kQ0 : -1;
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    const unsigned m_live = __ballot_sync(kFull, live);
    const unsigned m_rel = __ballot_sync(kFull, live && next == NEXT_RELOCATE);
    unsigned m_q[kNQ];
#pragma unroll
    for (int qq = 0; qq < kNQ; ++qq) m_q[qq] = __ballot_sync(kFull, q == qq);
    uint32_t mine = 0;
    if (lane == 0) { if (m_live) mine = atomicAdd(&cnt->count[parity ^ 1][species], __popc(m_live)); }
    else if (lane == 1) { if (m_rel) mine = atomicAdd(&cnt->n_reloc, __popc(m_rel)); }
    else if (lane < 2 + kNQ) {
      unsigned mq = 0;
#pragma unroll
      for (int qq = 0; qq < kNQ; ++qq) if (lane == 2 + qq) mq = m_q[qq];
      if (mq) mine = atomicAdd(&cnt->n_inter[kQ0 + lane - 2], __popc(mq));
    }
    const uint32_t j = __shfl_sync(kFull, mine, 0) + __popc(m_live & lt);
    const uint32_t k_rel = __shfl_sync(kFull, mine, 1) + __popc(m_rel & lt);
    uint32_t k_q = 0;
#pragma unroll
    for (int qq = 0; qq < kNQ; ++qq) {
      const uint32_t bq = __shfl_sync(kFull, mine, 2 + qq);
      if (q == qq) k_q = bq + __popc(m_q[qq] & lt);
    }
    if (live) {
      o.post.step = in.step + 1;
      if (j < c.capacity) {
        store_track(slot.buf[parity ^ 1][species], j, o.post);
        const uint32_t entry = (static_cast<uint32_t>(species) << 30) | j;
        if (next == NEXT_RELOCATE) slot.reloc_queue[k_rel] = entry;
        else if (q >= 0) slot.inter_queue[static_cast<size_t>(kQ0 + q) * c.capacity + k_q] = entry;
      } else {
        cnt->overflow = 1;
      }
    }
    append_secondaries(c, slot, parity, active, in.event, u, o, tally);   // at-rest annihilation photons
  }
  flush_tally(tally, lt, slot, species);
}

template <bool BVH>
__global__ void __launch_bounds__(kBlock) relocate_kernel(const __grid_constant__ DevCtx c, const __grid_constant__ DevSlot slot,
                                                          int parity) {
  SlotCounters* cnt = slot.counters;
  const uint32_t n = cnt->n_reloc;
  __shared__ BlockTally tally;
  if (threadIdx.x == 0) tally = BlockTally{};
  __syncthreads();
  LaneTally lt;
  const uint32_t n_round = (n + 31u) & ~31u;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_round; i += gridDim.x * blockDim.x) {
    const bool active = i < n;
    uint32_t entry = 0;
    if (active) entry = slot.reloc_queue[i];
    const int species = entry >> 30;
    const uint32_t j = entry & 0x3fffffffu;
    const TrackSoA& b = slot.buf[parity ^ 1][species];
    double x = 0.0, y = 0.0, z = 0.0;
    if (active) { x = b.x[j]; y = b.y[j]; z = b.z[j]; }
    const int nv = nav_locate<BVH>(c, c.navigator, active, x, y, z);
    if (!active) continue;
    tally.touched = 1;
    if (nv >= 0) {
      b.vol[j] = static_cast<uint32_t>(nv);
      atomicAdd(&tally.outcomes[ADEPT_OUT_BOUNDARY], 1ull);
    } else {
      Track t = load_track(b, j, species);
      b.vol[j] = kDeadVolume;
      lt.esc += carried_energy(species, t.ekin);
      record_leak(c, slot, t, species);
      atomicAdd(&tally.outcomes[ADEPT_OUT_ESCAPED], 1ull);
    }
  }
  {
    const int lane = threadIdx.x & 31;
    const double esc = warp_sum(lt.esc);
    if (lane == 0 && esc != 0.0) atomicAdd(&tally.ledger[2], esc);
    __syncthreads();
    if (threadIdx.x == 0 && tally.touched) {
      if (tally.ledger[2] != 0.0) atomicAdd(slot.ledger + 2, tally.ledger[2]);
      if (tally.outcomes[ADEPT_OUT_BOUNDARY]) atomicAdd(&slot.stats->outcomes[ADEPT_OUT_BOUNDARY], tally.outcomes[ADEPT_OUT_BOUNDARY]);
      if (tally.outcomes[ADEPT_OUT_ESCAPED]) atomicAdd(&slot.stats->outcomes[ADEPT_OUT_ESCAPED], tally.outcomes[ADEPT_OUT_ESCAPED]);
    }
  }
}

// Every warp works on one process queue at a time, so the rejection loops of different processes never
// share a warp (PAPER.md:101 names divergence between processes as a main cost).
__global__ void __launch_bounds__(kBlock, ADEPT_MINB_I) interact_kernel(const __grid_constant__ DevCtx c, const __grid_constant__ DevSlot slot,
                                                          int parity) {
  SlotCounters* cnt = slot.counters;
  __shared__ BlockTally tally;
  __shared__ uint32_t warp_begin[kNumInterQueues + 1];   // prefix of 32-lane groups per queue
  if (threadIdx.x == 0) {
    tally = BlockTally{};
    uint32_t acc = 0;
    for (int q = 0; q < kNumInterQueues; ++q) { warp_begin[q] = acc; acc += (cnt->n_inter[q] + 31u) >> 5; }
    warp_begin[kNumInterQueues] = acc;
  }
  __syncthreads();
  LaneTally lt;
  const int lane = threadIdx.x & 31;
  const uint32_t warps_per_grid = gridDim.x * (blockDim.x >> 5);
  const uint32_t total = warp_begin[kNumInterQueues];
  for (uint32_t w = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); w < total; w += warps_per_grid) {
    int q = 0;
    while (w >= warp_begin[q + 1]) ++q;
    const uint32_t i = ((w - warp_begin[q]) << 5) + lane;
    const bool active = i < cnt->n_inter[q];
    StepOut o;
    Stream u;
    Track t{};
    uint32_t j = 0;
    int species = 0;
    if (active) {
      const uint32_t entry = slot.inter_queue[static_cast<size_t>(q) * c.capacity + i];
      species = entry >> 30;
      j = entry & 0x3fffffffu;
      t = load_track(slot.buf[parity ^ 1][species], j, species);
      init_out(o, t, true);
      u.init(t.event, c.seed, t.id, t.step - 1);          // the stream of the step that chose the process
      const int mat = volume(c, t.vol).material;
      run_process(c, inter_queue_process(q), species, mat, o, u);
      const TrackSoA& b = slot.buf[parity ^ 1][species];
      if (o.alive) { b.dx[j] = o.post.dx; b.dy[j] = o.post.dy; b.dz[j] = o.post.dz; b.ekin[j] = o.post.ekin; }
      else b.vol[j] = kDeadVolume;
      lt.cut += o.edep_cut;
      atomicAdd(&tally.outcomes[o.outcome], 1ull);
      tally.touched = 1;
    } else {
      init_out(o, t, false);
      u.init(0, 0, 0, 0);
    }
    score(slot.edep, t.vol, o.edep_cut, active);
    append_secondaries(c, slot, parity, active, t.event, u, o, tally);
  }
  flush_tally(tally, lt, slot, 0);
}

// End of one population step: the just-consumed buffers become the next step's output buffers.
__global__ void finish_iteration_kernel(const __grid_constant__ DevSlot slot, int parity) {
  SlotCounters* cnt = slot.counters;
  const uint32_t before = cnt->count[parity][0] + cnt->count[parity][1] + cnt->count[parity][2];
  cnt->count[parity][0] = cnt->count[parity][1] = cnt->count[parity][2] = 0;
  const uint32_t live = cnt->count[parity ^ 1][0] + cnt->count[parity ^ 1][1] + cnt->count[parity ^ 1][2];
  cnt->live = live;
  cnt->n_reloc = 0;
  for (int q = 0; q < 8; ++q) cnt->n_inter[q] = 0;
  if (before) {
    slot.stats->iterations += 1;
    if (before > slot.stats->peak_population) slot.stats->peak_population = before;
  }
}

// Places primaries (G5: volume = Locate(p + eps d)) and appends them to the parity-0 buffers.
__global__ void __launch_bounds__(kBlock) enqueue_kernel(const __grid_constant__ DevCtx c, const __grid_constant__ DevSlot slot,
                                                         const adept_track* __restrict__ prim, int n, uint32_t* bad) {
  const int n_round = (n + 31) & ~31;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_round; i += gridDim.x * blockDim.x) {
    const bool active = i < n;
    adept_track p{};
    if (active) p = prim[i];
    const int v = nav_locate(c, c.navigator, active, p.pos[0] + c.eps_push * p.dir[0], p.pos[1] + c.eps_push * p.dir[1],
                             p.pos[2] + c.eps_push * p.dir[2]);
    if (active && (v < 0 || p.species < 0 || p.species > 2)) { atomicAdd(bad, 1u); continue; }
    if (!active) continue;
    const uint32_t j = atomicAdd(&slot.counters->count[0][p.species], 1u);
    if (j >= c.capacity) { slot.counters->overflow = 1; continue; }
    Track t;
    t.x = p.pos[0]; t.y = p.pos[1]; t.z = p.pos[2]; t.dx = p.dir[0]; t.dy = p.dir[1]; t.dz = p.dir[2];
    t.ekin = p.ekin; t.id = p.id; t.event = p.event; t.step = 0; t.vol = static_cast<uint32_t>(v); t.species = p.species;
    store_track(slot.buf[0][p.species], j, t);
    atomicAdd(slot.ledger + 4, carried_energy(p.species, p.ekin));
    atomicAdd(&slot.counters->live, 1u);
  }
}

// Test hook: exactly one step per track, results in input order.
__global__ void __launch_bounds__(kBlock) frozen_kernel(const __grid_constant__ DevCtx c, const adept_track* __restrict__ in,
                                                        adept_step_result* __restrict__ out, adept_track* __restrict__ sec,
                                                        int n) {
  const int n_round = (n + 31) & ~31;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_round; i += gridDim.x * blockDim.x) {
    const bool active = i < n;
    Track t{};
    if (active) {
      const adept_track& a = in[i];
      t.x = a.pos[0]; t.y = a.pos[1]; t.z = a.pos[2]; t.dx = a.dir[0]; t.dy = a.dir[1]; t.dz = a.dir[2];
      t.ekin = a.ekin; t.id = a.id; t.event = a.event; t.step = a.step; t.vol = a.volume; t.species = a.species;
    }
    StepOut o;
    step_track<MODE_ANY>(c, c.navigator, active, t, o);
    if (!active) continue;
    adept_step_result& r = out[i];
    r.post.pos[0] = o.post.x; r.post.pos[1] = o.post.y; r.post.pos[2] = o.post.z;
    r.post.dir[0] = o.post.dx; r.post.dir[1] = o.post.dy; r.post.dir[2] = o.post.dz;
    r.post.ekin = o.post.ekin; r.post.id = o.post.id; r.post.event = o.post.event; r.post.step = o.post.step;
    r.post.volume = o.post.vol; r.post.species = t.species;
    r.alive = o.alive; r.outcome = o.outcome; r.n_sec = o.n_sec; r.chords = o.chords;
    r.s = o.s; r.edep_dep = o.edep_dep; r.edep_cut = o.edep_cut; r.escaped = o.escaped; r.killed = o.killed;
    Stream u;
    u.init(t.event, c.seed, t.id, t.step);
    for (int k = 0; k < 2; ++k) {
      adept_track& s = sec[2 * i + k];
      s = adept_track{};
      if (k < o.n_sec) {
        s.pos[0] = o.post.x; s.pos[1] = o.post.y; s.pos[2] = o.post.z;
        s.dir[0] = o.sec[k].dx; s.dir[1] = o.sec[k].dy; s.dir[2] = o.sec[k].dz;
        s.ekin = o.sec[k].ekin; s.id = u.child_id(o.sec[k].child); s.event = t.event; s.step = 0;
        s.volume = o.post.vol; s.species = o.sec[k].species;
      }
    }
  }
}

__global__ void __launch_bounds__(kBlock) distance_kernel(const __grid_constant__ DevCtx c, int nav, int n, const double* pos,
                                                          const double* dir, const uint32_t* vol, const double* smax,
                                                          double* out) {
  const int n_round = (n + 31) & ~31;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_round; i += gridDim.x * blockDim.x) {
    const bool a = i < n;
    const int k = a ? i : 0;
    const double r = nav_distance(c, nav, a, pos[3 * k], pos[3 * k + 1], pos[3 * k + 2], dir[3 * k], dir[3 * k + 1],
                                  dir[3 * k + 2], vol[k], smax[k]);
    if (a) out[i] = r;
  }
}

__global__ void __launch_bounds__(kBlock) locate_kernel(const __grid_constant__ DevCtx c, int nav, int n, const double* pos,
                                                        long long* out) {
  const int n_round = (n + 31) & ~31;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_round; i += gridDim.x * blockDim.x) {
    const bool a = i < n;
    const int k = a ? i : 0;
    const int r = nav_locate(c, nav, a, pos[3 * k], pos[3 * k + 1], pos[3 * k + 2]);
    if (a) out[i] = r;
  }
}

}  // namespace adept
