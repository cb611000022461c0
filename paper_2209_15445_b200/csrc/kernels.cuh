// Transport kernels: population stepping over per-species SoA track buffers  (SURVEY.md §8 rows A0,
// A9, A10).  Differences from the paper's design: the per-species
// "current/next" arrays hold the track records themselves (SoA, ping-pong) instead of indices into
// an append-only store, so every read and write of track state is coalesced and finished slots are
// reclaimed every step; survivors and secondaries are appended with warp-aggregated atomics.
#pragma once
#include "step.cuh"

namespace adept {

constexpr int kBlock = 128;

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
  const unsigned peers = __match_any_sync(kFull, has ? vol : kDeadVolume);
  const int lane = threadIdx.x & 31;
  double sum = 0.0;
  unsigned m = peers;
  while (m) {  // sum over the group (groups are disjoint; every lane walks its own peer mask)
    const int src = __ffs(m) - 1;
    m &= m - 1;
    sum += __shfl_sync(peers, e, src);
  }
  if (has && lane == __ffs(peers) - 1) atomicAdd(edep + vol, sum);
}

struct BlockTally {
  double ledger[4];                       // deposited, below_cut, escaped, killed
  unsigned long long steps, chords;
  unsigned long long outcomes[ADEPT_N_OUTCOMES];
  unsigned long long secondaries[3];
};

// Steps every track of one species queue once.  grid.y selects the species of a charged launch.
template <int MODE>
__global__ void __launch_bounds__(kBlock) step_kernel(const __grid_constant__ DevCtx c, const __grid_constant__ DevSlot slot,
                                                      int parity) {
  const int species = MODE == MODE_GAMMA ? ADEPT_GAMMA : static_cast<int>(blockIdx.y);
  const TrackSoA& cur = slot.buf[parity][species];
  SlotCounters* cnt = slot.counters;
  const uint32_t n = cnt->count[parity][species];
  const int lane = threadIdx.x & 31;

  __shared__ BlockTally tally;
  if (threadIdx.x == 0) tally = BlockTally{};
  __syncthreads();

  double l_dep = 0.0, l_cut = 0.0, l_esc = 0.0, l_kill = 0.0;
  unsigned l_steps = 0, l_chords = 0;

  const uint32_t n_round = (n + 31u) & ~31u;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_round; i += gridDim.x * blockDim.x) {
    const bool active = i < n;
    Track in{};
    if (active) in = load_track(cur, i, species);
    in.species = species;
    StepOut o;
    step_track<MODE>(c, c.navigator, active, in, o);

    // scoring (A9) and ledger
    score(slot.edep, in.vol, o.edep_dep + o.edep_cut, active);
    if (active) {
      l_dep += o.edep_dep; l_cut += o.edep_cut; l_esc += o.escaped; l_kill += o.killed;
      ++l_steps; l_chords += o.chords;
      atomicAdd(&tally.outcomes[o.outcome], 1ull);
    }
    // survivors -> next buffer of the same species
    const bool live = active && o.alive;
    {
      const uint32_t j = warp_append(&cnt->count[parity ^ 1][species], live);
      if (live) {
        if (j < c.capacity) store_track(slot.buf[parity ^ 1][species], j, o.post);
        else cnt->overflow = 1;
      }
    }
    // secondaries -> next buffers, one warp-aggregated append per (slot k, species)
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      const int ss = (active && k < o.n_sec) ? o.sec[k].species : -1;
      if (__ballot_sync(kFull, ss >= 0) == 0) continue;
      uint64_t cid = 0;
      if (ss >= 0) {
        Stream u;
        u.init(in.event, c.seed, in.id, in.step);
        cid = u.child_id(o.sec[k].child);
      }
#pragma unroll
      for (int sp = 0; sp < 3; ++sp) {
        const bool want = ss == sp;
        const uint32_t j = warp_append(&cnt->count[parity ^ 1][sp], want);
        if (want) {
          if (j < c.capacity) {
            Track s;
            s.x = o.post.x; s.y = o.post.y; s.z = o.post.z;
            s.dx = o.sec[k].dx; s.dy = o.sec[k].dy; s.dz = o.sec[k].dz;
            s.ekin = o.sec[k].ekin; s.id = cid; s.event = in.event; s.step = 0; s.vol = o.post.vol; s.species = sp;
            store_track(slot.buf[parity ^ 1][sp], j, s);
            atomicAdd(&tally.secondaries[sp], 1ull);
          } else {
            cnt->overflow = 1;
          }
        }
      }
    }
    // outgoing particles
    if (active && o.outcome == ADEPT_OUT_ESCAPED) {
      const uint32_t j = atomicAdd(&cnt->n_leaked, 1u);
      if (j < c.leak_capacity) {
        adept_track& L = slot.leaked[j];
        L.pos[0] = o.post.x; L.pos[1] = o.post.y; L.pos[2] = o.post.z;
        L.dir[0] = o.post.dx; L.dir[1] = o.post.dy; L.dir[2] = o.post.dz;
        L.ekin = o.post.ekin; L.id = in.id; L.event = in.event; L.step = in.step + 1; L.volume = kDeadVolume;
        L.species = species;
      }
    }
  }

  // block-level tallies -> one set of global atomics per block
  l_dep = warp_sum(l_dep); l_cut = warp_sum(l_cut); l_esc = warp_sum(l_esc); l_kill = warp_sum(l_kill);
  if (lane == 0) {
    if (l_dep != 0.0) atomicAdd(&tally.ledger[0], l_dep);
    if (l_cut != 0.0) atomicAdd(&tally.ledger[1], l_cut);
    if (l_esc != 0.0) atomicAdd(&tally.ledger[2], l_esc);
    if (l_kill != 0.0) atomicAdd(&tally.ledger[3], l_kill);
  }
  if (l_steps) { atomicAdd(&tally.steps, static_cast<unsigned long long>(l_steps)); atomicAdd(&tally.chords, static_cast<unsigned long long>(l_chords)); }
  __syncthreads();
  if (threadIdx.x == 0 && tally.steps) {
    for (int k = 0; k < 4; ++k) if (tally.ledger[k] != 0.0) atomicAdd(slot.ledger + k, tally.ledger[k]);
    atomicAdd(&slot.stats->steps[species], tally.steps);
    atomicAdd(&slot.stats->chords, tally.chords);
    for (int k = 0; k < ADEPT_N_OUTCOMES; ++k) if (tally.outcomes[k]) atomicAdd(&slot.stats->outcomes[k], tally.outcomes[k]);
    for (int k = 0; k < 3; ++k) if (tally.secondaries[k]) atomicAdd(&slot.stats->secondaries[k], tally.secondaries[k]);
  }
}

// End of one population step: the just-consumed buffers become the next step's output buffers.
__global__ void finish_iteration_kernel(const __grid_constant__ DevSlot slot, int parity) {
  SlotCounters* cnt = slot.counters;
  const uint32_t before = cnt->count[parity][0] + cnt->count[parity][1] + cnt->count[parity][2];
  cnt->count[parity][0] = cnt->count[parity][1] = cnt->count[parity][2] = 0;
  const uint32_t live = cnt->count[parity ^ 1][0] + cnt->count[parity ^ 1][1] + cnt->count[parity ^ 1][2];
  cnt->live = live;
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
