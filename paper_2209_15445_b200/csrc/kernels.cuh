// Transport kernels: population stepping over per-species SoA track buffers  (SURVEY.md §8 rows A0,
// A9, A10).  Differences from the paper's design: the per-species
// "current/next" arrays hold the track records themselves (SoA, ping-pong) instead of indices into
// an append-only store, so every read and write of track state is coalesced and finished slots are
// reclaimed every step.  A thread block works on tiles of kBlock consecutive tracks; everything a tile
// appends (survivors, staged interactions, secondaries) is reserved with ONE global atomic per
// destination queue and tile, and every queue counter has its own 128 B line.
#pragma once
#include "step.cuh"

namespace adept {

#ifndef ADEPT_BLOCK
#define ADEPT_BLOCK 128
#endif
constexpr int kBlock = ADEPT_BLOCK;
constexpr int kWarps = kBlock / 32;
// minimum resident blocks per SM asked of the compiler (register caps chosen from measurement)
#ifndef ADEPT_MINB_I
#define ADEPT_MINB_I 4   // 128 registers: measured 9.75 ms per config-2 pass against 9.9 (5 blocks) and 10.1 (6, spills)
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

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
  return v;
}

// ------------------------------------------------------------------------------------------------
// A0: tile loads.  A tile is kBlock consecutive entries of a species buffer (or staging queue): eleven
// contiguous SoA slices, fetched by ONE thread with eleven TMA bulk copies (cp.async.bulk, SASS UBLKCP)
// into a double-buffered shared-memory tile that completes on an mbarrier.  The copy of tile k+1 is in
// flight while the block computes tile k, so the HBM latency of the track state is hidden without
// spending registers or occupancy on it.  Buffers are allocated in multiples of kBlock entries, so a
// full tile can always be read (entries past the live count are ignored).
template <int N>
struct alignas(128) TrackTileT {
  double d[7][N];      // x, y, z, dx, dy, dz, ekin
  uint64_t id[N];
  uint32_t u[3][N];    // event, step, vol
  static constexpr uint32_t kBytes = 8u * N * 8u + 3u * N * 4u;
};
using TrackTile = TrackTileT<kBlock>;
constexpr uint32_t kTileBytes = TrackTile::kBytes;
static_assert(sizeof(TrackTile) % 128 == 0 && sizeof(TrackTile) >= kTileBytes, "TrackTile layout");
static_assert(sizeof(TrackTileT<32>) % 128 == 0 && sizeof(TrackTileT<32>) >= TrackTileT<32>::kBytes, "warp tile layout");

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra WAIT_DONE;\n"
      "bra WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_load(void* smem_dst, const void* gmem_src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(smem_dst)),
               "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// issued by one thread: tile `tile` (N entries) of buffer b -> shared tile t, completion on bar
template <int N>
__device__ __forceinline__ void tile_issue(TrackTileT<N>& t, const TrackSoA& b, uint32_t tile, uint64_t* bar) {
  const size_t base = static_cast<size_t>(tile) * N;
  mbar_expect_tx(bar, TrackTileT<N>::kBytes);
  bulk_load(t.d[0], b.x + base, N * 8, bar); bulk_load(t.d[1], b.y + base, N * 8, bar);
  bulk_load(t.d[2], b.z + base, N * 8, bar); bulk_load(t.d[3], b.dx + base, N * 8, bar);
  bulk_load(t.d[4], b.dy + base, N * 8, bar); bulk_load(t.d[5], b.dz + base, N * 8, bar);
  bulk_load(t.d[6], b.ekin + base, N * 8, bar); bulk_load(t.id, b.id + base, N * 8, bar);
  bulk_load(t.u[0], b.event + base, N * 4, bar); bulk_load(t.u[1], b.step + base, N * 4, bar);
  bulk_load(t.u[2], b.vol + base, N * 4, bar);
}

// same for the first g entries of a tile (g a power of two >= 4, so every copy is a multiple of 16 B):
// sparse tiles of a small population (charged.cuh)
__device__ __forceinline__ void tile_issue_n(TrackTile& t, const TrackSoA& b, size_t base, uint32_t g, uint64_t* bar) {
  mbar_expect_tx(bar, g * 76u);
  bulk_load(t.d[0], b.x + base, g * 8, bar); bulk_load(t.d[1], b.y + base, g * 8, bar);
  bulk_load(t.d[2], b.z + base, g * 8, bar); bulk_load(t.d[3], b.dx + base, g * 8, bar);
  bulk_load(t.d[4], b.dy + base, g * 8, bar); bulk_load(t.d[5], b.dz + base, g * 8, bar);
  bulk_load(t.d[6], b.ekin + base, g * 8, bar); bulk_load(t.id, b.id + base, g * 8, bar);
  bulk_load(t.u[0], b.event + base, g * 4, bar); bulk_load(t.u[1], b.step + base, g * 4, bar);
  bulk_load(t.u[2], b.vol + base, g * 4, bar);
}

__device__ __forceinline__ Track tile_read(const TrackTile& t, int k, int species) {
  Track r;
  r.x = t.d[0][k]; r.y = t.d[1][k]; r.z = t.d[2][k];
  r.dx = t.d[3][k]; r.dy = t.d[4][k]; r.dz = t.d[5][k];
  r.ekin = t.d[6][k]; r.id = t.id[k];
  r.event = t.u[0][k]; r.step = t.u[1][k]; r.vol = t.u[2][k];
  r.species = species;
  return r;
}

// generic-proxy writes to a tile must be ordered before the TMA (async proxy) refill of the same buffer
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

struct TilePipe {
  TrackTile tile[2];
  uint64_t bar[2];
};
__device__ __forceinline__ void pipe_init(TilePipe& p) {
  if (threadIdx.x == 0) { mbar_init(&p.bar[0], 1); mbar_init(&p.bar[1], 1); mbar_fence_init(); }
  __syncthreads();
}

// ------------------------------------------------------------------------------------------------
// A0: block-aggregated append.  Every lane asks for cnt[d] (0..3) consecutive entries of destination
// queue d; the block adds its total to each queue counter with one atomic and every lane gets the
// index of its first entry.  Must be called by all threads of the block (two __syncthreads); the
// caller alternates `phase` between consecutive calls so that a fast warp cannot overwrite the
// per-warp totals a slow warp still reads.
template <int ND>
struct BlockReserve {
  uint32_t wtot[2][kWarps][ND];
  uint32_t wbase[2][kWarps][ND];   // first entry of each warp's share
};

// second half: one thread per destination turns the per-warp totals into per-warp bases
template <int ND, typename CounterOf>
__device__ __forceinline__ void block_reserve_commit(BlockReserve<ND>& br, int phase, CounterOf counter_of) {
  __syncthreads();
  if (threadIdx.x < ND) {
    const int d = threadIdx.x;
    uint32_t w[kWarps], tot = 0;
#pragma unroll
    for (int k = 0; k < kWarps; ++k) { w[k] = br.wtot[phase][k][d]; tot += w[k]; }
    uint32_t base = tot ? atomicAdd(counter_of(d), tot) : 0u;
#pragma unroll
    for (int k = 0; k < kWarps; ++k) { br.wbase[phase][k][d] = base; base += w[k]; }
  }
  __syncthreads();
}

template <int ND, typename CounterOf>
__device__ __forceinline__ void block_reserve(BlockReserve<ND>& br, int phase, const uint32_t (&cnt)[ND], uint32_t (&first)[ND],
                                              CounterOf counter_of) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned lt = (1u << lane) - 1u;
  uint32_t pre[ND];
#pragma unroll
  for (int d = 0; d < ND; ++d) {
    const unsigned b0 = __ballot_sync(kFull, cnt[d] & 1u), b1 = __ballot_sync(kFull, cnt[d] & 2u);
    pre[d] = __popc(b0 & lt) + 2 * __popc(b1 & lt);
    if (lane == 0) br.wtot[phase][warp][d] = __popc(b0) + 2 * __popc(b1);
  }
  block_reserve_commit<ND>(br, phase, counter_of);
#pragma unroll
  for (int d = 0; d < ND; ++d) first[d] = br.wbase[phase][warp][d] + pre[d];
}

// Steps a lane may take of its own track within one launch of a move kernel (adept_config::steps_per_launch).
// Automatic choice: one while the species' population fills the lanes of the grid -- a lane that goes on
// stepping leaves the finished lanes of its warp idle -- and more the emptier the GPU is: below a few
// thousand tracks a population step is a chain of dependent launches whose cost does not depend on the
// population, and the tracks that outlive the shower by thousands of steps (e+- spiralling in vacuum, 16
// chords per step) advance one step per launch triple (PAPER.md:91-99 names these idle gaps).  Random
// numbers are keyed by (event, track, step), so the result does not depend on the choice.
#ifndef ADEPT_INNER_MAX
#define ADEPT_INNER_MAX 32
#endif
// e+- in a field and a BVH geometry (configs 4-5), where a looper's step is 16 chords with a traversal each and the
// showers of the other primaries go on beside it: config 4 ms per pass / config 5 events/s (3 resident blocks) with
// 32: 980 / 28.6, 16: 937 / 28.7, 12: 918 / 28.4, 8: 897 / 28.1; with the two-block variant for small populations
// (charged.cuh LOWOCC) 8: 905 / 32.3, 6: 890 / 31.7, 4: 884 / 30.8
#ifndef ADEPT_INNER_MAX_BVH
#define ADEPT_INNER_MAX_BVH 8
#endif
// Photons and field-free e+- do not loop: their long-lived tracks are few steps from an interaction, and a lane that
// holds on to its track keeps the secondaries of the others waiting.  Measured (profiles/r2_summary.md): at most 3
// steps per launch for them, config 1 4.42 -> 3.10 ms, config 2 34.19 -> 33.78 ms per pass (2: 3.19 / 33.73;
// 4: 3.32 / 33.88; 8: 3.98 / 34.06); e+- in a field keep ADEPT_INNER_MAX.
#ifndef ADEPT_INNER_MAX_STRAIGHT
#define ADEPT_INNER_MAX_STRAIGHT 3
#endif
// `cap`: ADEPT_INNER_MAX for e+- in a field (the loopers), ADEPT_INNER_MAX_STRAIGHT for photons and field-free e+-
__device__ __forceinline__ int inner_steps(const DevCtx& c, uint32_t n, uint32_t lanes, int cap = ADEPT_INNER_MAX) {
  if (c.steps_per_launch > 0) return c.steps_per_launch;
  int k = ADEPT_INNER_MAX;
  if (n >= lanes) k = 1;
  else if (n >= lanes / 4) k = 2;
  else if (n >= lanes / 16) k = 4;
  else if (n >= lanes / 64) k = 8;
  else if (n >= lanes / 256) k = 16;
  return min(k, cap);
}

// A9: scoring.  Every depositing lane issues one fp64 reduction (RED.ADD.F64, no return value, so the
// warp does not wait for it).  With 100 scoring slabs all deposits of a calorimeter fall on seven 128 B
// lines, two or three of them hot at the shower maximum, and one L2 slice retires an fp64 atomic on one
// line every ~3.5 cycles: with a single array the atomic unit of the hottest slice was busy 60 % (gamma
// move) and 86 % (charged move) of the kernel time and serialised the two concurrent step kernels.  The
// deposits therefore go to one of several replicas of the array, chosen per warp, which spreads them over
// as many L2 slices; adept_read_scoring folds the replicas in a fixed order.  Combining the lanes of a
// warp by volume first (match_any + shuffles, one atomic per group) was measured 5 % slower per config-2
// pass once the replicas had removed the contention: the ~40 instructions per warp cost more than the
// reductions they save.
__device__ __forceinline__ void score(const DevSlot& slot, uint32_t vol, double e, bool active) {
  if (active && e != 0.0) {
    const uint32_t rep = (blockIdx.x * kWarps + (threadIdx.x >> 5)) & slot.edep_mask;
    atomicAdd(slot.edep + static_cast<size_t>(rep) * slot.edep_stride + vol, e);
  }
}

// Folds the replicas into replica 0 (fixed order, so the result does not depend on scheduling) and
// clears the others.
__global__ void fold_edep_kernel(const __grid_constant__ DevSlot slot, int n_vol) {
  const int v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= n_vol) return;
  double s = slot.edep[v];
  for (uint32_t r = 1; r <= slot.edep_mask; ++r) {
    double* p = slot.edep + static_cast<size_t>(r) * slot.edep_stride + v;
    s += *p;
    *p = 0.0;
  }
  slot.edep[v] = s;
}

// Per-block statistics, folded into the slot's counters once at the end of the kernel.
struct BlockTally {
  double ledger[4];                       // deposited, below_cut, escaped, killed
  unsigned long long chords;
  unsigned int steps;
  unsigned int outcomes[ADEPT_N_OUTCOMES];
  unsigned int secondaries[3];
};

__device__ __forceinline__ void tally_init(BlockTally& t) {
  if (threadIdx.x == 0) t = BlockTally{};
  __syncthreads();
}

// warp-aggregated count of the lanes whose outcome is `which`
__device__ __forceinline__ void tally_outcome(BlockTally& t, bool active, int outcome, int which) {
  const unsigned m = __ballot_sync(kFull, active && outcome == which);
  if (m && (threadIdx.x & 31) == 0) atomicAdd(&t.outcomes[which], static_cast<unsigned>(__popc(m)));
}

__device__ __forceinline__ void tally_flush(BlockTally& t, const DevSlot& slot, int species, double dep, double cut) {
  dep = warp_sum(dep);
  cut = warp_sum(cut);
  if ((threadIdx.x & 31) == 0) {
    if (dep != 0.0) atomicAdd(&t.ledger[0], dep);
    if (cut != 0.0) atomicAdd(&t.ledger[1], cut);
  }
  __syncthreads();
  for (int k = threadIdx.x; k < 32 + ADEPT_N_OUTCOMES; k += kBlock) {   // (one pass for blocks of 64 threads and more)
    if (k < 4) { if (t.ledger[k] != 0.0) atomicAdd(slot.ledger + k, t.ledger[k]); }
    else if (k == 4) { if (t.steps) atomicAdd(&slot.stats->steps[species], static_cast<unsigned long long>(t.steps)); }
    else if (k == 5) { if (t.chords) atomicAdd(&slot.stats->chords, t.chords); }
    else if (k < 6 + 3) { if (t.secondaries[k - 6]) atomicAdd(&slot.stats->secondaries[k - 6], static_cast<unsigned long long>(t.secondaries[k - 6])); }
    else if (k >= 32) {
      if (t.outcomes[k - 32]) atomicAdd(&slot.stats->outcomes[k - 32], static_cast<unsigned long long>(t.outcomes[k - 32]));
    }
  }
}

__device__ __forceinline__ void record_leak(const DevCtx& c, const DevSlot& slot, const Track& t, int species) {
  const uint32_t j = atomicAdd(&slot.counters->n_leaked.v, 1u);
  if (j < c.leak_capacity) {
    adept_track& L = slot.leaked[j];
    L.pos[0] = t.x; L.pos[1] = t.y; L.pos[2] = t.z;
    L.dir[0] = t.dx; L.dir[1] = t.dy; L.dir[2] = t.dz;
    L.ekin = t.ekin; L.id = t.id; L.event = t.event; L.step = t.step; L.volume = kDeadVolume;
    L.species = species;
  }
}

__device__ __forceinline__ Track make_secondary(const StepOut& o, int k, uint32_t event, const Stream& u) {
  Track s;
  s.x = o.post.x; s.y = o.post.y; s.z = o.post.z;
  s.dx = o.sec[k].dx; s.dy = o.sec[k].dy; s.dz = o.sec[k].dz;
  s.ekin = o.sec[k].ekin; s.id = u.child_id(o.sec[k].child); s.event = event; s.step = 0; s.vol = o.post.vol;
  s.species = o.sec[k].species;
  return s;
}

// ------------------------------------------------------------------------------------------------
// Interaction staging queues: see kNumStage in types.cuh.
__device__ __forceinline__ int stage_queue(int process, int species) {
  if (species == ADEPT_GAMMA) return process - ADEPT_OUT_COMPTON;                       // 0, 1, 2
  if (species == ADEPT_ELECTRON) return process == ADEPT_OUT_BREM ? 3 : 4;
  return process == ADEPT_OUT_BREM ? 5 : (process == ADEPT_OUT_IONI ? 6 : 7);
}
__device__ __forceinline__ int stage_process(int q) {
  constexpr int p[kNumStage] = {ADEPT_OUT_COMPTON, ADEPT_OUT_PAIR, ADEPT_OUT_PHOTO, ADEPT_OUT_BREM, ADEPT_OUT_IONI,
                                ADEPT_OUT_BREM, ADEPT_OUT_IONI, ADEPT_OUT_ANNI};
  return p[q];
}
__device__ __forceinline__ int stage_species(int q) { return q < 3 ? ADEPT_GAMMA : (q < 5 ? ADEPT_ELECTRON : ADEPT_POSITRON); }

// Outcome counters of the move kernel, packed one byte per field in a per-thread 64-bit word.
enum { MC_STEPS = 0, MC_BOUNDARY, MC_ESCAPED, MC_STOPPED, MC_KILLED, MC_LOSS, MC_TRUNCATED, MC_PHOTO, MC_N };
__device__ __forceinline__ int move_count_field(int outcome) {
  switch (outcome) {
    case ADEPT_OUT_BOUNDARY: return MC_BOUNDARY;
    case ADEPT_OUT_ESCAPED: return MC_ESCAPED;
    case ADEPT_OUT_STOPPED: return MC_STOPPED;
    case ADEPT_OUT_KILLED: return MC_KILLED;
    case ADEPT_OUT_LOSS: return MC_LOSS;
    case ADEPT_OUT_TRUNCATED: return MC_TRUNCATED;
    default: return MC_PHOTO;
  }
}
__device__ __forceinline__ void move_counts_flush(BlockTally& t, unsigned long long& packed) {
  constexpr int which[MC_N] = {-1, ADEPT_OUT_BOUNDARY, ADEPT_OUT_ESCAPED, ADEPT_OUT_STOPPED, ADEPT_OUT_KILLED, ADEPT_OUT_LOSS,
                               ADEPT_OUT_TRUNCATED, ADEPT_OUT_PHOTO};
#pragma unroll
  for (int f = 0; f < MC_N; ++f) {
    const unsigned v = __reduce_add_sync(kFull, static_cast<unsigned>((packed >> (8 * f)) & 255ull));
    if ((threadIdx.x & 31) == 0 && v) {
      if (f == MC_STEPS) atomicAdd(&t.steps, v);
      else atomicAdd(&t.outcomes[which[f]], v);
    }
  }
  packed = 0;
}

// End of one population step: the just-consumed buffers become the next step's output buffers.  Run by
// the last block of the interaction kernel to finish (ticket counter), so a population step is three
// launches; every other block has completed its appends (they precede its ticket) when this runs.
__device__ __forceinline__ void finish_iteration(const DevCtx& c, const DevSlot& slot, int parity) {
  SlotCounters* cnt = slot.counters;
  const int k = threadIdx.x;
  uint32_t before = 0, live = 0, in_sp[3];
  for (int sp = 0; sp < 3; ++sp) {   // a counter can run past the capacity when its queue overflowed (the stores are guarded)
    in_sp[sp] = min(__ldcg(&cnt->count[parity][sp].v), c.capacity);
    before += in_sp[sp];
    live += min(__ldcg(&cnt->count[parity ^ 1][sp].v), c.capacity);
  }
  __syncthreads();
  if (k < 3) cnt->count[parity][k].v = 0;
  else if (k < 3 + kNumStage) cnt->n_stage[k - 3].v = 0;
  else if (k == 3 + kNumStage) {
    cnt->live.v = live;
    cnt->ticket.v = 0;
    if (before) {
      slot.stats->iterations += 1;
      if (before > slot.stats->peak_population) slot.stats->peak_population = before;
      const uint32_t j = *slot.trace_n;
      if (j < ADEPT_TRACE_CAPACITY) {
        unsigned long long now;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(now));
        slot.trace_t[j] = now; *slot.trace_n = j + 1;
        for (int sp = 0; sp < 3; ++sp) slot.trace_pop[3 * j + sp] = in_sp[sp];
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Interaction kernel: a tile is kBlock staged tracks of ONE queue, so a whole block runs the rejection
// loop of one process (PAPER.md:101 names divergence between processes as a main cost).  The updated
// parent and the secondaries are appended to the next buffers.
__global__ void __launch_bounds__(kBlock, ADEPT_MINB_I)
interact_kernel(const __grid_constant__ DevCtx c, const __grid_constant__ DevSlot slot, int parity) {
  SlotCounters* cnt = slot.counters;
  __shared__ BlockTally tally;
  __shared__ BlockReserve<3> br;
  __shared__ TilePipe pipe;
  __shared__ uint32_t tile_begin[kNumStage + 1];   // prefix of tiles per queue
  __shared__ uint32_t n_staged[kNumStage];
  __shared__ bool is_last;
  uint32_t total = 0;
#pragma unroll
  for (int q = 0; q < kNumStage; ++q) total += (min(__ldcg(&cnt->n_stage[q].v), c.stage_capacity) + kBlock - 1) / kBlock;
  if (blockIdx.x >= total) {   // no tile for this block (tail of a shower: most blocks); it only takes its ticket
    if (threadIdx.x == 0) is_last = atomicAdd(&cnt->ticket.v, 1u) == gridDim.x - 1;
    __syncthreads();
    if (is_last) finish_iteration(c, slot, parity);
    return;
  }
  if (threadIdx.x == 0) {
    uint32_t acc = 0;
    for (int q = 0; q < kNumStage; ++q) {
      const uint32_t nq = min(cnt->n_stage[q].v, c.stage_capacity);
      n_staged[q] = nq;
      tile_begin[q] = acc;
      acc += (nq + kBlock - 1) / kBlock;
    }
    tile_begin[kNumStage] = acc;
  }
  tally_init(tally);
  pipe_init(pipe);
  double sum_cut = 0.0;
  unsigned long long pk_out = 0, pk_sec = 0;
  const auto counts_flush = [&]() {
#pragma unroll
    for (int f = 0; f < 7; ++f) {
      const unsigned v = __reduce_add_sync(kFull, static_cast<unsigned>((pk_out >> (8 * f)) & 255ull));
      if ((threadIdx.x & 31) == 0 && v) atomicAdd(&tally.outcomes[f == 6 ? ADEPT_OUT_CLOSED : ADEPT_OUT_COMPTON + f], v);
    }
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const unsigned v = __reduce_add_sync(kFull, static_cast<unsigned>((pk_sec >> (16 * d)) & 65535ull));
      if ((threadIdx.x & 31) == 0 && v) atomicAdd(&tally.secondaries[d], v);
    }
    pk_out = 0; pk_sec = 0;
  };
  const auto queue_of = [&](uint32_t tile) { int q = 0; while (tile >= tile_begin[q + 1]) ++q; return q; };
  if (threadIdx.x == 0 && blockIdx.x < total) {
    const int q = queue_of(blockIdx.x);
    tile_issue(pipe.tile[0], slot.stage[q], blockIdx.x - tile_begin[q], &pipe.bar[0]);
  }
  uint32_t k = 0;
  for (uint32_t tile = blockIdx.x; tile < total; tile += gridDim.x, ++k) {
    const int phase = k & 1;
    if (threadIdx.x == 0 && tile + gridDim.x < total) {
      const int qn = queue_of(tile + gridDim.x);
      tile_issue(pipe.tile[phase ^ 1], slot.stage[qn], tile + gridDim.x - tile_begin[qn], &pipe.bar[phase ^ 1]);
    }
    const int q = queue_of(tile);
    const uint32_t i = (tile - tile_begin[q]) * kBlock + threadIdx.x;
    const bool active = i < n_staged[q];
    const int species = stage_species(q);
    mbar_wait(&pipe.bar[phase], (k >> 1) & 1);
    StepOut o;
    Stream u;
    Track t = tile_read(pipe.tile[phase], threadIdx.x, species);
    if (active) {
      init_out(o, t, true);
      u.init(t.event, c.seed, t.id, t.step - 1);          // the stream of the step that chose the process
      const int mat = volume(c, t.vol).material;
      run_process(c, stage_process(q), species, mat, o, u);
      sum_cut += o.edep_cut;
    } else {
      t = Track{};
      init_out(o, t, false);
      u.init(0, 0, 0, 0);
    }
    score(slot, t.vol, o.edep_cut, active);
    const int s0 = active ? o.sec[0].species : -1;
    const int s1 = active ? o.sec[1].species : -1;
    const bool live = active && o.alive;
    // per-thread counters: outcomes one byte per field (COMPTON..ANNI -> 0..5, CLOSED -> 6), secondaries
    // 16 bits per species; folded into the block tally every 127 tiles
    if (active) {
      pk_out += 1ull << (8 * (o.outcome == ADEPT_OUT_CLOSED ? 6 : o.outcome - ADEPT_OUT_COMPTON));
      if (s0 >= 0) pk_sec += 1ull << (16 * s0);
      if (s1 >= 0) pk_sec += 1ull << (16 * s1);
    }
    uint32_t want[3], first[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) want[d] = (live && species == d ? 1u : 0u) + (s0 == d ? 1u : 0u) + (s1 == d ? 1u : 0u);
    block_reserve<3>(br, phase, want, first, [&](int d) -> uint32_t* { return &cnt->count[parity ^ 1][d].v; });
    // within a destination the lane's entries are ordered: surviving parent, secondary 0, secondary 1
    const auto sel = [&](int d) { return d == 0 ? first[0] : (d == 1 ? first[1] : first[2]); };
    if (live) {
      const uint32_t j = sel(species);
      if (j < c.capacity) store_track(slot.buf[parity ^ 1][species], j, o.post);
      else cnt->overflow.v = 1;
    }
#pragma unroll
    for (int kk = 0; kk < 2; ++kk) {
      const int ss = kk == 0 ? s0 : s1;
      if (ss < 0) continue;
      const uint32_t j = sel(ss) + ((live && species == ss) ? 1u : 0u) + ((kk == 1 && s0 == ss) ? 1u : 0u);
      if (j < c.capacity) store_track(slot.buf[parity ^ 1][ss], j, make_secondary(o, kk, t.event, u));
      else cnt->overflow.v = 1;
    }
    if (k % 127u == 126u) counts_flush();
  }
  counts_flush();
  tally_flush(tally, slot, 0, 0.0, sum_cut);
  // the last block to get here ends the population step
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    is_last = atomicAdd(&cnt->ticket.v, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (is_last) finish_iteration(c, slot, parity);
}

// Places primaries (G5: volume = Locate(p + eps d)).  pending == nullptr: appends them to the parity-0
// buffers.  Otherwise (staggered injection) stores the located primary i at pending[i]; inject_kernel
// moves it into the population later.
__global__ void __launch_bounds__(kBlock) enqueue_kernel(const __grid_constant__ DevCtx c, const __grid_constant__ DevSlot slot,
                                                         const adept_track* __restrict__ prim, int n, uint32_t* bad,
                                                         adept_track* __restrict__ pending) {
  const int n_round = (n + 31) & ~31;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_round; i += gridDim.x * blockDim.x) {
    const bool active = i < n;
    adept_track p{};
    if (active) p = prim[i];
    const int v = nav_locate(c, c.navigator, active, p.pos[0] + c.eps_push * p.dir[0], p.pos[1] + c.eps_push * p.dir[1],
                             p.pos[2] + c.eps_push * p.dir[2]);
    if (active && (v < 0 || p.species < 0 || p.species > 2)) { atomicAdd(bad, 1u); continue; }
    if (!active) continue;
    if (pending) {
      p.volume = static_cast<uint32_t>(v); p.step = 0;
      pending[i] = p;
      atomicAdd(slot.ledger + 4, carried_energy(p.species, p.ekin));
      continue;
    }
    const uint32_t j = atomicAdd(&slot.counters->count[0][p.species].v, 1u);
    if (j >= c.capacity) { slot.counters->overflow.v = 1; continue; }
    Track t;
    t.x = p.pos[0]; t.y = p.pos[1]; t.z = p.pos[2]; t.dx = p.dir[0]; t.dy = p.dir[1]; t.dz = p.dir[2];
    t.ekin = p.ekin; t.id = p.id; t.event = p.event; t.step = 0; t.vol = static_cast<uint32_t>(v); t.species = p.species;
    store_track(slot.buf[0][p.species], j, t);
    atomicAdd(slot.ledger + 4, carried_energy(p.species, p.ekin));
    atomicAdd(&slot.counters->live.v, 1u);
  }
}

// Staggered injection: appends the pending primaries [first, first + n) to
// the buffers the population step about to start reads (launched before its move kernels on the same
// stream).  One atomic per warp and species.
__global__ void __launch_bounds__(kBlock) inject_kernel(const __grid_constant__ DevCtx c, const __grid_constant__ DevSlot slot,
                                                        int parity, uint32_t first, uint32_t n) {
  const uint32_t n_round = (n + 31u) & ~31u;
  const int lane = threadIdx.x & 31;
  const unsigned lt = (1u << lane) - 1u;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_round; i += gridDim.x * blockDim.x) {
    const bool active = i < n;
    adept_track p{};
    if (active) p = slot.pending[first + i];
    const int sp = active ? p.species : -1;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const unsigned b = __ballot_sync(kFull, sp == d);
      if (!b) continue;
      uint32_t base = 0;
      if (lane == __ffs(b) - 1) base = atomicAdd(&slot.counters->count[parity][d].v, static_cast<uint32_t>(__popc(b)));
      base = __shfl_sync(kFull, base, __ffs(b) - 1);
      if (sp == d) {
        const uint32_t j = base + __popc(b & lt);
        if (j >= c.capacity) { slot.counters->overflow.v = 1; continue; }
        Track t;
        t.x = p.pos[0]; t.y = p.pos[1]; t.z = p.pos[2]; t.dx = p.dir[0]; t.dy = p.dir[1]; t.dz = p.dir[2];
        t.ekin = p.ekin; t.id = p.id; t.event = p.event; t.step = 0; t.vol = p.volume; t.species = d;
        store_track(slot.buf[parity][d], j, t);
      }
    }
  }
}

// Test hook adept_step_population: scatters tracks, taken as given (volume, step, id), into the parity-0
// buffers of an empty slot; their carried energy is the ledger's "primary".
__global__ void __launch_bounds__(kBlock) load_tracks_kernel(const __grid_constant__ DevCtx c, const __grid_constant__ DevSlot slot,
                                                             const adept_track* __restrict__ in, int n) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const adept_track p = in[i];
    const uint32_t j = atomicAdd(&slot.counters->count[0][p.species].v, 1u);
    if (j >= c.capacity) { slot.counters->overflow.v = 1; continue; }
    Track t;
    t.x = p.pos[0]; t.y = p.pos[1]; t.z = p.pos[2]; t.dx = p.dir[0]; t.dy = p.dir[1]; t.dz = p.dir[2];
    t.ekin = p.ekin; t.id = p.id; t.event = p.event; t.step = p.step; t.vol = p.volume; t.species = p.species;
    store_track(slot.buf[0][p.species], j, t);
    atomicAdd(slot.ledger + 4, carried_energy(p.species, p.ekin));
    atomicAdd(&slot.counters->live.v, 1u);
  }
}

// ... and copies the first n[sp] entries of the three buffers of `parity` to out, species after species.
__global__ void __launch_bounds__(kBlock) gather_tracks_kernel(const __grid_constant__ DevSlot slot, int parity, uint32_t n0, uint32_t n1,
                                                               uint32_t n2, adept_track* __restrict__ out) {
  const uint32_t total = n0 + n1 + n2;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < total; i += gridDim.x * blockDim.x) {
    const int sp = i < n0 ? 0 : (i < n0 + n1 ? 1 : 2);
    const uint32_t j = i - (sp == 0 ? 0u : (sp == 1 ? n0 : n0 + n1));
    const Track t = load_track(slot.buf[parity][sp], j, sp);
    adept_track& o = out[i];
    o.pos[0] = t.x; o.pos[1] = t.y; o.pos[2] = t.z; o.dir[0] = t.dx; o.dir[1] = t.dy; o.dir[2] = t.dz;
    o.ekin = t.ekin; o.id = t.id; o.event = t.event; o.step = t.step; o.volume = t.vol; o.species = sp;
  }
}

// Relocation hints (geom.cuh nav_relocate), built once per context: thread (v, f) locates the point
// eps_push outside the centre of face f of box volume v.  Hints are only ever candidates that the
// relocation verifies, so a face whose neighbourhood is not uniform costs speed, never correctness.
__global__ void __launch_bounds__(kBlock) hint_kernel(const __grid_constant__ DevCtx c, int32_t* __restrict__ nbr) {
  const int n = 6 * c.n_vol, n_round = (n + 31) & ~31;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_round; i += gridDim.x * blockDim.x) {
    const int vi = i / 6, f = i - 6 * vi;
    bool active = i < n;
    double g[3] = {0.0, 0.0, 0.0};
    if (active) {
      const DevVolume& v = volume(c, vi);
      active = v.solid == ADEPT_BOX;
      double l[3] = {0.0, 0.0, 0.0};
      l[f >> 1] = (f & 1) ? v.dims[f >> 1] + c.eps_push : -(v.dims[f >> 1] + c.eps_push);
      to_global(c, vi, v, l, g);
    }
    const int r = nav_locate(c, c.navigator, active, g[0], g[1], g[2]);
    if (i < n) nbr[i] = r;   // -1: non-box volume or outside the world
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
    sec[2 * i] = adept_track{};
    sec[2 * i + 1] = adept_track{};
    int n_out = 0;
#pragma unroll
    for (int k = 0; k < 2; ++k) {      // created secondaries, in child order, packed at the front
      if (o.sec[k].species < 0) continue;
      adept_track& s = sec[2 * i + n_out++];
      s.pos[0] = o.post.x; s.pos[1] = o.post.y; s.pos[2] = o.post.z;
      s.dir[0] = o.sec[k].dx; s.dir[1] = o.sec[k].dy; s.dir[2] = o.sec[k].dz;
      s.ekin = o.sec[k].ekin; s.id = u.child_id(o.sec[k].child); s.event = t.event; s.step = 0;
      s.volume = o.post.vol; s.species = o.sec[k].species;
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

// Ray-cast validator of the navigator (Fig. 1): ray i starts at pos[i] along
// dir[i] and is marched boundary by boundary -- distance to boundary (A4), push, relocation (A5), exactly the
// calls a photon step makes -- until it leaves the world or has crossed max_crossings boundaries.
// column[i] = sum of path x density [g/cm^2], crossings[i] = boundaries crossed (-1: start outside the world).
// R = double: the transport path's navigator.  R = float: the single-precision geometry mode.
template <typename R>
__global__ void __launch_bounds__(kBlock) raycast_kernel(const __grid_constant__ DevCtx c, int nav, int n, const double* __restrict__ pos,
                                                         const double* __restrict__ dir, int max_crossings, double* __restrict__ column,
                                                         int32_t* __restrict__ crossings) {
  constexpr bool kDouble = std::is_same<R, double>::value;
  const R eps = kDouble ? static_cast<R>(c.eps_push) : static_cast<R>(kPushF32);
  const int n_round = (n + 31) & ~31;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_round; i += gridDim.x * blockDim.x) {
    const bool a = i < n;
    const int k = a ? i : 0;
    R px = static_cast<R>(pos[3 * k]), py = static_cast<R>(pos[3 * k + 1]), pz = static_cast<R>(pos[3 * k + 2]);
    const R dx = static_cast<R>(dir[3 * k]), dy = static_cast<R>(dir[3 * k + 1]), dz = static_cast<R>(dir[3 * k + 2]);
    int vol = nav_locate<true, R>(c, nav, a, px, py, pz);
    bool alive = a && vol >= 0;
    R col = R(0);
    int nx = alive ? 0 : -1;
    NavCache cache;
    nav_cache_reset(cache);
    while (__any_sync(kFull, alive)) {
      int face;
      const R s = nav_distance<true, R>(c, nav, alive, px, py, pz, dx, dy, dz, alive ? static_cast<uint32_t>(vol) : 0u, Geo<R>::inf(), face,
                                        kDouble ? &cache : nullptr);
      if (alive) {
        col += s * static_cast<R>(mat_scalar(c, Geo<R>::vol(c, vol).material, S_RHO));
        px += s * dx; py += s * dy; pz += s * dz;
        px += eps * dx; py += eps * dy; pz += eps * dz;
      }
      const int nv = nav_relocate<true, R>(c, nav, alive, alive ? static_cast<uint32_t>(vol) : 0u, px, py, pz, face);
      if (alive) {
        ++nx;
        if constexpr (kDouble) { if (nav == ADEPT_NAV_BVH) nav_cache_left_daughter(c, cache, static_cast<uint32_t>(vol), nv, px, py, pz); }
        vol = nv;
        if (nv < 0 || nx >= max_crossings) alive = false;
      }
    }
    if (a) { column[i] = static_cast<double>(col); crossings[i] = nx; }
  }
}

// Test hook for A5: relocation of point i starting from volume from[i] (any volume of the tree).
__global__ void __launch_bounds__(kBlock) relocate_kernel(const __grid_constant__ DevCtx c, int nav, int n, const double* pos,
                                                          const uint32_t* from, const int32_t* face, long long* out) {
  const int n_round = (n + 31) & ~31;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_round; i += gridDim.x * blockDim.x) {
    const bool a = i < n;
    const int k = a ? i : 0;
    const int r = nav_relocate(c, nav, a, from[k], pos[3 * k], pos[3 * k + 1], pos[3 * k + 2], face ? face[k] : -1);
    if (a) out[i] = r;
  }
}

}  // namespace adept
