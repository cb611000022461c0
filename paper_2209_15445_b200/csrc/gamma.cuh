// Gamma move kernel, hand-specialised (§8(c) S1).
//
// Same arithmetic, in the same order, as step_move<MODE_GAMMA> (step.cuh), which stays the reference
// implementation behind the frozen-step hook.  What differs is where the track lives: the step kernels
// are bound by instruction latency at 4 resident warps per scheduler (profiles/r1b_summary.md), and the
// resident warps are set by registers.  Here a lane's track stays in its slot of the shared-memory tile
// the TMA pipeline filled and every phase reads only the fields it needs, at the point of use, so nothing
// but the position, the step length and three flags is live across the two navigator phases (which are
// inlined: as calls they cost 4 % of a config-2 pass).  The discrete process is chosen (U1) before the
// propagation -- it depends on nothing the propagation computes -- so neither the cross sections nor
// the Philox state survive phase A.
//
// Two instantiations (adept.cu picks one per host round from the slot's population): MULTI = false takes one
// step per track and launch; MULTI = true lets a lane go on stepping its own track while it stays in the
// gamma buffer (kernels.cuh inner_steps), with the whole state kept in the lane's tile slot between steps.
// The loop costs registers (spills at the 5-block cap) and 2-5 % of a full-GPU pass, hence the lean variant.
#pragma once
#include "kernels.cuh"

namespace adept {

// resident blocks per SM asked of the compiler (measured, profiles/r2_summary.md): without a BVH 6 (80 registers, a few
// bytes of spill; config-2 pass 35.65 -> 35.17 ms over 5 blocks; 7 and 8 blocks: 36.3, 38.2); with the traversal code 4 (128 registers; the gamma kernel of a config-4 pass 134.9 -> 124.0 ms over 5 blocks,
// config 5 32.3 -> 32.9 events/s; 3 blocks: 147.5 ms)
#ifndef ADEPT_MINB_G2
#define ADEPT_MINB_G2 6
#endif
#ifndef ADEPT_MINB_G2B
#define ADEPT_MINB_G2B 4
#endif

// per-thread outcome counters, 10 bits per field, folded into the block tally every 1023 tiles
enum { GC_STEPS = 0, GC_BOUNDARY, GC_ESCAPED, GC_STOPPED, GC_KILLED, GC_PHOTO, GC_N };

__device__ __forceinline__ void gamma_counts_flush(BlockTally& t, unsigned long long& packed) {
  constexpr int which[GC_N] = {-1, ADEPT_OUT_BOUNDARY, ADEPT_OUT_ESCAPED, ADEPT_OUT_STOPPED, ADEPT_OUT_KILLED, ADEPT_OUT_PHOTO};
#pragma unroll
  for (int f = 0; f < GC_N; ++f) {
    const unsigned v = __reduce_add_sync(kFull, static_cast<unsigned>((packed >> (10 * f)) & 1023ull));
    if ((threadIdx.x & 31) == 0 && v) {
      if (f == GC_STEPS) atomicAdd(&t.steps, v);
      else atomicAdd(&t.outcomes[which[f]], v);
    }
  }
  packed = 0;
}

// One gamma step of lane `t` of a tile (phases A-C and the outcome); warp-convergent.  On return `post` is
// the state to store if `live` (dest 0 = next gamma buffer, 1.. = staging queue of the process), and
// (has_pe, T_pe) describe the photoelectron.  MULTI: the post-step position, step count and volume also go
// back into the lane's tile slot (a photon's direction and energy do not change in a move), so that the slot
// is the pre-step state of the lane's next step within this launch.
struct GammaLane {
  Track post;
  double edep, T_pe;
  bool active, live, has_pe;
  int dest;
  uint32_t vol;   // pre-step volume (scoring)
};

template <bool BVH, bool MULTI, int N>
__device__ __forceinline__ void gamma_lane(const DevCtx& c, const DevSlot& slot, BlockTally& tally, TrackTileT<N>& T, int t,
                                           bool in_range, unsigned long long& packed, GammaLane& r, NavCache* cache = nullptr) {
  constexpr int species = ADEPT_GAMMA;
  enum { FATE_NONE = 0, FATE_KILLED, FATE_STOPPED, FATE_GO };
    const uint32_t vol = T.u[2][t];
    const bool active = in_range && vol != kDeadVolume;

    // ---- phase A: step-start rules, physics step limit, process choice (S1, A2)
    int fate = FATE_NONE, process = 0, mat = 0;
    double s_phys = ADEPT_INF;
    if (active) {
      const uint32_t step = T.u[1][t];
      const double T0 = T.d[6][t];
      if (step >= c.max_steps) {
        fate = FATE_KILLED;
      } else if (T0 < kTmin) {
        fate = FATE_STOPPED;
      } else {
        fate = FATE_GO;
        mat = volume(c, vol).material;
        {  // the rows of a vacuum are zero (adept_init), so no material flag has to be read first.
          // Order: the two dependent loads of this phase (material of the volume, then the table rows) are each
          // followed by arithmetic that does not need them -- the grid position and the Philox block, then -ln U0
          // -- so that their latency is covered by the lane's own work (a photon in vacuum computes them in vain).
          const GridPos gp = grid_pos(c, T0);
          Stream u;
          u.init(T.u[0][t], c.seed, T.id[t], step);
          const double u0 = u.uniform(0), u1 = u.uniform(1);
          const double* tab = c.tab_g + (static_cast<size_t>(mat) * kNGrid + gp.i) * kRowG;
          const Row4 r0 = load_row4(tab), r1 = load_row4(tab + kRowG);
          const double nlu0 = -log_pos(u0);
          const double x0 = lerp_col(r0, r1, 0, gp.f);                                 // Compton
          const double x1 = T0 > 2.0 * kMe ? lerp_col(r0, r1, 1, gp.f) : 0.0;          // pair, exact threshold (P2)
          const double se = lerp_col(r0, r1, 2, gp.f);                                 // photoelectric
          const double stot = x0 + x1 + se;
          if (stot > 0.0) {
            s_phys = div_pos(nlu0, stot);
            process = ADEPT_OUT_PHOTO;
            if (u1 * stot < x0) process = ADEPT_OUT_COMPTON;
            else if (u1 * stot < x0 + x1) process = ADEPT_OUT_PAIR;
          }
        }
      }
    }
    const bool go = fate == FATE_GO;

    // ---- phase B: straight-line propagation to min(s_phys, boundary) (A4), push (G5)
    double px = T.d[0][t], py = T.d[1][t], pz = T.d[2][t];
    bool cross = false;
    int face = -1;
    {
      const double dx = T.d[3][t], dy = T.d[4][t], dz = T.d[5][t];
      const double s_geo = nav_distance<BVH>(c, c.navigator, go, px, py, pz, dx, dy, dz, vol, s_phys, face, cache);
      if (go) {
        cross = s_geo < s_phys;
        const double s = cross ? s_geo : s_phys;
        px += s * dx; py += s * dy; pz += s * dz;
        if (cross) { px += c.eps_push * dx; py += c.eps_push * dy; pz += c.eps_push * dz; }
      }
    }
    // ---- phase C: relocation (A5)
    const int nv = nav_relocate<BVH>(c, c.navigator, cross, vol, px, py, pz, face);

    // ---- outcome.  Everything still needed of the track is read from the tile here, before the
    // reservation barriers: after them thread 0 may already refill this tile buffer.
    Track post;
    post.x = px; post.y = py; post.z = pz;
    post.dx = T.d[3][t]; post.dy = T.d[4][t]; post.dz = T.d[5][t];
    post.ekin = T.d[6][t]; post.id = T.id[t];
    post.event = T.u[0][t]; post.step = T.u[1][t] + 1; post.vol = vol; post.species = species;
    double edep = 0.0, T_pe = 0.0;
    bool live = false, has_pe = false;
    int dest = -1;
    if (active) {
      packed += 1ull << (10 * GC_STEPS);
      if (fate == FATE_KILLED) {
        atomicAdd(&tally.ledger[3], post.ekin);
        packed += 1ull << (10 * GC_KILLED);
      } else if (fate == FATE_STOPPED) {
        edep = post.ekin;
        packed += 1ull << (10 * GC_STOPPED);
      } else if (cross) {
        if (nv < 0) {
          atomicAdd(&tally.ledger[2], post.ekin);
          record_leak(c, slot, post, species);
          packed += 1ull << (10 * GC_ESCAPED);
        } else {
          post.vol = static_cast<uint32_t>(nv);
          live = true; dest = 0;
          packed += 1ull << (10 * GC_BOUNDARY);
          if (MULTI && BVH && cache) nav_cache_left_daughter(c, *cache, vol, nv, px, py, pz);
        }
      } else if (process == ADEPT_OUT_PHOTO) {   // P3: no sampling involved, done here rather than staged
        const double BK = photo_binding(c, mat, post.ekin, post.event, post.id, post.step - 1);
        if (post.ekin > BK) {
          edep = BK;
          T_pe = post.ekin - BK;
          if (T_pe < mat_scalar(c, mat, S_TCUT)) edep += T_pe;   // M5: below the production cut
          else has_pe = true;
        } else {
          edep = post.ekin;
        }
        packed += 1ull << (10 * GC_PHOTO);
      } else {                                   // Compton / pair: staged for the interaction kernel
        live = true; dest = 1 + process - ADEPT_OUT_COMPTON;
      }
      if (MULTI) {
        T.d[0][t] = px; T.d[1][t] = py; T.d[2][t] = pz;
        T.u[1][t] = post.step; T.u[2][t] = post.vol;
      }
    }
    r.post = post; r.edep = edep; r.T_pe = T_pe; r.active = active; r.live = live; r.has_pe = has_pe; r.dest = dest; r.vol = vol;
}

// (the body of the kernel, so that the merged move kernel of charged.cuh can run it in the blocks it gives to photons; the
// block's shared memory comes from the kernel)
template <bool BVH, bool MULTI>
__device__ __forceinline__ void gamma_move_body(const DevCtx& c, const DevSlot& slot, int parity, BlockTally& tally, BlockReserve<5>& br,
                                                TilePipe& pipe) {
  constexpr int species = ADEPT_GAMMA;
  const TrackSoA& cur = slot.buf[parity][species];
  SlotCounters* cnt = slot.counters;
  // (a counter can run past the capacity when its queue overflowed: the stores are guarded, the reads clamped)
  const uint32_t n = min(cnt->count[parity][species].v, c.capacity);

  // destinations: 0 = next gamma buffer, 1..3 = Compton / pair / (unused) staging queues, 4 = next
  // electron buffer (photoelectrons)
  constexpr int ND = 5;
  if (blockIdx.x >= (n + kBlock - 1) / kBlock) return;   // no tile for this block (tail of a shower: most blocks)
  tally_init(tally);
  pipe_init(pipe);
  double sum_cut = 0.0;
  unsigned long long packed = 0;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned lt = (1u << lane) - 1u;
  const int t = threadIdx.x;
  int k_inner = MULTI ? min(inner_steps(c, n, gridDim.x * kBlock, ADEPT_INNER_MAX_STRAIGHT), 1023) : 1;
  // full GPU, BVH geometry: only the passage through the gap a track has just entered from a daughter is taken in
  // the same launch (geom.cuh NavCache: the daughter's neighbour list answers its query without a traversal)
  const bool transit_only = MULTI && BVH && k_inner == 1 && c.transit;
  if (transit_only) k_inner = 2;
  NavCache nav_cache;
  nav_cache_reset(nav_cache);
  NavCache* const cache = (MULTI && BVH) ? &nav_cache : nullptr;

  const uint32_t n_tiles = (n + kBlock - 1) / kBlock;
  if (t == 0 && blockIdx.x < n_tiles) tile_issue(pipe.tile[0], cur, blockIdx.x, &pipe.bar[0]);
  uint32_t k = 0;
  for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++k) {
    const int phase = k & 1;
    if (t == 0 && tile + gridDim.x < n_tiles) tile_issue(pipe.tile[phase ^ 1], cur, tile + gridDim.x, &pipe.bar[phase ^ 1]);
    mbar_wait(&pipe.bar[phase], (k >> 1) & 1);
    GammaLane r;
    if (!MULTI) {
      gamma_lane<BVH, false>(c, slot, tally, pipe.tile[phase], t, tile * kBlock + t < n, packed, r);
      score(slot, r.vol, r.edep, r.active);
      sum_cut += r.edep;
      if ((k & 1023u) == 1022u) gamma_counts_flush(tally, packed);
    } else {
      // A lane steps its track until it leaves the gamma buffer (interaction, absorption, escape, ...) or has
      // taken k_inner steps; the warp goes round together because the navigator is warp-convergent.  A lane
      // that is done keeps the result of its last step in `r`.
      bool cont = tile * kBlock + t < n;
      for (int it = 0;; ++it) {
        GammaLane q;
        gamma_lane<BVH, true>(c, slot, tally, pipe.tile[phase], t, cont, packed, q, cache);
        score(slot, q.vol, q.edep, q.active);
        sum_cut += q.edep;
        if (q.active || it == 0) r = q;
        cont = q.active && q.live && q.dest == 0 && it + 1 < k_inner;
        if (transit_only) cont = cont && nav_cache.reach > 0.0 && nav_cache.vol == q.post.vol;
        if (!__any_sync(kFull, cont)) break;
      }
      gamma_counts_flush(tally, packed);
      fence_proxy_async_smem();   // the tile writes (generic proxy) before the TMA refill of this buffer
    }
    Track post = r.post;
    const double T_pe = r.T_pe;
    const bool live = r.live, has_pe = r.has_pe;
    const int dest = r.dest;

    // ---- reservation and stores (A0)
    uint32_t pre = 0;
#pragma unroll
    for (int d = 0; d < 4; ++d) {
      const unsigned b = __ballot_sync(kFull, dest == d);
      if (dest == d) pre = __popc(b & lt);
      if (lane == 0) br.wtot[phase][warp][d] = __popc(b);
    }
    const unsigned bpe = __ballot_sync(kFull, has_pe);
    const uint32_t pre_pe = __popc(bpe & lt);
    if (lane == 0) {
      br.wtot[phase][warp][4] = __popc(bpe);
      if (bpe) atomicAdd(&tally.secondaries[ADEPT_ELECTRON], static_cast<unsigned>(__popc(bpe)));
    }
    block_reserve_commit<ND>(br, phase, [&](int d) -> uint32_t* {
      if (d == 0) return &cnt->count[parity ^ 1][species].v;
      if (d == 4) return &cnt->count[parity ^ 1][ADEPT_ELECTRON].v;
      return &cnt->n_stage[d - 1].v;
    });
    if (live) {
      const uint32_t j = br.wbase[phase][warp][dest] + pre;
      const bool staged = dest != 0;
      const TrackSoA& dst = staged ? slot.stage[dest - 1] : slot.buf[parity ^ 1][species];
      if (j < (staged ? c.stage_capacity : c.capacity)) store_track(dst, j, post);
      else cnt->overflow.v = 1;
    }
    if (has_pe) {   // photoelectron along the photon direction, child 0 of this step's stream (R3)
      const uint32_t j = br.wbase[phase][warp][4] + pre_pe;
      Stream u;
      u.init(post.event, c.seed, post.id, post.step - 1);
      post.ekin = T_pe; post.id = u.child_id(0); post.step = 0; post.species = ADEPT_ELECTRON;
      if (j < c.capacity) store_track(slot.buf[parity ^ 1][ADEPT_ELECTRON], j, post);
      else cnt->overflow.v = 1;
    }
  }
  gamma_counts_flush(tally, packed);
  tally_flush(tally, slot, species, 0.0, sum_cut);
}

template <bool BVH, bool MULTI>
__global__ void __launch_bounds__(kBlock, BVH ? ADEPT_MINB_G2B : ADEPT_MINB_G2)
gamma_move_kernel(const __grid_constant__ DevCtx c, const __grid_constant__ DevSlot slot, int parity) {
  __shared__ BlockTally tally;
  __shared__ BlockReserve<5> br;
  __shared__ TilePipe pipe;
  gamma_move_body<BVH, MULTI>(c, slot, parity, tally, br, pipe);
}

}  // namespace adept
