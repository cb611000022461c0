// Charged (e-/e+) move kernel, hand-specialised (§8(c) S1-S4).
//
// Same arithmetic, in the same order, as step_move<MODE_CHARGED> (step.cuh), which stays the reference
// implementation behind the frozen-step hook.  The generic kernel needs 166 registers, i.e. three
// resident blocks (12 warps) per SM, and at that occupancy it issues 0.39 instructions per cycle and
// scheduler with `wait` (fixed-latency fp64 dependencies) as its top stall (profiles/r1d_summary.md):
// throughput is set by the number of resident warps.  As in gamma.cuh the lane's track stays in its
// slot of the shared-memory tile and is read at the point of use; in addition the lane WRITES its
// post-step direction and energy back into that slot before the relocation call, so the tile is the
// lane's spill space and little is live across the two navigator phases (inlined: calls cost 4-20 %).
// The discrete process is chosen (U1, same Philox block as U0) before the propagation; the MSC draws
// (U2, U3) and the at-rest annihilation draws (U4, U5) are regenerated from the key where they are used.
// As in gamma.cuh there is a lean instantiation (one step per track and launch) and MULTI = true, in which a
// lane goes on stepping its own track while it stays in its species buffer (kernels.cuh inner_steps).
#pragma once
#include "kernels.cuh"

namespace adept {

// resident blocks per SM asked of the compiler: 6 (80 registers) without a field -- measured 1.3 % of a
// config-2 pass over 5 -- and 4 (128 registers) with the chord loop, which spills 700 B at 96 registers
// (config 4: 3.92 -> 3.72 s per pass over 5 blocks; 3 blocks, no spills at all, are no faster)
#ifndef ADEPT_MINB_C2
#define ADEPT_MINB_C2 6
#endif
// fewest lanes per track (as a shift) that take the chord loop in its wide form (field.cuh propagate_wide)
#ifndef ADEPT_WIDE_MIN_SHIFT
#define ADEPT_WIDE_MIN_SHIFT 2
#endif
#ifndef ADEPT_MINB_C2F
#define ADEPT_MINB_C2F 4
#endif
// field + BVH (configs 4-5): 3 blocks (168 registers) for the populations that fill the GPU, and a second
// instantiation with 2 (255 registers, no spills) for the small ones (LOWOCC below).  Measured, config 4 ms per pass /
// config 5 events/s: 4 blocks everywhere 1 012 / 25.9; 3: 980 / 28.6; 2: 972 / 33.1 (with 16 steps per launch);
// 3 and 2 below 262 144 tracks: 904 / 32.3 (below 65 536: 908 / 32.0, below 16 384: 900 / 29.9), all with 8 steps
// per launch (kernels.cuh ADEPT_INNER_MAX_BVH)
#ifndef ADEPT_MINB_C2FB
#define ADEPT_MINB_C2FB 3
#endif
#ifndef ADEPT_MINB_LOW
#define ADEPT_MINB_LOW 2
#endif

// One e-/e+ step of the track in tile slot `t`; warp-convergent.  The post-step direction and energy are written
// into the tile slot (MULTI: position, step count and volume as well, so that the slot is the pre-step state of
// the lane's next step).  On return (px, py, pz, vol_post) complete the post-step state; `live` and `dest` say
// where it goes (0 = next buffer of the species, 1.. = staging queue q0 + dest - 1), `has_ph` that two
// annihilation photons start at the end point.
struct ChargedLane {
  double px, py, pz;
  uint32_t vol_post;
  bool live, has_ph;
  int dest;
};

template <int FIELD, bool BVH, bool MULTI>
__device__ __forceinline__ void charged_lane(const DevCtx& c, const DevSlot& slot, BlockTally& tally, TrackTile& T, int t, bool in_range,
                                             int species, int q0, unsigned long long& packed, double& sum_dep, double& sum_cut,
                                             unsigned& chords_sum, ChargedLane& r, NavCache* cache, int32_t* cand, int wide_shift = 0) {
  enum { FATE_NONE = 0, FATE_KILLED, FATE_STOPPED, FATE_GO };
  const bool positron = species == ADEPT_POSITRON;
    if (MULTI && wide_shift) __syncwarp();   // the slot as the group's first lane left it after the previous step
    const uint32_t vol = T.u[2][t];
    const bool active = in_range && vol != kDeadVolume;

    // ---- phase A: step-start rules, physics step limit (A3), process choice (U1)
    int fate = FATE_NONE, process = 0, mat = 0;
    bool vacuum = true, lim_disc = false, range_out = false;
    double s_phys = 0.0, S = 0.0, R = ADEPT_INF;
    if (active) {
      const uint32_t step = T.u[1][t];
      const double T0 = T.d[6][t];
      if (step >= c.max_steps) {
        fate = FATE_KILLED;
      } else if (T0 < kTmin) {
        fate = FATE_STOPPED;
        mat = volume(c, vol).material;
      } else {
        fate = FATE_GO;
        mat = volume(c, vol).material;
        vacuum = mat_scalar(c, mat, S_VACUUM) != 0.0;
        double x0 = 0.0, x1 = 0.0, sa = 0.0;
        if (!vacuum) {
          const GridPos gp = grid_pos(c, T0);
          if (positron) {
            const double* tab = c.tab_ep + static_cast<size_t>(mat) * kNGrid * kRowEp;
            x0 = interp(tab, kRowEp, 0, gp); x1 = interp(tab, kRowEp, 1, gp); sa = interp(tab, kRowEp, 2, gp);
            S = interp(tab, kRowEp, 3, gp); R = interp(tab, kRowEp, 4, gp);
          } else {
            const double* tab = c.tab_em + (static_cast<size_t>(mat) * kNGrid + gp.i) * kRowEm;
            const Row4 r0 = load_row4(tab), r1 = load_row4(tab + kRowEm);
            x0 = lerp_col(r0, r1, 0, gp.f); x1 = lerp_col(r0, r1, 1, gp.f);
            S = lerp_col(r0, r1, 2, gp.f); R = lerp_col(r0, r1, 3, gp.f);
          }
        }
        const double stot = x0 + x1 + sa;
        double s_disc = ADEPT_INF;
        if (stot > 0.0) {
          Stream u;
          u.init(T.u[0][t], c.seed, T.id[t], step);
          s_disc = div_pos(-log_pos(u.uniform(0)), stot);
          const double u1 = u.uniform(1);
          process = ADEPT_OUT_BREM;
          if (u1 * stot < x0) process = ADEPT_OUT_BREM;
          else if (!positron || u1 * stot < x0 + x1) process = ADEPT_OUT_IONI;
          else process = ADEPT_OUT_ANNI;
        }
        range_out = R <= c.rho_R;
        const double s_loss = range_out ? R : c.alpha_R * R + c.rho_R * (1.0 - c.alpha_R) * (2.0 - c.rho_R / R);
        lim_disc = s_disc < s_loss;
        s_phys = lim_disc ? s_disc : s_loss;
      }
    }
    bool go = fate == FATE_GO;

    // ---- phase B: propagation (A4, A6)
    double px = T.d[0][t], py = T.d[1][t], pz = T.d[2][t];
    double s = 0.0;
    int flag = 0, face = -1;
    double pdx, pdy, pdz;   // push direction
    if (FIELD == ADEPT_FIELD_NONE) {
      // straight line: one geometry query (what propagate() does when the field vanishes)
      const double dx = T.d[3][t], dy = T.d[4][t], dz = T.d[5][t];
      const bool query = go && !(0.0 >= s_phys);
      int f;
      const double s_geo = nav_distance<BVH>(c, c.navigator, query, px, py, pz, dx, dy, dz, vol, s_phys, f, cache, cand);
      if (query) {
        if (s_geo < s_phys) { px += s_geo * dx; py += s_geo * dy; pz += s_geo * dz; s = s_geo; flag = 1; face = f; }
        else { px += s_phys * dx; py += s_phys * dy; pz += s_phys * dz; s = s_phys; }
      }
      pdx = dx; pdy = dy; pdz = dz;
    } else {
      double pos[3] = {px, py, pz}, dir[3] = {T.d[3][t], T.d[4][t], T.d[5][t]}, pushdir[3];
      int chords = 0;
      if (MULTI && wide_shift) {
        // sparse tiles: the 2^wide_shift lanes that share tile slot t take the chord loop of its track together
        // (field.cuh propagate_wide); only the first of them has run phase A
        const double ekin = T.d[6][t];
        __syncwarp();   // every lane of the group has read the slot before its first lane writes the post-step state into it
        const int g0 = (threadIdx.x & 31) & ~((1 << wide_shift) - 1);
        flag = propagate_wide<FIELD, BVH>(c, c.navigator, wide_shift, __shfl_sync(kFull, go, g0), positron ? +1 : -1, ekin, pos, dir, vol,
                                          __shfl_sync(kFull, s_phys, g0), s, chords, pushdir, face, cache, cand);
      } else
      flag = propagate<FIELD, BVH>(c, c.navigator, go, positron ? +1 : -1, T.d[6][t], pos, dir, vol, s_phys, s, chords, pushdir, face,
                                   cache, cand);
      px = pos[0]; py = pos[1]; pz = pos[2];
      pdx = pushdir[0]; pdy = pushdir[1]; pdz = pushdir[2];
      if (go) { T.d[3][t] = dir[0]; T.d[4][t] = dir[1]; T.d[5][t] = dir[2]; chords_sum += chords; }
    }

    // ---- along-step actions (A7): continuous loss, stop test, MSC; the post-step direction and energy
    // go back into the lane's tile slot
    bool cross = go && flag == 1;
    bool ann_rest = false;
    double edep_dep = 0.0, edep_cut = 0.0;
    if (fate == FATE_STOPPED) {
      edep_cut += T.d[6][t];
      T.d[6][t] = 0.0;
      ann_rest = positron;
    }
    if (go) {
      const double T0 = T.d[6][t];
      double dE = 0.0;
      if (!vacuum) {
        if (flag == 0 && !lim_disc && range_out) dE = T0;
        else if (s <= 0.01 * R) dE = S * s;
        else {
          const double* tab = positron ? c.tab_ep + static_cast<size_t>(mat) * kNGrid * kRowEp
                                       : c.tab_em + static_cast<size_t>(mat) * kNGrid * kRowEm;
          dE = T0 - inverse_range(c, tab, positron ? kRowEp : kRowEm, positron ? 4 : 3,
                                  c.rhint + (2 * mat + (positron ? 1 : 0)) * kHintStride, R - s);
        }
        dE = fmin(fmax(dE, 0.0), T0);
      }
      edep_dep += dE;
      double T1 = T0 - dE;
      if (T1 < kTmin) {
        edep_cut += T1; T1 = 0.0;
        ann_rest = positron;
        fate = FATE_STOPPED;
        go = false; cross = false;
      }
      T.d[6][t] = T1;
      if (go && !vacuum && s > 0.0) {  // P9 Highland MSC at the pre-step energy, U2 and U3 of this step
        const double X0 = mat_scalar(c, mat, S_X0);
        const double pbeta = T0 * (T0 + 2.0 * kMe) / (T0 + kMe);
        const double beta2 = T0 * (T0 + 2.0 * kMe) / ((T0 + kMe) * (T0 + kMe));
        const double corr = fmax(0.0, 1.0 + 0.038 * log_pos(s / (X0 * beta2)));
        const double th0 = (13.6 / pbeta) * sqrt(s / X0) * corr;
        Stream u;
        u.init(T.u[0][t], c.seed, T.id[t], T.u[1][t]);
        const double u2 = u.uniform(2), u3 = u.uniform(3);
        const double th = th0 * sqrt(-2.0 * log_pos(u2));
        double sn, cs, dn[3];
        sincos(th, &sn, &cs);
        const double dir[3] = {T.d[3][t], T.d[4][t], T.d[5][t]};
        rotate(dir, cs, sn, 2.0 * u3, dn);
        T.d[3][t] = dn[0]; T.d[4][t] = dn[1]; T.d[5][t] = dn[2];
      }
      if (cross) { px += c.eps_push * pdx; py += c.eps_push * pdy; pz += c.eps_push * pdz; }   // G5
    }
    // at-rest annihilation (P8): both photons carry m; below the gamma cut they are deposited (M5)
    bool has_ph = false;
    if (ann_rest) {
      if (kMe < mat_scalar(c, mat, S_KCUT)) { edep_cut += kMe; edep_cut += kMe; }
      else has_ph = true;
    }

    // ---- relocation (A5), warp-convergent
    const int nv = nav_relocate<BVH>(c, c.navigator, cross, vol, px, py, pz, face);

    // ---- outcome
    bool live = false;
    int dest = -1;
    uint32_t vol_post = vol;
    if (active) {
      packed += 1ull << (8 * MC_STEPS);
      sum_dep += edep_dep; sum_cut += edep_cut;
      if (fate == FATE_KILLED) {
        atomicAdd(&tally.ledger[3], carried_energy(species, T.d[6][t]));
        packed += 1ull << (8 * MC_KILLED);
      } else if (fate == FATE_STOPPED) {
        packed += 1ull << (8 * MC_STOPPED);
      } else if (cross) {
        if (nv < 0) {
          Track post;
          post.x = px; post.y = py; post.z = pz;
          post.dx = T.d[3][t]; post.dy = T.d[4][t]; post.dz = T.d[5][t];
          post.ekin = T.d[6][t]; post.id = T.id[t];
          post.event = T.u[0][t]; post.step = T.u[1][t] + 1; post.vol = vol; post.species = species;
          atomicAdd(&tally.ledger[2], carried_energy(species, post.ekin));
          record_leak(c, slot, post, species);
          packed += 1ull << (8 * MC_ESCAPED);
        } else {
          vol_post = static_cast<uint32_t>(nv);
          live = true; dest = 0;
          packed += 1ull << (8 * MC_BOUNDARY);
          if (MULTI && BVH && cache) nav_cache_left_daughter(c, *cache, vol, nv, px, py, pz);
        }
      } else if (flag == 2) {
        live = true; dest = 0;
        packed += 1ull << (8 * MC_TRUNCATED);
      } else if (!lim_disc) {
        live = true; dest = 0;
        packed += 1ull << (8 * MC_LOSS);
      } else {
        live = true; dest = 1 + stage_queue(process, species) - q0;
      }
      if (MULTI) {
        T.d[0][t] = px; T.d[1][t] = py; T.d[2][t] = pz;
        T.u[1][t] += 1; T.u[2][t] = vol_post;
      }
      r.px = px; r.py = py; r.pz = pz; r.vol_post = vol_post; r.live = live; r.dest = dest; r.has_ph = has_ph;
    }
    score(slot, vol, edep_dep + edep_cut, active);
}

template <int FIELD, bool BVH, bool MULTI>
__device__ __forceinline__ void charged_move_body(const DevCtx& c, const DevSlot& slot, int parity, int species, BlockTally& tally,
                                                  BlockReserve<5>& br, TilePipe& pipe, int32_t* cand_lists) {
  const bool positron = species == ADEPT_POSITRON;
  const TrackSoA& cur = slot.buf[parity][species];
  SlotCounters* cnt = slot.counters;
  // (a counter can run past the capacity when its queue overflowed: the stores are guarded, the reads clamped)
  const uint32_t n = min(cnt->count[parity][species].v, c.capacity);

  // destinations: 0 = next buffer of the species, 1..3 = its staging queues, 4 = next gamma buffer (the
  // photons of an annihilation at rest)
  constexpr int ND = 5;
  const int q0 = positron ? 5 : 3;
  // Tracks per tile.  A population smaller than the grid's lanes is spread over all blocks and warps
  // (g tracks per tile, one lane in every 128/g): the warp-cooperative BVH serves the queries of a warp
  // one after the other, so a few hundred loopers packed into a few warps would take 32 x 16 chord queries
  // in sequence per step (measured 4 ms per population step on config 4), spread out they run in parallel.
  // (the two species share the resident blocks: the tiles of both together must fit one wave -- DevCtx::sparse_waves of
  // them in a BVH geometry in a field when the slot has the GPU to itself, adept.cu --; at most a warp per track)
  // (without a field the other species is taken to be as numerous: nothing hangs on it there, and the kernel that fills
  // the GPU on the bench configuration reads one counter less)
  const uint32_t n_other = FIELD == ADEPT_FIELD_NONE ? n : min(cnt->count[parity][species ^ 1].v, c.capacity);   // e- = 0, e+ = 1
  uint32_t g = kBlock;
  while (g > (kBlock / 32 > 4 ? kBlock / 32 : 4) && (n + (g >> 1) - 1) / (g >> 1) + (n_other + (g >> 1) - 1) / (g >> 1) <= gridDim.x * ((FIELD == ADEPT_FIELD_NONE || !BVH) ? 1u : static_cast<uint32_t>(c.sparse_waves))) g >>= 1;
  const int lane_shift = __ffs(kBlock / g) - 1;            // every (1 << lane_shift)-th lane takes a track
  const uint32_t n_tiles = (n + g - 1) / g;
  if (blockIdx.x >= n_tiles) return;   // no tile for this block
  // candidate lists of the chord queries in a BVH volume (geom.cuh NavCache): one per lane, kept across the
  // tiles and steps of the launch
  constexpr bool kLists = BVH;
  NavCache nav_cache;
  nav_cache_reset(nav_cache);
  NavCache* const cache = kLists ? &nav_cache : nullptr;
  tally_init(tally);
  pipe_init(pipe);
  double sum_dep = 0.0, sum_cut = 0.0;
  unsigned chords_sum = 0;
  unsigned long long packed = 0;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned lt = (1u << lane) - 1u;
  const int t = threadIdx.x >> lane_shift;                 // this lane's entry of the tile
  const bool mine = (threadIdx.x & ((1u << lane_shift) - 1u)) == 0;
  // eight or more lanes per track: they take its chord loop together (field.cuh propagate_wide)
  const int wide_shift = (MULTI && FIELD != ADEPT_FIELD_NONE && lane_shift >= ADEPT_WIDE_MIN_SHIFT) ? lane_shift : 0;
  int k_inner = MULTI ? min(inner_steps(c, n, gridDim.x * kBlock, FIELD == ADEPT_FIELD_NONE ? ADEPT_INNER_MAX_STRAIGHT : BVH ? ADEPT_INNER_MAX_BVH : ADEPT_INNER_MAX), 255) : 1;
  // full GPU, BVH geometry: only the passage through the gap a track has just entered from a daughter is taken in
  // the same launch (geom.cuh NavCache)
  const bool transit_only = MULTI && BVH && k_inner == 1 && c.transit;
  if (transit_only) k_inner = 2;

  if (threadIdx.x == 0) tile_issue_n(pipe.tile[0], cur, static_cast<size_t>(blockIdx.x) * g, g, &pipe.bar[0]);
  uint32_t k = 0;
  for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++k) {
    const int phase = k & 1;
    if (threadIdx.x == 0 && tile + gridDim.x < n_tiles)
      tile_issue_n(pipe.tile[phase ^ 1], cur, static_cast<size_t>(tile + gridDim.x) * g, g, &pipe.bar[phase ^ 1]);
    mbar_wait(&pipe.bar[phase], (k >> 1) & 1);
    TrackTile& T = pipe.tile[phase];
    ChargedLane r;
    r.px = 0.0; r.py = 0.0; r.pz = 0.0; r.vol_post = 0; r.live = false; r.has_ph = false; r.dest = -1;
    if (!MULTI) {
      charged_lane<FIELD, BVH, false>(c, slot, tally, T, t, mine && tile * g + t < n, species, q0, packed, sum_dep, sum_cut, chords_sum, r,
                                      cache, cand_lists);
      if (k % 255u == 254u) move_counts_flush(tally, packed);
    } else {
      // A lane steps its track until it leaves the species buffer (interaction, stop, escape, ...) or has taken
      // k_inner steps; the warp goes round together because the navigator is warp-convergent.
      bool cont = mine && tile * g + t < n;
      for (int it = 0;; ++it) {
        charged_lane<FIELD, BVH, true>(c, slot, tally, T, t, cont, species, q0, packed, sum_dep, sum_cut, chords_sum, r, cache, cand_lists,
                                       wide_shift);
        cont = cont && r.live && r.dest == 0 && it + 1 < k_inner;
        if (transit_only) cont = cont && nav_cache.reach > 0.0 && nav_cache.vol == r.vol_post;
        if (!__any_sync(kFull, cont)) break;
      }
      move_counts_flush(tally, packed);
    }
    // Everything still needed of the track is read from the tile here, before the reservation barriers:
    // after them thread 0 may already refill this tile buffer.
    Track post;
    post.x = r.px; post.y = r.py; post.z = r.pz;
    post.dx = T.d[3][t]; post.dy = T.d[4][t]; post.dz = T.d[5][t];
    post.ekin = T.d[6][t]; post.id = T.id[t];
    post.event = T.u[0][t]; post.step = MULTI ? T.u[1][t] : T.u[1][t] + 1; post.vol = r.vol_post; post.species = species;
    const bool live = r.live, has_ph = r.has_ph;
    const int dest = r.dest;
    fence_proxy_async_smem();

    // ---- reservation and stores (A0)
    uint32_t pre = 0;
#pragma unroll
    for (int d = 0; d < 4; ++d) {
      const unsigned b = __ballot_sync(kFull, dest == d);
      if (dest == d) pre = __popc(b & lt);
      if (lane == 0) br.wtot[phase][warp][d] = __popc(b);
    }
    const unsigned bph = __ballot_sync(kFull, has_ph);
    const uint32_t pre_ph = 2 * __popc(bph & lt);
    if (lane == 0) {
      br.wtot[phase][warp][4] = 2 * __popc(bph);
      if (bph) atomicAdd(&tally.secondaries[ADEPT_GAMMA], static_cast<unsigned>(2 * __popc(bph)));
    }
    block_reserve_commit<ND>(br, phase, [&](int d) -> uint32_t* {
      if (d == 0) return &cnt->count[parity ^ 1][species].v;
      if (d == 4) return &cnt->count[parity ^ 1][ADEPT_GAMMA].v;
      return &cnt->n_stage[q0 + d - 1].v;
    });
    if (live) {
      const uint32_t j = br.wbase[phase][warp][dest] + pre;
      const bool staged = dest != 0;
      const TrackSoA& dst = staged ? slot.stage[q0 + dest - 1] : slot.buf[parity ^ 1][species];
      if (j < (staged ? c.stage_capacity : c.capacity)) store_track(dst, j, post);
      else cnt->overflow.v = 1;
    }
    if (has_ph) {   // two back-to-back photons: cos(theta) = 2 U4 - 1, phi = 2 pi U5; children 0 and 1 (R3)
      const uint32_t j = br.wbase[phase][warp][4] + pre_ph;
      Stream u;
      u.init(post.event, c.seed, post.id, post.step - 1);
      const double u4 = u.uniform(4), u5 = u.uniform(5);
      const double cos_t = 2.0 * u4 - 1.0, sin_t = sqrt(fmax(0.0, 1.0 - cos_t * cos_t));
      double sp, cp;
      sincospi(2.0 * u5, &sp, &cp);
      const uint64_t id0 = u.child_id(0), id1 = u.child_id(1);
      post.dx = sin_t * cp; post.dy = sin_t * sp; post.dz = cos_t;
      post.ekin = kMe; post.step = 0; post.species = ADEPT_GAMMA; post.id = id0;
      if (j + 1 < c.capacity) {
        store_track(slot.buf[parity ^ 1][ADEPT_GAMMA], j, post);
        post.dx = -post.dx; post.dy = -post.dy; post.dz = -post.dz; post.id = id1;
        store_track(slot.buf[parity ^ 1][ADEPT_GAMMA], j + 1, post);
      } else {
        cnt->overflow.v = 1;
      }
    }
  }
  move_counts_flush(tally, packed);
  {
    const unsigned long long ch = __reduce_add_sync(kFull, chords_sum);
    if (lane == 0 && ch) atomicAdd(&tally.chords, ch);
  }
  tally_flush(tally, slot, species, sum_dep, sum_cut);
}

// LOWOCC: the same kernel compiled for ADEPT_MINB_LOW resident blocks per SM (255 registers, no spills), which the host
// launches while the population is small (adept.cu round_variant).  BVH geometry in a field only: there a launch of
// a small population lasts as long as its longest chain of chords and traversals, and the spills of the
// 128-register form are on that chain.
template <int FIELD, bool BVH, bool MULTI, bool LOWOCC = false>
__global__ void __launch_bounds__(kBlock, FIELD == ADEPT_FIELD_NONE ? ADEPT_MINB_C2 : LOWOCC ? ADEPT_MINB_LOW : BVH ? ADEPT_MINB_C2FB : ADEPT_MINB_C2F)
charged_move_kernel(const __grid_constant__ DevCtx c, const __grid_constant__ DevSlot slot, int parity) {
  __shared__ BlockTally tally;
  __shared__ BlockReserve<5> br;
  __shared__ TilePipe pipe;
  __shared__ int32_t cand_lists[BVH ? kBlock * kCandCap : 1];
  charged_move_body<FIELD, BVH, MULTI>(c, slot, parity, static_cast<int>(blockIdx.y) /* e- or e+ */, tally, br, pipe, cand_lists);
}

// Without a field and without a BVH the photon and the e+- kernel need the same registers (80) and the same shared
// memory, so one launch serves all three species of a population step: blockIdx.y = 0 photons (the longest, scheduled
// first), 1 electrons, 2 positrons.  One launch and no fork/join between two streams per population step; the
// per-kernel timing mode and the other field kinds keep the two kernels.
template <bool MULTI>
__global__ void __launch_bounds__(kBlock, ADEPT_MINB_C2)
move_kernel(const __grid_constant__ DevCtx c, const __grid_constant__ DevSlot slot, int parity) {
  __shared__ BlockTally tally;
  __shared__ BlockReserve<5> br;
  __shared__ TilePipe pipe;
  if (blockIdx.y == 0) gamma_move_body<false, MULTI>(c, slot, parity, tally, br, pipe);
  else charged_move_body<ADEPT_FIELD_NONE, false, MULTI>(c, slot, parity, static_cast<int>(blockIdx.y) - 1, tally, br, pipe, nullptr);
}

}  // namespace adept
