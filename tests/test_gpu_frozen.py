"""Frozen single-step parity, CUDA path (through the C ABI) vs oracle, on states drawn from the oracle's
own showers (SURVEY.md §8(d) "parity gates"; BASELINE.json:north_star: discrete outcomes bit-exact, continuous
outputs to 1e-12 relative).

Two arms per case.  `population`: adept_step_population runs exactly one population step of the kernels
adept_transport launches -- gamma_move_kernel, charged_move_kernel<FIELD, BVH>, interact_kernel, with their
grids, tile pipeline, sparse tiles and staging queues -- and the next population they write is matched to the
oracle's step results track by track.  `generic`: adept_step_frozen runs the per-lane any-species form of the
step (csrc/step.cuh), which also reports the per-track path length, deposits and outcome code."""
import multiprocessing as mp
import os

import numpy as np
import pytest

from parity import compare_population, compare_steps, deposit_tolerance, energy_scale

pytestmark = pytest.mark.gpu

M = 0.51099895


def _states(o, prim, per_species, stride):
    """>= per_species pre-step states of each species recorded from the oracle's own showers."""
    out = []
    for sp in range(3):
        o.set_recorder(1 << sp, stride, per_species)
        o.run(o.make_tracks(prim))
        out.append(o.recorded())
    o.set_recorder(0, 1, 0)
    return np.concatenate(out)


def _x0(g, scal, pre):
    x0 = scal[g.material[pre["volume"]], 0]
    return np.where(scal[g.material[pre["volume"]], 5] != 0, np.inf, x0)


def _dedx(o, g, scal, pre):
    """Restricted stopping power S(T0) of the pre-step material for e- / e+ (0 in vacuum and for photons)."""
    mat = g.material[pre["volume"]]
    out = np.zeros(len(pre))
    for i in np.where((pre["species"] != 2) & (scal[mat, 5] == 0) & (pre["ekin"] > 0))[0]:
        out[i] = o.lookup(int(mat[i]), 5 if pre["species"][i] == 0 else 10, float(pre["ekin"][i]))
    return out


def _bmax(fld):
    return float(np.abs(fld.bz).max()) if fld.kind == 2 else float(np.linalg.norm(fld.B))


def check_population(a, o, g, scal, fld, pre, ores, osec, slot=0, dedx=None):
    """One population step of the transport kernels on `pre` against the oracle's results (ores, osec)."""
    n_vol = g.n_volumes
    st0 = a.stats(slot)
    out = a.step_population(pre, slot=slot)
    edep, led = a.read_scoring(slot)
    leaked, n_leak = a.read_leaked(slot, cap=max(len(pre), 1))
    st = a.stats(slot)
    x0 = _x0(g, scal, pre)
    if dedx is None:
        dedx = _dedx(o, g, scal, pre)
    ds, worst = compare_population(pre, out, ores, osec, x0=x0, b_max=_bmax(fld), dedx=dedx)
    tol = deposit_tolerance(pre, ds, dedx)
    # counters: steps per species, every outcome code, secondaries per species -- exact
    assert [st.steps[k] - st0.steps[k] for k in range(3)] == np.bincount(pre["species"], minlength=3).tolist()
    assert [st.outcomes[k] - st0.outcomes[k] for k in range(13)] == np.bincount(ores["outcome"], minlength=13).tolist()
    sec_species = np.concatenate([osec[ores["n_sec"] > k, k]["species"] for k in range(2)])
    assert [st.secondaries[k] - st0.secondaries[k] for k in range(3)] == np.bincount(sec_species, minlength=3).tolist()
    assert st.chords - st0.chords == int(ores["chords"].sum())
    # per-volume deposits: sum of the oracle's per-track deposits of that volume, within the sum of their tolerances
    want = np.bincount(pre["volume"], weights=ores["edep_dep"] + ores["edep_cut"], minlength=n_vol)
    cnt = np.bincount(pre["volume"], minlength=n_vol)
    tol_v = np.bincount(pre["volume"], weights=tol, minlength=n_vol) + 4e-16 * np.sqrt(cnt + 1.0) * want
    bad = np.abs(edep - want) > tol_v
    assert not bad.any(), (np.where(bad)[0][:5], edep[bad][:5], want[bad][:5], tol_v[bad][:5])
    # ledger buckets
    tot = tol.sum() + 4e-16 * np.sqrt(len(pre)) * energy_scale(pre).sum()
    assert led.primary == pytest.approx(energy_scale(pre).sum(), rel=1e-11)      # n fp64 atomics in any order
    for name in ("edep_dep", "edep_cut", "escaped", "killed"):
        got = {"edep_dep": led.deposited, "edep_cut": led.below_cut, "escaped": led.escaped, "killed": led.killed}[name]
        assert abs(got - ores[name].sum()) <= tot, (name, got, ores[name].sum())
    carried_out = energy_scale(out).sum()
    assert abs(led.total() + carried_out - led.primary) <= 1e-9 * led.primary      # nothing lost in the step
    # outgoing tracks = the oracle's escaped ones
    esc = ores["outcome"] == 10
    assert n_leak == esc.sum() == len(leaked)
    key = lambda t: sorted(zip(t["event"].tolist(), t["id"].tolist()))
    assert key(leaked) == key(pre[esc])
    return worst


def check_generic(a, g, scal, fld, pre, ores, osec, dedx):
    res, sec = a.step_frozen(pre)
    return compare_steps(pre, res, sec, ores, osec, x0=_x0(g, scal, pre), b_max=_bmax(fld), dedx=dedx)[1]


def check_per_track_deposits(a, g, scal, fld, pre, ores, osec, dedx, n_chunks=48):
    """Batches in which every track sits in a volume of its own: the per-volume deposit the kernels score IS that
    track's deposit, compared at the single-step tolerance."""
    order = np.argsort(pre["volume"], kind="stable")
    vol = pre["volume"][order]
    rank = np.arange(len(vol)) - np.searchsorted(vol, vol, side="left")      # k-th state of its volume
    checked = 0
    for c in range(n_chunks):
        idx = order[rank == c]
        if len(idx) == 0:
            break
        out = a.step_population(pre[idx])
        edep, led = a.read_scoring(0)
        a.read_leaked(0)
        ds, _ = compare_population(pre[idx], out, ores[idx], osec[idx], x0=_x0(g, scal, pre[idx]), b_max=_bmax(fld), dedx=dedx[idx])
        tol = deposit_tolerance(pre[idx], ds, dedx[idx])
        got = edep[pre["volume"][idx]]
        want = ores["edep_dep"][idx] + ores["edep_cut"][idx]
        assert np.all(np.abs(got - want) <= tol), (c, np.abs(got - want).max())
        assert edep.sum() == pytest.approx(got.sum(), rel=1e-15, abs=0)          # nothing scored elsewhere
        checked += len(idx)
    return checked


def _run_case(ob, geom_set, fld, prim, per_species, stride, elements=None, **cfg):
    from paper_2209_15445_b200 import adept
    g, _, tabs, scal = geom_set[:4]
    o = ob.Oracle(g, tabs, scal, fld, elements=elements)
    pre = _states(o, prim, per_species, stride)
    counts = np.bincount(pre["species"], minlength=3)
    ores, osec = o.step(pre)
    dedx = _dedx(o, g, scal, pre)
    a = adept.Adept(g, tabs, scal, fld, track_capacity=1 << 18, leak_capacity=1 << 18, elements=elements, **cfg)
    worst_p = check_population(a, o, g, scal, fld, pre, ores, osec, dedx=dedx)
    # small batches take the sparse-tile path of the charged kernel: 32, 16 and 8 lanes per track, i.e. in a field the
    # wide chord loop with one and with two rounds of chords per step (csrc/field.cuh propagate_wide)
    for m in (700, 2000, 4000):
        few = np.concatenate([np.where(pre["species"] == sp)[0][:m] for sp in range(3)])
        check_population(a, o, g, scal, fld, pre[few], ores[few], osec[few], dedx=dedx[few])
    n_single = check_per_track_deposits(a, g, scal, fld, pre, ores, osec, dedx)
    worst_g = check_generic(a, g, scal, fld, pre, ores, osec, dedx)
    a.close()
    return counts, worst_p, worst_g, ores, n_single


@pytest.mark.parametrize("bz", [0.0, 1.0])
def test_calorimeter_frozen_steps(ob, calo, bz):
    """Configs 1-3: >= 1e5 states per species; several tiles of 128 threads plus a ragged tail."""
    from paper_2209_15445_b200.inputs import field, primaries
    fld = field.uniform_field(0, 0, bz) if bz else field.no_field()
    prim = primaries.beam(24, 10000.0, spread=1.0)
    prim["species"][1::3] = 1
    prim["species"][2::3] = 2
    counts, worst_p, worst_g, ores, n_single = _run_case(ob, calo, fld, prim, 100003, 1)
    assert np.all(counts >= 100000), counts
    seen = set(np.unique(ores["outcome"]).tolist())
    assert {0, 1, 2, 3, 4, 5, 6, 7, 9, 10}.issubset(seen), seen      # every process and fate is exercised
    assert n_single > 2000
    print("worst scaled errors: population", worst_p, "generic", worst_g)


def test_barrel_patch_frozen_steps(ob, barrel_patch):
    """Config 4 ingredients on a 12x12 crystal patch: tubes, rotated boxes, BVH (144 daughters), RK4 field map."""
    from paper_2209_15445_b200.inputs import field, primaries
    prim = primaries.barrel_events(1, 40, 1e3, 2e4, mode="cfg5")
    d = np.array([np.cos(0.1), np.sin(0.1), 0.01])
    prim["dir"][:] = d / np.linalg.norm(d)
    counts, worst_p, worst_g, ores, n_single = _run_case(ob, barrel_patch, field.solenoid_map(), prim, 40000, 1)
    assert np.all(counts >= 20000), counts
    assert 8 in set(np.unique(ores["outcome"]).tolist())             # truncated (chord budget) steps occur
    print("worst scaled errors: population", worst_p, "generic", worst_g)


def test_compound_crystals_frozen_steps(ob, barrel_patch_compound):
    """the crystal patch in the real compound PbWO4 = Pb + W + 4 O, whose
    photoelectric absorptions pick their target element (and its K-shell binding energy) with uniform U6."""
    from paper_2209_15445_b200.inputs import field, primaries
    g, mats, tabs, scal, elements = barrel_patch_compound
    prim = primaries.barrel_events(1, 40, 1e3, 2e4, mode="cfg5")
    d = np.array([np.cos(0.1), np.sin(0.1), 0.01])
    prim["dir"][:] = d / np.linalg.norm(d)
    counts, worst_p, worst_g, ores, n_single = _run_case(ob, barrel_patch_compound, field.solenoid_map(), prim, 40000, 1,
                                                         elements=elements)
    assert np.all(counts >= 20000), counts
    pe = ores["outcome"] == 3
    assert pe.sum() > 2000
    # both heavy elements were chosen: deposits of the two K-shell binding energies occur among the absorptions
    bk = elements[1][2]
    dep = ores["edep_cut"][pe]
    assert np.isclose(dep, bk[0], rtol=1e-12).sum() > 100 and np.isclose(dep, bk[1], rtol=1e-12).sum() > 50
    print("worst scaled errors: population", worst_p, "generic", worst_g)


# ---- full barrel: the loop-navigator oracle over 61 212 volumes runs in a process pool
def _full_barrel_worker(job):
    pre, = job
    from oracle import binding as ob
    from paper_2209_15445_b200.inputs import field, geometry, materials
    g = geometry.barrel()
    _, tabs, scal = materials.build_material_set(g.material_names)
    o = ob.Oracle(g, tabs, scal, field.solenoid_map())
    keep = np.zeros(len(pre), dtype=bool)
    for i in range(len(pre)):
        v = o.locate(pre["pos"][i])
        if v >= 0:
            pre["volume"][i] = v
            keep[i] = True
    pre = pre[keep]
    ores, osec = o.step(pre)
    return pre, ores, osec, _dedx(o, g, scal, pre)


def test_full_barrel_sampled_frozen_steps(ob, barrel_full):
    """Config 4 at full size (61 200 crystals): >= 2e4 states per species recorded from showers in the patch
    geometry are replayed in the full geometry (same shells, mother and crystal placement formula; volume ids
    re-located by the oracle) through the transport kernels; the oracle steps them in a process pool."""
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field, geometry, primaries
    g, _, tabs, scal = barrel_full
    fld = field.solenoid_map()
    gp = geometry.barrel(n_eta=12, n_phi=12)
    op = ob.Oracle(gp, tabs, scal, fld)
    prim = primaries.barrel_events(1, 40, 1e3, 2e4, mode="cfg5")
    d = np.array([np.cos(0.1), np.sin(0.1), 0.01])
    prim["dir"][:] = d / np.linalg.norm(d)                  # into the patch; states are re-located in the workers
    pre = _states(op, prim, 21000, 3)
    # shift a third of the states to other crystals of the full barrel: rotate about z by a multiple of the column pitch
    rng = np.random.default_rng(11)
    k = rng.integers(0, 360, len(pre)) * (rng.random(len(pre)) < 0.34)
    ang = k * (2 * np.pi / 360)
    cs, sn = np.cos(ang), np.sin(ang)
    for f in ("pos", "dir"):
        x, y = pre[f][:, 0].copy(), pre[f][:, 1].copy()
        pre[f][:, 0], pre[f][:, 1] = cs * x - sn * y, sn * x + cs * y
    n_proc = min(os.cpu_count() or 1, 16)
    jobs = [(pre[i::n_proc].copy(),) for i in range(n_proc)]
    with mp.get_context("spawn").Pool(n_proc) as pool:
        parts = pool.map(_full_barrel_worker, jobs)
    pre = np.concatenate([p[0] for p in parts]); ores = np.concatenate([p[1] for p in parts])
    osec = np.concatenate([p[2] for p in parts]); dedx = np.concatenate([p[3] for p in parts])
    counts = np.bincount(pre["species"], minlength=3)
    assert np.all(counts >= 20000), counts
    assert (pre["volume"] >= 12).sum() > 20000 and len(np.unique(pre["volume"])) > 1000
    o = ob.Oracle(g, tabs, scal, fld)
    a = adept.Adept(g, tabs, scal, fld, track_capacity=1 << 17, leak_capacity=1 << 17)
    worst_p = check_population(a, o, g, scal, fld, pre, ores, osec, dedx=dedx)
    few = np.arange(0, len(pre), 97)
    check_population(a, o, g, scal, fld, pre[few], ores[few], osec[few], dedx=dedx[few])
    worst_g = check_generic(a, g, scal, fld, pre, ores, osec, dedx)
    a.close()
    # 6e4 tracks are below config.low_occupancy_below: the steps above ran the two-block build of the e+- kernel.
    # The same states through the three-block build, which transport launches for the populations that fill the GPU:
    a = adept.Adept(g, tabs, scal, fld, track_capacity=1 << 17, leak_capacity=1 << 17, low_occupancy_below=-1)
    worst_p3 = check_population(a, o, g, scal, fld, pre, ores, osec, dedx=dedx)
    a.close()
    print("worst scaled errors: population", worst_p, "three-block build", worst_p3, "generic", worst_g)


def test_degenerate_states(ob, calo):
    """Edge cases of the step: sub-keV tracks, the step cap, exactly axis-parallel and z-aligned directions."""
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field
    g, _, tabs, scal = calo
    fld = field.uniform_field(0, 0, 1.0)
    o = ob.Oracle(g, tabs, scal, fld, max_steps=50)
    a = adept.Adept(g, tabs, scal, fld, track_capacity=1 << 10, max_steps=50)
    pre = np.zeros(3 * 6, dtype=ob.TRACK)
    k = 0
    for sp in range(3):
        for ekin, step, d, pos, vol in ((5e-4, 0, (1, 0, 0), (0.1, 0, 0), 52), (3.0, 50, (1, 0, 0), (0.1, 0, 0), 52),
                                        (8.0, 1, (0, 0, 1), (0.1, 0, 0), 52), (8.0, 2, (0, 0, -1), (0.3, 1, 1), 53),
                                        (50.0, 3, (-1, 0, 0), (-5.0, 0, 0), 0), (0.02, 4, (0, 1, 0), (0.4, 0, 19.9), 53)):
            pre[k]["species"], pre[k]["ekin"], pre[k]["step"], pre[k]["dir"], pre[k]["pos"] = sp, ekin, step, d, pos
            pre[k]["volume"], pre[k]["id"], pre[k]["event"] = vol, 100 + k, 7
            k += 1
    ores, osec = o.step(pre)
    dedx = _dedx(o, g, scal, pre)
    check_population(a, o, g, scal, fld, pre, ores, osec, dedx=dedx)
    res, sec = a.step_frozen(pre)
    compare_steps(pre, res, sec, ores, osec, x0=_x0(g, scal, pre), b_max=_bmax(fld), dedx=dedx)
    assert set(ores["outcome"][[0, 6, 12]]) == {7} and set(ores["outcome"][[1, 7, 13]]) == {11}
    # an empty batch is a no-op; a slot that still holds tracks refuses the hook
    r0, s0 = a.step_frozen(np.zeros(0, dtype=ob.TRACK))
    assert len(r0) == 0 and len(a.step_population(np.zeros(0, dtype=ob.TRACK))) == 0
    a.close()
