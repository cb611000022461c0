"""Full-shower parity (BASELINE.json:north_star: mean edep per layer/volume within 0.5 % or 3 sigma of the
combined statistical error, whichever is larger; per-event ledger closing to 1e-9) and the API edge cases."""
import numpy as np
import pytest

from parity import layer_stats

pytestmark = pytest.mark.gpu

M = 0.51099895


def _oracle_events(o, tr, n_vol):
    """Per-event edep arrays from the oracle (one orc_run per event)."""
    ev = np.unique(tr["event"])
    out = np.zeros((len(ev), n_vol))
    led = []
    for k, e in enumerate(ev):
        _, l, _ = o.run(tr[tr["event"] == e], out[k])
        led.append(l)
    return out, led


def _check_layers(gpu_mean, o_mean, o_err):
    tol = np.maximum(0.005 * np.abs(o_mean), 3.0 * np.sqrt(2.0) * o_err)
    bad = np.abs(gpu_mean - o_mean) > tol
    assert not bad.any(), (np.where(bad)[0], gpu_mean[bad], o_mean[bad], tol[bad])


@pytest.mark.parametrize("sync_interval", [8, 1])
def test_config1_calorimeter_256_electrons(ob, calo, sync_interval):
    """BASELINE.json:configs[0]: 256 e- at 1 GeV, seed 1, edep per layer; one slot per group of events so the
    per-event ledgers are checked too."""
    import torch
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field, primaries
    g, _, tabs, scal = calo
    prim = primaries.beam(256, 1000.0)
    o = ob.Oracle(g, tabs, scal, field.no_field())
    tr = o.make_tracks(prim)
    o_ev, o_led = _oracle_events(o, tr, g.n_volumes)
    o_mean, o_err = layer_stats(o_ev)
    a = adept.Adept(g, tabs, scal, field.no_field(), track_capacity=1 << 18, n_event_slots=2, sync_interval=sync_interval,
                    stage_capacity=(1 << 17 if sync_interval == 1 else 0))
    # slot 0: all 256 events in one population; slot 1: single events, ledger per event
    a.enqueue(prim, slot=0)
    a.transport(0, torch.cuda.current_stream())
    e, led = a.read_scoring(0)
    assert led.primary == 256 * 1000.0
    assert abs(led.total() - led.primary) <= 1e-9 * led.primary
    gpu_mean = e[52:152].reshape(50, 2).sum(axis=1) / 256
    _check_layers(gpu_mean, o_mean, o_err)
    # identical random streams: short of a threshold flip the showers are the same, track for track
    np.testing.assert_allclose(e, o_ev.sum(axis=0), rtol=1e-9, atol=1e-9)
    for i in (0, 17, 255):
        one = {k: v[i:i + 1] for k, v in prim.items()}
        a.enqueue(one, slot=1)
        a.transport(1, torch.cuda.current_stream())
        ei, li = a.read_scoring(1)
        assert abs(li.total() - li.primary) <= 1e-9 * li.primary and li.primary == 1000.0
        np.testing.assert_allclose(ei, o_ev[i], rtol=1e-9, atol=1e-10)
        assert li.escaped == pytest.approx(o_led[i].escaped, rel=1e-9, abs=1e-12)
    st = a.stats(0)
    assert st.outcomes[11] == 0 and st.iterations > 50
    a.close()


@pytest.mark.parametrize("species", [0, 2])
def test_config3_uniform_field(ob, calo, species):
    """BASELINE.json:configs[2] at reduced statistics: 1 T along +z, exact helix, e- and gamma runs."""
    import torch
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field, primaries
    g, _, tabs, scal = calo
    fld = field.uniform_field(0, 0, 1.0)
    prim = primaries.beam(48, 10000.0, species=species, spread=1.0)
    o = ob.Oracle(g, tabs, scal, fld)
    tr = o.make_tracks(prim)
    o_ev, _ = _oracle_events(o, tr, g.n_volumes)
    o_mean, o_err = layer_stats(o_ev)
    a = adept.Adept(g, tabs, scal, fld, track_capacity=1 << 19)
    a.enqueue(prim)
    a.transport(0, torch.cuda.current_stream())
    e, led = a.read_scoring(0)
    st = a.stats(0)
    a.close()
    assert abs(led.total() - led.primary) <= 1e-9 * led.primary
    _check_layers(e[52:152].reshape(50, 2).sum(axis=1) / 48, o_mean, o_err)
    # per material (config 2 asks for it): Pb and LAr totals
    slabs_g, slabs_o = e[52:152].reshape(50, 2).sum(axis=0), o_ev.sum(axis=0)[52:152].reshape(50, 2).sum(axis=0)
    np.testing.assert_allclose(slabs_g, slabs_o, rtol=5e-3)
    assert st.chords > 0


def test_config4_full_barrel_showers(ob, barrel_full):
    """BASELINE.json:configs[3] on the FULL barrel (61 200 crystals, 10 Si shells, solenoid map, RK4, BVH
    navigator) at reduced energies so the loop-navigator oracle finishes in seconds: 3 events of 4 e-/gamma
    primaries, 0.2-2 GeV log-uniform, isotropic in phi, |eta| < 1.4.  Identical Philox streams: every event
    must reproduce the oracle's per-volume deposits, step counts and leaked energy."""
    import torch
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field, primaries
    g, _, tabs, scal = barrel_full
    fld = field.solenoid_map()
    n_ev, n_per = 3, 4
    prim = primaries.barrel_events(n_ev, n_per, 200.0, 2000.0, mode="cfg4")
    o = ob.Oracle(g, tabs, scal, fld)
    tr = o.make_tracks(prim)
    o_ev, o_led, o_steps, o_outcomes = np.zeros((n_ev, g.n_volumes)), [], np.zeros(3, dtype=np.int64), None
    for e in range(n_ev):
        _, led_e, st_e = o.run(tr[tr["event"] == e], o_ev[e])
        o_led.append(led_e)
        o_steps += np.array(list(st_e.steps), dtype=np.int64)
        o_outcomes = np.array(list(st_e.outcomes), dtype=np.int64) + (0 if o_outcomes is None else o_outcomes)
    # both builds of the e+- kernel of a BVH geometry in a field (include/adept.h low_occupancy_below): the one for small
    # populations (default here) and the one transport launches when the population fills the GPU
    for below in (0, -1):
        a = adept.Adept(g, tabs, scal, fld, track_capacity=1 << 16, n_event_slots=n_ev + 1, sync_interval=8,
                        low_occupancy_below=below)
        same = 0
        for e in range(n_ev):
            sel = prim["event"] == e
            a.enqueue_primaries(e, e, prim["species"][sel], prim["pos"][sel], prim["dir"][sel], prim["ekin"][sel])
            a.transport(e, torch.cuda.current_stream())
            hits, led = a.read_scoring(e)
            assert abs(led.total() - led.primary) <= 1e-9 * led.primary
            assert led.primary == pytest.approx(o_led[e].primary, rel=1e-14)
            if np.allclose(hits, o_ev[e], rtol=1e-8, atol=1e-8):
                same += 1
                assert led.escaped == pytest.approx(o_led[e].escaped, rel=1e-9, abs=1e-9)
            else:    # a threshold flip: the shower legitimately diverges, totals stay statistically close
                assert hits.sum() == pytest.approx(o_ev[e].sum(), rel=0.05)
        assert same >= n_ev - 1
        # all events in one population: counts of every outcome equal the oracle's
        a.enqueue(prim, slot=n_ev)
        a.transport(n_ev, torch.cuda.current_stream())
        hits, led = a.read_scoring(n_ev)
        st = a.stats(n_ev)
        a.close()
        if same == n_ev:
            assert list(st.steps) == list(o_steps) and list(st.outcomes) == list(o_outcomes)
            np.testing.assert_allclose(hits, o_ev.sum(axis=0), rtol=1e-8, atol=1e-8)
        assert st.chords > 0 and hits[12:].sum() > 0          # RK4 chords ran, crystals were hit


@pytest.mark.parametrize("navigator", [1, 0])
def test_config5_concurrent_events_on_streams(ob, barrel_patch, navigator):
    """BASELINE.json:configs[4] on the crystal patch: 16 events on 16 CUDA streams, per-event per-volume hits
    copied back to the host and checked against the oracle event by event."""
    import torch
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field, primaries
    g, _, tabs, scal = barrel_patch
    fld = field.solenoid_map()
    n_ev, n_per = 16, 10
    prim = primaries.barrel_events(n_ev, n_per, 100.0, 5e3, mode="cfg5")
    rng = np.random.default_rng(4)
    phi, z = rng.uniform(0.03, 0.17, n_ev * n_per), rng.uniform(-0.08, 0.08, n_ev * n_per)
    d = np.stack([np.cos(phi), np.sin(phi), z], axis=1)
    prim["dir"][:] = d / np.linalg.norm(d, axis=1, keepdims=True)      # into the patch
    o = ob.Oracle(g, tabs, scal, fld)
    tr = o.make_tracks(prim)
    o_ev, o_led = _oracle_events(o, tr, g.n_volumes)
    a = adept.Adept(g, tabs, scal, fld, track_capacity=1 << 16, n_event_slots=n_ev, sync_interval=4, navigator=navigator)
    streams = [torch.cuda.Stream() for _ in range(n_ev)]
    for e in range(n_ev):
        sel = prim["event"] == e
        a.enqueue_primaries(e, e, prim["species"][sel], prim["pos"][sel], prim["dir"][sel], prim["ekin"][sel])
    a.transport_many(list(range(n_ev)), streams)
    total_tol = 0
    for e in range(n_ev):
        hits, led = a.read_scoring(e, streams[e])
        assert abs(led.total() - led.primary) <= 1e-9 * led.primary
        assert led.primary == pytest.approx(o_led[e].primary, rel=1e-14)
        # same streams => same shower unless a threshold flip happened; allow statistical agreement otherwise
        if np.allclose(hits, o_ev[e], rtol=1e-8, atol=1e-8):
            total_tol += 1
        else:
            assert hits.sum() == pytest.approx(o_ev[e].sum(), rel=0.05)
        leaked, n_leak = a.read_leaked(e)
        assert n_leak == len(leaked) and led.escaped == pytest.approx(
            (leaked["ekin"] + np.where(leaked["species"] == 1, 2 * M, 0)).sum(), rel=1e-12, abs=1e-12)
    assert total_tol >= n_ev - 1
    a.close()


def _full_barrel_run_worker(job):
    tracks, max_steps = job
    from oracle import binding as ob
    from paper_2209_15445_b200.inputs import field, geometry, materials
    g = geometry.barrel()
    _, tabs, scal = materials.build_material_set(g.material_names)
    o = ob.Oracle(g, tabs, scal, field.solenoid_map(), max_steps=max_steps)
    edep, led, st = o.run(tracks)
    nz = np.nonzero(edep)[0]
    return nz, edep[nz], (led.deposited, led.below_cut, led.escaped, led.killed, led.primary), list(st.steps), list(st.outcomes)


def test_config5_full_barrel_200_primaries(ob, barrel_full):
    """BASELINE.json:configs[4] at its stated structure: 16 events x 200 primaries (e-, e+, gamma 2:1:2) on 16 CUDA
    streams in the FULL barrel (61 200 crystals, BVH, solenoid map), per-event hits copied back per event.  The
    energies are lowered to 20-200 MeV log-uniform and the step cap to 300 so that the loop-navigator oracle (3 ms
    per step in a gap between crystals) finishes two whole events in a process pool: events 0 and 1 are compared
    with the oracle crystal by crystal, the other 14 by their ledgers and against a second, sequential transport
    of the same event (random streams are keyed by event, track and step, so the schedule must not matter)."""
    import multiprocessing as mp
    import os
    import torch
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field, primaries
    g, _, tabs, scal = barrel_full
    n_ev, n_per, max_steps = 16, 200, 300
    prim = primaries.barrel_events(n_ev, n_per, 20.0, 200.0, mode="cfg5")
    o = ob.Oracle(g, tabs, scal, field.solenoid_map(), max_steps=max_steps)
    a = adept.Adept(g, tabs, scal, field.solenoid_map(), track_capacity=1 << 16, n_event_slots=n_ev + 1, max_steps=max_steps)
    streams = [torch.cuda.Stream() for _ in range(n_ev)]
    sel = [prim["event"] == e for e in range(n_ev)]
    for e in range(n_ev):
        a.enqueue_primaries(e, e, prim["species"][sel[e]], prim["pos"][sel[e]], prim["dir"][sel[e]], prim["ekin"][sel[e]])
    a.transport_many(list(range(n_ev)), streams)
    hits, leds, stats = [], [], []
    for e in range(n_ev):
        h, led = a.read_scoring(e, streams[e])
        hits.append(h); leds.append(led); stats.append(a.stats(e))
        assert abs(led.total() - led.primary) <= 1e-9 * led.primary
        assert led.primary == pytest.approx((prim["ekin"][sel[e]] + np.where(prim["species"][sel[e]] == 1, 2 * M, 0)).sum(), rel=1e-12)
    assert sum(h[12:].sum() for h in hits) > 0 and sum(l.killed for l in leds) > 0    # crystals hit; curlers reached the cap
    # events 2..15: the same event alone, sequentially, in the spare slot
    for e in range(2, n_ev):
        a.enqueue_primaries(n_ev, e, prim["species"][sel[e]], prim["pos"][sel[e]], prim["dir"][sel[e]], prim["ekin"][sel[e]])
        st0 = a.stats(n_ev)
        a.transport(n_ev, torch.cuda.current_stream())
        h, led = a.read_scoring(n_ev)
        st1 = a.stats(n_ev)
        np.testing.assert_allclose(h, hits[e], rtol=1e-9, atol=1e-10)
        assert [st1.steps[k] - st0.steps[k] for k in range(3)] == list(stats[e].steps)
        assert [st1.outcomes[k] - st0.outcomes[k] for k in range(13)] == list(stats[e].outcomes)
        assert led.killed == pytest.approx(leds[e].killed, rel=1e-9, abs=1e-9)
    a.close()
    # events 0 and 1 against the oracle: the primaries of each spread over half of a process pool (deposits add)
    n_proc = min(os.cpu_count() or 2, 16)
    per_ev = max(n_proc // 2, 1)
    jobs, owner = [], []
    for e in (0, 1):
        tr = o.make_tracks({k: v[sel[e]] for k, v in prim.items()})
        tr["id"] = np.arange(len(tr))
        for i in range(per_ev):
            jobs.append((tr[i::per_ev].copy(), max_steps)); owner.append(e)
    with mp.get_context("spawn").Pool(len(jobs)) as pool:
        parts = pool.map(_full_barrel_run_worker, jobs)
    for e in (0, 1):
        want, led = np.zeros(g.n_volumes), np.zeros(5)
        steps, outcomes = np.zeros(3, dtype=np.int64), np.zeros(13, dtype=np.int64)
        for (nz, val, l, st, oc), ev in zip(parts, owner):
            if ev != e:
                continue
            want[nz] += val
            led += np.array(l)
            steps += np.array(st, dtype=np.int64)
            outcomes += np.array(oc, dtype=np.int64)
        assert list(stats[e].steps) == steps.tolist() and list(stats[e].outcomes) == outcomes.tolist()
        np.testing.assert_allclose(hits[e], want, rtol=1e-8, atol=1e-9)
        assert leds[e].escaped == pytest.approx(led[2], rel=1e-9, abs=1e-9)
        assert leds[e].killed == pytest.approx(led[3], rel=1e-9, abs=1e-9)
        assert (want[12:] > 0).sum() > 20


def test_compound_crystals_showers(ob, barrel_patch_compound):
    """showers in crystals of the real compound PbWO4 with the element selector; identical random
    streams, so every counter and every per-volume deposit equals the oracle's."""
    import torch
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field, primaries
    g, mats, tabs, scal, elements = barrel_patch_compound
    fld = field.solenoid_map()
    prim = primaries.barrel_events(6, 6, 200.0, 3e3, mode="cfg5")
    rng = np.random.default_rng(7)
    phi, z = rng.uniform(0.03, 0.17, 36), rng.uniform(-0.08, 0.08, 36)
    d = np.stack([np.cos(phi), np.sin(phi), z], axis=1)
    prim["dir"][:] = d / np.linalg.norm(d, axis=1, keepdims=True)
    o = ob.Oracle(g, tabs, scal, fld, elements=elements)
    oe, ol, ost = o.run(o.make_tracks(prim))
    # without the element tables the result differs: the selector is really in the path
    oe1, _, ost1 = ob.Oracle(g, tabs, scal, fld).run(o.make_tracks(prim))
    assert list(ost1.outcomes) != list(ost.outcomes) or not np.allclose(oe1, oe, rtol=1e-9, atol=1e-9)
    a = adept.Adept(g, tabs, scal, fld, track_capacity=1 << 17, elements=elements)
    a.enqueue(prim)
    a.transport(0, torch.cuda.current_stream())
    e, led = a.read_scoring(0)
    st = a.stats(0)
    a.close()
    assert abs(led.total() - led.primary) <= 1e-9 * led.primary
    assert list(st.steps) == list(ost.steps) and list(st.outcomes) == list(ost.outcomes)
    assert list(st.secondaries) == list(ost.secondaries)
    np.testing.assert_allclose(e, oe, rtol=1e-9, atol=1e-9)
    assert led.escaped == pytest.approx(ol.escaped, rel=1e-9, abs=1e-9)


def test_empty_and_error_paths(ob, calo):
    import ctypes as C
    import torch
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field, primaries
    g, _, tabs, scal = calo
    a = adept.Adept(g, tabs, scal, field.no_field(), track_capacity=64, leak_capacity=4)
    # empty slot: transport returns at once, scoring is zero
    a.transport(0, torch.cuda.current_stream())
    e, led = a.read_scoring(0)
    assert e.sum() == 0 and led.primary == 0
    a.enqueue({k: v[:0] for k, v in primaries.beam(1, 10.0).items()})
    # bad slot / primary outside the world / unknown species
    with pytest.raises(adept.AdeptError) as ei:
        a.transport(3)
    assert ei.value.code == adept.EINVAL
    p = primaries.beam(2, 10.0)
    p["pos"][1] = (100.0, 0, 0)
    with pytest.raises(adept.AdeptError) as ei:
        a.enqueue(p)
    assert ei.value.code == adept.EINVAL
    a.close()
    # a slot listed twice is refused and leaves nothing marked live
    a = adept.Adept(g, tabs, scal, field.no_field(), track_capacity=1 << 14, n_event_slots=2)
    s = torch.cuda.current_stream()
    with pytest.raises(adept.AdeptError) as ei:
        a.transport_many([0, 1, 0], [s, s, s])
    assert ei.value.code == adept.EINVAL
    a.enqueue(primaries.beam(2, 50.0))                      # ESTATE if a slot had stayed live
    a.transport_many([0, 1], [s, torch.cuda.Stream()])
    assert a.read_scoring(0)[1].primary == 100.0
    a.close()
    # workspace too small: adept_init refuses it
    a = adept.Adept(g, tabs, scal, field.no_field(), track_capacity=64)
    assert a.workspace_bytes > 1024
    with pytest.raises(adept.AdeptError) as ei:
        adept.Adept(g, tabs, scal, field.no_field(), track_capacity=64, _workspace_bytes=a.workspace_bytes - 256)
    assert ei.value.code == adept.ENOMEM
    a.close()


def test_queue_overflow_is_reported_and_the_slot_stays_usable(ob, calo):
    """ADEPT_EOVERFLOW instead of out-of-range reads: a batch that overflows the track buffers by far more than a
    tile, with the host looking only every 16 population steps; the CUDA context survives, the slot is reset,
    and a batch that fits then gives the oracle's result.  Same for a staging queue that is too small."""
    import torch
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field, primaries
    g, _, tabs, scal = calo
    small = primaries.beam(4, 200.0, spread=1.0)
    o = ob.Oracle(g, tabs, scal, field.no_field())
    oe, ol, ost = o.run(o.make_tracks(small))
    for cfg in (dict(track_capacity=4096), dict(track_capacity=1 << 16, stage_capacity=64)):
        a = adept.Adept(g, tabs, scal, field.no_field(), sync_interval=16, **cfg)
        for rep in range(2):
            a.enqueue(primaries.beam(64, 10000.0, spread=1.0))        # peaks at ~3e4 live tracks
            with pytest.raises(adept.AdeptError) as ei:
                a.transport(0, torch.cuda.current_stream())
            assert ei.value.code == adept.EOVERFLOW
            torch.cuda.synchronize()                                  # no sticky CUDA error
            a.enqueue(small)
            a.transport(0, torch.cuda.current_stream())
            e, led = a.read_scoring(0)
            assert led.primary == 800.0 and abs(led.total() - led.primary) <= 1e-9 * led.primary
            np.testing.assert_allclose(e, oe, rtol=1e-9, atol=1e-9)
        a.reset_slot(0)
        assert a.read_scoring(0)[0].sum() == 0.0
        a.close()


def test_full_size_config2_properties(ob, calo):
    """Config 2 at the size and launch configuration bench.py times (10 000 x 10 GeV): properties that hold at
    any size (ledger, conservation), and -- random streams being keyed by (event, track, step) -- the first 48
    events transported again in a second slot of the same context must equal the oracle's exactly: every step,
    outcome and secondary counter, deposits to 1e-9."""
    import torch
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field, primaries
    g, _, tabs, scal = calo
    n = 10000
    prim = primaries.beam(n, 10000.0, spread=1.0)
    a = adept.Adept(g, tabs, scal, field.no_field(), track_capacity=1024 * n, n_event_slots=2, time_kernels=1)
    a.set_kernel_timing(False)
    a.enqueue(prim)
    a.transport(0, torch.cuda.current_stream())
    e, led = a.read_scoring(0)
    st = a.stats(0)
    assert led.primary == n * 10000.0
    assert abs(led.total() - led.primary) <= 1e-9 * led.primary
    assert e[:52].sum() == 0 and np.all(e >= 0)
    assert sum(st.outcomes) == sum(st.steps) and st.outcomes[11] == 0
    # the oracle on the first 48 events
    o = ob.Oracle(g, tabs, scal, field.no_field())
    first = {k: v[:48] for k, v in prim.items()}
    oe, ol, ost = o.run(o.make_tracks(first))
    a.enqueue(first, slot=1)
    a.transport(1, torch.cuda.current_stream())
    e1, led1 = a.read_scoring(1)
    st1 = a.stats(1)
    a.close()
    assert list(st1.steps) == list(ost.steps) and list(st1.outcomes) == list(ost.outcomes)
    assert list(st1.secondaries) == list(ost.secondaries)
    np.testing.assert_allclose(e1, oe, rtol=1e-9, atol=1e-9)
    assert led1.escaped == pytest.approx(ol.escaped, rel=1e-9)
    # and the 10 000-event means agree with that sample within its statistical error
    o_ev, _ = _oracle_events(o, o.make_tracks(first), g.n_volumes)
    o_mean, o_err = layer_stats(o_ev)
    gpu_mean = e[52:152].reshape(50, 2).sum(axis=1) / n
    tol = np.maximum(0.005 * o_mean, 3.5 * o_err * np.sqrt(1 + 48 / n))
    assert np.all(np.abs(gpu_mean - o_mean) <= tol)
    assert sum(st.steps) / n == pytest.approx(sum(ost.steps) / 48, rel=0.08)


@pytest.mark.parametrize("chunk", [1, 7, 64])
def test_staggered_injection_gives_the_same_showers(ob, calo, chunk):
    """primaries injected `chunk` per population step instead of all at once.
    Random streams are keyed by (event, track, step), so every shower is the same track for track: equal
    step / outcome / secondary counters, equal deposits up to the order of the fp64 sums, the oracle's
    deposits, and a lower peak population."""
    import torch
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field, primaries
    g, _, tabs, scal = calo
    prim = primaries.beam(96, 500.0, spread=1.0)
    prim["species"][1::3] = 1
    prim["species"][2::3] = 2
    o = ob.Oracle(g, tabs, scal, field.no_field())
    oe, _, ost = o.run(o.make_tracks(prim))
    res = []
    for c in (0, chunk):
        a = adept.Adept(g, tabs, scal, field.no_field(), track_capacity=1 << 17, inject_chunk=c, pending_capacity=128)
        for rep in range(2):       # the slot is reusable after a staggered pass
            a.enqueue(prim)
            a.transport(0, torch.cuda.current_stream())
            e, led = a.read_scoring(0)
            assert abs(led.total() - led.primary) <= 1e-9 * led.primary
            assert led.primary == pytest.approx(sum(500.0 + (2 * M if s == 1 else 0.0) for s in prim["species"]), rel=1e-12)
        st = a.stats(0)
        res.append((e, st))
        if c:
            with pytest.raises(adept.AdeptError):      # more primaries than the pending store holds
                a.enqueue({k: np.concatenate([v, v]) for k, v in prim.items()})
        a.close()
    (e0, s0), (e1, s1) = res
    assert list(s1.steps) == list(s0.steps) == [2 * x for x in ost.steps]
    assert list(s1.outcomes) == list(s0.outcomes) and list(s1.secondaries) == list(s0.secondaries)
    np.testing.assert_allclose(e1, e0, rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(e1, oe, rtol=1e-9, atol=1e-9)
    assert s1.iterations >= s0.iterations
    if chunk < 64:
        assert s1.peak_population < s0.peak_population


def test_hybrid_buffer_threshold_and_flush(ob, calo):
    """tracks handed over one at a time, a batch transported whenever the
    threshold is reached, Flush for the rest; accumulated deposits and ledger equal one transport of all
    tracks (and the oracle's), outgoing tracks are the leaked ones."""
    import torch
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field, primaries
    g, _, tabs, scal = calo
    prim = primaries.beam(50, 300.0, spread=1.0)
    prim["species"][1::3] = 1
    prim["species"][2::3] = 2
    prim["dir"][::7] = [0.0, 1.0, 0.0]            # some tracks start in front of the calorimeter and leave the world
    prim["pos"][::7, 0] = -5.0                    # sideways: outgoing particles
    o = ob.Oracle(g, tabs, scal, field.no_field())
    oe, ol, ost = o.run(o.make_tracks(prim))
    a = adept.Adept(g, tabs, scal, field.no_field(), track_capacity=1 << 16, n_event_slots=2)
    a.enqueue(prim, slot=1)
    a.transport(1, torch.cuda.current_stream())
    e_all, led_all = a.read_scoring(1)
    leaked_all, _ = a.read_leaked(1)
    buf = adept.HybridBuffer(a, threshold=16, slot=0, stream=torch.cuda.current_stream())
    flushed = 0
    for i in range(50):
        flushed += buf.add(prim["event"][i], 0, prim["species"][i], prim["pos"][i], prim["dir"][i], prim["ekin"][i])
    assert flushed == 3 and buf.pending()[0] == 2 and buf.pending()[2] == 3
    assert buf.flush() and not buf.flush()        # Flush transports the remaining two; nothing left afterwards
    assert buf.pending()[0] == 0 and buf.pending()[2] == 4
    e, led, out = buf.take()
    np.testing.assert_allclose(e, e_all, rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(e, oe, rtol=1e-9, atol=1e-9)
    assert led.primary == pytest.approx(led_all.primary, rel=1e-13)
    assert abs(led.total() - led.primary) <= 1e-9 * led.primary
    assert led.escaped == pytest.approx(led_all.escaped, rel=1e-9) and led.escaped == pytest.approx(ol.escaped, rel=1e-9)
    assert len(out) == len(leaked_all) > 0
    key = lambda t: (int(t["event"]), int(t["id"]), int(t["step"]))
    assert sorted(map(key, out)) == sorted(map(key, leaked_all))
    assert sum(float(t["ekin"]) + (2 * M if t["species"] == 1 else 0.0) for t in out) == pytest.approx(led.escaped, rel=1e-9)
    e2, led2, out2 = buf.take()                   # taking clears
    assert e2.sum() == 0.0 and led2.primary == 0.0 and len(out2) == 0
    with pytest.raises(adept.AdeptError):
        buf.add(0, 0, 5, prim["pos"][0], prim["dir"][0], 1.0)
    buf.close()
    a.close()


def test_measurement_modes_do_not_change_the_showers(ob, calo):
    """The measurement switches of the C ABI -- species kernels on one stream or two, CUDA events around every
    launch, the iteration trace -- change the schedule, never the result."""
    import torch
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field, primaries
    g, _, tabs, scal = calo
    prim = primaries.beam(40, 400.0, spread=1.0)
    prim["species"][1::2] = 2
    ref = None
    for conc, timed in ((1, 0), (0, 0), (1, 1), (0, 1)):
        a = adept.Adept(g, tabs, scal, field.no_field(), track_capacity=1 << 16, concurrent_species=conc, time_kernels=timed)
        if not timed:
            with pytest.raises(adept.AdeptError):
                a.set_kernel_timing(True)           # context was not created with time_kernels
        a.enqueue(prim)
        a.iteration_trace()
        a.transport(0, torch.cuda.current_stream())
        e, led = a.read_scoring(0)
        st = a.stats(0)
        t, pop = a.iteration_trace()
        assert len(t) == st.iterations and list(pop[0]) == [20, 0, 20]
        assert (np.diff(t.astype(np.int64)) > 0).all() and pop.sum(axis=1).max() == st.peak_population
        assert len(a.iteration_trace()[0]) == 0     # reading clears
        if timed:
            ms, n = a.kernel_times(0)
            # no field, no BVH: with concurrent species the gamma and the e+- kernel are the blocks of one launch, timed
            # as kernel [0] while [1] stays empty (adept.h); with concurrent_species = 0 all three are launched and timed
            used = [0, 2] if conc else [0, 1, 2]
            assert (n[used] >= st.iterations).all() and (ms[used] > 0).all()
            if conc:
                assert n[1] == 0 and ms[1] == 0
            a.set_kernel_timing(False)
            a.enqueue(prim)
            a.transport(0, torch.cuda.current_stream())
            e2, _ = a.read_scoring(0)
            assert (a.kernel_times(0)[1] == 0).all()
            np.testing.assert_allclose(e2, e, rtol=1e-9, atol=1e-9)
        key = (list(st.steps), list(st.outcomes), list(st.secondaries), st.iterations)
        if ref is None:
            ref = (key, e, led.total())
        else:
            assert key == ref[0]
            np.testing.assert_allclose(e, ref[1], rtol=1e-9, atol=1e-9)
            assert led.total() == pytest.approx(ref[2], rel=1e-12)
        a.close()
