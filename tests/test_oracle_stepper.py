"""Pins of the oracle's step functions and event loop."""
import math

import numpy as np
import pytest

from paper_2209_15445_b200.inputs import field, geometry, materials, primaries

M = 0.51099895


def mk(ob, n, species, ekin, pos=(0.0, 0.0, 0.0), direc=(1.0, 0.0, 0.0), volume=52, event=0):
    t = np.zeros(n, dtype=ob.TRACK)
    t["pos"], t["dir"], t["ekin"] = pos, direc, ekin
    t["id"] = np.arange(n)
    t["event"] = event
    t["volume"] = volume
    t["species"] = species
    return t


def slab(ob, material, half=1e4, **kw):
    """One huge box of `material` (index 0 of its own material list)."""
    g = geometry._finish([0], [(half, half, half)], [0], [-1], np.eye(3).reshape(1, 9), [(0.0, 0, 0)], [material], "slab")
    mats, tabs, scal = materials.build_material_set([material])
    return ob.Oracle(g, tabs, scal, kw.pop("fld", field.no_field()), **kw), mats[0], tabs[0], scal[0]


@pytest.mark.parametrize("fld", ["none", "uniform"])
def test_energy_ledger_closes_per_event(ob, calo, fld):
    """north_star: deposited + escaped + below-cut (+ killed) = primary, to 1e-9 relative, per event."""
    g, _, tabs, scal = calo
    o = ob.Oracle(g, tabs, scal, field.no_field() if fld == "none" else field.uniform_field(0, 0, 1.0))
    prim = primaries.beam(6, 1000.0, spread=1.0)
    prim["species"][1] = 1; prim["species"][2] = 2
    tr = o.make_tracks(prim)
    for i in range(6):
        edep, led, st = o.run(tr[i:i + 1])
        carried = 1000.0 + (2 * M if prim["species"][i] == 1 else 0.0)
        assert led.primary == carried
        assert abs(led.total() - carried) <= 1e-9 * carried
        assert edep.sum() == pytest.approx(led.deposited + led.below_cut, rel=1e-12)
        assert edep[:52].sum() == 0.0                        # vacuum mothers score nothing
        assert led.killed == 0.0 and led.escaped < 0.2 * carried


def test_energy_ledger_closes_per_event_in_the_field_map(ob, barrel_patch):
    """Same invariant through the ORC_FIELD_MAP_RZ branch of the chord loop (RK4, F2' clamp, boundary hits with
    interpolated tangents): tubes, rotated crystals and the solenoid map of configs 4-5, one event at a time."""
    g, _, tabs, scal = barrel_patch
    o = ob.Oracle(g, tabs, scal, field.solenoid_map())
    prim = primaries.barrel_events(5, 5, 500.0, 3000.0, mode="cfg5")     # e-, e-, e+, gamma, gamma per event
    d = np.array([np.cos(0.1), np.sin(0.1), 0.01])
    prim["dir"][:] = d / np.linalg.norm(d)                      # into the 12 x 12 crystal patch
    tr = o.make_tracks(prim)
    chords, in_crystals, photons = 0, 0.0, 0.0
    for e in range(5):
        sel = tr[tr["event"] == e]
        edep, led, st = o.run(sel)
        carried = float(sum(t["ekin"] + (2 * M if t["species"] == 1 else 0.0) for t in sel))
        assert led.primary == pytest.approx(carried, rel=1e-15)
        assert abs(led.total() - carried) <= 1e-9 * carried
        assert edep.sum() == pytest.approx(led.deposited + led.below_cut, rel=1e-12)
        in_crystals += edep[12:].sum()
        photons += float(sel["ekin"][sel["species"] == 2].sum())
        chords += st.chords
    # the photons fly straight into the crystals and shower there; the e+- spiral through the tracker shells
    assert in_crystals > 0.5 * photons and chords > 1000


def test_unscattered_photon_fraction(ob, calo):
    """G pins: fraction of photons crossing the first 5 layers without interacting = exp(-sum Sigma t)."""
    g, _, tabs, scal = calo
    o = ob.Oracle(g, tabs, scal, field.no_field())
    k, n = 2.0, 20000
    sig = [sum(o.lookup(m, t, k) for t in (0, 1, 2)) for m in (1, 2)]
    want = math.exp(-5 * (sig[0] * 0.23 + sig[1] * 0.57))
    tr = mk(ob, n, 2, k)
    alive = np.ones(n, dtype=bool)
    for _ in range(40):                                       # boundary steps only; stop at x >= 4
        idx = np.where(alive & (tr["pos"][:, 0] < 4.0))[0]
        if idx.size == 0:
            break
        res, _ = o.step(tr[idx])
        ok = res["outcome"] == 0
        alive[idx[~ok]] = False
        tr[idx[ok]] = res["post"][ok]
    frac = alive.mean()
    assert abs(frac - want) < 4 * math.sqrt(want * (1 - want) / n)
    assert np.all(tr["ekin"][alive] == k) and np.allclose(tr["dir"][alive], [1.0, 0, 0])


def test_process_fractions_follow_cross_sections(ob):
    o, mat, tab, scal = slab(ob, "Pb")
    k, n = 3.0, 20000
    res, _ = o.step(mk(ob, n, 2, k, volume=0))
    sig = np.array([o.lookup(0, t, k) for t in (0, 1, 2)])
    for proc, s in zip((1, 2, 3), sig):
        f, p = (res["outcome"] == proc).mean(), s / sig.sum()
        assert abs(f - p) < 4.5 * math.sqrt(p * (1 - p) / n)
    # free path is exponential with mean 1/Sigma
    assert res["s"].mean() == pytest.approx(1 / sig.sum(), rel=0.03)


def test_csda_range_with_discrete_processes_closed(ob):
    """An e- below k_c and 2 T_c only loses energy continuously: total path = tabulated range."""
    o, mat, tab, scal = slab(ob, "Pb")
    T0 = 0.15
    assert T0 < scal[2] and T0 < 2 * scal[1]
    tr = mk(ob, 1, 0, T0, volume=0)
    R0 = o.lookup(0, 6, T0)
    path, dep, steps = 0.0, 0.0, 0
    while True:
        res, _ = o.step(tr)
        path += res["s"][0]; dep += res["edep_dep"][0] + res["edep_cut"][0]; steps += 1
        assert res["outcome"][0] in (7, 9)
        if not res["alive"][0]:
            break
        # the step function: s = alpha R + rho (1-alpha)(2 - rho/R) for R > rho, else R
        tr = res["post"].copy()
    assert path == pytest.approx(R0, rel=2e-3)
    assert dep == pytest.approx(T0, rel=1e-12)
    assert steps < 40


def test_step_function_and_loss(ob):
    o, mat, tab, scal = slab(ob, "LAr")
    T = 50.0
    R, S = o.lookup(0, 6, T), o.lookup(0, 5, T)
    res, _ = o.step(mk(ob, 4000, 0, T, volume=0))
    lossy = res["outcome"] == 9
    assert lossy.any()
    s_loss = 0.2 * R + 0.1 * 0.8 * (2 - 0.1 / R)
    np.testing.assert_allclose(res["s"][lossy], s_loss, rtol=1e-13)
    assert res["s"].max() <= s_loss * (1 + 1e-13)
    # energy after a step of length s: R(T') = R(T) - s
    Tn = res["post"]["ekin"][lossy][0]
    assert o.lookup(0, 6, Tn) == pytest.approx(R - s_loss, rel=1e-9)
    # short steps use S*s
    short = (res["s"] <= 0.01 * R) & (res["alive"] == 1)
    if short.any():
        np.testing.assert_allclose(res["edep_dep"][short], S * res["s"][short], rtol=1e-13)


def test_highland_msc_width(ob):
    """P9 pin: <theta^2> = 2 theta0^2 and theta^2/(2 theta0^2) exponential for fixed (T, s)."""
    o, mat, tab, scal = slab(ob, "LAr")
    T = 30.0
    res, _ = o.step(mk(ob, 60000, 0, T, volume=0))
    sel = res["outcome"] == 9                                  # identical step length s_loss
    s = res["s"][sel][0]
    X0 = scal[0]
    pbeta = T * (T + 2 * M) / (T + M)
    beta2 = T * (T + 2 * M) / (T + M) ** 2
    th0 = 13.6 / pbeta * math.sqrt(s / X0) * (1 + 0.038 * math.log(s / (X0 * beta2)))
    th = np.arccos(np.clip(res["post"]["dir"][sel] @ [1.0, 0, 0], -1, 1))
    x = th ** 2 / (2 * th0 ** 2)
    n = sel.sum()
    assert n > 1500
    assert x.mean() == pytest.approx(1.0, abs=4 / math.sqrt(n))
    assert (x > 1).mean() == pytest.approx(math.exp(-1), abs=4 * math.sqrt(0.23 / n))
    phi = np.arctan2(res["post"]["dir"][sel][:, 2], res["post"]["dir"][sel][:, 1])
    assert abs(np.cos(phi).mean()) < 4 / math.sqrt(n) and abs(np.sin(phi).mean()) < 4 / math.sqrt(n)


def test_stopping_and_at_rest_annihilation(ob):
    o, mat, tab, scal = slab(ob, "LAr")
    res, sec = o.step(mk(ob, 2000, 1, 5e-4, volume=0))         # below 1 keV at step start
    assert np.all(res["outcome"] == 7) and np.all(res["alive"] == 0) and np.all(res["n_sec"] == 2)
    np.testing.assert_allclose(res["edep_cut"], 5e-4)
    assert np.all(sec["ekin"] == M) and np.all(sec["species"] == 2)
    np.testing.assert_allclose(sec[:, 0]["dir"], -sec[:, 1]["dir"])
    cz = sec[:, 0]["dir"][:, 2]
    assert abs(cz.mean()) < 4 / math.sqrt(3 * 2000) and abs((cz ** 2).mean() - 1 / 3) < 0.03   # isotropic
    res, sec = o.step(mk(ob, 5, 0, 5e-4, volume=0))
    assert np.all(res["outcome"] == 7) and np.all(res["n_sec"] == 0)
    res, sec = o.step(mk(ob, 5, 2, 5e-4, volume=0))
    assert np.all(res["outcome"] == 7) and np.all(res["edep_cut"] == 5e-4)


def test_vacuum_and_escape(ob):
    o, mat, tab, scal = slab(ob, "vacuum", half=10.0)
    for sp in (0, 1, 2):
        res, _ = o.step(mk(ob, 3, sp, 7.0, volume=0))
        assert np.all(res["outcome"] == 10) and np.all(res["alive"] == 0)
        np.testing.assert_allclose(res["escaped"], 7.0 + (2 * M if sp == 1 else 0))
        np.testing.assert_allclose(res["s"], 10.0)
        assert np.all(res["edep_dep"] == 0) and np.all(res["post"]["dir"] == [1.0, 0, 0])


def test_step_cap_kills_and_books_energy(ob):
    """S4 / PAPER.md:67: unfinished tracks are killed and accounted for."""
    o, mat, tab, scal = slab(ob, "vacuum", half=10.0, max_steps=5)
    t = mk(ob, 2, 1, 3.0, volume=0)
    t["step"] = 5
    res, _ = o.step(t)
    assert np.all(res["outcome"] == 11) and np.all(res["alive"] == 0)
    np.testing.assert_allclose(res["killed"], 3.0 + 2 * M)


def test_pair_threshold_guard(ob, calo):
    """The interpolated pair table is positive just below 2m; the step must not pick pair there."""
    g, _, tabs, scal = calo
    o = ob.Oracle(g, tabs, scal, field.no_field())
    k = 2 * M * (1 - 1e-5)
    assert k < 2 * M and o.lookup(1, 1, k) > 0
    res, _ = o.step(mk(ob, 5000, 2, k, pos=(0.1, 0, 0)))
    assert not np.any(res["outcome"] == 2)
