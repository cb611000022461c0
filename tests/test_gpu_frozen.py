"""Frozen single-step parity, CUDA path (through the C ABI) vs oracle, on states drawn from the oracle's
own showers (SURVEY.md §8(d) "parity gates"; BASELINE.json:north_star)."""
import numpy as np
import pytest

from parity import compare_steps

pytestmark = pytest.mark.gpu


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


def _bmax(fld):
    return float(np.abs(fld.bz).max()) if fld.kind == 2 else float(np.linalg.norm(fld.B))


def _run_case(ob, geom_set, fld, prim, per_species, stride, **cfg):
    from paper_2209_15445_b200 import adept
    g, _, tabs, scal = geom_set
    o = ob.Oracle(g, tabs, scal, fld)
    pre = _states(o, prim, per_species, stride)
    counts = np.bincount(pre["species"], minlength=3)
    a = adept.Adept(g, tabs, scal, fld, track_capacity=1 << 12, **cfg)
    res, sec = a.step_frozen(pre)
    a.close()
    ores, osec = o.step(pre)
    flips, worst = compare_steps(pre, res, sec, ores, osec, x0=_x0(g, scal, pre), b_max=_bmax(fld))
    return counts, flips, worst, ores


@pytest.mark.parametrize("bz", [0.0, 1.0])
def test_calorimeter_frozen_steps(ob, calo, bz):
    """Configs 1-3: >= 1e5 states per species; several tiles of 128 threads plus a ragged tail."""
    from paper_2209_15445_b200.inputs import field, primaries
    fld = field.uniform_field(0, 0, bz) if bz else field.no_field()
    prim = primaries.beam(24, 10000.0, spread=1.0)
    prim["species"][1::3] = 1
    prim["species"][2::3] = 2
    counts, flips, worst, ores = _run_case(ob, calo, fld, prim, 100003, 1)
    assert np.all(counts >= 100000), counts
    seen = set(np.unique(ores["outcome"]).tolist())
    assert {0, 1, 2, 3, 4, 5, 6, 7, 9, 10}.issubset(seen), seen      # every process and fate is exercised
    print("flips", flips, "worst scaled errors", worst)


def test_barrel_patch_frozen_steps(ob, barrel_patch):
    """Config 4 ingredients on a 12x12 crystal patch: tubes, rotated boxes, BVH (144 daughters), RK4 field map."""
    from paper_2209_15445_b200.inputs import field, primaries
    prim = primaries.barrel_events(1, 40, 1e3, 2e4, mode="cfg5")
    d = np.array([np.cos(0.1), np.sin(0.1), 0.01])
    prim["dir"][:] = d / np.linalg.norm(d)
    counts, flips, worst, ores = _run_case(ob, barrel_patch, field.solenoid_map(), prim, 40000, 1)
    assert np.all(counts >= 20000), counts
    assert 8 in set(np.unique(ores["outcome"]).tolist())             # truncated (chord budget) steps occur
    print("flips", flips, "worst scaled errors", worst)


def test_full_barrel_sampled_frozen_steps(ob, barrel_full):
    """Config 4 at full size (61 200 crystals): the oracle's loop navigator is slow, so a sample of states
    recorded in the patch geometry is replayed in the full geometry (same shells, mother and crystal
    placement formula; volume ids re-located by the oracle)."""
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field, geometry, materials, primaries
    g, _, tabs, scal = barrel_full
    fld = field.solenoid_map()
    o = ob.Oracle(g, tabs, scal, fld)
    gp = geometry.barrel(n_eta=12, n_phi=12)
    op = ob.Oracle(gp, tabs, scal, fld)
    prim = primaries.barrel_events(1, 12, 1e3, 1e4, mode="cfg5")
    d = np.array([np.cos(0.1), np.sin(0.1), 0.01])
    prim["dir"][:] = d / np.linalg.norm(d)                  # into the patch; states are re-located below
    op.set_recorder(7, 41, 600)
    op.run(op.make_tracks(prim))
    pre = op.recorded()
    keep = []
    for i in range(len(pre)):
        v = o.locate(pre["pos"][i])
        if v >= 0:
            pre["volume"][i] = v
            keep.append(i)
    pre = pre[keep]
    assert len(pre) > 300
    a = adept.Adept(g, tabs, scal, fld, track_capacity=1 << 12)
    res, sec = a.step_frozen(pre)
    a.close()
    ores, osec = o.step(pre)
    flips, worst = compare_steps(pre, res, sec, ores, osec, x0=_x0(g, scal, pre), b_max=_bmax(fld))
    print("flips", flips, "worst scaled errors", worst)


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
    res, sec = a.step_frozen(pre)
    ores, osec = o.step(pre)
    compare_steps(pre, res, sec, ores, osec, flip_budget=0, x0=_x0(g, scal, pre), b_max=_bmax(fld))
    assert set(ores["outcome"][[0, 6, 12]]) == {7} and set(ores["outcome"][[1, 7, 13]]) == {11}
    # an empty batch is a no-op
    r0, s0 = a.step_frozen(np.zeros(0, dtype=ob.TRACK))
    assert len(r0) == 0
    a.close()
