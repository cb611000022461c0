"""Element-by-element comparison of CUDA step results with the oracle's (DESIGN.md §3 "tolerances").

Discrete outcomes (outcome code, alive flag, secondary count/species/ids, next volume) must be
bit-exact; BASELINE.json:north_star allows a flip only where a sampled value lies within 1e-12 of a
threshold, so a budget of 1e-5 of the batch is tolerated and everything else must be identical.
Continuous outputs agree to 1e-12 relative to the scale of the quantities that enter them: energies
relative to the track's pre-step energy, lengths relative to max(1 cm, |position|, path length),
direction cosines absolute (they are O(1)).

One propagated term is added: the Highland angle (P9) is theta0(s) ~ sqrt(s), so on the very short steps
a track takes right after a boundary (s ~ 1e-9 cm, known to ~1e-15 cm absolute, i.e. 1e-6 relative) a
rounding-level difference in s moves the scattered direction by theta * |ds| / (2 s).  The direction
tolerance therefore adds 8 theta0 (|ds|/s) (1/2 + 0.038/corr), with |ds| the *observed* difference of
the two path lengths (itself bounded by the length tolerance); the energy tolerance adds S_max |ds|.
In a magnetic field the tangent turns at rate kappa = 2.998 |B| / p per cm, and at grazing incidence the
boundary distance amplifies rounding by 1/cos(incidence), so the direction tolerance also adds
kappa_max |ds| (b_max = largest field of the configuration).
"""
import numpy as np

M = 0.51099895
RTOL = 1e-12


S_MAX = 50.0   # MeV/cm, above every restricted stopping power in the tables (used when no dE/dx is given)


def _msc_slack(pre, ores, ds, x0):
    """8 theta0 (|ds|/s) (1/2 + 0.038/corr) for charged steps in matter, else 0."""
    T, s = pre["ekin"], ores["s"]
    with np.errstate(all="ignore"):
        pbeta = T * (T + 2 * M) / (T + M)
        beta2 = T * (T + 2 * M) / (T + M) ** 2
        corr = np.maximum(1e-3, 1 + 0.038 * np.log(s / (x0 * beta2)))
        th0 = 13.6 / pbeta * np.sqrt(s / x0) * corr
        slack = 8 * th0 * (ds / s) * (0.5 + 0.038 / corr)
    charged = (pre["species"] != 2) & np.isfinite(x0) & (s > 0)
    return np.where(charged & np.isfinite(slack), slack, 0.0)


def energy_scale(pre):
    """The energy a track carries into its step: T, or T + 2m for a positron."""
    return pre["ekin"] + np.where(pre["species"] == 1, 2 * M, 0.0)


def compare_steps(pre, res, sec, ores, osec, flip_budget=0.0, x0=None, b_max=0.0, dedx=None):
    """x0: radiation length of each pre-step volume's material (inf for vacuum); None = no MSC slack.
    b_max: largest |B| [T] of the configuration (curvature slack for charged tracks).
    dedx: restricted stopping power S(T0) [MeV/cm] of each pre-step state (0 in vacuum and for photons), the
    factor that carries the observed |ds| into the continuous loss; None = the blanket bound S_MAX.
    flip_budget: fraction of the batch whose discrete outcome may differ (north_star allows a flip only where a
    sampled value lies within 1e-12 of a threshold; none has ever been observed, so the default is 0)."""
    n = len(pre)
    disc = (res["outcome"] != ores["outcome"]) | (res["alive"] != ores["alive"]) | (res["n_sec"] != ores["n_sec"])
    both_alive = (res["alive"] == 1) & (ores["alive"] == 1) & ~disc
    disc |= both_alive & (res["post"]["volume"] != ores["post"]["volume"])
    for k in range(2):
        m = ~disc & (ores["n_sec"] > k)
        disc[m] |= (sec[m, k]["species"] != osec[m, k]["species"]) | (sec[m, k]["id"] != osec[m, k]["id"]) | \
                   (sec[m, k]["volume"] != osec[m, k]["volume"])
    n_flip = int(disc.sum())
    assert n_flip <= int(flip_budget * n), f"{n_flip} discrete mismatches in {n} steps: first {np.where(disc)[0][:5]}"
    ok = ~disc
    e_scale = energy_scale(pre)
    l_scale = np.maximum(1.0, np.maximum(np.abs(pre["pos"]).max(axis=1), ores["s"]))
    worst = {}

    with np.errstate(invalid="ignore"):
        ds = np.where(np.isfinite(ores["s"]), np.abs(res["s"] - ores["s"]), 0.0)
    dir_slack = _msc_slack(pre, ores, ds, x0) if x0 is not None else np.zeros(n)
    e_slack = (S_MAX if dedx is None else 1.001 * dedx) * ds
    if b_max > 0.0:
        pmom = np.sqrt(pre["ekin"] * (pre["ekin"] + 2 * M))
        with np.errstate(all="ignore"):
            dir_slack = dir_slack + np.where(pre["species"] != 2, 2.99792458 * b_max / pmom * ds, 0.0)

    def chk(name, a, b, scale, sel, slack=None):
        if not sel.any():
            return
        err = np.abs(a[sel] - b[sel])
        if err.ndim > 1:
            err = err.max(axis=1)
        if slack is not None:
            err = np.maximum(err - slack[sel], 0.0)
        rel = err / scale[sel]
        worst[name] = float(rel.max())
        assert rel.max() <= RTOL, f"{name}: max scaled error {rel.max():.3e} at step {np.where(sel)[0][rel.argmax()]}"

    alive = ok & (ores["alive"] == 1)
    one = np.ones(n)
    chk("pos", res["post"]["pos"], ores["post"]["pos"], l_scale, alive)
    chk("dir", res["post"]["dir"], ores["post"]["dir"], one, alive, dir_slack)
    chk("ekin", res["post"]["ekin"], ores["post"]["ekin"], e_scale, alive, e_slack)
    assert np.array_equal(res["post"]["step"][alive], ores["post"]["step"][alive])
    for f in ("edep_dep", "edep_cut", "escaped", "killed"):
        chk(f, res[f], ores[f], e_scale, ok, e_slack)
    chk("s", res["s"], ores["s"], l_scale, ok & np.isfinite(ores["s"]))
    assert np.array_equal(res["chords"][ok], ores["chords"][ok])
    for k in range(2):
        m = ok & (ores["n_sec"] > k)
        chk(f"sec{k}.ekin", sec[:, k]["ekin"], osec[:, k]["ekin"], e_scale, m, e_slack)
        chk(f"sec{k}.dir", sec[:, k]["dir"], osec[:, k]["dir"], one, m, dir_slack)
        chk(f"sec{k}.pos", sec[:, k]["pos"], osec[:, k]["pos"], l_scale, m)
    return n_flip, worst


def _key(t):
    """(event, id, step) of every track as one structured key array."""
    k = np.zeros(len(t), dtype=[("event", "u4"), ("id", "u8"), ("step", "u4")])
    k["event"], k["id"], k["step"] = t["event"], t["id"], t["step"]
    return k


def compare_population(pre, out, ores, osec, x0=None, b_max=0.0, dedx=None):
    """One population step of the transport kernels (adept_step_population) against the oracle's orc_step of the
    same pre-step states.  `out` is the next population the kernels wrote (survivors and secondaries, any
    order).  Tracks are matched by (event, id, step): a survivor of (e, i, s) is (e, i, s + 1), a secondary
    carries the child id the oracle derives from its parent's stream and step 0.  Discrete results -- which
    tracks exist, their species and volume -- must be identical; positions, directions and energies agree to
    1e-12 of the scale of what enters them, with the same first-order propagation of the path difference as
    compare_steps.  The population carries no path length, so |ds| is bounded from the positions: the observed
    end-point difference (a track's end point is its start plus s times a unit vector) plus one unit in the last
    place of the largest coordinate -- a distance to a boundary is a difference of coordinates of that size and
    cannot be known better, whoever computes it (the steps of 1e-9 cm right after a boundary, at |x| ~ 150 cm,
    have |ds| ~ 2e-15 cm = 0.1 ulp(x) and a Highland angle that moves by theta |ds| / (2 s) ~ 1e-9).
    Returns ds per pre-step state (for the deposit tolerances) and the worst errors."""
    n = len(pre)
    exp_t, exp_parent, exp_kind = [], [], []
    alive = ores["alive"] == 1
    exp_t.append(ores["post"][alive]); exp_parent.append(np.where(alive)[0]); exp_kind.append(np.zeros(alive.sum(), dtype=int))
    for k in range(2):
        m = ores["n_sec"] > k
        exp_t.append(osec[m, k]); exp_parent.append(np.where(m)[0]); exp_kind.append(np.full(m.sum(), 1 + k))
    exp_t, exp_parent, exp_kind = np.concatenate(exp_t), np.concatenate(exp_parent), np.concatenate(exp_kind)
    ke, kg = _key(exp_t), _key(out)
    assert len(np.unique(ke)) == len(ke), "oracle keys are not unique"
    assert len(np.unique(kg)) == len(kg), "the kernels wrote a track twice"
    oe, og = np.argsort(ke, order=("event", "id", "step")), np.argsort(kg, order=("event", "id", "step"))
    missing = np.setdiff1d(ke, kg)
    extra = np.setdiff1d(kg, ke)
    assert len(missing) == 0 and len(extra) == 0, f"{len(missing)} tracks missing, {len(extra)} unexpected: {missing[:3]} {extra[:3]}"
    e, g, parent = exp_t[oe], out[og], exp_parent[oe]
    assert np.array_equal(_key(e), _key(g))
    assert np.array_equal(e["species"], g["species"]), "species of a matched track differs"
    bad_vol = e["volume"] != g["volume"]
    assert not bad_vol.any(), f"{bad_vol.sum()} matched tracks in a different volume: parents {parent[bad_vol][:5]}"
    p = pre[parent]
    e_scale = energy_scale(p)
    l_scale = np.maximum(1.0, np.maximum(np.abs(p["pos"]).max(axis=1), np.where(np.isfinite(ores["s"][parent]), ores["s"][parent], 0.0)))
    dpos = np.linalg.norm(g["pos"] - e["pos"], axis=1)
    ds_pre = np.zeros(n)
    np.maximum.at(ds_pre, parent, dpos)
    ds_pre += np.spacing(np.abs(pre["pos"]).max(axis=1))
    ds = ds_pre[parent]
    dir_slack = _msc_slack(p, ores[parent], ds, x0[parent]) if x0 is not None else np.zeros(len(e))
    if b_max > 0.0:
        pmom = np.sqrt(p["ekin"] * (p["ekin"] + 2 * M))
        with np.errstate(all="ignore"):
            dir_slack = dir_slack + np.where(p["species"] != 2, 2.99792458 * b_max / pmom * ds, 0.0)
    e_slack = (S_MAX if dedx is None else 1.001 * dedx[parent]) * ds
    worst = {}
    for name, err, scale, slack in (("pos", np.abs(g["pos"] - e["pos"]).max(axis=1), l_scale, None),
                                    ("dir", np.abs(g["dir"] - e["dir"]).max(axis=1), np.ones(len(e)), dir_slack),
                                    ("ekin", np.abs(g["ekin"] - e["ekin"]), e_scale, e_slack)):
        if slack is not None:
            err = np.maximum(err - slack, 0.0)
        rel = err / scale
        worst[name] = float(rel.max()) if len(rel) else 0.0
        assert worst[name] <= RTOL, f"{name}: max scaled error {worst[name]:.3e} for the track of parent {parent[rel.argmax()]}"
    return ds_pre, worst


def deposit_tolerance(pre, ds, dedx=None):
    """Per pre-step state: the tolerance on what its step deposits (1e-12 of the carried energy plus S |ds|)."""
    return RTOL * energy_scale(pre) + (S_MAX if dedx is None else 1.001 * dedx) * ds


def layer_stats(edep_events, first_slab=52, n_layers=50):
    """per-event edep arrays [n_events, n_vol] -> (mean per layer, std error per layer)."""
    lay = edep_events[:, first_slab:first_slab + 2 * n_layers].reshape(edep_events.shape[0], n_layers, 2).sum(axis=2)
    return lay.mean(axis=0), lay.std(axis=0, ddof=1) / np.sqrt(lay.shape[0])
