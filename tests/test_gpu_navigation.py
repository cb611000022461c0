"""Navigation parity: the warp-cooperative BVH navigator must return exactly what the loop navigator
returns (a min over the same set), and both must match the oracle (rows A4, A5)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _rays(rng, n, r_lo, r_hi, phi_hi, z_half):
    r, phi, z = rng.uniform(r_lo, r_hi, n), rng.uniform(0, phi_hi, n), rng.uniform(-z_half, z_half, n)
    pos = np.stack([r * np.cos(phi), r * np.sin(phi), z], axis=1)
    d = rng.normal(size=(n, 3))
    return pos, d / np.linalg.norm(d, axis=1, keepdims=True)


def test_full_barrel_bvh_equals_loop_bit_for_bit(barrel_full):
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field
    g, _, tabs, scal = barrel_full
    a = adept.Adept(g, tabs, scal, field.no_field(), track_capacity=1 << 10)
    rng = np.random.default_rng(1)
    n = 4099                                            # several tiles and a ragged tail
    pos, d = _rays(rng, n, 127.6, 152.9, 2 * np.pi, 289.0)
    vol_bvh = a.locate_batch(pos, adept.NAV_BVH)
    vol_loop = a.locate_batch(pos, adept.NAV_LOOP)
    assert np.array_equal(vol_bvh, vol_loop)
    assert (vol_bvh >= 12).sum() > 1000 and (vol_bvh == 11).sum() > 200
    smax = np.where(rng.random(n) < 0.3, rng.uniform(0.01, 5.0, n), np.inf)
    s_bvh = a.distance_batch(pos, d, vol_bvh, smax, adept.NAV_BVH)
    s_loop = a.distance_batch(pos, d, vol_bvh, smax, adept.NAV_LOOP)
    assert np.array_equal(s_bvh, s_loop)               # bit-exact
    assert np.all(s_bvh <= smax) and np.all(s_bvh >= 0) and np.all(np.isfinite(s_bvh[np.isfinite(smax)]))
    # rays started in the mother volume (gaps between crystals) exercise the BVH ray query
    in_gap = vol_bvh == 11
    assert np.array_equal(s_bvh[in_gap], s_loop[in_gap]) and in_gap.sum() > 100
    # points outside the world
    out = a.locate_batch(np.array([[400.0, 0, 0], [0, 0, 301.0]]), adept.NAV_BVH)
    assert list(out) == [-1, -1]
    a.close()


def test_navigation_matches_oracle(ob, barrel_patch, calo):
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field
    rng = np.random.default_rng(2)
    for geom_set, args in ((barrel_patch, (110.0, 160.0, 0.22, 20.0)), (barrel_patch, (0.0, 120.0, 2 * np.pi, 290.0))):
        g, _, tabs, scal = geom_set
        o = ob.Oracle(g, tabs, scal, field.no_field())
        a = adept.Adept(g, tabs, scal, field.no_field(), track_capacity=1 << 10)
        n = 1500
        pos, d = _rays(rng, n, *args)
        vol = a.locate_batch(pos)
        want = np.array([o.locate(p) for p in pos])
        assert np.array_equal(vol, want)
        s = a.distance_batch(pos, d, vol)
        ws = np.array([o.distance(pos[i], d[i], int(vol[i])) for i in range(n)])
        np.testing.assert_allclose(s, ws, rtol=0, atol=1e-12 * 300.0)
        a.close()
    g, _, tabs, scal = calo
    o = ob.Oracle(g, tabs, scal, field.no_field())
    a = adept.Adept(g, tabs, scal, field.no_field(), track_capacity=1 << 10)
    pos = np.stack([rng.uniform(-19, 59, 2000), rng.uniform(-29, 29, 2000), rng.uniform(-29, 29, 2000)], axis=1)
    d = rng.normal(size=(2000, 3)); d /= np.linalg.norm(d, axis=1, keepdims=True)
    vol = a.locate_batch(pos)
    assert np.array_equal(vol, np.array([o.locate(p) for p in pos]))
    s = a.distance_batch(pos, d, vol)
    ws = np.array([o.distance(pos[i], d[i], int(vol[i])) for i in range(2000)])
    np.testing.assert_allclose(s, ws, rtol=0, atol=1e-12 * 60.0)
    a.close()


@pytest.mark.parametrize("navigator", [1, 0])
def test_relocation_from_any_volume_equals_locate(ob, barrel_full, calo, navigator):
    """A5: the move kernel relocates locally (climb from the old volume, then descend, neighbours of the
    daughter just left first).  Whatever volume the climb starts from, the answer must be Locate(q) from
    the world down, which is the oracle's only relocation routine."""
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field
    rng = np.random.default_rng(7)
    # calorimeter: points anywhere in the world, starts in every kind of volume (world, box, layer, slab)
    g, _, tabs, scal = calo
    o = ob.Oracle(g, tabs, scal, field.no_field())
    a = adept.Adept(g, tabs, scal, field.no_field(), track_capacity=1 << 10, navigator=navigator)
    n = 4099
    pos = np.stack([rng.uniform(-21, 61, n), rng.uniform(-31, 31, n), rng.uniform(-31, 31, n)], axis=1)
    # half the points sit a push (1e-7 cm) past a slab face, where real relocations happen
    k = rng.integers(0, 50, n // 2)
    pos[: n // 2, 0] = 0.8 * k + rng.choice([0.0, 0.23], n // 2) + rng.choice([-1e-7, 1e-7], n // 2)
    pos[: n // 2, 1:] = rng.uniform(-19.9, 19.9, (n // 2, 2))
    frm = rng.integers(0, g.n_volumes, n)
    want = a.locate_batch(pos, navigator)
    assert np.array_equal(want[:600], np.array([o.locate(p) for p in pos[:600]]))
    assert np.array_equal(a.relocate_batch(pos, frm, navigator), want)
    # neighbouring start volumes (the common case): slab of the previous / next layer
    near = np.clip(want + rng.choice([-2, -1, 1, 2], n), 52, g.n_volumes - 1)
    assert np.array_equal(a.relocate_batch(pos, near, navigator), want)
    assert (want < 0).sum() > 10 and (want >= 52).sum() > 1000
    # relocation hints (the volume beyond each box face, built by adept_init) are candidates that are
    # verified: any face, right or wrong, from any volume gives Locate(q)
    for f in (0, 1, 2, 5):
        assert np.array_equal(a.relocate_batch(pos, near, navigator, face=f), want)
    assert np.array_equal(a.relocate_batch(pos, frm, navigator, face=rng.integers(-1, 6, n)), want)
    # the right face: a point a push beyond the +x / -x face of slab v is in the next / previous slab
    slabs = np.arange(52, g.n_volumes - 1)
    px = np.array([g.trans[v][0] + g.dims[v][0] + 1e-7 for v in slabs])
    q = np.stack([px, rng.uniform(-19, 19, len(slabs)), rng.uniform(-19, 19, len(slabs))], axis=1)
    assert np.array_equal(a.relocate_batch(q, slabs, navigator, face=1), slabs + 1)
    assert np.array_equal(a.locate_batch(q, navigator), slabs + 1)
    a.close()
    # barrel: crystals (BVH mother), gaps, shells, outside
    g, _, tabs, scal = barrel_full
    a = adept.Adept(g, tabs, scal, field.no_field(), track_capacity=1 << 10, navigator=navigator)
    n = 3001 if navigator == 1 else 257
    pos, _ = _rays(rng, n, 0.0, 305.0, 2 * np.pi, 305.0)
    pos[: n // 2], _ = _rays(rng, n // 2, 127.6, 152.9, 2 * np.pi, 289.0)
    frm = rng.integers(0, g.n_volumes, n)
    want = a.locate_batch(pos, navigator)
    assert np.array_equal(a.relocate_batch(pos, frm, navigator), want)
    assert np.array_equal(a.relocate_batch(pos, np.maximum(want, 0), navigator), want)
    assert np.array_equal(a.relocate_batch(pos, np.maximum(want, 0), navigator, face=rng.integers(-1, 6, n)), want)
    a.close()


def _oracle_raycast(o, scal, g, pos, direc, max_crossings=10000, eps=1e-7):
    """The same march with the oracle's Locate and loop-navigator distance (G3-G5), one ray at a time."""
    col, nx = np.zeros(len(pos)), np.zeros(len(pos), dtype=np.int32)
    for i, (p, d) in enumerate(zip(pos, direc)):
        p = p.copy()
        v = o.locate(p)
        if v < 0:
            nx[i] = -1
            continue
        while v >= 0 and nx[i] < max_crossings:
            s = o.distance(p, d, v)
            col[i] += s * scal[g.material[v]][7]
            p = p + s * d
            p = p + eps * d
            nx[i] += 1
            v = o.locate(p)
    return col, nx


def test_raycast_validator(ob, barrel_patch, barrel_full, tmp_path):
    """SURVEY.md 8(f)3 / PAPER.md:49, Fig. 1: a picture of the geometry taken with the navigation calls of the
    transport path.  Patch: equals the oracle's march (crossings exact, column density to rounding).  Full
    barrel: the BVH picture equals the loop navigator's picture bit for bit; PPM written headless."""
    from paper_2209_15445_b200 import adept, raycast
    from paper_2209_15445_b200.inputs import field
    g, _, tabs, scal = barrel_patch
    o = ob.Oracle(g, tabs, scal, field.no_field())
    a = adept.Adept(g, tabs, scal, field.no_field(), track_capacity=1 << 10)
    rng = np.random.default_rng(11)
    # rays from the origin into the patch (12 x 12 crystals around eta = 0, phi = 0..12 columns), and a few away from it
    phi = rng.uniform(-0.02, 0.23, 300)
    eta = rng.uniform(-0.12, 0.12, 300)
    th = 2.0 * np.arctan(np.exp(-eta))
    d = np.stack([np.sin(th) * np.cos(phi), np.sin(th) * np.sin(phi), np.cos(th)], axis=1)
    d[-20:] = -d[-20:]
    pos = np.zeros_like(d)
    pos[-5:] = [400.0, 0.0, 0.0]                       # outside the world
    col, nx, _ = a.raycast(pos, d, adept.NAV_BVH)
    ocol, onx = _oracle_raycast(o, scal, g, pos, d)
    assert np.array_equal(nx, onx) and (nx[-5:] == -1).all() and nx[:280].max() >= 8
    np.testing.assert_allclose(col, ocol, rtol=1e-12, atol=1e-12)
    col2, nx2, _ = a.raycast(pos, d, adept.NAV_LOOP)
    assert np.array_equal(nx2, nx) and np.array_equal(col2, col)
    a.close()
    # full barrel: BVH == loop, bit for bit, on an eta-phi picture
    g, _, tabs, scal = barrel_full
    a = adept.Adept(g, tabs, scal, field.no_field(), track_capacity=1 << 10)
    w, h = 96, 40
    p, d = raycast.barrel_rays(w, h)
    cb, nb, _ = a.raycast(p, d, adept.NAV_BVH)
    cl, nl, _ = a.raycast(p, d, adept.NAV_LOOP)
    assert np.array_equal(nb, nl) and np.array_equal(cb, cl)
    inside = np.abs(-1.45 + (np.arange(h) + 0.5) * 2.9 / h) < 1.3
    # 10 shells in and out, mother, at least one crystal, mother, world; >= 20 cm of PbWO4 on a line of sight of the
    # barrel; the crystals point at the origin and cover 97.7 % of the row / column pitch, so about one pixel in
    # twenty looks straight down a gap between them
    assert (nb.reshape(h, w)[inside] >= 23).mean() > 0.9
    assert (cb.reshape(h, w)[inside] > 8.28 * 20.0).mean() > 0.9
    assert (nb.reshape(h, w)[inside] >= 21).all()      # every line of sight crosses the ten shells and enters the mother
    out = tmp_path / "barrel.ppm"
    raycast.write_ppm(str(out), cb, w, h)
    data = out.read_bytes()
    assert data.startswith(b"P6\n96 40\n255\n") and len(data) == len(b"P6\n96 40\n255\n") + 3 * w * h
    a.close()


def test_single_precision_geometry_raycast(ob, barrel_patch, barrel_full):
    """the single-precision geometry mode (every solid, transform and BVH box in
    fp32) validated the paper's way, by comparing its ray-cast picture with the double-precision one, and against the
    oracle's march.  fp32 positions at r ~ 150 cm resolve 1.5e-5 cm and the fp32 march pushes 1e-3 cm past every
    boundary, so per crossing a path length is off by at most the push plus a few spacings: the column density agrees
    within crossings x (1e-3 + 2e-4) cm x the largest density, and the crossing count is the same except on rays
    that graze an edge within that distance."""
    from paper_2209_15445_b200 import adept, raycast
    from paper_2209_15445_b200.inputs import field
    rho_max = 8.28
    # patch: against the oracle's fp64 march
    g, _, tabs, scal = barrel_patch
    o = ob.Oracle(g, tabs, scal, field.no_field())
    a = adept.Adept(g, tabs, scal, field.no_field(), track_capacity=1 << 10)
    rng = np.random.default_rng(12)
    phi, eta = rng.uniform(-0.02, 0.23, 300), rng.uniform(-0.12, 0.12, 300)
    th = 2.0 * np.arctan(np.exp(-eta))
    d = np.stack([np.sin(th) * np.cos(phi), np.sin(th) * np.sin(phi), np.cos(th)], axis=1)
    pos = np.zeros_like(d)
    ocol, onx = _oracle_raycast(o, scal, g, pos, d)
    for nav in (adept.NAV_BVH_F32, adept.NAV_LOOP_F32):
        col, nx, _ = a.raycast(pos, d, nav)
        same = nx == onx
        assert same.mean() > 0.97, same.mean()
        tol = (np.maximum(nx, onx) + 1) * 1.2e-3 * rho_max
        assert np.all(np.abs(col - ocol)[same] <= tol[same]), np.abs(col - ocol)[same].max()
    cb, nb, _ = a.raycast(pos, d, adept.NAV_BVH_F32)
    cl, nl, _ = a.raycast(pos, d, adept.NAV_LOOP_F32)
    assert np.array_equal(nb, nl) and np.array_equal(cb, cl)      # the fp32 BVH culls, the fp32 solids decide
    a.close()
    # full barrel: fp32 picture against the fp64 picture, pixel for pixel
    g, _, tabs, scal = barrel_full
    a = adept.Adept(g, tabs, scal, field.no_field(), track_capacity=1 << 10)
    w, h = 256, 96
    p, d = raycast.barrel_rays(w, h)
    c64, n64, ms64 = a.raycast(p, d, adept.NAV_BVH)
    c32, n32, ms32 = a.raycast(p, d, adept.NAV_BVH_F32)
    same = n64 == n32
    assert same.mean() > 0.98, same.mean()
    tol = (n64 + 1) * 1.2e-3 * rho_max
    assert np.all(np.abs(c32 - c64)[same] <= tol[same])
    assert np.abs(c32 - c64)[same].max() > 0.0                    # it really is another arithmetic
    # pictures agree to a grey level almost everywhere (a differing pixel is a ray down an edge of a crystal)
    top = c64.max()
    assert (np.abs(c32 - c64) > top / 255.0).mean() < 0.02
    print(f"ray-cast {w}x{h}: fp64 {ms64:.2f} ms, fp32 {ms32:.2f} ms, ratio {ms64 / ms32:.2f}; same crossings {same.mean():.4f}")
    a.close()
