"""Pins of the oracle's solids, loop navigator and Locate."""
import ctypes
import math

import numpy as np
import pytest

from paper_2209_15445_b200.inputs import field


def _p(a):
    # data_as keeps the (possibly temporary) array alive for the duration of the call
    return np.ascontiguousarray(a, dtype=np.float64).ctypes.data_as(ctypes.c_void_p)


def _rand_dirs(rng, n):
    v = rng.normal(size=(n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


def _inside_solid(solid, dims, p):
    if solid == 0:
        return bool(np.all(np.abs(p) <= dims))
    r2 = p[0] ** 2 + p[1] ** 2
    return dims[0] ** 2 <= r2 <= dims[1] ** 2 and abs(p[2]) <= dims[2]


def _march(solid, dims, p, d, want_inside, tmax, n=1500):
    """First parameter t in (0, tmax] where inside() becomes `want_inside`, by dense march + bisection."""
    ts = np.linspace(0, tmax, n + 1)
    prev = 0.0
    for t in ts[1:]:
        if _inside_solid(solid, dims, p + t * d) == want_inside:
            lo, hi = prev, t
            for _ in range(60):
                mid = 0.5 * (lo + hi)
                if _inside_solid(solid, dims, p + mid * d) == want_inside:
                    hi = mid
                else:
                    lo = mid
            return hi
        prev = t
    return math.inf


@pytest.mark.parametrize("solid,dims", [(0, (1.1, 1.1, 11.5)), (0, (0.115, 20.0, 20.0)),
                                         (1, (0.0, 3.0, 5.0)), (1, (2.0, 2.5, 4.0)), (1, (50.0, 50.03, 280.0))])
def test_solid_distances_against_ray_march(ob, solid, dims):
    rng = np.random.default_rng(11)
    dims = np.array(dims)
    ext = np.array([dims[0], dims[1], dims[2]]) if solid == 0 else np.array([dims[1], dims[1], dims[2]])
    n_in = n_out = 0
    for it in range(200):
        p = (rng.random(3) * 2 - 1) * ext * 1.6
        if it % 2 == 0:                                    # force a point inside the solid
            if solid == 0:
                p = (rng.random(3) * 2 - 1) * dims
            else:
                r, phi = rng.uniform(dims[0], dims[1]), rng.uniform(0, 2 * math.pi)
                p = np.array([r * math.cos(phi), r * math.sin(phi), rng.uniform(-dims[2], dims[2])])
        d = _rand_dirs(rng, 1)[0]
        if _inside_solid(solid, dims, p):
            got = ob.lib.orc_solid_exit(solid, _p(dims), _p(p), _p(d))
            want = _march(solid, dims, p, d, False, 4 * np.linalg.norm(ext))
            n_in += 1
        else:
            got = ob.lib.orc_solid_entry(solid, _p(dims), _p(p), _p(d))
            want = _march(solid, dims, p, d, True, 6 * np.linalg.norm(ext))
            n_out += 1
        if math.isinf(want):
            # the march may step over a grazing hit shorter than its resolution; a reported hit must be real
            if not math.isinf(got):
                assert _inside_solid(solid, dims, p + (got + 1e-9) * d) or _inside_solid(solid, dims, p + (got - 1e-9) * d)
        else:
            assert got <= want + 1e-9
            if abs(got - want) > 1e-7:   # an earlier, thinner crossing the march missed
                assert _inside_solid(solid, dims, p + (got + 1e-9) * d) != _inside_solid(solid, dims, p + (got - 1e-9) * d)
    assert n_in > 20 and n_out > 20


def test_tube_analytic_cases(ob):
    dims = np.array([2.0, 3.0, 5.0])
    z = np.zeros(3)
    # from the axis along +x: enters at rmin; from inside the wall: exits at rmax / re-enters the hole at rmin
    assert ob.lib.orc_solid_entry(1, _p(dims), _p(z), _p([1.0, 0, 0])) == pytest.approx(2.0, abs=1e-14)
    assert ob.lib.orc_solid_exit(1, _p(dims), _p([2.5, 0, 0]), _p([1.0, 0, 0])) == pytest.approx(0.5, abs=1e-14)
    assert ob.lib.orc_solid_exit(1, _p(dims), _p([2.5, 0, 0]), _p([-1.0, 0, 0])) == pytest.approx(0.5, abs=1e-14)
    assert ob.lib.orc_solid_exit(1, _p(dims), _p([2.5, 0, 1.0]), _p([0, 0, 1.0])) == pytest.approx(4.0, abs=1e-14)
    # from outside through the end cap, and a miss through the hole
    assert ob.lib.orc_solid_entry(1, _p(dims), _p([2.5, 0, 9.0]), _p([0, 0, -1.0])) == pytest.approx(4.0, abs=1e-14)
    assert math.isinf(ob.lib.orc_solid_entry(1, _p(dims), _p([0.5, 0, 9.0]), _p([0, 0, -1.0])))
    # tangent-free chord through the wall from outside
    assert ob.lib.orc_solid_entry(1, _p(dims), _p([10.0, 0, 0]), _p([-1.0, 0, 0])) == pytest.approx(7.0, abs=1e-14)
    # oblique ray from the axis: hits the inner cylinder at slant length rmin / sin(theta)
    th = 0.7
    assert ob.lib.orc_solid_entry(1, _p(dims), _p(z), _p([math.sin(th), 0, math.cos(th)])) == pytest.approx(2.0 / math.sin(th), rel=1e-14)


def test_box_analytic_cases(ob):
    dims = np.array([1.0, 2.0, 3.0])
    assert ob.lib.orc_solid_exit(0, _p(dims), _p([0.25, 0, 0]), _p([1.0, 0, 0])) == 0.75
    assert ob.lib.orc_solid_entry(0, _p(dims), _p([-5.0, 0, 0]), _p([1.0, 0, 0])) == 4.0
    assert math.isinf(ob.lib.orc_solid_entry(0, _p(dims), _p([-5.0, 2.5, 0]), _p([1.0, 0, 0])))
    assert math.isinf(ob.lib.orc_solid_entry(0, _p(dims), _p([-5.0, 0, 0]), _p([-1.0, 0, 0])))
    assert ob.lib.orc_solid_entry(0, _p(dims), _p([0.5, 0, 0]), _p([0, 1.0, 0])) == 0.0
    # a point a hair outside: exit distance is clamped at zero (G3 reading in DESIGN.md)
    assert ob.lib.orc_solid_exit(0, _p(dims), _p([1.0 + 1e-12, 0, 0]), _p([1.0, 0, 0])) == 0.0


def test_calorimeter_boundaries_are_analytic(ob, calo):
    """Along +x the boundaries sit at x = 0.8 i and 0.8 i + 0.23 (SURVEY.md §8(c) G pins)."""
    g, _, tabs, scal = calo
    o = ob.Oracle(g, tabs, scal, field.no_field())
    x, d = 1e-7, np.array([1.0, 0, 0])
    vol = o.locate([x, 0.3, -0.2])
    assert vol == 52
    bounds = []
    for _ in range(101):
        s = o.distance([x, 0.3, -0.2], d, vol)
        bounds.append(x + s)
        x = x + s + 1e-7
        vol = o.locate([x, 0.3, -0.2])
    want = sorted([0.8 * i + 0.23 for i in range(50)] + [0.8 * (i + 1) for i in range(50)]) + [60.0]
    np.testing.assert_allclose(bounds, want, atol=1e-9)
    assert vol == -1                                         # left the world at x = 60
    assert o.locate([45.0, 0, 0]) == 0 and o.locate([20.0, 25.0, 0]) == 0 and o.locate([20.0, 31.0, 0]) == -1
    # an oblique ray: the distance scales with 1/cos
    dd = np.array([math.cos(0.3), math.sin(0.3), 0.0])
    assert o.distance([0.05, 0, 0], dd, 52) == pytest.approx(0.18 / math.cos(0.3), rel=1e-13)
    # s_max caps the result
    assert o.distance([0.05, 0, 0], d, 52, 0.01) == 0.01


def _brute_locate(o, g, p):
    """Deepest touchable containing p whose whole ancestor chain contains p."""
    best, best_depth = -1, -1
    for v in range(g.n_volumes):
        if not o.inside(p, v):
            continue
        depth, m, ok = 0, g.mother[v], True
        while m >= 0:
            ok = ok and o.inside(p, m)
            m = g.mother[m]
            depth += 1
        if ok and depth > best_depth:
            best, best_depth = v, depth
    return best


def test_locate_against_brute_force(ob, calo, barrel_patch):
    rng = np.random.default_rng(3)
    g, _, tabs, scal = calo
    o = ob.Oracle(g, tabs, scal, field.no_field())
    for _ in range(300):
        p = np.array([rng.uniform(-25, 65), rng.uniform(-32, 32), rng.uniform(-32, 32)])
        assert o.locate(p) == _brute_locate(o, g, p)
    g, _, tabs, scal = barrel_patch
    o = ob.Oracle(g, tabs, scal, field.no_field())
    hits = 0
    for _ in range(400):
        r, phi, z = rng.uniform(120, 160), rng.uniform(-0.02, 0.25), rng.uniform(-15, 15)
        p = np.array([r * math.cos(phi), r * math.sin(phi), z])
        v = o.locate(p)
        assert v == _brute_locate(o, g, p)
        hits += v >= 12
    assert hits > 50
    for r in (3.01, 14.9, 110.02):                            # inside Si shells
        assert 1 <= o.locate([r, 0, 0]) <= 10


def test_loop_navigator_in_barrel_patch(ob, barrel_patch):
    """From the origin towards a crystal centre: shells at their radii, mother at 127.5, crystal face at 129."""
    g, _, tabs, scal = barrel_patch
    o = ob.Oracle(g, tabs, scal, field.no_field())
    c = 12 + 6 * 12 + 5                                       # a crystal near eta = 0
    axis = g.rot[c].reshape(3, 3)[:, 2]
    front = g.trans[c] - 11.5 * axis
    d = front / np.linalg.norm(front)
    p, vol, seen = np.zeros(3), 0, []
    for _ in range(40):
        s = o.distance(p, d, vol)
        p = p + (s + 1e-7) * d
        seen.append((vol, np.linalg.norm(p)))
        vol = o.locate(p)
        if vol == c:
            break
    assert vol == c
    radii = [r for v, r in seen if v == 0]
    sin_t = math.hypot(d[0], d[1])
    want = [(3.0 + 107.0 * i / 9.0) / sin_t for i in range(10)] + [127.5 / sin_t]
    np.testing.assert_allclose(radii, want, atol=1e-6)
    assert np.linalg.norm(p) == pytest.approx(np.linalg.norm(front), abs=1e-6)
    # through the crystal along its axis: 23 cm
    assert o.distance(p, axis, c) == pytest.approx(23.0, abs=1e-5)
