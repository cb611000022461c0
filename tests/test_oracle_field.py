"""Pins of the oracle's field propagation."""
import ctypes
import math

import numpy as np
import pytest

from paper_2209_15445_b200.inputs import field, geometry, materials

M = 0.51099895
CB = 2.99792458


def _p(a):
    return np.ascontiguousarray(a, dtype=np.float64).ctypes.data_as(ctypes.c_void_p)


def helix(ob, B, q, pmom, h, p, d):
    p1, d1 = np.zeros(3), np.zeros(3)
    ob.lib.orc_helix(_p(B), q, pmom, h, _p(p), _p(d), _p(p1), _p(d1))
    return p1, d1


def test_helix_is_the_analytic_circle(ob):
    B, pm = np.array([0.0, 0.0, 1.0]), 100.0
    R = pm / (CB * 1.0)                                       # 33.356 cm
    p0, d0 = np.zeros(3), np.array([1.0, 0.0, 0.0])
    for q in (-1, +1):
        # e- (q=-1) in +z field turns towards +y: centre (0, -q R ... ) -> check via the circle equation
        centre = np.array([0.0, -q * R, 0.0])
        for h in (0.1, 5.0, 60.0, 200.0):
            p1, d1 = helix(ob, B, q, pm, h, p0, d0)
            assert np.linalg.norm(p1 - centre) == pytest.approx(R, rel=1e-13)
            ang = h / R
            np.testing.assert_allclose(p1, [R * math.sin(ang), -q * R * (1 - math.cos(ang)), 0.0], atol=1e-11)
            np.testing.assert_allclose(d1, [math.cos(ang), -q * math.sin(ang), 0.0], atol=1e-13)
    # after one full turn the track is back at its transverse start, advanced along B by pitch
    d0 = np.array([math.cos(0.4), 0.0, math.sin(0.4)])
    Rt = pm * math.cos(0.4) / CB
    turn = 2 * math.pi * Rt / math.cos(0.4)
    p1, d1 = helix(ob, B, -1, pm, turn, p0, d0)
    np.testing.assert_allclose(p1, [0.0, 0.0, turn * math.sin(0.4)], atol=1e-10)
    np.testing.assert_allclose(d1, d0, atol=1e-12)


def test_helix_general_field_direction_and_unit_tangent(ob):
    rng = np.random.default_rng(2)
    for _ in range(50):
        B = rng.normal(size=3) * 2
        d = rng.normal(size=3); d /= np.linalg.norm(d)
        p = rng.normal(size=3) * 10
        pm, h = rng.uniform(1, 1e3), rng.uniform(0.01, 50)
        q = int(rng.choice([-1, 1]))
        p1, d1 = helix(ob, B, q, pm, h, p, d)
        assert np.linalg.norm(d1) == pytest.approx(1.0, abs=1e-14)
        b = B / np.linalg.norm(B)
        assert d1 @ b == pytest.approx(d @ b, abs=1e-14)                # pitch conserved
        assert (p1 - p) @ b == pytest.approx(h * (d @ b), abs=1e-11)
        # equation of motion F1 by central difference of the tangent
        e = 1e-4
        _, dp = helix(ob, B, q, pm, h + e, p, d)
        _, dm = helix(ob, B, q, pm, h - e, p, d)
        np.testing.assert_allclose((dp - dm) / (2 * e), q * CB / pm * np.cross(d1, B), atol=1e-7)


def _vac_oracle(ob, fld, **kw):
    """A big vacuum box world (one volume)."""
    g = geometry._finish([0], [(500.0, 500.0, 500.0)], [0], [-1], np.eye(3).reshape(1, 9), [(0.0, 0, 0)], ["vacuum"], "vac")
    _, tabs, scal = materials.build_material_set(["vacuum"])
    return ob.Oracle(g, tabs, scal, fld, **kw)


def test_rk4_converges_to_helix_with_fifth_order_local_error(ob):
    fm = field.solenoid_map(b0=2.0, r_scale=1e9)                        # uniform 2 T as a map
    o = _vac_oracle(ob, fm)
    np.testing.assert_allclose(o.field_at([10.0, 20.0, 30.0]), [0, 0, 2.0], atol=1e-12)
    B, pm = np.array([0, 0, 2.0]), 50.0
    p, d = np.array([1.0, 2.0, 3.0]), np.array([0.6, 0.0, 0.8])
    errs = []
    for h in (8.0, 4.0, 2.0):
        p1, d1 = o.rk4(-1, pm, h, p, d)
        pe, de = helix(ob, B, -1, pm, h, p, d)
        assert np.linalg.norm(d1) == pytest.approx(1.0, abs=1e-14)
        errs.append(np.linalg.norm(p1 - pe))
    assert 24 < errs[0] / errs[1] < 40 and 24 < errs[1] / errs[2] < 40   # error ~ h^5
    assert errs[2] < 1e-4


def test_field_map_bilinear_and_clamped(ob):
    o = _vac_oracle(ob, field.solenoid_map())
    bz = lambda r: 3.8 * (1 - (r / 300.0) ** 2)
    assert o.field_at([0, 0, 0])[2] == pytest.approx(3.8)
    assert o.field_at([30.0, 40.0, -100.0])[2] == pytest.approx(bz(50.0), rel=1e-14)
    r = 77.25
    want = bz(77) + 0.25 * (bz(78) - bz(77))                             # linear between nodes
    assert o.field_at([r, 0, 12.5])[2] == pytest.approx(want, rel=1e-13)
    assert o.field_at([400.0, 0, 0])[2] == 0.0 and o.field_at([0, 0, 1e4])[2] == pytest.approx(3.8)


def test_chord_loop_sagitta_budget_and_boundary(ob):
    """each chord's deflection <= threshold; PAPER.md:67 / F4: at most `budget` chords."""
    delta = 1e-3
    o = _vac_oracle(ob, field.uniform_field(0, 0, 1.0), delta_chord=delta)
    T = 100.0
    pm = math.sqrt(T * (T + 2 * M))
    R = pm / CB
    flag, p, d, s, ch, push = o.propagate(-1, T, [0, 0, 0], [1.0, 0, 0], 0, 5.0)
    hmax = math.sqrt(8 * delta * R)
    assert flag == 0 and s == 5.0 and ch == math.ceil(5.0 / hmax)
    assert R * (1 - math.cos(0.5 * hmax / R)) == pytest.approx(delta, rel=1e-3)       # sagitta of a chord
    assert np.linalg.norm(p - np.array([0.0, R, 0.0])) == pytest.approx(R, rel=1e-12)  # on the circle
    # chord budget
    flag, p, d, s, ch, push = o.propagate(-1, T, [0, 0, 0], [1.0, 0, 0], 0, 1e4)
    assert flag == 2 and ch == 16 and s == pytest.approx(16 * hmax, rel=1e-13)
    # straight track (d parallel to B) reaches the world face: boundary at 500 cm, no chords
    flag, p, d, s, ch, push = o.propagate(+1, T, [0, 0, 0], [0, 0, 1.0], 0, math.inf)
    assert flag == 1 and ch == 0 and s == 500.0
    # a high-momentum track hits the x = 500 face: crossing point within delta of the true circle
    T = 5e4
    pm = math.sqrt(T * (T + 2 * M)); R = pm / CB
    o2 = _vac_oracle(ob, field.uniform_field(0, 0, 1.0), delta_chord=delta, chord_budget=10000)
    flag, p, d, s, ch, push = o2.propagate(-1, T, [0, 0, 0], [1.0, 0, 0], 0, 1e5)
    assert flag == 1 and p[0] == pytest.approx(500.0, abs=1e-9)
    y_true = R - math.sqrt(R * R - 500.0 ** 2)
    assert abs(p[1] - y_true) < delta
    assert s == pytest.approx(R * math.asin(500.0 / R), abs=2e-3)
    assert np.linalg.norm(d) == pytest.approx(1.0, abs=1e-14)
    # no field: straight line to the physics limit
    o3 = _vac_oracle(ob, field.no_field())
    flag, p, d, s, ch, push = o3.propagate(-1, 10.0, [1.0, 2.0, 3.0], [0, 1.0, 0], 0, 7.0)
    assert flag == 0 and ch == 0 and s == 7.0
    np.testing.assert_allclose(p, [1.0, 9.0, 3.0])
