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


# ---------------------------------------------------------------------------------------------------
# The ORC_FIELD_MAP_RZ branch of orc_propagate: RK4 chords, the F2' clamp and the linear
# tangent interpolation at a boundary hit.  None of these tests calls the oracle's own formula for the
# expected value: the chord count is a number worked out here, the end point is the analytic helix or an
# independent adaptive integrator (scipy DOP853) of the equation of motion F1 in the same bilinear field.
def _rk4_local_bound(omega):
    """Local position error of one classical RK4 step over a turning angle omega on a circle of unit radius:
    the leading term of the Taylor remainder, omega^5 / 120."""
    return omega ** 5 / 120.0


def test_map_chord_count_is_the_sagitta_limit_when_it_binds(ob):
    """Track perpendicular to B: h_max = sqrt(8 delta R) (F2) is far below the F2' clamp 0.5 R, so a step of
    length s takes ceil(s / sqrt(8 delta R)) chords and ends on the analytic circle within the h^5 bound."""
    delta, b0 = 1e-3, 2.0
    o = _vac_oracle(ob, field.solenoid_map(b0=b0, r_scale=1e9), delta_chord=delta, chord_budget=100000)
    T = 20.0
    pm = math.sqrt(T * (T + 2 * M))
    R = pm / (CB * b0)
    h_sag, h_clamp = math.sqrt(8 * delta * R), 0.5 * R
    assert h_sag < h_clamp
    s = 9.0
    flag, p, d, s_done, ch, push = o.propagate(-1, T, [0, 0, 0], [1.0, 0, 0], 0, s)
    assert flag == 0 and s_done == s and ch == math.ceil(s / h_sag)
    pe, de = helix(ob, np.array([0, 0, b0]), -1, pm, s, np.zeros(3), np.array([1.0, 0, 0]))
    bound = 2.0 * ch * R * _rk4_local_bound(h_sag / R)
    assert 0.0 < np.linalg.norm(p - pe) < bound and bound < 1e-6
    assert np.linalg.norm(d) == pytest.approx(1.0, abs=1e-14)
    np.testing.assert_allclose(d, de, atol=2.0 * ch * _rk4_local_bound(h_sag / R))


@pytest.mark.parametrize("angle", [0.01, 0.05, 0.15])
def test_map_chord_count_is_the_half_radian_clamp_when_it_binds(ob, angle):
    """F2': a track nearly parallel to B has a huge local radius p / (c B_perp), so the sagitta rule would allow
    chords that turn the direction about B by radians; the clamp h <= 0.5 p / (2.998 |B|) limits the turn to
    0.5 rad.  The chord count is that number, and the end point is the exact helix within the RK4 bound."""
    delta, b0 = 1e-3, 2.0
    o = _vac_oracle(ob, field.solenoid_map(b0=b0, r_scale=1e9), delta_chord=delta, chord_budget=100000)
    pm = 1.0
    T = math.sqrt(pm * pm + M * M) - M
    Rfull = pm / (CB * b0)                      # radius of a track perpendicular to B
    d0 = np.array([math.sin(angle), 0.0, math.cos(angle)])
    h_sag = math.sqrt(8 * delta * Rfull / math.sin(angle))
    h_clamp = 0.5 * Rfull
    assert h_clamp < h_sag                       # the clamp binds
    s = 1.0
    flag, p, d, s_done, ch, push = o.propagate(+1, T, [1.0, 2.0, 3.0], d0, 0, s)
    assert flag == 0 and s_done == s
    assert ch == math.ceil(s / h_clamp)          # = 12: a factor 1 instead of 0.5 gives 6, no clamp gives <= 3
    pe, de = helix(ob, np.array([0, 0, b0]), +1, pm, s, np.array([1.0, 2.0, 3.0]), d0)
    # transverse radius R sin(angle); every chord turns by 0.5 rad
    bound = 2.0 * ch * Rfull * math.sin(angle) * _rk4_local_bound(0.5)
    err = np.linalg.norm(p - pe)
    assert 0.0 < err < bound
    assert np.linalg.norm(d) == pytest.approx(1.0, abs=1e-14)
    # without the clamp one RK4 step over 2.9 rad (angle 0.01) misses by far more than this bound
    if angle == 0.01:
        p_one, _ = o.rk4(+1, pm, s, [1.0, 2.0, 3.0], d0)
        assert np.linalg.norm(p_one - pe) > 20 * bound


def test_map_boundary_hit_point_tangent_and_push_direction(ob):
    """F3 at a boundary in a field map: the crossing point lies within delta_chord of the analytic circle, the
    returned tangent (linear interpolation of the chord's end tangents, renormalised) has unit length and is
    within (h/R)^2 of the exact tangent, the push direction is the unit chord, s_done the arc up to the hit."""
    delta, b0 = 1e-3, 1.0
    o = _vac_oracle(ob, field.solenoid_map(b0=b0, r_scale=1e9, r_max=600.0, z_half=600.0, step=50.0),
                    delta_chord=delta, chord_budget=100000)
    T = 5e4
    pm = math.sqrt(T * (T + 2 * M))
    R = pm / (CB * b0)
    h = math.sqrt(8 * delta * R)
    for q in (-1, +1):
        flag, p, d, s_done, ch, push = o.propagate(q, T, [0, 0, 0], [1.0, 0, 0], 0, 1e5)
        assert flag == 1 and p[0] == pytest.approx(500.0, abs=1e-9)      # on the world's x = +500 face
        y_true = -q * (R - math.sqrt(R * R - 500.0 ** 2))
        assert abs(p[1] - y_true) < delta and p[2] == 0.0
        th = math.asin(500.0 / R)
        assert s_done == pytest.approx(R * th, abs=2e-3)
        assert np.linalg.norm(d) == pytest.approx(1.0, abs=1e-15)
        d_true = np.array([math.cos(th), -q * math.sin(th), 0.0])
        assert np.linalg.norm(d - d_true) < (h / R) ** 2
        assert np.linalg.norm(d - d_true) > 0.0                           # interpolated, not the exact tangent
        assert np.linalg.norm(push) == pytest.approx(1.0, abs=1e-15)
        # the chord that hit: from the last chord start (a multiple of h along the arc) to its end
        k = math.floor(R * th / h)
        a0, a1 = k * h / R, (k + 1) * h / R
        c0 = np.array([R * math.sin(a0), -q * R * (1 - math.cos(a0)), 0.0])
        c1 = np.array([R * math.sin(a1), -q * R * (1 - math.cos(a1)), 0.0])
        np.testing.assert_allclose(push, (c1 - c0) / np.linalg.norm(c1 - c0), atol=1e-9)
        assert ch == k + 1


def test_map_chord_loop_follows_the_equation_of_motion_in_a_non_uniform_field(ob):
    """The RK4 chord loop in the real solenoid map (Bz falls with r) against an adaptive 8th-order integration
    of F1, dx/ds = d, dd/ds = (q c / p) d x B(x), with the bilinear field evaluated here in numpy."""
    from scipy.integrate import solve_ivp
    fm = field.solenoid_map()
    o = _vac_oracle(ob, fm, chord_budget=100000)
    bz = fm.bz

    def b_at(x):
        r = math.hypot(x[0], x[1])
        fr = min(max((r - fm.r0) / fm.dr, 0.0), fm.nr - 1.0)
        fz = min(max((x[2] - fm.z0) / fm.dz, 0.0), fm.nz - 1.0)
        ir, iz = min(int(fr), fm.nr - 2), min(int(fz), fm.nz - 2)
        a, b = fr - ir, fz - iz
        lo = bz[iz, ir] + a * (bz[iz, ir + 1] - bz[iz, ir])
        hi = bz[iz + 1, ir] + a * (bz[iz + 1, ir + 1] - bz[iz + 1, ir])
        return np.array([0.0, 0.0, lo + b * (hi - lo)])

    for q, pm, p0, d0, s in ((-1, 50.0, [100.0, 0.0, 10.0], [0.6, 0.3, 0.2], 60.0),
                             (+1, 400.0, [10.0, -20.0, -50.0], [0.5, 0.5, 0.1], 250.0)):
        d0 = np.array(d0) / np.linalg.norm(d0)
        T = math.sqrt(pm * pm + M * M) - M
        rhs = lambda _, y: np.concatenate([y[3:], q * CB / pm * np.cross(y[3:], b_at(y[:3]))])
        sol = solve_ivp(rhs, (0.0, s), np.concatenate([p0, d0]), method="DOP853", rtol=1e-12, atol=1e-13, max_step=0.5)
        flag, p, d, s_done, ch, push = o.propagate(q, T, p0, d0, 0, s)
        assert flag == 0 and s_done == s and ch > 50
        # the field's kinks at the grid nodes limit both integrators to ~1e-7 cm here
        np.testing.assert_allclose(p, sol.y[:3, -1], atol=5e-6)
        np.testing.assert_allclose(d, sol.y[3:, -1], atol=5e-7)
        rr = np.hypot(sol.y[0], sol.y[1])
        assert rr.max() - rr.min() > 5.0                # the track really crossed regions of different field
