"""Pins of the oracle's closed-form cross sections and table builder.

Each closed-form total is checked against numerical quadrature of its *differential* cross
section (a different formula), plus textbook values from tests/golden/closed_form_pins.txt.
"""
import math
import os

import numpy as np
import pytest
from scipy.integrate import quad

M = 0.51099895
RE = 2.8179403262e-13
GOLD = os.path.join(os.path.dirname(__file__), "golden", "closed_form_pins.txt")
PB = (82.0, 207.2, 11.35)
LAR = (18.0, 39.95, 1.396)


def gold(kind):
    return [l.split()[1:] for l in open(GOLD) if l.split() and l.split()[0] == kind]


def test_klein_nishina_golden_and_thomson_limit(ob):
    sig_t = 8 * math.pi * RE ** 2 / 3
    for kap, want in gold("kn_ratio"):
        assert ob.lib.orc_sigma_compton(float(kap) * M) / sig_t == pytest.approx(float(want), abs=1e-6)
    assert ob.lib.orc_sigma_compton(1e-9) / sig_t == pytest.approx(1.0, abs=1e-8)
    # the series and the full expression meet at the switch point kappa = 2e-3
    lo, hi = ob.lib.orc_sigma_compton(M * 1.9999999e-3), ob.lib.orc_sigma_compton(M * 2.0000001e-3)
    assert lo / hi == pytest.approx(1.0, abs=1e-9)


@pytest.mark.parametrize("kappa", [0.01, 0.1, 1.0, 10.0, 1000.0])
def test_klein_nishina_total_is_integral_of_differential(ob, kappa):
    def dsde(e):
        t = (1 - e) / (kappa * e)
        return math.pi * RE ** 2 / kappa * (e + 1 / e - t * (2 - t))
    val, _ = quad(dsde, 1 / (1 + 2 * kappa), 1, epsabs=0, epsrel=1e-12)
    assert ob.lib.orc_sigma_compton(kappa * M) == pytest.approx(val, rel=1e-10)


@pytest.mark.parametrize("k", [1.03, 1.1, 2.0, 10.0, 1e4])
def test_pair_polynomial_is_integral_of_shape(ob, k):
    a = M / k
    val, _ = quad(lambda e: 1 - 4 / 3 * e * (1 - e), a, 1 - a, epsabs=0, epsrel=1e-13)
    assert ob.lib.orc_pair_shape(k) == pytest.approx(val, rel=1e-11, abs=1e-16)
    assert ob.lib.orc_pair_shape(2 * M) == 0.0 and ob.lib.orc_pair_shape(0.5) == 0.0


def test_pair_high_energy_limit(ob):
    assert ob.lib.orc_pair_shape(1e8) == pytest.approx(7 / 9, rel=1e-7)


def test_photoelectric_power_law(ob):
    assert ob.lib.orc_sigma_photo(0.2, 82) / ob.lib.orc_sigma_photo(0.1, 82) == pytest.approx(2 ** -3.5, rel=1e-13)
    assert ob.lib.orc_sigma_photo(0.1, 82) / ob.lib.orc_sigma_photo(0.1, 41) == pytest.approx(32.0, rel=1e-13)


@pytest.mark.parametrize("T,kc", [(1.0, 0.1), (100.0, 0.0175), (1e4, 0.174), (0.5, 0.174)])
def test_brem_closed_forms_are_integrals(ob, T, kc):
    E = T + M
    d = lambda k: (4 / 3 - 4 / 3 * (k / E) + (k / E) ** 2) / k
    val, _ = quad(d, kc, T, epsabs=0, epsrel=1e-13)
    assert ob.lib.orc_brem_shape(T, kc) == pytest.approx(val, rel=1e-11)
    ku = min(kc, T)
    val, _ = quad(lambda k: k * d(k), 0, ku, epsabs=0, epsrel=1e-13)
    assert ob.lib.orc_srad_shape(T, kc) == pytest.approx(val, rel=1e-11)
    assert ob.lib.orc_brem_shape(kc * 0.9, kc) == 0.0


def test_unrestricted_radiative_loss_tends_to_T_over_X0(ob):
    T = 1e7
    assert ob.lib.orc_srad_shape(T, T) / T == pytest.approx(1.0, rel=1e-6)


def _moller_diff(T):
    g = 1 + T / M
    b2 = 1 - 1 / g ** 2
    b = (2 * g - 1) / g ** 2
    pref = 2 * math.pi * RE ** 2 / (b2 * (g - 1))
    return lambda e: pref * ((g - 1) ** 2 / g ** 2 + (1 / e) * (1 / e - b) + (1 / (1 - e)) * (1 / (1 - e) - b))


def _bhabha_diff(T):
    g = 1 + T / M
    b2 = 1 - 1 / g ** 2
    y = 1 / (g + 1)
    w = 1 - 2 * y
    B1, B2, B3, B4 = 2 - y * y, w * (3 + y * y), w ** 2 + w ** 3, w ** 3
    pref = 2 * math.pi * RE ** 2 / (g - 1)
    return lambda e: pref * (1 / (b2 * e * e) - B1 / e + B2 - B3 * e + B4 * e * e)


@pytest.mark.parametrize("T", [0.01, 1.0, 100.0, 1e4])
@pytest.mark.parametrize("x", [1e-3, 0.1, 0.4])
def test_moller_bhabha_totals_are_integrals(ob, T, x):
    Tc = x * T
    val, _ = quad(_moller_diff(T), x, 0.5, epsabs=0, epsrel=1e-13)
    assert ob.lib.orc_sigma_moller(T, Tc) == pytest.approx(val, rel=1e-10)
    val, _ = quad(_bhabha_diff(T), x, 1.0, epsabs=0, epsrel=1e-13)
    assert ob.lib.orc_sigma_bhabha(T, Tc) == pytest.approx(val, rel=1e-10)
    assert ob.lib.orc_sigma_moller(T, 0.5 * T) == 0.0 and ob.lib.orc_sigma_bhabha(T, T) == 0.0


@pytest.mark.parametrize("T", [1e-3, 0.1, 1.0, 100.0, 1e4])
def test_annihilation_total_is_integral_of_heitler_differential(ob, T):
    g = 1 + T / M
    root = math.sqrt((g - 1) / (g + 1))
    d = lambda e: math.pi * RE ** 2 / (g - 1) / e * (1 + 2 * g / (g + 1) ** 2 - e - 1 / ((g + 1) ** 2 * e))
    val, _ = quad(d, 0.5 - 0.5 * root, 0.5 + 0.5 * root, epsabs=0, epsrel=1e-13)
    assert ob.lib.orc_sigma_annihilation(T) == pytest.approx(val, rel=1e-9)


@pytest.mark.parametrize("T", [1.0, 100.0, 1e4])
@pytest.mark.parametrize("positron", [0, 1])
def test_restricted_stopping_power_invariant(ob, T, positron):
    """P7: S_coll(T;T2) - S_coll(T;T1) = n_el * first moment of the P5/P6 differential."""
    Z, A, rho = PB
    n_el = Z * 6.02214076e23 * rho / A
    T1, T2 = 0.01 * T, 0.3 * T
    diff = _bhabha_diff(T) if positron else _moller_diff(T)
    val, _ = quad(lambda e: e * T * diff(e), T1 / T, T2 / T, epsabs=0, epsrel=1e-13)
    lhs = ob.lib.orc_s_coll(T, Z, A, rho, T2, positron) - ob.lib.orc_s_coll(T, Z, A, rho, T1, positron)
    assert lhs == pytest.approx(n_el * val, rel=1e-9)


def test_collision_stopping_power_sane(ob):
    for Z, A, rho in (PB, LAR):
        s = [ob.lib.orc_s_coll(T, Z, A, rho, -1.0, 0) / rho for T in np.geomspace(1e-3, 1e5, 60)]
        assert min(s) > 0.9 and min(s) < 1.6          # minimum-ionising ~1-1.5 MeV cm^2/g
    # unrestricted >= restricted, equal once the cut exceeds the kinematic limit
    assert ob.lib.orc_s_coll(10.0, *PB, 1.0, 0) < ob.lib.orc_s_coll(10.0, *PB, -1.0, 0)
    assert ob.lib.orc_s_coll(10.0, *PB, 6.0, 0) == ob.lib.orc_s_coll(10.0, *PB, -1.0, 0)


def test_radiation_lengths_textbook(ob):
    for name, Z, A, rho, want in gold("x0_gcm2"):
        _, scal = ob.build_material(float(Z), float(A), float(rho))
        assert scal[0] * float(rho) == pytest.approx(float(want), abs=0.006)


def test_tables_structure_and_cuts(ob):
    tab, scal = ob.build_material(*PB)
    assert np.all(np.isfinite(tab)) and np.all(tab >= 0)
    X0, Tc, kc, BK = scal[:4]
    T = np.exp(np.log(1e-3) + np.arange(2048) * (np.log(1e8) - np.log(1e-3)) / 2047)
    # range tables increase strictly; dR/dT = 1/S
    for tr, ts in ((6, 5), (11, 10)):
        assert np.all(np.diff(tab[tr]) > 0)
        i = 1200
        assert (tab[tr][i + 1] - tab[tr][i - 1]) / (T[i + 1] - T[i - 1]) == pytest.approx(1 / tab[ts][i], rel=1e-3)
    # discrete cross sections vanish below their thresholds
    assert np.all(tab[3][T <= kc] == 0) and np.all(tab[4][T <= 2 * Tc] == 0) and np.all(tab[8][T <= Tc] == 0)
    assert np.all(tab[1][T <= 2 * M] == 0)
    # M4: the cut energies reproduce 0.7 mm
    assert 5.0 / np.interp(np.log(kc), np.log(T), tab[0] + tab[1] + tab[2]) == pytest.approx(0.07, rel=2e-3)
    assert BK == pytest.approx(13.605693e-6 * 81 ** 2)
    # vacuum
    vt, vs = ob.build_material(0, 0, 0)
    assert vs[5] == 1.0 and np.all(vt[[0, 1, 2, 3, 4, 5, 7, 8, 9, 10]] == 0)


def test_lookup_interpolates_linearly_in_lnT(ob, calo):
    from paper_2209_15445_b200.inputs import field
    g, mats, tabs, scal = calo
    o = ob.Oracle(g, tabs, scal, field.no_field())
    u0, du = math.log(1e-3), (math.log(1e8) - math.log(1e-3)) / 2047
    for i, f in ((0, 0.0), (17, 0.25), (1000, 0.5), (2046, 0.999)):
        T = math.exp(u0 + du * (i + f))
        want = tabs[1, 5, i] + f * (tabs[1, 5, i + 1] - tabs[1, 5, i])
        assert o.lookup(1, 5, T) == pytest.approx(want, rel=1e-10)
    # inverse range inverts the range lookup
    for T in (0.01, 1.0, 350.0):
        R = o.lookup(1, 6, T)
        assert o.inverse_range(1, 6, R) == pytest.approx(T, rel=1e-9)
    assert o.inverse_range(1, 6, 0.5 * tabs[1, 6, 0]) == 0.0
