"""Pins of the oracle's final-state samplers.

Sampled spectra are compared by chi-square with the differential cross sections (formulas that
the sampler does not contain), final states are checked for energy and momentum balance.
"""
import ctypes
import math

import numpy as np
import pytest
from scipy.integrate import quad
from scipy.stats import chi2

from paper_2209_15445_b200.inputs import field

M = 0.51099895
N = 20000


def _p(a):
    return np.ascontiguousarray(a, dtype=np.float64).ctypes.data_as(ctypes.c_void_p)


@pytest.fixture(scope="module")
def orc(ob, calo):
    g, mats, tabs, scal = calo
    return ob.Oracle(g, tabs, scal, field.no_field()), mats, scal


def tracks(ob, species, ekin, n=N, direc=(0.6, 0.0, 0.8)):
    t = np.zeros(n, dtype=ob.TRACK)
    t["dir"] = direc
    t["ekin"] = ekin
    t["id"] = np.arange(n) + 1000
    t["event"] = 5
    t["step"] = 3
    t["volume"] = 52
    t["species"] = species
    return t


def chi2_check(samples, pdf, lo, hi, bins=40, log=False):
    edges = np.geomspace(lo, hi, bins + 1) if log else np.linspace(lo, hi, bins + 1)
    obs, _ = np.histogram(samples, edges)
    assert obs.sum() == len(samples), "samples outside the kinematic range"
    exp = np.array([quad(pdf, a, b, epsrel=1e-10)[0] for a, b in zip(edges[:-1], edges[1:])])
    exp *= len(samples) / exp.sum()
    keep = exp > 5
    stat = ((obs[keep] - exp[keep]) ** 2 / exp[keep]).sum()
    assert stat < chi2.ppf(0.9999, keep.sum() - 1), (stat, keep.sum())


def pvec(T, d, massless=False):
    p = T if massless else np.sqrt(T * (T + 2 * M))
    return p[:, None] * d


@pytest.mark.parametrize("k", [0.05, 1.0, 20.0, 5000.0])
def test_compton(ob, orc, k):
    o, mats, scal = orc
    t = tracks(ob, 2, k)
    res, sec = o.interact(1, t, 1)
    kap = k / M
    eps = np.where(res["alive"] == 1, res["post"]["ekin"], k - sec[:, 0]["ekin"]) / k
    made = res["n_sec"] == 1
    # energy: k = k' + T_e (+ below-cut deposit)
    tot = np.where(res["alive"] == 1, res["post"]["ekin"], 0) + np.where(made, sec[:, 0]["ekin"], 0) + res["edep_cut"]
    np.testing.assert_allclose(tot, k, rtol=1e-14)
    # the cut rule (M5): electrons are made iff T_e >= T_c(Pb)
    Te = k - eps * k
    alive = res["alive"] == 1
    assert np.all(made[alive] == (Te[alive] >= scal[1, 1]))
    # momentum balance where the electron exists
    if made.any():
        pin = k * t["dir"][made]
        pout = pvec(res["post"]["ekin"][made], res["post"]["dir"][made], True) + pvec(sec[:, 0]["ekin"][made], sec[:, 0]["dir"][made])
        np.testing.assert_allclose(pout, pin, atol=1e-9 * max(k, 1))
    # scattering angle <-> energy (Compton formula)
    cos_t = np.einsum("ij,ij->i", res["post"]["dir"], t["dir"])[alive]
    np.testing.assert_allclose(1 / eps[alive] - 1, kap * (1 - cos_t), atol=1e-9 * (1 + kap))

    def pdf(e):
        tt = (1 - e) / (kap * e)
        return e + 1 / e - tt * (2 - tt)
    sel = alive if k > 0.01 else slice(None)
    chi2_check(eps[sel], pdf, 1 / (1 + 2 * kap), 1.0, log=kap > 10)
    # azimuth uniform
    d = res["post"]["dir"][alive]
    e2 = np.array([0.0, 1.0, 0.0])
    e1 = np.cross(e2, t["dir"][0])
    phi = np.arctan2(d @ e2, d @ e1)
    chi2_check(phi, lambda x: 1.0, -math.pi, math.pi, bins=20)


@pytest.mark.parametrize("k", [1.5, 10.0, 3000.0])
def test_pair(ob, orc, k):
    o, mats, scal = orc
    res, sec = o.interact(2, tracks(ob, 2, k), 1)
    assert np.all(res["alive"] == 0)
    a = M / k
    pos = np.where(res["n_sec"] == 2, sec[:, 1]["ekin"], sec[:, 0]["ekin"])     # e+ always made (child 1)
    assert np.all(np.where(res["n_sec"] == 2, sec[:, 1]["species"], sec[:, 0]["species"]) == 1)
    eps = (pos + M) / k
    chi2_check(eps, lambda e: 1 - 4 / 3 * e * (1 - e), a, 1 - a)
    tot = res["edep_cut"] + pos + 2 * M + np.where(res["n_sec"] == 2, sec[:, 0]["ekin"], 0)
    np.testing.assert_allclose(tot, k, rtol=1e-13)
    two = res["n_sec"] == 2
    if two.any():
        assert np.all(sec[two, 0]["species"] == 0) and np.all(sec[two, 0]["ekin"] >= scal[1, 1])
        # polar angles m/E about the photon direction, opposite azimuths
        d0 = np.array([0.6, 0.0, 0.8])
        cm = sec[two, 0]["dir"] @ d0
        np.testing.assert_allclose(np.arccos(np.clip(cm, -1, 1)), M / (sec[two, 0]["ekin"] + M), atol=1e-7)
        tm = sec[two, 0]["dir"] - cm[:, None] * d0
        cp = sec[two, 1]["dir"] @ d0
        tp = sec[two, 1]["dir"] - cp[:, None] * d0
        cosd = np.einsum("ij,ij->i", tm, tp) / (np.linalg.norm(tm, axis=1) * np.linalg.norm(tp, axis=1))
        np.testing.assert_allclose(cosd, -1.0, atol=1e-6)


def test_photoelectric(ob, orc):
    o, mats, scal = orc
    BK, Tc = scal[1, 3], scal[1, 1]
    for k in (0.05, 0.5, 3.0):
        res, sec = o.interact(3, tracks(ob, 2, k, n=10), 1)
        assert np.all(res["alive"] == 0)
        if k - BK >= Tc:
            assert np.all(res["n_sec"] == 1) and np.allclose(sec[:, 0]["ekin"], k - BK)
            np.testing.assert_allclose(res["edep_cut"], BK)
            np.testing.assert_allclose(sec[:, 0]["dir"], [[0.6, 0.0, 0.8]] * 10)
        else:
            assert np.all(res["n_sec"] == 0)
            np.testing.assert_allclose(res["edep_cut"], k)


@pytest.mark.parametrize("T,species", [(2.0, 0), (100.0, 1), (1e4, 0)])
def test_bremsstrahlung(ob, orc, T, species):
    o, mats, scal = orc
    kc = scal[1, 2]
    res, sec = o.interact(4, tracks(ob, species, T), 1)
    assert np.all(res["alive"] == 1) and np.all(res["n_sec"] == 1) and np.all(res["outcome"] == 4)
    kg = sec[:, 0]["ekin"]
    np.testing.assert_allclose(kg + res["post"]["ekin"], T, rtol=1e-14)
    E = T + M
    chi2_check(kg, lambda k: (4 / 3 - 4 / 3 * k / E + (k / E) ** 2) / k, kc, T, log=True)
    np.testing.assert_allclose(res["post"]["dir"], [[0.6, 0.0, 0.8]] * N)          # parent keeps its direction
    np.testing.assert_allclose(np.arccos(np.clip(sec[:, 0]["dir"] @ [0.6, 0.0, 0.8], -1, 1)), M / E, atol=1e-7)
    # kinematically closed below the cut
    res, _ = o.interact(4, tracks(ob, species, 0.9 * kc, n=5), 1)
    assert np.all(res["outcome"] == 12) and np.all(res["n_sec"] == 0) and np.all(res["post"]["ekin"] == 0.9 * kc)


def _moller_pdf(T):
    g = 1 + T / M
    b = (2 * g - 1) / g ** 2
    return lambda e: (g - 1) ** 2 / g ** 2 + (1 / e) * (1 / e - b) + (1 / (1 - e)) * (1 / (1 - e) - b)


def _bhabha_pdf(T):
    g = 1 + T / M
    b2 = 1 - 1 / g ** 2
    y = 1 / (g + 1); w = 1 - 2 * y
    B1, B2, B3, B4 = 2 - y * y, w * (3 + y * y), w ** 2 + w ** 3, w ** 3
    return lambda e: 1 / (b2 * e * e) - B1 / e + B2 - B3 * e + B4 * e * e


@pytest.mark.parametrize("T,species", [(3.0, 0), (50.0, 0), (2.0, 1), (50.0, 1), (1e4, 1)])
def test_ionisation(ob, orc, T, species):
    o, mats, scal = orc
    Tc = scal[1, 1]
    t = tracks(ob, species, T)
    res, sec = o.interact(5, t, 1)
    assert np.all(res["n_sec"] == 1) and np.all(res["alive"] == 1)
    Td = sec[:, 0]["ekin"]
    np.testing.assert_allclose(Td + res["post"]["ekin"], T, rtol=1e-14)
    pdf, hi = (_moller_pdf(T), 0.5) if species == 0 else (_bhabha_pdf(T), 1.0)
    chi2_check(Td / T, pdf, Tc / T, hi, log=True)
    # momentum balance
    pout = pvec(res["post"]["ekin"], res["post"]["dir"]) + pvec(Td, sec[:, 0]["dir"])
    np.testing.assert_allclose(pout, pvec(t["ekin"], t["dir"]), atol=1e-9 * T)
    # closed
    closed_T = (1.9 if species == 0 else 0.95) * Tc
    res, _ = o.interact(5, tracks(ob, species, closed_T, n=5), 1)
    assert np.all(res["outcome"] == 12) and np.all(res["n_sec"] == 0)


@pytest.mark.parametrize("T", [0.01, 1.0, 200.0])
def test_annihilation_in_flight(ob, orc, T):
    o, mats, scal = orc
    t = tracks(ob, 1, T)
    res, sec = o.interact(6, t, 2)                      # LAr: k_c = 17.5 keV, both photons survive
    assert np.all(res["alive"] == 0)
    g = 1 + T / M
    two = res["n_sec"] == 2
    assert two.mean() > 0.99
    k1, k2 = sec[two, 0]["ekin"], sec[two, 1]["ekin"]
    np.testing.assert_allclose(k1 + k2, T + 2 * M, rtol=1e-14)
    pout = pvec(k1, sec[two, 0]["dir"], True) + pvec(k2, sec[two, 1]["dir"], True)
    np.testing.assert_allclose(pout, pvec(t["ekin"][two], t["dir"][two]), atol=1e-9 * (T + 1))
    root = math.sqrt((g - 1) / (g + 1))
    pdf = lambda e: (1 / e) * (1 + 2 * g / (g + 1) ** 2 - e - 1 / ((g + 1) ** 2 * e))
    chi2_check(k1 / (T + 2 * M), pdf, 0.5 - 0.5 * root, 0.5 + 0.5 * root, log=T > 10)


def test_rotation_convention(ob):
    rng = np.random.default_rng(0)
    out = np.zeros(3)
    for _ in range(200):
        d = rng.normal(size=3); d /= np.linalg.norm(d)
        th, phi = rng.uniform(0, math.pi), rng.uniform(0, 2 * math.pi)
        ob.lib.orc_rotate(_p(d), math.cos(th), math.sin(th), phi, _p(out))
        assert np.linalg.norm(out) == pytest.approx(1.0, abs=1e-15)
        assert out @ d == pytest.approx(math.cos(th), abs=1e-14)
        # azimuth measured in the (e1, e2) frame of P10
        rho = math.hypot(d[0], d[1])
        e1 = np.array([d[0] * d[2], d[1] * d[2], -rho * rho]) / rho
        e2 = np.array([-d[1], d[0], 0.0]) / rho
        assert math.atan2(out @ e2, out @ e1) % (2 * math.pi) == pytest.approx(phi, abs=1e-9)
    for dz in (1.0, -1.0):                               # rho = 0 branch
        ob.lib.orc_rotate(_p([0.0, 0.0, dz]), math.cos(0.3), math.sin(0.3), 0.0, _p(out))
        np.testing.assert_allclose(out, [dz * math.sin(0.3), 0.0, dz * math.cos(0.3)], atol=1e-15)


def test_secondary_ids_follow_R3(ob, orc):
    o, _, _ = orc
    t = tracks(ob, 1, 5.0, n=3)
    res, sec = o.interact(6, t, 2)
    for i in range(3):
        for c in range(2):
            assert sec[i, c]["id"] == ob.lib.orc_child_id(5, 1, int(t["id"][i]), 3, c)
            assert sec[i, c]["step"] == 0 and sec[i, c]["event"] == 5 and sec[i, c]["volume"] == 52
