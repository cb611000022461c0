"""Materials, production cuts and the 12 tables per material.

This is the product's host-side table builder (numpy, fp64).  The tables it returns are the
`adept_tables` input of `adept_init` (include/adept.h).  The test oracle has its own builder
(oracle/tables.cpp, long double) and the two are compared in tests/test_tables.py.

Units: MeV, cm, g/cm^3.
"""
from dataclasses import dataclass
import math

import numpy as np

from .constants import (ALPHA, DU, ELECTRON_MASS, N_AVOGADRO, N_GRID, N_TABLES, PRODUCTION_CUT_CM,
                        R_E, RYDBERG_EV, T_GRID_MIN, U0, TAB_G_COMPTON, TAB_G_PAIR, TAB_G_PHOTO,
                        TAB_EM_BREM, TAB_EM_IONI, TAB_EM_DEDX, TAB_EM_RANGE, TAB_EP_BREM,
                        TAB_EP_IONI, TAB_EP_ANNI, TAB_EP_DEDX, TAB_EP_RANGE)

M = ELECTRON_MASS
TWO_PI_RE2 = 2.0 * math.pi * R_E * R_E
VACUUM_RANGE = 1.0e99          # range-table filler for vacuum (no loss, never limits a step)


@dataclass
class Material:
    name: str
    Z: float
    A: float
    rho: float                  # 0 => vacuum
    # derived
    n_at: float = 0.0
    n_el: float = 0.0
    X0: float = math.inf        # [cm]
    I: float = 0.0              # [MeV]
    hwp: float = 0.0            # plasma energy [MeV]
    B_K: float = 0.0            # K-shell binding [MeV] (compound: of its first element)
    e_cut: float = 0.0          # T_c [MeV]
    g_cut: float = 0.0          # k_c [MeV]
    # compounds (DESIGN.md §3 C1-C5): per element (Z, A, atoms per formula unit), number density, B_K
    elements: tuple = ()
    n_i: tuple = ()
    B_K_i: tuple = ()

    @property
    def vacuum(self):
        return self.rho <= 0.0


def make_material(name, Z, A, rho):
    """M1-M3: densities, Tsai radiation length, mean excitation energy, plasma energy, B_K (one element)."""
    mat = Material(name, float(Z), float(A), float(rho))
    if mat.vacuum:
        return mat
    mat.n_at = N_AVOGADRO * rho / A
    mat.n_el = Z * mat.n_at
    a = ALPHA * Z
    a2 = a * a
    f_c = a2 * (1.0 / (1.0 + a2) + 0.20206 - 0.0369 * a2 + 0.0083 * a2 ** 2 - 0.002 * a2 ** 3)
    l_rad = math.log(184.15 * Z ** (-1.0 / 3.0))
    lp_rad = math.log(1194.0 * Z ** (-2.0 / 3.0))
    inv_x0 = 4.0 * ALPHA * R_E ** 2 * mat.n_at * (Z * Z * (l_rad - f_c) + Z * lp_rad)
    mat.X0 = 1.0 / inv_x0
    i_ev = Z * (12.0 + 7.0 / Z) if Z < 13 else Z * (9.76 + 58.8 * Z ** (-1.19))
    mat.I = i_ev * 1.0e-6
    mat.hwp = 28.816e-6 * math.sqrt(rho * Z / A)
    mat.B_K = RYDBERG_EV * 1.0e-6 * (Z - 1.0) ** 2
    return mat


def _tsai_per_atom(Z):
    a2 = (ALPHA * Z) ** 2
    f_c = a2 * (1.0 / (1.0 + a2) + 0.20206 - 0.0369 * a2 + 0.0083 * a2 ** 2 - 0.002 * a2 ** 3)
    return Z * Z * (math.log(184.15 * Z ** (-1.0 / 3.0)) - f_c) + Z * math.log(1194.0 * Z ** (-2.0 / 3.0))


def _mean_excitation(Z):
    return (Z * (12.0 + 7.0 / Z) if Z < 13 else Z * (9.76 + 58.8 * Z ** (-1.19))) * 1.0e-6


def make_compound(name, elements, rho):
    """C1-C3: a compound of (Z, A, atoms per formula unit) triples.  Number densities n_i = N_A rho nu_i / A_mol;
    1/X0 additive over the atoms (Tsai); ln I = sum n_i Z_i ln I_i / n_el (Bragg); plasma energy from the total
    electron density."""
    elements = tuple((float(z), float(a), float(nu)) for z, a, nu in elements)
    a_mol = sum(nu * a for _, a, nu in elements)
    z_mol = sum(nu * z for z, _, nu in elements)
    mat = Material(name, z_mol / sum(nu for _, _, nu in elements), a_mol, float(rho), elements=elements)
    mat.n_i = tuple(N_AVOGADRO * rho * nu / a_mol for _, _, nu in elements)
    mat.n_at = sum(mat.n_i)
    mat.n_el = sum(n * z for n, (z, _, _) in zip(mat.n_i, elements))
    mat.X0 = 1.0 / sum(4.0 * ALPHA * R_E ** 2 * n * _tsai_per_atom(z) for n, (z, _, _) in zip(mat.n_i, elements))
    mat.I = math.exp(sum(n * z * math.log(_mean_excitation(z)) for n, (z, _, _) in zip(mat.n_i, elements)) / mat.n_el)
    mat.hwp = 28.816e-6 * math.sqrt(rho * z_mol / a_mol)
    mat.B_K_i = tuple(RYDBERG_EV * 1.0e-6 * (z - 1.0) ** 2 for z, _, _ in elements)
    mat.B_K = mat.B_K_i[0]
    return mat


def photo_macro(mat, k):
    """Macroscopic photoelectric cross section [1/cm]: sum over the elements of a compound."""
    if mat.elements:
        return sum(n * sigma_photo_atom(k, z) for n, (z, _, _) in zip(mat.n_i, mat.elements))
    return mat.n_at * sigma_photo_atom(k, mat.Z)


# the materials BASELINE.json:configs names (A_eff of the PbWO4 stand-in: SURVEY.md M1); "PbWO4_true" is the real
# compound, Pb + W + 4 O
def standard_materials():
    return {
        "PbWO4_true": make_compound("PbWO4_true", [(82.0, 207.2, 1), (74.0, 183.84, 1), (8.0, 15.999, 4)], 8.28),
        "vacuum": make_material("vacuum", 0.0, 0.0, 0.0),
        "Pb": make_material("Pb", 82.0, 207.2, 11.35),
        "LAr": make_material("LAr", 18.0, 39.95, 1.396),
        "Si": make_material("Si", 14.0, 28.0855, 2.33),
        "PbWO4": make_material("PbWO4", 73.0, 176.69, 8.28),
    }


def energy_grid():
    return np.exp(U0 + DU * np.arange(N_GRID))


# ---------------------------------------------------------------- cross sections (per electron)
def sigma_compton(k):
    """P1 Klein-Nishina total cross section per electron [cm^2]; series below kappa = 2e-3."""
    kap = np.asarray(k, dtype=np.float64) / M
    l = np.log1p(2.0 * kap)
    full = TWO_PI_RE2 * ((1.0 + kap) / kap ** 2 * (2.0 * (1.0 + kap) / (1.0 + 2.0 * kap) - l / kap)
                         + l / (2.0 * kap) - (1.0 + 3.0 * kap) / (1.0 + 2.0 * kap) ** 2)
    sig_t = 8.0 * math.pi * R_E ** 2 / 3.0
    ser = sig_t * (1.0 - 2.0 * kap + 26.0 * kap ** 2 / 5.0 - 133.0 * kap ** 3 / 10.0
                   + 1144.0 * kap ** 4 / 35.0 - 544.0 * kap ** 5 / 7.0)
    return np.where(kap < 2.0e-3, ser, full)


def pair_shape(k):
    """P2: (7/9 - 2a + 4a^2/3 - 8a^3/9), a = m/k, zero below threshold; Sigma = shape / X0."""
    k = np.asarray(k, dtype=np.float64)
    a = M / k
    return np.where(k > 2.0 * M, 7.0 / 9.0 - 2.0 * a + 4.0 * a ** 2 / 3.0 - 8.0 * a ** 3 / 9.0, 0.0)


def sigma_photo_atom(k, Z):
    """P3 Born K-shell x 5/4 [cm^2 per atom]."""
    sig_t = 8.0 * math.pi * R_E ** 2 / 3.0
    return 1.25 * 4.0 * math.sqrt(2.0) * ALPHA ** 4 * Z ** 5 * sig_t * (M / np.asarray(k)) ** 3.5


def brem_shape(T, k_c):
    """P4: X0 * Sigma_brem(T; k_c)."""
    T = np.asarray(T, dtype=np.float64)
    E = T + M
    with np.errstate(divide="ignore", invalid="ignore"):
        val = (4.0 / 3.0) * np.log(T / k_c) - (4.0 / 3.0) * (T - k_c) / E \
            + (T * T - k_c * k_c) / (2.0 * E * E)
    return np.where(T > k_c, val, 0.0)


def srad_shape(T, k_c):
    """P4: X0 * S_rad(T; k_c) [MeV]; k_c = inf gives the unrestricted loss."""
    T = np.asarray(T, dtype=np.float64)
    E = T + M
    ku = np.minimum(k_c, T)
    return (4.0 / 3.0) * ku - (2.0 / 3.0) * ku ** 2 / E + ku ** 3 / (3.0 * E * E)


def sigma_moller(T, T_c):
    """P5 per electron [cm^2], zero for T <= 2 T_c."""
    T = np.asarray(T, dtype=np.float64)
    g = 1.0 + T / M
    b2 = 1.0 - 1.0 / (g * g)
    with np.errstate(divide="ignore", invalid="ignore"):
        x = T_c / T
        val = TWO_PI_RE2 / (b2 * (g - 1.0)) * (
            (g - 1.0) ** 2 / g ** 2 * (0.5 - x) + 1.0 / x - 1.0 / (1.0 - x)
            - (2.0 * g - 1.0) / g ** 2 * np.log((1.0 - x) / x))
    return np.where(T > 2.0 * T_c, val, 0.0)


def sigma_bhabha(T, T_c):
    """P6 per electron [cm^2], zero for T <= T_c."""
    T = np.asarray(T, dtype=np.float64)
    g = 1.0 + T / M
    b2 = 1.0 - 1.0 / (g * g)
    y = 1.0 / (g + 1.0)
    B1 = 2.0 - y * y
    B2 = (1.0 - 2.0 * y) * (3.0 + y * y)
    B3 = (1.0 - 2.0 * y) ** 2 + (1.0 - 2.0 * y) ** 3
    B4 = (1.0 - 2.0 * y) ** 3
    with np.errstate(divide="ignore", invalid="ignore"):
        x = T_c / T
        val = TWO_PI_RE2 / (g - 1.0) * ((1.0 / b2) * (1.0 / x - 1.0) + B1 * np.log(x)
                                        + B2 * (1.0 - x) - B3 * (1.0 - x * x) / 2.0
                                        + B4 * (1.0 - x ** 3) / 3.0)
    return np.where(T > T_c, val, 0.0)


def sigma_annihilation(T):
    """P8 Heitler, per electron [cm^2]."""
    g = 1.0 + np.asarray(T, dtype=np.float64) / M
    sq = np.sqrt(g * g - 1.0)
    return math.pi * R_E ** 2 / (g + 1.0) * ((g * g + 4.0 * g + 1.0) / (g * g - 1.0) * np.log(g + sq)
                                             - (g + 3.0) / sq)


def s_coll(T, mat, T_c, positron):
    """P7 restricted Bethe-Bloch (Berger-Seltzer) [MeV/cm]; T_c = inf => unrestricted."""
    T = np.asarray(T, dtype=np.float64)
    tau = T / M
    g = tau + 1.0
    b2 = 1.0 - 1.0 / (g * g)
    tau_max = tau if positron else 0.5 * tau
    tu = np.minimum(T_c / M, tau_max)
    # density effect (M3)
    bg = np.sqrt(tau * (tau + 2.0))
    delta = np.maximum(0.0, 2.0 * (math.log(mat.hwp / mat.I) + np.log(bg) - 0.5))
    if positron:
        y = 1.0 / (g + 1.0)
        F = np.log(tau * tu) - (b2 / tau) * (tau + 2.0 * tu - 1.5 * tu ** 2 * y
                                             - (tu - tu ** 3 / 3.0) * y ** 2
                                             - (tu ** 2 / 2.0 - tau * tu ** 3 / 3.0 + tu ** 4 / 4.0) * y ** 3)
    else:
        F = -1.0 - b2 + np.log((tau - tu) * tu) + tau / (tau - tu) \
            + (tu ** 2 / 2.0 + (2.0 * tau + 1.0) * np.log(1.0 - tu / tau)) / (g * g)
    return TWO_PI_RE2 * M * mat.n_el / b2 * (np.log(2.0 * (g + 1.0) / (mat.I / M) ** 2) + F - delta)


def _range_table(T, S):
    """M6: R_0 = T_0/S_0, then trapezoid in ln T of T/S."""
    f = T / S
    R = np.empty_like(T)
    R[0] = f[0]
    R[1:] = R[0] + np.cumsum(0.5 * DU * (f[1:] + f[:-1]))
    return R


def _interp_crossing_lnT(u_lo, y_lo, y_hi, target):
    return u_lo + DU * (target - y_lo) / (y_hi - y_lo)


def compute_cuts(mat):
    """M4: 0.7 mm -> (T_c for e-/e+, k_c for gamma), both clamped to >= 1 keV."""
    if mat.vacuum:
        return 0.0, 0.0
    T = energy_grid()
    # e-: CSDA range under the unrestricted total stopping power
    S = s_coll(T, mat, math.inf, False) + srad_shape(T, math.inf) / mat.X0
    R = _range_table(T, S)
    if R[0] >= PRODUCTION_CUT_CM:
        e_cut = T_GRID_MIN
    else:
        j = int(np.searchsorted(R, PRODUCTION_CUT_CM, side="right")) - 1
        e_cut = math.exp(_interp_crossing_lnT(U0 + DU * j, R[j], R[j + 1], PRODUCTION_CUT_CM))
    # gamma: falling low-energy branch where 5 / Sigma_tot = cut
    sig = mat.n_el * sigma_compton(T) + pair_shape(T) / mat.X0 + photo_macro(mat, T)
    target = 5.0 / PRODUCTION_CUT_CM
    if sig[0] <= target:
        g_cut = T_GRID_MIN
    else:
        j = int(np.argmax(sig < target)) - 1          # sig[j] >= target > sig[j+1]
        g_cut = math.exp(_interp_crossing_lnT(U0 + DU * j, sig[j], sig[j + 1], target))
    return max(e_cut, T_GRID_MIN), max(g_cut, T_GRID_MIN)


def build_tables(mat):
    """M6: the 12 x 2048 table block of one material (fills mat.e_cut / mat.g_cut)."""
    tab = np.zeros((N_TABLES, N_GRID), dtype=np.float64)
    if mat.vacuum:
        tab[TAB_EM_RANGE] = VACUUM_RANGE
        tab[TAB_EP_RANGE] = VACUUM_RANGE
        return tab
    mat.e_cut, mat.g_cut = compute_cuts(mat)
    T = energy_grid()
    tab[TAB_G_COMPTON] = mat.n_el * sigma_compton(T)
    tab[TAB_G_PAIR] = pair_shape(T) / mat.X0
    tab[TAB_G_PHOTO] = photo_macro(mat, T)
    brem = brem_shape(T, mat.g_cut) / mat.X0
    srad = srad_shape(T, mat.g_cut) / mat.X0
    tab[TAB_EM_BREM] = brem
    tab[TAB_EM_IONI] = mat.n_el * sigma_moller(T, mat.e_cut)
    tab[TAB_EM_DEDX] = s_coll(T, mat, mat.e_cut, False) + srad
    tab[TAB_EM_RANGE] = _range_table(T, tab[TAB_EM_DEDX])
    tab[TAB_EP_BREM] = brem
    tab[TAB_EP_IONI] = mat.n_el * sigma_bhabha(T, mat.e_cut)
    tab[TAB_EP_ANNI] = mat.n_el * sigma_annihilation(T)
    tab[TAB_EP_DEDX] = s_coll(T, mat, mat.e_cut, True) + srad
    tab[TAB_EP_RANGE] = _range_table(T, tab[TAB_EP_DEDX])
    return tab


N_MAT_SCALARS = 8


def material_scalars(mat):
    """Per-material scalar block of the C ABI: X0, T_c, k_c, B_K, n_el, vacuum flag, Z, rho."""
    return np.array([mat.X0 if not mat.vacuum else 1.0e99, mat.e_cut, mat.g_cut, mat.B_K, mat.n_el,
                     1.0 if mat.vacuum else 0.0, mat.Z, mat.rho], dtype=np.float64)


MAX_ELEMENTS = 4


def element_tables(mats):
    """C5, the element selector's inputs (adept_tables.n_elem / elem_bk / pe_cum): per material the number of
    elements, their K-shell binding energies, and on the ln T grid the cumulative share of elements 0..j in the
    photoelectric cross section (1 from the last element on).  None if every material is a single element."""
    if not any(len(m.elements) > 1 for m in mats):
        return None
    n_elem = np.ones(len(mats), dtype=np.int32)
    bk = np.zeros((len(mats), MAX_ELEMENTS))
    cum = np.ones((len(mats), N_GRID, MAX_ELEMENTS))
    T = energy_grid()
    for i, m in enumerate(mats):
        if not m.elements:
            bk[i, 0] = m.B_K
            continue
        n = len(m.elements)
        assert n <= MAX_ELEMENTS
        n_elem[i] = n
        bk[i, :n] = m.B_K_i
        part = np.stack([ni * sigma_photo_atom(T, z) for ni, (z, _, _) in zip(m.n_i, m.elements)], axis=1)
        share = np.cumsum(part, axis=1) / part.sum(axis=1, keepdims=True)
        cum[i, :, :n - 1] = share[:, :n - 1]
    return n_elem, np.ascontiguousarray(bk), np.ascontiguousarray(cum)


def build_material_set(names):
    """-> (list[Material], tables (n,12,2048), scalars (n,8)) for the named standard materials."""
    std = standard_materials()
    mats = [std[n] for n in names]
    tabs = np.stack([build_tables(m) for m in mats])
    scal = np.stack([material_scalars(m) for m in mats])
    return mats, np.ascontiguousarray(tabs), np.ascontiguousarray(scal)
