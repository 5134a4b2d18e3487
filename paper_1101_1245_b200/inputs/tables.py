"""Closed-form cross-section / stopping-power tables (input data only).

GPUMCD reads its cross sections and stopping powers from pre-interpolated
tables (Sec. II.C.2) that come from EGSnrc data files which are
not available here.  BASELINE.json's north_star fixes the substitute: tables
"generated in-build from closed-form models (Klein-Nishina; a Z^n/E^3
photoelectric parameterisation; a Bethe-Heitler-style pair model; Bethe-Bloch
restricted stopping power; Moller; a screened bremsstrahlung parameterisation)
and shared as data only".  This module is that generator.  Its output is a
bundle of float32 arrays handed unchanged to ``gpumcd_create`` and to the CPU
oracle; neither transport implementation imports anything from here.

All columns are *mass* coefficients (per g/cm^2) on a grid that is uniform in
ln(E) between ``e_min`` and ``e_max``; the transport codes multiply by the
voxel density (Eq. 2).  Energies are kinetic, in MeV.

Column order
    photon  [n_mat][3][n_E]: compton, photoelectric, pair            (cm^2/g)
    electron[n_mat][4][n_E]: L_restricted (MeV cm^2/g),
                             moller_hard, brems_hard, inv_lambda1    (cm^2/g)
    ms_a    [n_K]           : screening parameter a(K) of the one-parameter
                              multiple-scattering distribution on a uniform
                              ln(K) grid.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Sequence

import numpy as np

from .materials import ELEMENTS, Material

# physical constants (CODATA), units MeV / cm / g
M_E = 0.51099895          # electron rest energy, MeV
R_E = 2.8179403e-13       # classical electron radius, cm
N_A = 6.02214076e23       # Avogadro
ALPHA = 1.0 / 137.035999  # fine-structure constant
ZETA3 = 1.2020569031595942

PHOTO_TAU0 = 4.94         # cm^2/g, water at 10 keV (anchor of the Z^n/E^3 parameterisation)
PHOTO_ZREF = 7.42         # effective Z of water under the 2.94-power rule
PHOTO_ZEXP = 2.94


@dataclass
class TableBundle:
    """What both transport implementations receive (all float32, C order)."""
    n_materials: int
    n_energy: int
    e_min: float
    e_max: float
    photon: np.ndarray        # [n_mat, 3, n_E]
    electron: np.ndarray      # [n_mat, 4, n_E]
    n_K: int
    lnK_min: float
    lnK_max: float
    ms_a: np.ndarray          # [n_K]
    e_cut: float              # electron kinetic cutoff = K_cut of the tables
    p_cut: float              # photon cutoff = k_c of the brems tables
    names: tuple

    def energy_grid(self) -> np.ndarray:
        return np.exp(np.linspace(np.log(self.e_min), np.log(self.e_max), self.n_energy))


# ----------------------------------------------------------------------------
# photons
# ----------------------------------------------------------------------------
def sigma_kn(E):
    """Klein-Nishina total cross section per electron, cm^2."""
    k = np.asarray(E, dtype=np.float64) / M_E
    l = np.log1p(2.0 * k)
    return 2.0 * np.pi * R_E**2 * (
        (1.0 + k) / k**2 * (2.0 * (1.0 + k) / (1.0 + 2.0 * k) - l / k)
        + l / (2.0 * k)
        - (1.0 + 3.0 * k) / (1.0 + 2.0 * k) ** 2
    )


def compton_mass(mat: Material, E):
    return N_A * mat.za_ratio() * sigma_kn(E)


def photo_zeff(mat: Material) -> float:
    """Effective Z by the power rule over electron fractions."""
    za = {e: w * ELEMENTS[e][0] / ELEMENTS[e][1] for e, w in mat.weights.items()}
    tot = sum(za.values())
    return sum((v / tot) * ELEMENTS[e][0] ** PHOTO_ZEXP for e, v in za.items()) ** (1.0 / PHOTO_ZEXP)


def photo_mass(mat: Material, E):
    """Z^n/E^3 photoelectric parameterisation anchored on water at 10 keV."""
    E = np.asarray(E, dtype=np.float64)
    return PHOTO_TAU0 * (photo_zeff(mat) / PHOTO_ZREF) ** 3 * (0.01 / E) ** 3


def pair_F(E):
    """Unscreened Born pair cross section in units of alpha r_e^2 Z^2 (Maximon expansions)."""
    k = np.atleast_1d(np.asarray(E, dtype=np.float64) / M_E)
    F = np.zeros_like(k)
    lo = (k > 2.0) & (k <= 4.0)
    if lo.any():
        kk = k[lo]
        eps = (2.0 * kk - 4.0) / (2.0 + kk + 2.0 * np.sqrt(2.0 * kk))
        F[lo] = (2.0 * np.pi / 3.0) * ((kk - 2.0) / kk) ** 3 * (
            1.0 + eps / 2.0 + 23.0 * eps**2 / 40.0 + 11.0 * eps**3 / 60.0 + 29.0 * eps**4 / 960.0
        )
    hi = k > 4.0
    if hi.any():
        kk = k[hi]
        l = np.log(2.0 * kk)
        q = 2.0 / kk
        F[hi] = (
            28.0 * l / 9.0 - 218.0 / 27.0
            + q**2 * (6.0 * l - 3.5 + (2.0 / 3.0) * l**3 - l**2 - (np.pi**2 / 3.0) * l
                      + 2.0 * ZETA3 + np.pi**2 / 6.0)
            - q**4 * (3.0 * l / 16.0 + 1.0 / 8.0)
            - q**6 * (29.0 * l / 2304.0 - 77.0 / 13824.0)
        )
    return F


def pair_mass(mat: Material, E):
    """Bethe-Heitler-style nuclear pair production, Z^2 only, no triplet."""
    z2a = sum(w * ELEMENTS[e][0] ** 2 / ELEMENTS[e][1] for e, w in mat.weights.items())
    return N_A * z2a * ALPHA * R_E**2 * pair_F(E)


# ----------------------------------------------------------------------------
# electrons
# ----------------------------------------------------------------------------
def _beta2(tau):
    return tau * (tau + 2.0) / (tau + 1.0) ** 2


def density_effect(mat: Material, T):
    """Sternheimer-Peierls density-effect correction delta(T)."""
    T = np.asarray(T, dtype=np.float64)
    tau = T / M_E
    x = np.log10(np.sqrt(tau * (tau + 2.0)))          # log10(beta*gamma)
    if mat.sternheimer:
        Cbar, x0, x1, a, m = mat.sternheimer
    else:
        hnu_p = 28.816 * np.sqrt(mat.density * mat.za_ratio())   # plasma energy, eV
        Cbar = 2.0 * np.log(mat.I_eV / hnu_p) + 1.0
        m = 3.0
        if mat.gas:
            x1 = 4.0
            if Cbar < 10.0:
                x0 = 1.6
            elif Cbar < 10.5:
                x0 = 1.7
            elif Cbar < 11.0:
                x0 = 1.8
            elif Cbar < 11.5:
                x0 = 1.9
            elif Cbar < 12.25:
                x0 = 2.0
            elif Cbar < 13.804:
                x0, x1 = 2.0, 5.0
            else:
                x0, x1 = 0.326 * Cbar - 2.5, 5.0
        elif mat.I_eV < 100.0:
            x1 = 2.0
            x0 = 0.2 if Cbar < 3.681 else 0.326 * Cbar - 1.0
        else:
            x1 = 3.0
            x0 = 0.2 if Cbar < 5.215 else 0.326 * Cbar - 1.5
        a = (Cbar - 2.0 * np.log(10.0) * x0) / (x1 - x0) ** 3
    d = np.zeros_like(x)
    mid = (x >= x0) & (x < x1)
    d[mid] = 2.0 * np.log(10.0) * x[mid] - Cbar + a * (x1 - x[mid]) ** m
    top = x >= x1
    d[top] = 2.0 * np.log(10.0) * x[top] - Cbar
    return d


def collision_stopping_restricted(mat: Material, T, k_cut):
    """Restricted collision mass stopping power (Moller), MeV cm^2/g (Eq. 6).

    ``k_cut >= T/2`` gives the unrestricted Bethe value.
    """
    T = np.asarray(T, dtype=np.float64)
    tau = T / M_E
    b2 = _beta2(tau)
    eta = np.minimum(k_cut / T, 0.5)
    G = (-1.0 - b2 + np.log(4.0 * (1.0 - eta) * eta) + 1.0 / (1.0 - eta)
         + (1.0 - b2) * (tau**2 * eta**2 / 2.0 + (2.0 * tau + 1.0) * np.log(1.0 - eta)))
    pref = 2.0 * np.pi * R_E**2 * M_E * N_A * mat.za_ratio() / b2
    I = mat.I_eV * 1e-6
    return pref * (np.log(tau**2 * (tau + 2.0) / (2.0 * (I / M_E) ** 2)) + G - density_effect(mat, T))


def moller_dsigma_deps(mat: Material, T, eps):
    """Moller d(Sigma/rho)/d(eps), eps = W/T in (0, 1/2], cm^2/g."""
    tau = T / M_E
    b2 = _beta2(tau)
    g2 = (tau / (tau + 1.0)) ** 2
    g3 = (2.0 * tau + 1.0) / (tau + 1.0) ** 2
    r = eps / (1.0 - eps)
    return N_A * mat.za_ratio() * 2.0 * np.pi * R_E**2 / (b2 * tau) / eps**2 * (1.0 + g2 * eps**2 + r * (r - g3))


def moller_hard_mass(mat: Material, T, k_cut):
    """Total Moller cross section for energy transfers above k_cut, cm^2/g."""
    T = np.asarray(T, dtype=np.float64)
    tau = T / M_E
    b2 = _beta2(tau)
    eta = np.minimum(k_cut / T, 0.5)
    g2 = (tau / (tau + 1.0)) ** 2
    g3 = (2.0 * tau + 1.0) / (tau + 1.0) ** 2
    br = 1.0 / eta - 1.0 / (1.0 - eta) + g2 * (0.5 - eta) - g3 * np.log((1.0 - eta) / eta)
    out = N_A * mat.za_ratio() * 2.0 * np.pi * R_E**2 / (b2 * tau) * br
    return np.where(T > 2.0 * k_cut, out, 0.0)


def inv_radiation_length(mat: Material) -> float:
    """1/X0 in cm^2/g (Tsai's formula with Coulomb correction)."""
    tot = 0.0
    for e, w in mat.weights.items():
        Z, A = ELEMENTS[e]
        if Z == 1:
            Lrad, Lradp = 5.31, 6.144
        else:
            Lrad = np.log(184.15 * Z ** (-1.0 / 3.0))
            Lradp = np.log(1194.0 * Z ** (-2.0 / 3.0))
        az2 = (ALPHA * Z) ** 2
        fC = az2 * (1.0 / (1.0 + az2) + 0.20206 - 0.0369 * az2 + 0.0083 * az2**2 - 0.002 * az2**3)
        tot += w * 4.0 * ALPHA * R_E**2 * (N_A / A) * (Z * Z * (Lrad - fC) + Z * Lradp)
    return tot


def brems_hard_mass(mat: Material, T, k_c):
    """Complete-screening bremsstrahlung cross section for photon energies k in [k_c, T], cm^2/g."""
    T = np.asarray(T, dtype=np.float64)
    Et = T + M_E
    out = inv_radiation_length(mat) * (
        (4.0 / 3.0) * np.log(T / k_c) - (4.0 / 3.0) * (T - k_c) / Et + (T**2 - k_c**2) / (2.0 * Et**2)
    )
    return np.where(T > k_c, out, 0.0)


def brems_soft_stopping(mat: Material, T, k_c):
    """Radiative energy loss to photons below k_c, MeV cm^2/g (added to L)."""
    T = np.asarray(T, dtype=np.float64)
    Et = T + M_E
    kc = np.minimum(k_c, T)
    return inv_radiation_length(mat) * (4.0 * kc / 3.0 - 2.0 * kc**2 / (3.0 * Et) + kc**3 / (3.0 * Et**2))


def brems_total_stopping(mat: Material, T):
    """Total radiative stopping power of the same parameterisation (closed form)."""
    T = np.asarray(T, dtype=np.float64)
    return brems_soft_stopping(mat, T, T)


def inv_lambda1_mass(mat: Material, T):
    """Inverse first transport mean free path of screened-Rutherford scattering, cm^2/g."""
    T = np.asarray(T, dtype=np.float64)
    tau = T / M_E
    b2 = _beta2(tau)
    tot = np.zeros_like(T)
    for e, w in mat.weights.items():
        Z, A = ELEMENTS[e]
        eta_s = (ALPHA**2 * Z ** (2.0 / 3.0) / (4.0 * 0.885**2)) / (tau * (tau + 2.0)) * (
            1.13 + 3.76 * (ALPHA * Z) ** 2 / b2)
        tot += w * (N_A / A) * 2.0 * np.pi * R_E**2 * Z * (Z + 1.0) / (b2**2 * (tau + 1.0) ** 2) * (
            np.log((1.0 + eta_s) / eta_s) - 1.0 / (1.0 + eta_s))
    return tot


# ----------------------------------------------------------------------------
# multiple-scattering shape parameter
# ----------------------------------------------------------------------------
def ms_mean_mu2(a):
    """2<mu> = 1 - <cos theta> of the Wentzel shape p(mu) ~ (a+mu)^-2 on mu in [0,1]."""
    a = np.asarray(a, dtype=np.float64)
    x = 1.0 / a
    big = a > 1e3
    out = np.empty_like(a)
    aa = a[~big]
    out[~big] = 2.0 * aa * (1.0 + aa) * (np.log1p(1.0 / aa) - 1.0 / (1.0 + aa))
    xx = x[big]
    out[big] = 1.0 - xx / 3.0 + xx**2 / 6.0 - xx**3 / 10.0 + xx**4 / 15.0
    return out


def ms_a_table(n_K: int, lnK_min: float, lnK_max: float) -> np.ndarray:
    """Solve 2<mu>(a) = 1 - exp(-K) for a on a uniform ln K grid (bisection in ln a)."""
    lnK = np.linspace(lnK_min, lnK_max, n_K)
    target = -np.expm1(-np.exp(lnK))
    lo = np.full(n_K, np.log(1e-12))
    hi = np.full(n_K, np.log(1e12))
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        f = ms_mean_mu2(np.exp(mid))
        up = f < target
        lo = np.where(up, mid, lo)
        hi = np.where(up, hi, mid)
    return np.exp(0.5 * (lo + hi))


# ----------------------------------------------------------------------------
# bundle
# ----------------------------------------------------------------------------
def build_tables(materials: Sequence[Material], n_energy: int = 1024, e_min: float = 0.01,
                 e_max: float = 20.0, e_cut: float = 0.2, p_cut: float = 0.01,
                 n_K: int = 1024, K_min: float = 1e-6, K_max: float = 20.0) -> TableBundle:
    E = np.exp(np.linspace(np.log(e_min), np.log(e_max), n_energy))
    n_mat = len(materials)
    photon = np.zeros((n_mat, 3, n_energy))
    electron = np.zeros((n_mat, 4, n_energy))
    for i, mat in enumerate(materials):
        photon[i, 0] = compton_mass(mat, E)
        photon[i, 1] = photo_mass(mat, E)
        photon[i, 2] = pair_mass(mat, E)
        electron[i, 0] = collision_stopping_restricted(mat, E, e_cut) + brems_soft_stopping(mat, E, p_cut)
        electron[i, 1] = moller_hard_mass(mat, E, e_cut)
        electron[i, 2] = brems_hard_mass(mat, E, p_cut)
        electron[i, 3] = inv_lambda1_mass(mat, E)
    lnK_min, lnK_max = float(np.log(K_min)), float(np.log(K_max))
    return TableBundle(
        n_materials=n_mat, n_energy=n_energy, e_min=float(e_min), e_max=float(e_max),
        photon=np.ascontiguousarray(photon, dtype=np.float32),
        electron=np.ascontiguousarray(electron, dtype=np.float32),
        n_K=n_K, lnK_min=lnK_min, lnK_max=lnK_max,
        ms_a=np.ascontiguousarray(ms_a_table(n_K, lnK_min, lnK_max), dtype=np.float32),
        e_cut=float(e_cut), p_cut=float(p_cut), names=tuple(m.name for m in materials),
    )
