"""Pins of the closed-form input tables: identities, continuity, anchors.

The tables are input data shared by the oracle and the CUDA library, so they cannot affect
parity; these tests guard their physical plausibility and the generator itself.
"""
import numpy as np
import pytest
from scipy import integrate

from paper_1101_1245_b200.inputs import materials as M
from paper_1101_1245_b200.inputs import tables as T


def test_klein_nishina_limits_and_anchor():
    # Thomson limit (8 pi / 3) r_e^2 as E -> 0
    thomson = 8.0 * np.pi / 3.0 * T.R_E**2
    assert T.sigma_kn(1e-6) == pytest.approx(thomson, rel=1e-4)
    # total cross section equals the integral of the differential KN formula
    for E in (0.05, 2.0, 15.0):
        k = E / T.M_E

        def dsig(c):
            r = 1.0 / (1.0 + k * (1.0 - c))
            return np.pi * T.R_E**2 * r * r * (r + 1.0 / r - (1.0 - c * c))

        val, _ = integrate.quad(dsig, -1.0, 1.0)
        assert T.sigma_kn(E) == pytest.approx(val, rel=1e-9)
    # water at 2 MeV: tabulated incoherent coefficient 0.0490 cm^2/g
    assert T.compton_mass(M.WATER, 2.0) == pytest.approx(0.0490, rel=0.01)


def test_photoelectric_anchor_and_scaling():
    assert T.photo_zeff(M.WATER) == pytest.approx(7.42, abs=0.01)
    assert T.photo_mass(M.WATER, 0.01) == pytest.approx(4.94, rel=0.01)
    assert T.photo_mass(M.WATER, 0.02) / T.photo_mass(M.WATER, 0.01) == pytest.approx(1 / 8)
    assert T.photo_mass(M.BONE, 0.05) > T.photo_mass(M.WATER, 0.05)


def test_pair_threshold_continuity_and_asymptote():
    assert T.pair_F(2.0 * T.M_E) == 0.0 and T.pair_F(1.0) == 0.0
    lo = T.pair_F(4.0 * T.M_E * (1 - 1e-9))[0]
    hi = T.pair_F(4.0 * T.M_E * (1 + 1e-9))[0]
    assert lo == pytest.approx(hi, rel=5e-4)
    E = np.exp(np.linspace(np.log(1.03), np.log(20.0), 400))
    F = T.pair_F(E)
    assert np.all(np.diff(F) > 0)
    # high-energy unscreened limit 28/9 ln(2k) - 218/27
    k = 1e5
    assert T.pair_F(k * T.M_E)[0] == pytest.approx(28 / 9 * np.log(2 * k) - 218 / 27, rel=1e-6)


@pytest.mark.parametrize("mat", [M.WATER, M.BONE, M.LUNG, M.AIR, M.SOFT])
@pytest.mark.parametrize("Tk", [0.5, 1.0, 5.0, 20.0])
def test_restricted_plus_hard_moller_equals_unrestricted(mat, Tk):
    """L_col(T, K_cut) + int_{K_cut}^{T/2} W dSigma_Moller = S_col(T)  (Eq. 6 split)."""
    k_cut = 0.2
    hard, _ = integrate.quad(lambda e: e * Tk * T.moller_dsigma_deps(mat, Tk, e), k_cut / Tk, 0.5,
                             epsabs=0, epsrel=1e-10)
    total = T.collision_stopping_restricted(mat, np.array([Tk]), 1e9)[0]
    restricted = T.collision_stopping_restricted(mat, np.array([Tk]), k_cut)[0]
    assert restricted + hard == pytest.approx(total, rel=1e-8)


@pytest.mark.parametrize("Tk", [1.0, 15.0])
def test_moller_total_is_integral_of_differential(Tk):
    k_cut = 0.2
    val, _ = integrate.quad(lambda e: T.moller_dsigma_deps(M.WATER, Tk, e), k_cut / Tk, 0.5, epsrel=1e-10)
    assert T.moller_hard_mass(M.WATER, np.array([Tk]), k_cut)[0] == pytest.approx(val, rel=1e-8)
    assert T.moller_hard_mass(M.WATER, np.array([0.39]), k_cut)[0] == 0.0


def test_water_stopping_power_anchors():
    # ICRU-37-like values for liquid water (unrestricted collision): 1.849 / 1.968 at 1 / 10 MeV
    S = T.collision_stopping_restricted(M.WATER, np.array([1.0, 10.0]), 1e9)
    assert S[0] == pytest.approx(1.849, rel=0.01)
    assert S[1] == pytest.approx(1.968, rel=0.01)


@pytest.mark.parametrize("Tk", [1.0, 15.0])
def test_brems_hard_plus_soft(Tk):
    k_c = 0.01
    invX0 = T.inv_radiation_length(M.WATER)
    Et = Tk + T.M_E

    def shape(k):
        y = k / Et
        return invX0 / k * (4.0 / 3.0 * (1 - y) + y * y)

    sig, _ = integrate.quad(shape, k_c, Tk, epsrel=1e-10)
    assert T.brems_hard_mass(M.WATER, np.array([Tk]), k_c)[0] == pytest.approx(sig, rel=1e-8)
    soft, _ = integrate.quad(lambda k: k * shape(k), 0, k_c, epsrel=1e-10)
    assert T.brems_soft_stopping(M.WATER, np.array([Tk]), k_c)[0] == pytest.approx(soft, rel=1e-8)
    hard_loss, _ = integrate.quad(lambda k: k * shape(k), k_c, Tk, epsrel=1e-10)
    assert soft + hard_loss == pytest.approx(T.brems_total_stopping(M.WATER, np.array([Tk]))[0], rel=1e-8)
    assert 1.0 / invX0 == pytest.approx(36.08, rel=0.005)   # radiation length of water, g/cm^2


def test_transport_mfp_anchor_and_monotone():
    E = np.exp(np.linspace(np.log(0.01), np.log(20), 200))
    lam = 1.0 / T.inv_lambda1_mass(M.WATER, E)
    assert np.all(np.diff(lam) > 0)
    assert 1.0 / T.inv_lambda1_mass(M.WATER, np.array([1.0]))[0] == pytest.approx(0.51, rel=0.05)


def test_ms_shape_parameter_solves_its_equation():
    tb = T.build_tables([M.WATER])
    lnK = np.linspace(tb.lnK_min, tb.lnK_max, tb.n_K)
    a = tb.ms_a.astype(np.float64)
    assert np.all(np.diff(a) > 0)
    # <cos> of p(mu) ~ (a+mu)^-2 by quadrature equals exp(-K)
    for i in (0, 100, 400, 700, 900, 1000):
        ai = a[i]
        norm = 1.0 / ai - 1.0 / (1.0 + ai)
        pts = [10.0 ** e for e in range(-12, 0) if ai * 1e-2 < 10.0 ** e < 1]
        mean_mu, _ = integrate.quad(lambda mu: mu / (ai + mu) ** 2 / norm, 0, 1, epsrel=1e-12, points=pts or None,
                                    limit=400)
        assert 2.0 * mean_mu == pytest.approx(-np.expm1(-np.exp(lnK[i])), rel=2e-6)
    # anchors: a(0.01), a(1)
    assert np.interp(np.log(0.01), lnK, a) == pytest.approx(8.127e-4, rel=2e-3)
    assert np.interp(0.0, lnK, a) == pytest.approx(0.4618, rel=2e-3)


def test_bundle_layout():
    tb = T.build_tables([M.WATER, M.BONE])
    assert tb.photon.shape == (2, 3, 1024) and tb.photon.dtype == np.float32
    assert tb.electron.shape == (2, 4, 1024) and tb.electron.dtype == np.float32
    assert tb.ms_a.shape == (1024,)
    E = tb.energy_grid()
    assert E[0] == pytest.approx(0.01) and E[-1] == pytest.approx(20.0)
    assert np.all(tb.electron[:, 0] > 0) and np.all(tb.photon[:, 0] > 0)
    assert np.all(tb.electron[:, 1][:, E <= 0.4] == 0)
