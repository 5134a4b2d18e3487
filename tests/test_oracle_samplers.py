"""Distribution pins of the oracle's samplers: sampled histograms against the analytic
densities the paper names (chi-square, p > 0.01), moments against quadrature, closed-form
CDFs and kinematic identities.  Seeds are fixed, so the tests are deterministic."""
import numpy as np
import pytest
from scipy import integrate, stats

import oracle

M_E = 0.51099895
N = 200_000


def chi2_against_pdf(samples, pdf, lo, hi, nbins=40, log_bins=False):
    edges = np.geomspace(lo, hi, nbins + 1) if log_bins else np.linspace(lo, hi, nbins + 1)
    obs, _ = np.histogram(samples, bins=edges)
    assert obs.sum() == samples.size, "samples outside the support"
    p = np.array([integrate.quad(pdf, a, b, epsrel=1e-10)[0] for a, b in zip(edges[:-1], edges[1:])])
    p /= p.sum()
    exp = p * samples.size
    keep = exp > 5
    chi2 = ((obs[keep] - exp[keep]) ** 2 / exp[keep]).sum()
    return stats.chi2.sf(chi2, keep.sum() - 1)


@pytest.mark.parametrize("E", [0.05, 2.0, 15.0])
def test_compton_energy_distribution_is_klein_nishina(E):
    """Klein-Nishina for a free electron.  d sigma/d eps ~ 1/eps + eps - sin^2(theta)."""
    k = E / M_E
    eps0 = 1.0 / (1.0 + 2.0 * k)
    eps, cost, phi = oracle.batch_compton(E, seed=11, n=N)

    def pdf(e):
        t = (1.0 - e) / (k * e)
        return 1.0 / e + e - t * (2.0 - t)

    assert chi2_against_pdf(eps, pdf, eps0, 1.0) > 0.01
    norm = integrate.quad(pdf, eps0, 1.0)[0]
    mean = integrate.quad(lambda e: e * pdf(e), eps0, 1.0)[0] / norm
    sd = np.sqrt(integrate.quad(lambda e: e * e * pdf(e), eps0, 1.0)[0] / norm - mean**2)
    assert abs(eps.mean() - mean) < 4 * sd / np.sqrt(N)
    # Compton kinematics: E'/E = 1/(1 + k (1 - cos theta))
    np.testing.assert_allclose(eps, 1.0 / (1.0 + k * (1.0 - cost)), rtol=1e-12)
    # azimuth uniform
    assert stats.kstest(phi / (2 * np.pi), "uniform").pvalue > 0.01


@pytest.mark.parametrize("T", [1.0, 15.0])
def test_moller_energy_distribution(T):
    """Moller cross section for transfers above K_cut."""
    k_cut = 0.2
    tau = T / M_E
    g2 = (tau / (tau + 1)) ** 2
    g3 = (2 * tau + 1) / (tau + 1) ** 2
    eps, cp, cd = oracle.batch_moller(T, k_cut, seed=12, n=N)

    def pdf(e):
        r = e / (1 - e)
        return (1 + g2 * e * e + r * (r - g3)) / (e * e)

    assert chi2_against_pdf(eps, pdf, k_cut / T, 0.5, log_bins=True) > 0.01
    # two-body kinematics: transverse momenta of the two outgoing electrons cancel
    W = eps * T
    p_p = np.sqrt((T - W) * (T - W + 2 * M_E))
    p_d = np.sqrt(W * (W + 2 * M_E))
    np.testing.assert_allclose(p_p * np.sqrt(1 - cp**2), p_d * np.sqrt(1 - cd**2), rtol=1e-9)
    # and the longitudinal ones add up to the incident momentum
    np.testing.assert_allclose(p_p * cp + p_d * cd, np.sqrt(T * (T + 2 * M_E)), rtol=1e-12)


@pytest.mark.parametrize("T", [1.0, 15.0])
def test_brems_photon_energy_distribution(T):
    """photon energy above k_c; complete-screening shape."""
    k_c = 0.01
    k = oracle.batch_brems(T, k_c, seed=13, n=N)

    def pdf(x):
        y = x / (T + M_E)
        return (4.0 / 3.0 * (1 - y) + y * y) / x

    assert chi2_against_pdf(k, pdf, k_c, T, log_bins=True) > 0.01


@pytest.mark.parametrize("E", [0.25, 1.0, 20.0])
def test_sauter_angle_distribution(E):
    """Sauter K-shell photo-electron angular distribution."""
    gam = 1 + E / M_E
    beta = np.sqrt(E * (E + 2 * M_E)) / (E + M_E)
    A = 1 / beta - 1
    B = 0.5 * beta * gam * (gam - 1) * (gam - 2)
    nu = oracle.batch_sauter(E, seed=14, n=N)

    def pdf(v):
        return (2 - v) * (1 / (A + v) + B) * v / (A + v) ** 3

    # same density written in theta: sin^2(theta)/(1-beta cos)^4 [1 + gamma(gamma-1)(gamma-2)(1-beta cos)/2]
    for v in (0.1, 0.7, 1.5):
        c = 1 - v
        alt = (1 - c * c) / (1 - beta * c) ** 4 * (1 + 0.5 * gam * (gam - 1) * (gam - 2) * (1 - beta * c))
        assert pdf(v) / pdf(1.0) == pytest.approx(
            alt / ((1.0) / 1.0 * (1 + 0.5 * gam * (gam - 1) * (gam - 2))), rel=1e-9)
    assert chi2_against_pdf(nu, pdf, 0.0, 2.0) > 0.01


def test_pair_split_and_angles():
    """uniform energy split; polar density ~ (1 - beta cos)^-2."""
    E = 10.0
    T1, c1, c2 = oracle.batch_pair(E, seed=15, n=N)
    Tsum = E - 2 * M_E
    assert stats.kstest(T1 / Tsum, "uniform").pvalue > 0.01
    # angle of electron 1 for a narrow band of T1: analytic CDF of (1 - beta c)^-2 on [-1, 1]
    sel = (T1 > 4.0) & (T1 < 4.1)
    Tm = T1[sel].mean()
    beta = np.sqrt(Tm * (Tm + 2 * M_E)) / (Tm + M_E)

    def cdf(c):
        return ((1 / (1 - beta * c)) - 1 / (1 + beta)) / (1 / (1 - beta) - 1 / (1 + beta))

    assert sel.sum() > 1000
    assert stats.kstest(c1[sel], cdf).pvalue > 0.01
    # electron 2 carries T2 = Tsum - T1: same law with its own beta
    T2m = Tsum - Tm
    beta = np.sqrt(T2m * (T2m + 2 * M_E)) / (T2m + M_E)
    assert stats.kstest(c2[sel], cdf).pvalue > 0.01


@pytest.mark.parametrize("K", [1e-3, 0.05, 0.5, 3.0])
def test_multiple_scattering_mean_cosine(K, water_tables):
    """PAPER.md L100 substitute (R13): <cos theta> = exp(-K) with a = a(K) from the table."""
    tb = water_tables
    a = oracle.lookup(tb.ms_a, tb.lnK_min, tb.lnK_max, np.log(K))
    c = oracle.batch_ms(a, seed=16, n=N)
    assert np.all(c <= 1.0) and np.all(c >= -1.0)
    assert abs(c.mean() - np.exp(-K)) < 4 * c.std() / np.sqrt(N) + 2e-4 * (1 - np.exp(-K))
    mu = (1 - c) / 2
    assert stats.kstest(mu, lambda m: (1 + a) * m / (a + m)).pvalue > 0.01


def test_ms_isotropic_limit():
    c = oracle.batch_ms(1e9, seed=17, n=N)
    assert stats.kstest((c + 1) / 2, "uniform").pvalue > 0.01


def test_rotation_geometry():
    rng = np.random.default_rng(3)
    for _ in range(200):
        d = rng.standard_normal(3)
        d /= np.linalg.norm(d)
        cost = rng.uniform(-1, 1)
        phi = rng.uniform(0, 2 * np.pi)
        out = oracle.rotate(d, cost, phi)
        assert np.linalg.norm(out) == pytest.approx(1.0, abs=1e-12)
        assert np.dot(out, d) == pytest.approx(cost, abs=1e-9)
    # azimuth sweeps a full, evenly spaced circle about d
    d = np.array([0.3, -0.5, np.sqrt(1 - 0.09 - 0.25)])
    ring = np.array([oracle.rotate(d, 0.2, p) for p in np.linspace(0, 2 * np.pi, 8, endpoint=False)])
    assert np.allclose(ring.mean(axis=0), 0.2 * d, atol=1e-12)
    step = [np.dot(ring[i], ring[(i + 1) % 8]) for i in range(8)]
    assert np.allclose(step, step[0], atol=1e-12)
    # pole branch agrees with the general formula's limit
    for w in (1.0, -1.0):
        out = oracle.rotate([0.0, 0.0, w], 0.5, 0.3)
        assert out[2] == pytest.approx(0.5 * w)
        assert np.hypot(out[0], out[1]) == pytest.approx(np.sqrt(0.75))
    near = oracle.rotate([2e-5, 0.0, np.sqrt(1 - 4e-10)], 0.5, 0.3)
    pole = oracle.rotate([0.0, 0.0, 1.0], 0.5, 0.3)
    assert np.allclose(near, pole, atol=1e-4)


def test_lookup_matches_linear_interpolation(water_tables):
    tb = water_tables
    lnE = np.linspace(np.log(tb.e_min), np.log(tb.e_max), tb.n_energy)
    col = tb.electron[0, 0]
    rng = np.random.default_rng(5)
    for x in rng.uniform(lnE[0], lnE[-1], 200):
        assert oracle.lookup(col, lnE[0], lnE[-1], x) == pytest.approx(np.interp(x, lnE, col.astype(np.float64)),
                                                                        rel=1e-12)
    assert oracle.lookup(col, lnE[0], lnE[-1], lnE[0] - 1.0) == pytest.approx(float(col[0]))
    assert oracle.lookup(col, lnE[0], lnE[-1], lnE[-1] + 1.0) == pytest.approx(float(col[-1]))
    assert oracle.lookup(col, lnE[0], lnE[-1], lnE[17]) == pytest.approx(float(col[17]), rel=1e-9)


def test_majorants_bound_every_material(slab_tables):
    tb = slab_tables
    rho_max = np.array([1.0, 1.85, 0.26])
    mu_max, m_e = oracle.majorants(tb, rho_max)
    tot = tb.photon.astype(np.float64).sum(axis=1) * rho_max[:, None]
    assert np.all(mu_max >= tot.max(axis=0) * (1 - 1e-15))
    assert np.allclose(mu_max, tot.max(axis=0))
    hard = (tb.electron[:, 1].astype(np.float64) + tb.electron[:, 2]) * rho_max[:, None]
    assert np.all(np.diff(m_e) >= 0)
    assert np.all(m_e >= hard.max(axis=0) * (1 - 1e-15))
    assert np.allclose(m_e, np.maximum.accumulate(hard.max(axis=0)))
