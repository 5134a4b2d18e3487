"""The dose-comparison metrics of the paper's evaluation (Eq. 11-15) on cases with known answers."""
import numpy as np
import pytest

from paper_1101_1245_b200 import evaluation as ev


def ramp(n=24):
    z = np.arange(n, dtype=np.float64)
    return np.broadcast_to((10.0 + z)[:, None, None], (n, 3, 3)).copy()     # dose rising 1 unit per voxel along z


def test_gamma_of_identical_and_of_scaled_grids():
    d = ramp()
    g, sel = ev.gamma_index(d, d, 0.25)
    assert sel.all() and np.all(g == 0.0)
    # a uniform +1 % of D_max is half the 2 % dose criterion where no closer point helps (flat direction x, y;
    # along z the ramp lets the search find the same dose 0.33 voxel away: min over both, Eq. 14)
    flat = np.full((4, 4, 4), 50.0)
    g, _ = ev.gamma_index(flat, flat * 1.01, 0.25)
    assert np.allclose(g, 0.5)
    assert ev.gamma_pass_rate(flat, flat * 1.03, 0.25) == 0.0           # 3 % > 2 % everywhere, no distance helps


def test_gamma_distance_to_agreement_on_a_shifted_ramp():
    """Eq. 15: a grid shifted by s along its gradient passes through distance alone when s <= 2 mm."""
    d = ramp(40)
    h = 0.25                                                              # cm; one voxel = 1 unit of dose = 1/49 of D_max
    shifted = d + 0.4                                                     # = the same ramp moved by 0.4 voxel = 1 mm
    g, sel = ev.gamma_index(d, shifted, h, dd_frac=0.002)                 # dose criterion so tight that only distance counts
    inner = g[(np.argwhere(sel)[:, 0] > 2) & (np.argwhere(sel)[:, 0] < 37)]
    assert np.allclose(inner, 0.1 / 0.2, atol=0.03)                       # 1 mm / 2 mm
    far = d + 1.2                                                         # 3 mm: fails
    assert ev.gamma_pass_rate(d[3:37], far[3:37], h, dd_frac=0.002) < 0.2


def test_uncertainty_and_efficiency():
    dose = np.array([10.0, 5.0, 1.0, 0.0])
    sigma = np.array([0.1, 0.1, 0.5, 0.0])
    assert ev.relative_uncertainty(dose, sigma, 0.2) == pytest.approx(0.5 * (0.01 + 0.02))   # Eq. 12: D > 0.2 D_max
    assert ev.efficiency(0.01, 4.0) == pytest.approx(2500.0)                                   # Eq. 11
    m, s = ev.batch_mean_sigma(np.array([[1.0, 2.0], [3.0, 2.0]]))
    assert np.allclose(m, [2.0, 2.0]) and np.allclose(s, [1.0, 0.0])
    assert ev.voxel_agreement(np.array([1.0, 1.0]), np.array([0.1, 0.1]), np.array([1.2, 2.0]), np.array([0.0, 0.0]), 0.1, 3.0) == 0.5
