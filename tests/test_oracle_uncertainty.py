"""Pins of the oracle's history-by-history uncertainty (Eq. 11-13) and of the paper's own benchmark
geometries (L233-266).  The second moment is pinned to its definition by brute force: one run per history."""
import numpy as np
import pytest

import oracle
from paper_1101_1245_b200 import evaluation as ev
from paper_1101_1245_b200.inputs import ELECTRON, PHOTON, make_config, make_paper_geometry


def test_second_moment_is_the_sum_of_squared_single_history_deposits():
    """Eq. 13's <D^2>: run every history on its own, square its deposit, add (the definition)."""
    w = make_paper_geometry(2, ELECTRON)
    n = 60
    e, sq, _ = oracle.run_moments(w.density, w.material, w.voxel_cm, w.tables, w.source, n, w.seed)
    e1 = np.zeros_like(e)
    sq1 = np.zeros_like(e)
    for h in range(n):
        r = oracle.run(w.density, w.material, w.voxel_cm, w.tables, w.source, 1, w.seed, hist_begin=h)
        e1 += r.edep
        sq1 += r.edep ** 2
    assert np.allclose(e, e1, rtol=1e-12, atol=0)
    assert np.allclose(sq, sq1, rtol=1e-12, atol=0)
    assert sq.sum() > 0 and (sq > 0).sum() == (e > 0).sum()


def test_moments_run_leaves_the_first_moment_and_counters_unchanged():
    w = make_config(3)
    r = oracle.run_workload(w, 3000)
    e, sq, c = oracle.run_moments(w.density, w.material, w.voxel_cm, w.tables, w.source, 3000, w.seed, n_threads=3)
    assert np.allclose(e, r.edep, rtol=1e-12, atol=0)
    assert c["ch_steps"] == r.counters["ch_steps"] and c["photon_flights"] == r.counters["photon_flights"]
    # Cauchy-Schwarz per voxel: N sum(e_h^2) >= (sum e_h)^2
    assert np.all(3000 * sq >= e ** 2 * (1 - 1e-12))


def test_batch_estimate_converges_to_the_history_by_history_uncertainty():
    """The batch estimator the CUDA path uses (gpumcd_run_uncertainty) has the same expectation as Eq. 13:
    Var(batch mean)/B = sigma_h^2/N.  Checked on the oracle alone, averaged over the voxels of Eq. 12."""
    w = make_paper_geometry(1, PHOTON)
    n, nb = 160_000, 32
    e, sq, _ = oracle.run_moments(w.density, w.material, w.voxel_cm, w.tables, w.source, n, w.seed)
    u_h = oracle.uncertainty_from_moments(e, sq, n)
    m = n // nb
    xb = np.stack([oracle.run(w.density, w.material, w.voxel_cm, w.tables, w.source, m, w.seed, hist_begin=b * m).edep / m
                   for b in range(nb)])
    assert np.allclose(xb.mean(axis=0), e / n, rtol=1e-10, atol=1e-18)   # same histories, same first moment
    u_b = xb.std(axis=0, ddof=1) / np.sqrt(nb)
    d = e / n
    sel = d > 0.2 * d.max()
    assert sel.sum() > 500
    ratio2 = (u_b[sel] / u_h[sel]) ** 2                    # ~ chi2_{B-1}/(B-1) per voxel
    assert abs(ratio2.mean() - 1.0) < 0.05
    assert abs(ratio2.std() - np.sqrt(2.0 / (nb - 1))) < 0.08
    s_h = ev.relative_uncertainty(d, u_h, 0.2)
    s_b = ev.relative_uncertainty(d, u_b, 0.2)
    assert s_b == pytest.approx(s_h, rel=0.03)


def test_uncertainty_scales_as_one_over_sqrt_n():
    """L334: the uncertainty varies as 1/sqrt(N); so s^2 N (hence the efficiency x time, Eq. 11) is constant."""
    w = make_paper_geometry(1, ELECTRON)
    s = []
    for n in (20_000, 80_000):
        e, sq, _ = oracle.run_moments(w.density, w.material, w.voxel_cm, w.tables, w.source, n, w.seed)
        s.append(ev.relative_uncertainty(e / n, oracle.uncertainty_from_moments(e, sq, n), 0.2))
    assert s[0] / s[1] == pytest.approx(2.0, rel=0.06)
    assert ev.efficiency(s[1], 2.0) == pytest.approx(1.0 / (s[1] ** 2 * 2.0))


def test_paper_geometries():
    """L246-251, L262-264: box and slab positions on the 64^3 x 0.5 cm grid."""
    for part in (ELECTRON, PHOTON):
        w = make_paper_geometry(1, part)
        assert w.density.shape == (64, 64, 64) and w.voxel_cm == 0.5 and np.all(w.density == 1.0)
        assert w.n_histories == (1_000_000 if part == ELECTRON else 4_000_000)
        assert w.source.energy == 15.0 and w.source.particle == part
    w = make_paper_geometry(2, ELECTRON)
    lung = w.material == 1
    zz, yy, xx = np.nonzero(lung)
    assert (zz.min(), zz.max()) == (6, 13)          # 3 cm .. 7 cm
    assert (xx.min(), xx.max()) == (28, 35) and (yy.min(), yy.max()) == (28, 35)   # centred on the axis (16 cm)
    assert np.allclose(w.density[lung], 0.26) and np.allclose(w.density[~lung], 1.0)
    w = make_paper_geometry(2, PHOTON)
    zz = np.nonzero(w.material == 1)[0]
    assert (zz.min(), zz.max()) == (11, 23)         # 5.5 cm .. 12 cm
    w = make_paper_geometry(3, ELECTRON)
    assert list(w.material[:14, 0, 0]) == [0] * 4 + [1] * 4 + [2] * 4 + [0] * 2
    w = make_paper_geometry(3, PHOTON)
    assert list(w.material[:26, 5, 5]) == [0] * 6 + [1] * 4 + [2] * 14 + [0] * 2
    assert np.allclose(np.unique(w.density), [0.26, 1.04, 1.85])
    with pytest.raises(ValueError):
        make_paper_geometry(4, PHOTON)
