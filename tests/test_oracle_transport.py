"""Pins of the oracle's transport loop against closed forms and invariants
(SURVEY.md 8(c) "Pins": S3 attenuation, Woodcock invariance, S4 CSDA range, S5 energy
conservation, S6 one-voxel brute force) plus source, normalisation and replay properties."""
import dataclasses

import numpy as np
import pytest
from scipy import integrate

import oracle
from paper_1101_1245_b200.inputs import ELECTRON, PENCIL, PHOTON, RECTANGLE, Source, make_config, phantoms
from paper_1101_1245_b200.inputs import materials as M
from paper_1101_1245_b200.inputs import tables as T

M_E = 0.51099895


def mu_total(mat, E, rho):
    return rho * float(T.compton_mass(mat, E) + T.photo_mass(mat, E) + T.pair_mass(mat, E)[0])


# ------------------------------------------------------------------ S5
@pytest.mark.parametrize("cfg,n", [(1, 20000), (2, 2000), (3, 10000), (4, 10000)])
def test_energy_is_conserved_exactly(cfg, n):
    w = make_config(cfg)
    r = oracle.run_workload(w, n)
    c = r.counters
    out = c["e_dep_continuous"] + c["e_dep_cutoff"] + c["e_escaped"]
    assert abs(out / c["e_incident"] - 1.0) <= 1e-6          # BASELINE.json north_star
    assert abs(out / c["e_incident"] - 1.0) <= 1e-12         # what fp64 actually gives
    assert r.edep.sum() == pytest.approx(c["e_dep_continuous"] + c["e_dep_cutoff"], rel=1e-12)
    assert c["n_histories"] == n and c["e_incident"] == pytest.approx(n * w.source.energy)


def test_energy_is_conserved_with_pair_rest_deposited_locally():
    w = make_config(3)
    r = oracle.run_workload(w, 5000, oracle.Options(pair_mode=0))
    c = r.counters
    assert c["photon_pair"] > 100
    assert c["e_pair_rest"] == pytest.approx(2 * M_E * c["photon_pair"])
    out = c["e_dep_continuous"] + c["e_dep_cutoff"] + c["e_escaped"]
    assert abs(out / c["e_incident"] - 1.0) <= 1e-12


# ------------------------------------------------------------------ S3
@pytest.mark.parametrize("nz", [8, 16, 32])
def test_narrow_beam_attenuation_homogeneous(nz, water_tables):
    """Eq. 1: primaries that cross a slab of thickness x without a real interaction = exp(-mu x)."""
    rho, mat = phantoms.homogeneous(3, 3, nz, 1.0, 0)
    h, E, n = 0.5, 2.0, 200_000
    src = Source(PHOTON, PENCIL, 0.75, 0.75, energy=E)
    r = oracle.run(rho, mat, h, water_tables, src, n, seed=21, options=oracle.Options(photon_only=1),
                   want_trace=True)
    p = np.exp(-mu_total(M.WATER, E, 1.0) * nz * h)
    frac = np.mean(r.trace == 4)          # escaped as the very first recorded event
    assert abs(frac - p) < 3 * np.sqrt(p * (1 - p) / n)


def test_narrow_beam_attenuation_heterogeneous_and_woodcock_invariance(slab_tables):
    """Eq. 3 / L63: Woodcock tracking is exact in heterogeneous media, whatever the majorant."""
    rho, mat = phantoms.z_slabs(3, 3, 40, [(12, 1.0, 0), (8, 1.85, 1), (12, 0.26, 2), (None, 1.0, 0)])
    h, E, n = 0.25, 6.0, 200_000
    src = Source(PHOTON, PENCIL, 0.375, 0.375, energy=E)
    tau = h * (12 * mu_total(M.WATER, E, 1.0) + 8 * mu_total(M.BONE, E, 1.85) + 12 * mu_total(M.LUNG, E, 0.26)
               + 8 * mu_total(M.WATER, E, 1.0))
    p = np.exp(-tau)
    fict = []
    for scale in (1.0, 2.5):
        r = oracle.run(rho, mat, h, slab_tables, src, n, seed=22,
                       options=oracle.Options(photon_only=1, majorant_scale=scale), want_trace=True)
        frac = np.mean(r.trace == 4)
        assert abs(frac - p) < 3 * np.sqrt(p * (1 - p) / n)
        fict.append(r.counters["photon_fict"])
    assert fict[1] > 2 * fict[0] > 0


def test_dose_is_invariant_under_majorant_inflation():
    """L63 / L233: inflating mu_max and M_e changes only the number of fictitious events."""
    w = make_config(4)
    n, nb = 20000, 8
    curves = {}
    for scale in (1.0, 2.0):
        pdd = []
        for b in range(nb):
            r = oracle.run(w.density, w.material, w.voxel_cm, w.tables, w.source, n // nb, seed=100 + b,
                           options=oracle.Options(majorant_scale=scale))
            pdd.append(r.edep.sum(axis=(1, 2)))
        pdd = np.array(pdd)
        curves[scale] = (pdd.mean(axis=0), pdd.std(axis=0, ddof=1) / np.sqrt(nb), r.counters)
    m1, s1, c1 = curves[1.0]
    m2, s2, c2 = curves[2.0]
    sel = m1 > 0.2 * m1.max()
    z = (m1[sel] - m2[sel]) / np.sqrt(s1[sel] ** 2 + s2[sel] ** 2)
    assert np.mean(np.abs(z) < 3) >= 0.97 and np.abs(z).max() < 5
    assert abs(m1.sum() - m2.sum()) < 4 * np.sqrt((s1**2).sum() + (s2**2).sum())
    assert c2["hard_fict"] > 2 * c1["hard_fict"] and c2["photon_fict"] > 1.5 * c1["photon_fict"]


# ------------------------------------------------------------------ S4
@pytest.mark.parametrize("T0", [1.0, 6.0, 15.0])
def test_csda_range_matches_integral_of_the_table(T0, water_tables):
    """Eq. 5-8: with hard events and scattering switched off (their table columns zeroed) the
    path length down to E_cut equals int dT / (rho L(T)) of the same table within 0.5 %."""
    tb = dataclasses.replace(water_tables, electron=water_tables.electron.copy())
    tb.electron[:, 1:4] = 0.0
    rho, mat = phantoms.homogeneous(1, 1, 64, 1.0, 0)
    src = Source(ELECTRON, PENCIL, 0.125, 0.125, energy=T0)
    path = oracle.run_pathlen(rho, mat, 0.25, tb, src, 4, seed=31)
    lnE = np.linspace(np.log(tb.e_min), np.log(tb.e_max), tb.n_energy)
    L = tb.electron[0, 0].astype(np.float64)
    expected, _ = integrate.quad(lambda t: 1.0 / np.interp(np.log(t), lnE, L), tb.e_cut, T0, epsrel=1e-7, limit=500)
    assert np.allclose(path, path[0])                 # deterministic without scattering / hard events
    assert path[0] == pytest.approx(expected, rel=5e-3)


def test_csda_energy_loss_step_is_the_midpoint_rule(water_tables):
    """Eq. 8 (R3): one step of length s loses s * L(E0 - L(E0) s / 2)."""
    tb = dataclasses.replace(water_tables, electron=water_tables.electron.copy())
    tb.electron[:, 1:4] = 0.0
    rho, mat = phantoms.homogeneous(1, 1, 4, 1.0, 0)
    T0, h = 10.0, 0.25
    src = Source(ELECTRON, PENCIL, 0.125, 0.125, energy=T0)
    r = oracle.run(rho, mat, h, tb, src, 1, seed=1)
    # DESIGN.md 3, R34: the boundary carries scalars as float32, so both sides are fed the float32-rounded
    # grid limits and nudge; with those the step is the midpoint rule to fp64 rounding
    f32 = lambda v: float(np.float32(v))
    lnE = np.linspace(np.log(f32(tb.e_min)), np.log(f32(tb.e_max)), tb.n_energy)
    L = lambda t: np.interp(np.log(t), lnE, tb.electron[0, 0].astype(np.float64))
    s = h * (1 + f32(1e-4))                              # d_vox plus the boundary nudge
    dE = s * L(T0 - 0.5 * L(T0) * s)
    assert r.edep[0, 0, 0] == pytest.approx(dE, rel=1e-12)


# ------------------------------------------------------------------ S6
@pytest.mark.parametrize("E", [0.05, 2.0, 15.0])
def test_one_voxel_brute_force(E, water_tables):
    """One thin voxel, photon-only: first-interaction probabilities and mean deposit against
    a direct evaluation of Eq. 1-2 and quadrature of Klein-Nishina."""
    h, n = 0.02, 4_000_000
    rho, mat = phantoms.homogeneous(1, 1, 1, 1.0, 0)
    src = Source(PHOTON, PENCIL, h / 2, h / 2, energy=E)
    r = oracle.run(rho, mat, h, water_tables, src, n, seed=41, options=oracle.Options(photon_only=1, pair_mode=0),
                   want_trace=True)
    sc = float(T.compton_mass(M.WATER, E))
    sp = float(T.photo_mass(M.WATER, E))
    spp = float(T.pair_mass(M.WATER, E)[0])
    mu = sc + sp + spp
    p_int = -np.expm1(-mu * h)
    first = r.trace & np.uint64(7)
    for code, sig in ((1, sc), (2, sp), (3, spp)):
        p = p_int * sig / mu
        got = np.mean(first == code)
        assert abs(got - p) < 4 * np.sqrt(p * (1 - p) / n) + 1e-12
    k = E / M_E
    eps0 = 1 / (1 + 2 * k)
    pdf = lambda e: 1 / e + e - ((1 - e) / (k * e)) * (2 - (1 - e) / (k * e))
    mean_eps = integrate.quad(lambda e: e * pdf(e), eps0, 1)[0] / integrate.quad(pdf, eps0, 1)[0]
    expect = p_int * (sc / mu * E * (1 - mean_eps) + sp / mu * E + spp / mu * E)
    got = r.edep.sum() / n
    sigma = E * np.sqrt(p_int / n)
    second_order = mu * h * np.sqrt(3.0) * expect * 5        # scattered photon interacting again in the voxel
    assert abs(got - expect) < 4 * sigma + second_order
    assert abs(got - expect) < 0.03 * expect


# ------------------------------------------------------------------ source / normalisation / replay
def test_rectangular_source_is_uniform_over_the_field(water_tables):
    """An electron beam whose electrons are deposited where they are born maps the source."""
    rho, mat = phantoms.homogeneous(16, 16, 4, 1.0, 0)
    h, n = 0.5, 400_000
    src = Source(ELECTRON, RECTANGLE, 4.0, 3.5, 3.0, 2.0, energy=5.0)   # x in [2.5,5.5], y in [2.5,4.5]
    r = oracle.run(rho, mat, h, water_tables, src, n, seed=51, options=oracle.Options(photon_only=1))
    layer = r.edep[0] / 5.0
    assert r.edep[1:].sum() == 0.0
    assert layer.sum() == pytest.approx(n)
    inside = np.zeros_like(layer, bool)
    inside[5:9, 5:11] = True
    assert layer[~inside].sum() == 0.0
    exp = n / inside.sum()
    assert np.all(np.abs(layer[inside] - exp) < 5 * np.sqrt(exp))


def test_spectrum_source_mean_energy(water_tables):
    w = make_config(1)
    edges = np.linspace(0.1, 18.0, 65).astype(np.float32)
    c = 0.5 * (edges[:-1] + edges[1:])
    wts = ((18.0 / c - 1.0) * np.exp(-1.0 / c)).astype(np.float32)
    src = Source(PHOTON, PENCIL, 8.25, 8.25, spec_edges=edges, spec_weights=wts)
    n = 200_000
    r = oracle.run(w.density, w.material, w.voxel_cm, w.tables, src, n, seed=52, options=oracle.Options(photon_only=1))
    p = wts.astype(np.float64) / wts.astype(np.float64).sum()
    mean = (p * c).sum()
    width = float(edges[1] - edges[0])
    var = (p * (c**2 + width**2 / 12)).sum() - mean**2
    assert abs(r.counters["e_incident"] / n - mean) < 4 * np.sqrt(var / n)


def test_dose_normalisation():
    w = make_config(4)
    n = 2000
    r = oracle.run_workload(w, n)
    expect = r.edep / (w.density.astype(np.float64) * w.voxel_cm**3) / n
    np.testing.assert_allclose(r.dose, expect.astype(np.float32), rtol=1e-6)


def test_result_is_independent_of_thread_count_and_history_partition():
    """Counter-based streams: any partition of the history range reproduces the same tally."""
    w = make_config(3)
    n = 3000
    a = oracle.run_workload(w, n, n_threads=1)
    b = oracle.run_workload(w, n, n_threads=5)
    c1 = oracle.run_workload(w, 1000, n_threads=2)
    c2 = oracle.run_workload(w, 2000, n_threads=3, hist_begin=1000)
    for k in ("ch_steps", "photon_flights", "hard_moller", "hard_brems", "pushes_e", "pushes_g"):
        assert a.counters[k] == b.counters[k] == c1.counters[k] + c2.counters[k]
    scale = a.edep.max()
    assert np.abs(a.edep - b.edep).max() < 1e-12 * scale
    assert np.abs(a.edep - (c1.edep + c2.edep)).max() < 1e-12 * scale


def test_trace_codes_agree_with_counters():
    w = make_config(1)
    n = 50_000
    r = oracle.run_workload(w, n, oracle.Options(photon_only=1, pair_mode=0), want_trace=True)
    c = r.counters
    assert c["pushes_e"] == 0 and c["ch_steps"] == 0 and c["pushes_g"] == 0
    tr = r.trace.copy()
    counts = np.zeros(8, np.int64)
    while tr.any():
        counts += np.bincount((tr & np.uint64(7)).astype(np.int64), minlength=8)
        tr >>= np.uint64(3)
    # with no secondary photons every event belongs to a primary track
    assert counts[1] == c["photon_compton"] and counts[2] == c["photon_photo"] and counts[3] == c["photon_pair"]
    assert counts[2] + counts[3] + counts[4] + counts[5] == n        # every history ends exactly once


def test_run_time_ordering_follows_the_paper():
    """lung needs more electron steps, a dense slab more fictitious interactions."""
    n = 5000
    water = oracle.run_workload(make_config(3), n).counters
    w4 = make_config(4)
    src15 = dataclasses.replace(w4.source, energy=15.0, wx=10.0, wy=10.0)
    slabs = oracle.run(w4.density, w4.material, w4.voxel_cm, w4.tables, src15, n, seed=3).counters
    assert water["photon_fict"] == 0 and slabs["photon_fict"] > 0.3 * slabs["photon_flights"]
    assert slabs["ch_steps"] > water["ch_steps"]
