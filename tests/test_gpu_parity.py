"""-m gpu: the CUDA hot path against the CPU oracle on the same seeded inputs, through the C ABI.

Tolerances are BASELINE.json's north_star:
  * photon-only replay: per-history interaction sequences identical for >= 99.9 % of histories;
  * total deposited energy within 1e-5 relative;
  * per-voxel dose within 3 sqrt(s_gpu^2 + s_cpu^2) for >= 99 % of voxels above 10 % of the maximum;
  * gamma 2 %/2 mm pass rate >= 99 %.
Because both sides draw from the same Philox streams, agreement is much tighter than these bars;
the extra "replay" assertions below measure that.
"""
import dataclasses

import numpy as np
import pytest

import oracle
from gpu_util import run_gpu
from paper_1101_1245_b200 import evaluation as ev
from paper_1101_1245_b200.inputs import ELECTRON, PENCIL, PHOTON, RECTANGLE, Source, make_config, phantoms

pytestmark = pytest.mark.gpu

# Histories per config for parity.  Configs 1-3 run at BASELINE.json's full size; 4 and 5 at the
# largest size the oracle finishes in seconds on the GPU box's host cores.  The statistical bars
# (1e-5 on the total, gamma) only mean something at such sizes: about 0.5 % of the electron
# histories leave the oracle's path at an fp32 voxel-boundary decision (DESIGN.md "Replay
# fidelity"), which is noise that shrinks like 1/sqrt(N).
PARITY_N = {1: 100_000, 2: 1_000_000, 3: 4_000_000, 4: 4_000_000, 5: 8_000_000}
NB = 8
SCHEDULERS = [0, 1]
INT_KEYS = ("photon_flights", "photon_compton", "photon_photo", "photon_pair", "photon_fict", "ch_steps",
            "hard_moller", "hard_brems", "hard_fict", "pushes_e", "pushes_g")


@pytest.fixture(scope="module")
def workloads():
    return {i: make_config(i) for i in (1, 2, 3, 4, 5)}


_ORACLE_CACHE = {}


def oracle_batches(w, cfg):
    """Oracle tallies of the NB batches of a config (computed once, shared by both schedulers)."""
    if cfg not in _ORACLE_CACHE:
        n = PARITY_N[cfg]
        eds, cnt = [], None
        for b in range(NB):
            o = oracle.run(w.density, w.material, w.voxel_cm, w.tables, w.source, n // NB, seed=w.seed + 1000 * b)
            eds.append(o.edep.astype(np.float32) if cfg == 5 else o.edep)
            cnt = o.counters if cnt is None else {k: cnt[k] + v for k, v in o.counters.items()}
        _ORACLE_CACHE.clear()          # keep one config at a time (config 5 tallies are large)
        _ORACLE_CACHE[cfg] = (eds, cnt)
    return _ORACLE_CACHE[cfg]


def total_deposit(c):
    return c["e_dep_continuous"] + c["e_dep_cutoff"]


@pytest.mark.parametrize("scheduler", SCHEDULERS)
@pytest.mark.parametrize("cfg", [1, 3, 4, 5])
def test_photon_only_replay_sequences(cfg, scheduler, workloads):
    w = workloads[cfg]
    n = min(PARITY_N[cfg], 1_000_000)
    o = oracle.run_workload(w, n, oracle.Options(photon_only=1), want_trace=True)
    g = run_gpu(w, n, want_trace=True, want_edep=False, scheduler=scheduler)
    same = np.mean(o.trace == g["trace"])
    assert same >= 0.999, f"only {same:.5f} of the histories replay identically"
    for k in ("photon_flights", "photon_compton", "photon_photo", "photon_pair", "photon_fict"):
        assert abs(g["counters"][k] - o.counters[k]) <= 2e-4 * max(o.counters[k], 1000), k
    assert g["counters"]["ch_steps"] == 0 and g["counters"]["pushes_e"] == 0


@pytest.mark.parametrize("scheduler", SCHEDULERS)
@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_dose_parity(cfg, scheduler, workloads):
    w = workloads[cfg]
    n = PARITY_N[cfg]
    nb = NB
    og, oc = oracle_batches(w, cfg)
    gg = []
    gc = None
    for b in range(nb):
        g = run_gpu(w, n // nb, seed=w.seed + 1000 * b, scheduler=scheduler)
        gg.append(g["edep"].astype(np.float32) if cfg == 5 else g["edep"])
        gc = g["counters"] if gc is None else {k: gc[k] + v for k, v in g["counters"].items()}
        assert g["counters"]["overflow_count"] == 0
        # the dose grid is the energy tally divided by the voxel mass and the number of histories
        expect = g["edep"] / (w.density.astype(np.float64) * w.voxel_cm**3) / (n // nb)
        np.testing.assert_allclose(g["dose"], expect.astype(np.float32), rtol=2e-6, atol=0)
    # --- total deposited energy, 1e-5 relative
    rel = abs(total_deposit(gc) - total_deposit(oc)) / total_deposit(oc)
    assert rel <= 1e-5, f"total deposited energy differs by {rel:.2e}"
    # --- energy conservation on the GPU side
    bal = (total_deposit(gc) + gc["e_escaped"]) / gc["e_incident"] - 1.0
    assert abs(bal) <= 1e-6
    assert gc["e_incident"] == pytest.approx(oc["e_incident"], rel=1e-7)
    # --- event counts replay almost exactly
    for k in INT_KEYS:
        assert abs(gc[k] - oc[k]) <= 3e-3 * oc[k] + 50, (k, gc[k], oc[k])
    # --- per-voxel agreement within the combined statistical uncertainty
    om, os_ = ev.batch_mean_sigma(np.array(og))
    gm, gs = ev.batch_mean_sigma(np.array(gg))
    assert ev.voxel_agreement(om, os_, gm, gs, frac=0.1, k=3.0) >= 0.99
    # --- gamma 2 %/2 mm, reference = oracle
    mass = w.density.astype(np.float64) * w.voxel_cm**3
    assert ev.gamma_pass_rate(om / mass, gm / mass, w.voxel_cm, frac=0.1) >= 0.99
    # --- replay quality: the two dose grids differ far less than their statistical noise
    sel = om > 0.1 * om.max()
    noise = np.sqrt(np.mean(os_[sel] ** 2))
    diff = np.sqrt(np.mean((gm[sel] - om[sel]) ** 2))
    assert diff < 0.2 * noise, f"rms difference {diff:.3e} vs statistical noise {noise:.3e}"


@pytest.mark.parametrize("scheduler", SCHEDULERS)
def test_config1_full_size_sampled_voxels(scheduler, workloads):
    """Config 1 at BASELINE.json's full size and seed: every voxel on the beam axis."""
    w = workloads[1]
    o = oracle.run_workload(w)
    g = run_gpu(w, scheduler=scheduler)
    assert g["counters"]["n_histories"] == 100_000
    axis_o = o.edep[:, 16, 16]
    axis_g = g["edep"][:, 16, 16]
    np.testing.assert_allclose(axis_g, axis_o, rtol=2e-3)
    assert abs(g["edep"].sum() - o.edep.sum()) / o.edep.sum() <= 1e-5


@pytest.mark.parametrize("scheduler", SCHEDULERS)
def test_same_seed_is_reproducible(scheduler, workloads):
    w = workloads[3]
    a = run_gpu(w, 30_000, scheduler=scheduler)
    b = run_gpu(w, 30_000, scheduler=scheduler)
    for k in INT_KEYS:
        assert a["counters"][k] == b["counters"][k]
    scale = a["edep"].max()
    assert np.abs(a["edep"] - b["edep"]).max() <= 1e-12 * scale       # fp64 atomic-order noise only
    c = run_gpu(w, 30_000, seed=w.seed + 1, scheduler=scheduler)
    assert c["counters"]["ch_steps"] != a["counters"]["ch_steps"]


def test_schedulers_agree_exactly(workloads):
    """Scheduling only changes who runs which particle when: same draws, same events, same tally."""
    for cfg in (2, 4):
        w = workloads[cfg]
        a = run_gpu(w, 40_000, scheduler=0)
        b = run_gpu(w, 40_000, scheduler=1)
        for k in INT_KEYS:
            assert a["counters"][k] == b["counters"][k], k
        assert np.abs(a["edep"] - b["edep"]).max() <= 1e-12 * a["edep"].max()


def test_cta_size_does_not_change_the_result(workloads):
    """Scheduler 1 runs with 768 (default), 512 or 1024 threads per SM: which lane works a particle off does
    not matter."""
    for cfg in (2, 4):
        w = workloads[cfg]
        a = run_gpu(w, 60_000, scheduler=1, cta_threads=512)
        b = run_gpu(w, 60_000, scheduler=1, cta_threads=1024)
        c = run_gpu(w, 60_000, scheduler=1)
        for k in INT_KEYS:
            assert a["counters"][k] == b["counters"][k] == c["counters"][k], k
        assert np.abs(a["edep"] - b["edep"]).max() <= 1e-12 * a["edep"].max()
        assert np.abs(a["edep"] - c["edep"]).max() <= 1e-12 * a["edep"].max()


@pytest.mark.parametrize("scheduler", SCHEDULERS)
@pytest.mark.parametrize("n,wave", [(1, 1 << 20), (31, 1 << 20), (2500, 1000), (4097, 4096), (70_001, 1 << 15)])
def test_ragged_sizes_and_waves(n, wave, scheduler, workloads):
    """History counts that are not multiples of the block, the warp or the wave size."""
    w = workloads[3]
    o = oracle.run_workload(w, n)
    g = run_gpu(w, n, wave_size=wave, scheduler=scheduler)
    for k in INT_KEYS:
        assert abs(g["counters"][k] - o.counters[k]) <= 10 + 3e-3 * o.counters[k], k
    assert g["counters"]["e_incident"] == pytest.approx(n * 15.0, rel=1e-7)
    assert g["edep"].sum() == pytest.approx(o.edep.sum(), rel=1e-3 if n > 1000 else 0.2)


@pytest.mark.parametrize("scheduler", SCHEDULERS)
def test_wave_partition_does_not_change_the_result(scheduler, workloads):
    w = workloads[4]
    a = run_gpu(w, 50_000, wave_size=1 << 20, scheduler=scheduler)
    b = run_gpu(w, 50_000, wave_size=7000, scheduler=scheduler)
    for k in INT_KEYS:
        assert a["counters"][k] == b["counters"][k]
    assert np.abs(a["edep"] - b["edep"]).max() <= 1e-12 * a["edep"].max()
    if scheduler == 0:
        assert b["counters"]["bank_high_water"] <= 7000 * 8


def test_pair_rest_energy_deposited_locally(workloads):
    w = workloads[3]
    n = 400_000
    o = oracle.run_workload(w, n, oracle.Options(pair_mode=0))
    g = run_gpu(w, n, pair_mode=0)
    assert g["counters"]["photon_pair"] == pytest.approx(o.counters["photon_pair"], rel=1e-3)
    assert g["counters"]["e_pair_rest"] == pytest.approx(o.counters["e_pair_rest"], rel=1e-3)
    # 3e-5, not 1e-5: a 15 MeV photon beam deposits a quarter of its energy, with a per-history spread larger
    # than the mean, so the ~1e-3 of the histories that leave the oracle's path by an fp32 flip
    # move the total by ~1e-5 sqrt(4e6 / n); measured over three seeds: 6e-5 at n = 5e4, <= 1.5e-5 at 4e5,
    # <= 1.7e-5 at 4e6 (config 3 itself is held to 1e-5 at its full 4e6 histories in test_dose_parity)
    assert abs(g["edep"].sum() - o.edep.sum()) / o.edep.sum() <= 3e-5
    bal = (total_deposit(g["counters"]) + g["counters"]["e_escaped"]) / g["counters"]["e_incident"] - 1
    assert abs(bal) <= 1e-6


def test_electron_source_deposited_at_birth_maps_the_field(water_tables):
    rho, mat = phantoms.homogeneous(16, 16, 4, 1.0, 0)
    src = Source(ELECTRON, RECTANGLE, 4.0, 3.5, 3.0, 2.0, energy=5.0)
    w = dataclasses.replace(make_config(1), density=rho, material=mat, voxel_cm=0.5, tables=water_tables, source=src)
    n = 100_000
    o = oracle.run(rho, mat, 0.5, water_tables, src, n, seed=9, options=oracle.Options(photon_only=1))
    g = run_gpu(w, n, seed=9, photon_only=1)
    np.testing.assert_allclose(g["edep"], o.edep, rtol=1e-12, atol=1e-9)   # identical voxel for every primary
    assert g["counters"]["ch_steps"] == 0


def test_spectrum_source(workloads):
    w = workloads[5]
    n = 100_000
    o = oracle.run_workload(w, n, oracle.Options(photon_only=1))
    g = run_gpu(w, n, photon_only=1)
    assert g["counters"]["e_incident"] == pytest.approx(o.counters["e_incident"], rel=1e-6)
    assert abs(g["edep"].sum() - o.edep.sum()) / o.edep.sum() <= 1e-5


def test_majorant_inflation_changes_only_fictitious_counts(workloads):
    """Woodcock tracking is not an approximation."""
    w = workloads[4]
    n = 4_000_000
    a = run_gpu(w, n, scheduler=1)
    b = run_gpu(w, n, majorant_scale=2.0, scheduler=1)
    assert b["counters"]["photon_fict"] > 1.5 * a["counters"]["photon_fict"]
    da, db = a["edep"].sum(axis=(1, 2)), b["edep"].sum(axis=(1, 2))
    sel = da > 0.2 * da.max()
    # 4e6 histories: depth-dose curves agree to a fraction of a per cent per slice
    assert np.abs(db[sel] / da[sel] - 1).max() < 0.02
    assert abs(db.sum() / da.sum() - 1) < 0.003


def test_host_entry_points_match_device_entry_points(workloads):
    import paper_1101_1245_b200 as g

    w = workloads[1]
    n = 20_000
    ref = run_gpu(w, n)
    dose = np.empty(w.density.shape, np.float32)
    with g.gpumcd_create_host(w.density, w.material, w.voxel_cm, w.tables) as ctx:
        g.gpumcd_set_source(ctx, w.source)
        g.gpumcd_run_host(ctx, n, w.seed, dose)
        c = g.gpumcd_get_counters(ctx)
    assert c["ch_steps"] == ref["counters"]["ch_steps"]
    np.testing.assert_allclose(dose, ref["dose"], rtol=1e-6, atol=0)


def test_set_phantom_replaces_the_volumes_and_majorants(workloads):
    """A context re-targeted at another phantom of the same grid gives what a fresh context gives."""
    import torch

    import paper_1101_1245_b200 as g

    w4, n = workloads[4], 30_000
    ref = run_gpu(w4, n)
    water = np.ones_like(w4.density)
    zeros = np.zeros_like(w4.material)
    dev = torch.device("cuda:0")
    dose = np.empty(w4.density.shape, np.float32)
    with g.gpumcd_create_host(water, zeros, w4.voxel_cm, w4.tables) as ctx:       # starts as plain water
        g.gpumcd_set_source(ctx, w4.source)
        g.gpumcd_run_host(ctx, n, w4.seed, dose)
        c_water = g.gpumcd_get_counters(ctx)
        g.gpumcd_set_phantom_host(ctx, w4.density, w4.material)                  # host volumes
        g.gpumcd_run_host(ctx, n, w4.seed, dose)
        c_host = g.gpumcd_get_counters(ctx)
        np.testing.assert_allclose(dose, ref["dose"], rtol=1e-6, atol=0)
        g.gpumcd_set_phantom(ctx, torch.from_numpy(water).to(dev), torch.from_numpy(zeros).to(dev))
        g.gpumcd_set_phantom(ctx, torch.from_numpy(w4.density).to(dev), torch.from_numpy(w4.material).to(dev))
        g.gpumcd_run_host(ctx, n, w4.seed, dose)                                   # device volumes
        c_dev = g.gpumcd_get_counters(ctx)
        bad = w4.material.copy()
        bad[0, 0, 0] = 7
        with pytest.raises(g.GpumcdError) as e:
            g.gpumcd_set_phantom_host(ctx, w4.density, bad)
        assert e.value.status == -1
    for k in INT_KEYS:
        assert c_host[k] == ref["counters"][k] == c_dev[k], k
    assert c_water["photon_fict"] < 0.5 * c_host["photon_fict"]      # bone raises the majorant


def test_error_paths(workloads):
    import torch

    import paper_1101_1245_b200 as g

    w = workloads[1]
    dev = torch.device("cuda:0")
    rho = torch.from_numpy(w.density).to(dev)
    mat = torch.from_numpy(w.material).to(dev)
    dose = torch.empty(rho.shape, dtype=torch.float32, device=dev)
    with g.gpumcd_create(rho, mat, w.voxel_cm, w.tables) as ctx:
        with pytest.raises(g.GpumcdError) as e:
            g.gpumcd_run(ctx, 10, 1, dose)
        assert e.value.status == -5                                   # no source yet
        with pytest.raises(g.GpumcdError) as e:
            g.gpumcd_set_source(ctx, Source(PHOTON, PENCIL, 8.25, 8.25, energy=25.0))
        assert e.value.status == -6                                   # outside the tables
        with pytest.raises(g.GpumcdError) as e:
            g.gpumcd_set_source(ctx, Source(PHOTON, RECTANGLE, 1.0, 8.0, 4.0, 4.0, energy=2.0))
        assert e.value.status == -1                                   # field sticks out of the phantom
    bad = mat.clone()
    bad[3, 3, 3] = 5
    with pytest.raises(g.GpumcdError) as e:
        g.gpumcd_create(rho, bad, w.voxel_cm, w.tables)
    assert e.value.status == -1
    neg = rho.clone()
    neg[0, 0, 0] = 0.0
    with pytest.raises(g.GpumcdError):
        g.gpumcd_create(neg, mat, w.voxel_cm, w.tables)
    # a queue that is too small must be reported, never silently dropped (PAPER.md L166 discards)
    w2 = workloads[2]
    rho2 = torch.from_numpy(w2.density).to(dev)
    mat2 = torch.from_numpy(w2.material).to(dev)
    dose2 = torch.empty(rho2.shape, dtype=torch.float32, device=dev)
    # scheduler 0 banks the ~60000 knock-on electrons and ~32000 bremsstrahlung photons of 20000 electrons of
    # 15 MeV in global queues of 1 x 20000 slots
    opt = g.gpumcd_default_options(scheduler=0, wave_size=20000, bank_factor=1)
    with g.gpumcd_create(rho2, mat2, w2.voxel_cm, w2.tables, opt) as ctx:
        g.gpumcd_set_source(ctx, w2.source)
        with pytest.raises(g.GpumcdError) as e:
            g.gpumcd_run(ctx, 20000, 1, dose2)
            g.gpumcd_get_counters(ctx)
        assert e.value.status == -4
    # scheduler 1: a warp changes type before a stack fills up (persistent.cuh "Forced type changes"), so even the
    # smallest stacks the library accepts (256 records; smaller requests are raised to that) hold what a warp
    # banks: same events, no overflow
    ref = run_gpu(w2, 200_000, scheduler=1)
    small = run_gpu(w2, 200_000, scheduler=1, warp_stack=192)
    assert small["counters"]["overflow_count"] == 0 and small["counters"]["bank_high_water"] <= 256
    for k in INT_KEYS:
        assert small["counters"][k] == ref["counters"][k], k


def test_tally_probe(workloads):
    """gpumcd_probe_tally: a plausible fp64 atomic rate, and the context still works afterwards."""
    import torch

    import paper_1101_1245_b200 as g
    w = workloads[1]
    dev = torch.device("cuda:0")
    rho = torch.from_numpy(w.density).to(dev)
    mat = torch.from_numpy(w.material).to(dev)
    dose = torch.empty(rho.shape, dtype=torch.float32, device=dev)
    with g.gpumcd_create(rho, mat, w.voxel_cm, w.tables) as ctx:
        with pytest.raises(g.GpumcdError):
            g.gpumcd_probe_tally(ctx, 1000)                 # no source yet
        g.gpumcd_set_source(ctx, w.source)
        g.gpumcd_run(ctx, 20_000, 1, dose)
        before = g.gpumcd_get_counters(ctx)
        rate = g.gpumcd_probe_tally(ctx, 20_000_000)
        assert 1e9 < rate < 1e13
        g.gpumcd_run(ctx, 20_000, 1, dose)
        after = g.gpumcd_get_counters(ctx)
        assert after["ch_steps"] == before["ch_steps"]
        assert after["e_dep_continuous"] == pytest.approx(before["e_dep_continuous"], rel=1e-12)


@pytest.mark.parametrize("cfg,n_oracle", [(4, 1_000_000), (5, 1_000_000)])
def test_full_size_properties(cfg, n_oracle, workloads):
    """Configs 4 and 5 at BASELINE.json's full history counts (2e7, 1e8), default options = the launch
    configuration bench.py times.  The oracle cannot run these sizes in seconds, so what is checked is what
    holds at any size: the energy audit, the tally against its own total, and per-history averages and the
    laterally integrated depth dose against the oracle's bounded sample of the same stream family."""
    w = workloads[cfg]
    n = w.n_histories
    g = run_gpu(w, n)
    c = g["counters"]
    assert c["n_histories"] == n and c["overflow_count"] == 0
    out = total_deposit(c) + c["e_escaped"]
    assert abs(out / c["e_incident"] - 1.0) <= 1e-6                       # BASELINE.json: energy conservation
    assert g["edep"].sum() == pytest.approx(total_deposit(c), rel=1e-9)
    assert np.isfinite(g["dose"]).all() and (g["dose"] >= 0).all() and (g["edep"] >= 0).all()
    mass = w.density.astype(np.float64) * w.voxel_cm ** 3
    np.testing.assert_allclose(g["dose"], g["edep"] / mass / n, rtol=2e-6, atol=0)      # H8
    o = oracle.run_workload(w, n_oracle)
    if w.source.spec_edges is None:
        assert c["e_incident"] == pytest.approx(n * w.source.energy, rel=1e-7)
    else:
        assert c["e_incident"] / n == pytest.approx(o.counters["e_incident"] / n_oracle, rel=5e-3)
    # per-history averages: the oracle's sample is the first n_oracle histories of the same streams
    for k in INT_KEYS:
        assert c[k] / n == pytest.approx(o.counters[k] / n_oracle, rel=0.02), k
    assert total_deposit(c) / n == pytest.approx(total_deposit(o.counters) / n_oracle, rel=0.01)
    dg = g["edep"].sum(axis=(1, 2)) / n
    do = o.edep.sum(axis=(1, 2)) / n_oracle
    assert np.abs(dg - do).max() <= 0.03 * do.max()      # the oracle sample's noise per depth bin is ~1 %
