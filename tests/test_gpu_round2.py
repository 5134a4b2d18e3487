"""-m gpu: paths the round-1 suite did not reach: the tally modes, the device's random-number
layer bit for bit, the multi-GPU hook (history offsets, ids beyond 2^32), tables read from global memory, two
live contexts of different table sizes, small warp stacks on pair-heavy beams, kinematic thresholds (R33)."""
import dataclasses
import os

import numpy as np
import pytest

import oracle
from gpu_util import run_gpu
from paper_1101_1245_b200 import evaluation as ev
from paper_1101_1245_b200.inputs import ELECTRON, PENCIL, PHOTON, Source, make_config, phantoms
from paper_1101_1245_b200.inputs import materials as M
from paper_1101_1245_b200.inputs.tables import build_tables

pytestmark = pytest.mark.gpu

INT_KEYS = ("photon_flights", "photon_compton", "photon_photo", "photon_pair", "photon_fict", "ch_steps",
            "hard_moller", "hard_brems", "hard_fict", "pushes_e", "pushes_g")
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


def total(c):
    return c["e_dep_continuous"] + c["e_dep_cutoff"]


# ------------------------------------------------------------------ H9 on the device
def test_device_philox_known_answers_and_bitwise_equality_with_the_oracle():
    """the published vectors on the device, and host == device on 2^20 random counters;
    U(w) is the same number on both sides."""
    import torch

    import paper_1101_1245_b200 as g
    rows = [[int(x, 16) for x in l.split()] for l in open(GOLDEN) if l.strip() and not l.startswith("#")]
    kat = np.array([r[:6] for r in rows], np.uint32)
    want = np.array([r[6:10] for r in rows], np.uint32)
    rng = np.random.default_rng(9)
    rnd = rng.integers(0, 2**32, size=(1 << 20, 6), dtype=np.uint64).astype(np.uint32)
    # lineage-style counters too: small history / track / draw numbers, the top bit of the draw counter set
    small = np.stack([rng.integers(0, 1 << 20, 4096), np.zeros(4096), rng.integers(0, 2**32, 4096),
                      rng.integers(0, 64, 4096) | 0x80000000, np.full(4096, 5), np.zeros(4096)], 1).astype(np.uint32)
    inp = np.concatenate([kat, rnd, small])
    dev = torch.device("cuda:0")
    t_in = torch.from_numpy(inp.view(np.int32)).to(dev)
    t_out = torch.zeros((inp.shape[0], 4), dtype=torch.int32, device=dev)
    t_u = torch.zeros((inp.shape[0], 4), dtype=torch.float32, device=dev)
    g.gpumcd_selftest_philox(t_in, t_out, t_u)
    torch.cuda.synchronize()
    got = t_out.cpu().numpy().view(np.uint32)
    assert np.array_equal(got[:3], want)
    assert np.array_equal(got, oracle.philox_batch(inp))
    u = t_u.cpu().numpy().astype(np.float64)
    assert np.array_equal(u, ((got >> 9).astype(np.float64) + 0.5) / 8388608.0)      # = oracle.uniform, exactly
    assert u.min() > 0.0 and u.max() < 1.0
    for w in (0, 0x1FF, 0x12345678, 0xFFFFFFFF):
        assert oracle.uniform(w) == ((w >> 9) + 0.5) / 8388608.0


# ------------------------------------------------------------------ tally modes (north_star; gpumcd_options.tally_mode)
@pytest.mark.parametrize("cfg,n", [(1, 100_000), (2, 200_000), (3, 400_000), (4, 1_000_000), (5, 1_000_000)])
def test_tally_modes_give_the_same_tally(cfg, n):
    """Mode 1 (warp-aggregated) adds the same fp64 numbers in another order; mode 2 (fixed point) rounds each
    deposit to 2^-k MeV.  Same events, same tally to rounding, on all five configurations, against the oracle."""
    w = make_config(cfg)
    o = oracle.run_workload(w, n)
    ref = run_gpu(w, n, tally_mode=0)
    scale = ref["edep"].max()
    for mode in (1, 2):
        for sched in (1, 0):
            g = run_gpu(w, n, tally_mode=mode, scheduler=sched)
            for k in INT_KEYS:
                assert g["counters"][k] == ref["counters"][k], (mode, sched, k)
            assert g["counters"]["overflow_count"] == 0
            tol = 1e-12 if mode == 1 else 2e-9          # mode 2: <= 2^-32 MeV per deposit at these sizes
            assert np.abs(g["edep"] - ref["edep"]).max() <= tol * scale
            assert total(g["counters"]) == pytest.approx(total(ref["counters"]), rel=1e-9)
            mass = w.density.astype(np.float64) * w.voxel_cm ** 3
            np.testing.assert_allclose(g["dose"], (g["edep"] / mass / n).astype(np.float32), rtol=2e-6, atol=0)
            bal = (total(g["counters"]) + g["counters"]["e_escaped"]) / g["counters"]["e_incident"] - 1.0
            assert abs(bal) <= 1e-6
            # and against the oracle: BASELINE.json's bar on the total, 1e-5 at the size test_dose_parity runs
            # the configuration at (n_full); the difference is the statistical one of the few histories that an
            # fp32 flip takes off the oracle's path, so it grows as 1 / sqrt(n) below that size
            n_full = {1: 100_000, 2: 1_000_000, 3: 4_000_000, 4: 4_000_000, 5: 8_000_000}[cfg]
            assert abs(total(g["counters"]) - total(o.counters)) / total(o.counters) <= 1e-5 * np.sqrt(n_full / n)


@pytest.mark.parametrize("cfg,n", [(2, 150_000), (4, 600_000)])
def test_fixed_point_tally_is_bitwise_reproducible(cfg, n):
    """Integer additions commute: same seed, same bits, whichever lane, warp or scheduler adds them; the fp64
    tally is reproducible only up to the order of its additions."""
    w = make_config(cfg)
    a = run_gpu(w, n, tally_mode=2)
    b = run_gpu(w, n, tally_mode=2)
    c = run_gpu(w, n, tally_mode=2, scheduler=0)
    assert np.array_equal(a["edep"], b["edep"]) and np.array_equal(a["dose"], b["dose"])
    assert np.array_equal(a["edep"], c["edep"]) and np.array_equal(a["dose"], c["dose"])
    assert a["counters"]["e_dep_continuous"] + a["counters"]["e_dep_cutoff"] == pytest.approx(a["edep"].sum(), rel=1e-12)
    f = run_gpu(w, n, tally_mode=0)
    f2 = run_gpu(w, n, tally_mode=0)
    assert np.abs(f["edep"] - f2["edep"]).max() <= 1e-12 * f["edep"].max()
    assert np.abs(a["edep"] - f["edep"]).max() <= 2e-9 * f["edep"].max()


def test_fixed_point_scale_follows_the_run_size():
    """1e8 histories of up to 18 MeV: k = 31; the grid must not overflow and keeps 2^-31 MeV resolution."""
    w = make_config(5)
    n = 2_000_000
    a = run_gpu(w, n, tally_mode=2)
    f = run_gpu(w, n, tally_mode=0)
    assert np.abs(a["edep"] - f["edep"]).max() <= 2e-9 * f["edep"].max()
    # uncertainty runs share the machinery (per-batch finalize converts the integers in place)
    import torch

    import paper_1101_1245_b200 as g
    dev = torch.device("cuda:0")
    rho = torch.from_numpy(w.density).to(dev)
    mat = torch.from_numpy(w.material).to(dev)
    out = {}
    for mode in (0, 2):
        with g.gpumcd_create(rho, mat, w.voxel_cm, w.tables, g.gpumcd_default_options(tally_mode=mode)) as ctx:
            g.gpumcd_set_source(ctx, w.source)
            d = torch.empty(rho.shape, dtype=torch.float32, device=dev)
            s = torch.empty(rho.shape, dtype=torch.float32, device=dev)
            g.gpumcd_run_uncertainty(ctx, 200_000, 8, w.seed, d, s)
            torch.cuda.synchronize()
            out[mode] = (d.cpu().numpy(), s.cpu().numpy())
    np.testing.assert_allclose(out[2][0], out[0][0], rtol=1e-5, atol=1e-9 * out[0][0].max())
    np.testing.assert_allclose(out[2][1], out[0][1], rtol=1e-4, atol=1e-7 * out[0][1].max())


# ------------------------------------------------------------------ multi-GPU hook
@pytest.mark.parametrize("scheduler", [0, 1])
def test_two_contexts_with_history_offsets_sum_to_one_run(scheduler):
    """What bench.py --gpus 2 does, on one device: two contexts simulate the two halves of the history range;
    their tallies add up to the tally of one run over the whole range, event for event."""
    import torch

    import paper_1101_1245_b200 as g
    w = make_config(3)
    n = 100_001
    whole = run_gpu(w, n, scheduler=scheduler)
    dev = torch.device("cuda:0")
    rho = torch.from_numpy(w.density).to(dev)
    mat = torch.from_numpy(w.material).to(dev)
    from paper_1101_1245_b200.sharding import combine_dose, history_range
    spans = [history_range(n, r, 2) for r in (0, 1)]
    assert spans[0][0] == 0 and spans[1][0] == spans[0][1] and spans[0][1] + spans[1][1] == n
    parts = []
    for first, count in spans:
        with g.gpumcd_create(rho, mat, w.voxel_cm, w.tables, g.gpumcd_default_options(scheduler=scheduler)) as ctx:
            g.gpumcd_set_source(ctx, w.source)
            g.gpumcd_set_history_offset(ctx, first)
            dose = torch.empty(rho.shape, dtype=torch.float32, device=dev)
            g.gpumcd_run(ctx, count, w.seed, dose)
            e = torch.empty(rho.shape, dtype=torch.float64, device=dev)
            g.gpumcd_get_energy_tally(ctx, e)
            torch.cuda.synchronize()
            parts.append((e.cpu().numpy(), g.gpumcd_get_counters(ctx), dose.cpu().numpy(), count))
    for k in INT_KEYS:
        assert parts[0][1][k] + parts[1][1][k] == whole["counters"][k], k
    assert np.abs(parts[0][0] + parts[1][0] - whole["edep"]).max() <= 1e-12 * whole["edep"].max()
    # sharding.combine_dose: per-rank doses weighted by their share of the histories
    dose = sum(combine_dose(torch.from_numpy(p[2].astype(np.float64)), p[3], n).numpy() for p in parts)
    np.testing.assert_allclose(dose, whole["dose"], rtol=2e-6, atol=1e-12 * whole["dose"].max())
    # the offset run is the oracle's run over the same ids
    o = oracle.run_workload(w, spans[1][1], hist_begin=spans[1][0])
    # (the ~0.5 % of the histories that an fp32 flip takes off the oracle's path are independent samples, DESIGN.md
    # 4.5: a rare-event counter such as hard_fict, ~1000 here and clustered in few histories, then differs by a few
    # times sqrt(0.01 c), which the relative bar alone does not allow for at this size)
    for k in INT_KEYS:
        c = o.counters[k]
        assert abs(parts[1][1][k] - c) <= 10 + 3e-3 * c + np.sqrt(c), k
    assert parts[1][0].sum() == pytest.approx(o.edep.sum(), rel=2e-3)


@pytest.mark.parametrize("scheduler", [0, 1])
def test_history_ids_beyond_2_to_the_32(scheduler):
    """A range that crosses 2^32 (the high counter word changes inside the run; scheduler 1 splits the launch,
    scheduler 0 the wave) against the oracle over the same ids, and a trace run indexed from the offset."""
    import torch

    import paper_1101_1245_b200 as g
    w = make_config(3)
    first, n = 2**32 - 5000, 10_000
    o = oracle.run_workload(w, n, hist_begin=first)
    ot = oracle.run_workload(w, n, oracle.Options(photon_only=1), want_trace=True, hist_begin=first)
    lo = oracle.run_workload(w, n, hist_begin=0)
    dev = torch.device("cuda:0")
    rho = torch.from_numpy(w.density).to(dev)
    mat = torch.from_numpy(w.material).to(dev)
    with g.gpumcd_create(rho, mat, w.voxel_cm, w.tables, g.gpumcd_default_options(scheduler=scheduler)) as ctx:
        g.gpumcd_set_source(ctx, w.source)
        g.gpumcd_set_history_offset(ctx, first)
        dose = torch.empty(rho.shape, dtype=torch.float32, device=dev)
        g.gpumcd_run(ctx, n, w.seed, dose)
        c = g.gpumcd_get_counters(ctx)
        e = torch.empty(rho.shape, dtype=torch.float64, device=dev)
        g.gpumcd_get_energy_tally(ctx, e)
        tr = torch.zeros(n, dtype=torch.int64, device=dev)
        g.gpumcd_run_trace(ctx, n, w.seed, tr)
        torch.cuda.synchronize()
        edep = e.cpu().numpy()
        trace = tr.cpu().numpy().view(np.uint64)
    assert c["n_histories"] == n and c["overflow_count"] == 0
    for k in INT_KEYS:
        assert abs(c[k] - o.counters[k]) <= 10 + 3e-3 * o.counters[k], k
    assert c["ch_steps"] != lo.counters["ch_steps"]                       # not the histories 0 .. n-1
    assert edep.sum() == pytest.approx(o.edep.sum(), rel=1e-3)
    mass = w.density.astype(np.float64) * w.voxel_cm ** 3
    np.testing.assert_allclose(dose.cpu().numpy(), (edep / mass / n).astype(np.float32), rtol=2e-6, atol=0)
    assert np.mean(trace == ot.trace) >= 0.999


# ------------------------------------------------------------------ tables in global memory; two live contexts
def test_tables_read_from_global_memory_give_the_same_run():
    for cfg, n in ((2, 60_000), (5, 300_000)):
        w = make_config(cfg)
        a = run_gpu(w, n)
        b = run_gpu(w, n, table_memory=1)
        c = run_gpu(w, n, table_memory=1, tally_mode=2, hom_tol=0.1)
        d = run_gpu(w, n, tally_mode=2, hom_tol=0.1)
        for k in INT_KEYS:
            assert a["counters"][k] == b["counters"][k], k
            assert c["counters"][k] == d["counters"][k], k
        assert np.abs(a["edep"] - b["edep"]).max() <= 1e-12 * a["edep"].max()
        assert np.array_equal(c["edep"], d["edep"])
    w = make_config(1)
    t = run_gpu(w, 50_000, want_trace=True, want_edep=False)
    tg = run_gpu(w, 50_000, want_trace=True, want_edep=False, table_memory=1)
    assert np.array_equal(t["trace"], tg["trace"])


def test_eight_materials_do_not_fit_shared_memory_and_still_run():
    """8 materials x 7 columns x 1024 nodes = 236 KB > 227 KB: the library falls back to global-memory tables."""
    mats = [M.WATER, M.BONE, M.LUNG, M.SOFT, M.AIR, M.WATER, M.BONE, M.LUNG]
    tb8 = build_tables(mats)
    w4 = make_config(4)
    remap = np.array([5, 6, 7], np.uint8)[w4.material]                   # the same media under other ids
    w8 = dataclasses.replace(w4, tables=tb8, material=remap)
    n = 200_000
    a = run_gpu(w4, n)
    b = run_gpu(w8, n)
    for k in INT_KEYS:
        assert a["counters"][k] == b["counters"][k], k
    assert np.abs(a["edep"] - b["edep"]).max() <= 1e-12 * a["edep"].max()


def test_two_live_contexts_with_different_table_sizes():
    """the dynamic shared-memory limit belongs to the kernel, not to a context; a context with a
    small table blob created later must not break a live one with a larger blob."""
    import torch

    import paper_1101_1245_b200 as g
    w5, w1 = make_config(5), make_config(1)          # 4 materials (127 KB) / 1 material (41 KB)
    dev = torch.device("cuda:0")
    ref5, ref1 = run_gpu(w5, 100_000), run_gpu(w1, 50_000)
    r5, m5 = torch.from_numpy(w5.density).to(dev), torch.from_numpy(w5.material).to(dev)
    r1, m1 = torch.from_numpy(w1.density).to(dev), torch.from_numpy(w1.material).to(dev)
    d5 = torch.empty(r5.shape, dtype=torch.float32, device=dev)
    d1 = torch.empty(r1.shape, dtype=torch.float32, device=dev)
    with g.gpumcd_create(r5, m5, w5.voxel_cm, w5.tables) as big:
        g.gpumcd_set_source(big, w5.source)
        with g.gpumcd_create(r1, m1, w1.voxel_cm, w1.tables) as small:
            g.gpumcd_set_source(small, w1.source)
            for _ in range(2):
                g.gpumcd_run(small, 50_000, w1.seed, d1)
                c1 = g.gpumcd_get_counters(small)
                g.gpumcd_run(big, 100_000, w5.seed, d5)
                c5 = g.gpumcd_get_counters(big)
                for k in INT_KEYS:
                    assert c1[k] == ref1["counters"][k] and c5[k] == ref5["counters"][k], k
    np.testing.assert_allclose(d5.cpu().numpy(), ref5["dose"], rtol=1e-6, atol=0)


# ------------------------------------------------------------------ small stacks on pair-heavy beams
@pytest.mark.parametrize("cfg,n", [(3, 400_000), (5, 1_000_000)])
def test_small_warp_stacks_on_photon_beams(cfg, n):
    """Pair events push two electrons and two photons at once; the smallest stacks the library accepts must
    either hold what a warp banks (same events as the default) or report the overflow, never drop silently."""
    w = make_config(cfg)
    ref = run_gpu(w, n)
    for cap in (256, 384, 512):
        g = run_gpu(w, n, warp_stack=cap)
        assert g["counters"]["bank_high_water"] <= cap
        assert g["counters"]["overflow_count"] == 0, cap
        for k in INT_KEYS:
            assert g["counters"][k] == ref["counters"][k], (cap, k)
    assert ref["counters"]["bank_high_water"] <= 1024 and ref["counters"]["overflow_count"] == 0


def test_overflow_is_reported_by_run_host():
    import paper_1101_1245_b200 as g
    w = make_config(2)
    opt = g.gpumcd_default_options(scheduler=0, wave_size=20000, bank_factor=1)
    dose = np.empty(w.density.shape, np.float32)
    with g.gpumcd_create_host(w.density, w.material, w.voxel_cm, w.tables, opt) as ctx:
        g.gpumcd_set_source(ctx, w.source)
        with pytest.raises(g.GpumcdError) as e:
            g.gpumcd_run_host(ctx, 20000, 1, dose)
        assert e.value.status == -4


# ------------------------------------------------------------------ kinematic thresholds (R33)
def test_thresholds_on_the_device():
    """No Moller event at T <= 2 K_cut, no pair event at E <= 2m, no negative deposit with coarse tables; same
    events as the oracle."""
    tb = build_tables([M.WATER], n_energy=20)
    dens, mat = phantoms.homogeneous(16, 16, 64, 1.0, 0)
    base = make_config(1)
    w = dataclasses.replace(base, density=dens, material=mat, voxel_cm=0.25, tables=tb,
                            source=Source(PHOTON, PENCIL, 2.125, 2.125, energy=1.0))
    for sched in (0, 1):
        g = run_gpu(w, 200_000, seed=82, scheduler=sched)
        o = oracle.run(dens, mat, 0.25, tb, w.source, 200_000, seed=82)
        assert g["counters"]["photon_pair"] == 0 == o.counters["photon_pair"]
        assert (g["edep"] >= 0).all()
        for k in INT_KEYS:
            assert abs(g["counters"][k] - o.counters[k]) <= 10 + 3e-3 * o.counters[k], k
        we = dataclasses.replace(w, source=Source(ELECTRON, PENCIL, 2.125, 2.125, energy=0.39))
        g = run_gpu(we, 100_000, seed=83, scheduler=sched, majorant_scale=50.0)
        assert g["counters"]["hard_moller"] == 0 and g["counters"]["hard_fict"] > 10_000
        assert (g["edep"] >= 0).all()
    w2 = make_config(2)
    src = dataclasses.replace(w2.source, energy=0.3995)
    g = run_gpu(dataclasses.replace(w2, source=src), 300_000, majorant_scale=200.0)
    assert g["counters"]["hard_moller"] == 0 and g["counters"]["hard_fict"] > 100_000


# ------------------------------------------------------------------ steps per refill (the paper's N)
@pytest.mark.parametrize("cfg,n", [(2, 60_000), (5, 300_000)])
def test_steps_per_refill_changes_the_schedule_not_the_histories(cfg, n):
    """Several condensed-history steps between two looks at the stacks: who steps when changes, no history does."""
    w = make_config(cfg)
    ref = run_gpu(w, n, steps_per_refill=1)
    for nsteps in (0, 2, 4, 8):          # 0 = automatic (4 for config 2's electron beam, 1 for config 5)
        g = run_gpu(w, n, steps_per_refill=nsteps)
        for k in INT_KEYS:
            assert g["counters"][k] == ref["counters"][k], (nsteps, k)
        assert g["counters"]["overflow_count"] == 0
        assert np.abs(g["edep"] - ref["edep"]).max() <= 1e-12 * ref["edep"].max()
    m = run_gpu(w, n, steps_per_refill=4, hom_tol=0.1, tally_mode=2)
    m1 = run_gpu(w, n, steps_per_refill=1, hom_tol=0.1, tally_mode=2)
    assert np.array_equal(m["edep"], m1["edep"])


def test_scheduler_options_that_could_loop_for_ever_are_refused():
    """bank_low above one batch (two stacks holding 32 .. bank_low records would send a warp back and forth), and a
    high-water mark below bank_low (a warp would change to a type it leaves at once)."""
    import torch

    import paper_1101_1245_b200 as g
    w = make_config(1)
    rho = torch.from_numpy(w.density).to("cuda:0")
    mat = torch.from_numpy(w.material).to("cuda:0")
    for bad in ({"bank_low": 33}, {"bank_high_g": 4}, {"bank_high_e": 20, "bank_low": 24}, {"steps_per_refill": 65},
                {"cta_threads": 640}, {"tally_mode": 1, "cta_threads": 512}):
        with pytest.raises(g.GpumcdError) as e:
            g.gpumcd_create(rho, mat, w.voxel_cm, w.tables, g.gpumcd_default_options(**bad))
        assert e.value.status == g.GPUMCD_ERR_INVALID_ARG, bad
    # the extremes that are allowed run and agree with the default
    ref = run_gpu(w, 30_000)
    for ok in ({"bank_low": 32, "bank_high_g": 32, "bank_high_e": 32}, {"bank_low": 1}, {"steps_per_refill": 64},
               {"warp_stack": 256, "bank_high_g": 1000, "bank_high_e": 1000}):
        g2 = run_gpu(w, 30_000, **ok)
        for k in INT_KEYS:
            assert g2["counters"][k] == ref["counters"][k], (ok, k)
