"""-m gpu: the phase-space source (gpumcd_source.shape = 2, R35) through the C ABI
against the oracle: a mixed photon / electron phase space in the slab phantom of config 4, both schedulers;
records whose fate needs no transport; host and device record arrays; the error statuses."""
import dataclasses

import numpy as np
import pytest

import oracle
from gpu_util import run_gpu
from paper_1101_1245_b200 import evaluation as ev
from paper_1101_1245_b200.inputs import PHASE_SPACE, PHOTON, Source, make_config, synthetic_phase_space

pytestmark = pytest.mark.gpu

INT_KEYS = ("photon_flights", "photon_compton", "photon_photo", "photon_pair", "photon_fict", "ch_steps",
            "hard_moller", "hard_brems", "hard_fict", "pushes_e", "pushes_g")


def total(c):
    return c["e_dep_continuous"] + c["e_dep_cutoff"]


def phsp_workload(cfg, n_rec, seed, share=0.2, e0=6.0):
    w = make_config(cfg)
    c0 = 0.5 * w.density.shape[2] * w.voxel_cm
    ps = synthetic_phase_space(n_rec, seed, c0, c0, 5.0, 5.0, electron_share=share, e0=e0)
    return dataclasses.replace(w, source=Source(PHOTON, PHASE_SPACE, 0.0, 0.0, phsp=ps))


@pytest.mark.parametrize("scheduler", [0, 1])
def test_mixed_phase_space_parity(scheduler):
    """1e6 histories from 3e5 records (every record serves 3-4 histories), 20 % electrons, slab phantom: event
    counts, total deposit to 1e-5 (BASELINE.json's bar), per-voxel agreement and gamma over 8 batches a side."""
    w = phsp_workload(4, 300_000, 23)
    n, nb = 1_000_000, 8
    og, gg, oc, gc = [], [], None, None
    for b in range(nb):
        o = oracle.run(w.density, w.material, w.voxel_cm, w.tables, w.source, n // nb, seed=500 + b)
        g = run_gpu(w, n // nb, seed=500 + b, scheduler=scheduler)
        assert g["counters"]["overflow_count"] == 0
        og.append(o.edep); gg.append(g["edep"])
        oc = o.counters if oc is None else {k: oc[k] + v for k, v in o.counters.items()}
        gc = g["counters"] if gc is None else {k: gc[k] + v for k, v in g["counters"].items()}
    assert abs(total(gc) - total(oc)) / total(oc) <= 1e-5
    assert abs((total(gc) + gc["e_escaped"]) / gc["e_incident"] - 1.0) <= 1e-6
    assert gc["e_incident"] == pytest.approx(oc["e_incident"], rel=1e-7)
    for k in INT_KEYS:
        assert abs(gc[k] - oc[k]) <= 3e-3 * oc[k] + 50, (k, gc[k], oc[k])
    om, os_ = ev.batch_mean_sigma(np.array(og))
    gm, gs = ev.batch_mean_sigma(np.array(gg))
    assert ev.voxel_agreement(om, os_, gm, gs, frac=0.1, k=3.0) >= 0.99
    mass = w.density.astype(np.float64) * w.voxel_cm**3
    assert ev.gamma_pass_rate(om / mass, gm / mass, w.voxel_cm, frac=0.1) >= 0.99


@pytest.mark.parametrize("scheduler", [0, 1])
def test_records_whose_fate_needs_no_transport(scheduler):
    """Outside the phantom: escaped at birth; below the cutoff of its type: deposited in the voxel it lies in;
    history h takes record h mod 3 (the same case pins the oracle in test_oracle_phase_space.py)."""
    w = make_config(1)
    rec = np.array([[-1.0, 3.0, 2.0, 0, 0, 1, 5.0, 0],
                    [3.2, 4.7, 6.1, 0, 0, 1, 0.01, 0],
                    [10.0, 0.1, 15.99, 1, 0, 0, 0.15, 1]], np.float32)
    w = dataclasses.replace(w, tables=dataclasses.replace(w.tables, p_cut=0.02),
                            source=Source(PHOTON, PHASE_SPACE, 0.0, 0.0, phsp=rec))
    g = run_gpu(w, 10, seed=3, scheduler=scheduler)
    c = g["counters"]
    assert c["photon_flights"] == 0 and c["ch_steps"] == 0 and c["overflow_count"] == 0
    e_ph, e_el = float(np.float32(0.01)), float(np.float32(0.15))
    assert c["e_escaped"] == pytest.approx(20.0, rel=1e-12)
    assert g["edep"][12, 9, 6] == pytest.approx(3 * e_ph, rel=1e-12)
    assert g["edep"][31, 0, 20] == pytest.approx(3 * e_el, rel=1e-12)
    assert g["edep"].sum() == pytest.approx(3 * e_ph + 3 * e_el, rel=1e-12)
    assert c["e_incident"] == pytest.approx(20.0 + 3 * e_ph + 3 * e_el, rel=1e-12)


def test_one_record_phase_space_is_the_pencil_beam():
    w = make_config(1)
    s = w.source
    rec = np.array([[s.cx, s.cy, 0.0, 0.0, 0.0, 1.0, s.energy, 0.0]], np.float32)
    a = run_gpu(w, 50_000)
    b = run_gpu(dataclasses.replace(w, source=Source(PHOTON, PHASE_SPACE, 0.0, 0.0, phsp=rec)), 50_000)
    for k in INT_KEYS:
        assert a["counters"][k] == b["counters"][k], k
    assert np.abs(a["edep"] - b["edep"]).max() <= 1e-12 * a["edep"].max()


def test_device_records_equal_host_records_and_errors():
    import torch

    import paper_1101_1245_b200 as g
    w = phsp_workload(1, 5000, 4, share=0.1, e0=2.0)
    a = run_gpu(w, 30_000)
    dev_rec = torch.from_numpy(w.source.phsp).to("cuda:0")
    b = run_gpu(dataclasses.replace(w, source=dataclasses.replace(w.source, phsp=dev_rec)), 30_000)
    for k in INT_KEYS:
        assert a["counters"][k] == b["counters"][k], k
    rho = torch.from_numpy(w.density).to("cuda:0")
    mat = torch.from_numpy(w.material).to("cuda:0")
    with g.gpumcd_create(rho, mat, w.voxel_cm, w.tables) as ctx:
        for bad, status in (([8.0, 8.0, 0.0, 0, 0, 1, 25.0, 0], g.GPUMCD_ERR_TABLE_RANGE),
                            ([8.0, 8.0, 0.0, 0, 0, 1, 2.0, 2], g.GPUMCD_ERR_INVALID_ARG),
                            ([8.0, np.nan, 0.0, 0, 0, 1, 2.0, 0], g.GPUMCD_ERR_INVALID_ARG)):
            rec = np.array([[8.0, 8.0, 0.0, 0, 0, 1, 2.0, 0], bad], np.float32)
            with pytest.raises(g.GpumcdError) as e:
                g.gpumcd_set_source(ctx, Source(PHOTON, PHASE_SPACE, 0.0, 0.0, phsp=rec))
            assert e.value.status == status
        with pytest.raises(g.GpumcdError) as e:   # a failed set_source leaves the context without a source
            g.gpumcd_run(ctx, 10, 1, torch.empty(rho.shape, dtype=torch.float32, device="cuda:0"))
        assert e.value.status == g.GPUMCD_ERR_NO_SOURCE
    # the 1024-thread CTA exists for the ablation of plain sources only
    with g.gpumcd_create(rho, mat, w.voxel_cm, w.tables, g.gpumcd_default_options(cta_threads=1024)) as ctx:
        g.gpumcd_set_source(ctx, w.source)
        with pytest.raises(g.GpumcdError) as e:
            g.gpumcd_run(ctx, 10, 1, torch.empty(rho.shape, dtype=torch.float32, device="cuda:0"))
        assert e.value.status == g.GPUMCD_ERR_INVALID_ARG
