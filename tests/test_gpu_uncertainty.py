"""-m gpu: gpumcd_run_uncertainty (Eq. 11-13) and the paper's own benchmark geometries (L233-266)
against the oracle, through the C ABI."""
import numpy as np
import pytest

import oracle
from gpu_util import run_gpu
from paper_1101_1245_b200 import evaluation as ev
from paper_1101_1245_b200.inputs import ELECTRON, PHOTON, make_config, make_paper_geometry

pytestmark = pytest.mark.gpu

INT_KEYS = ("photon_flights", "photon_compton", "photon_photo", "photon_pair", "photon_fict", "ch_steps",
            "hard_moller", "hard_brems", "hard_fict", "pushes_e", "pushes_g")


def run_gpu_uncertainty(w, n, nb, **opts):
    import torch

    import paper_1101_1245_b200 as g
    dev = torch.device("cuda:0")
    rho = torch.from_numpy(np.ascontiguousarray(w.density)).to(dev)
    mat = torch.from_numpy(np.ascontiguousarray(w.material)).to(dev)
    with g.gpumcd_create(rho, mat, w.voxel_cm, w.tables, g.gpumcd_default_options(**opts)) as ctx:
        g.gpumcd_set_source(ctx, w.source)
        dose = torch.empty(rho.shape, dtype=torch.float32, device=dev)
        sig = torch.empty(rho.shape, dtype=torch.float32, device=dev)
        g.gpumcd_run_uncertainty(ctx, n, nb, w.seed, dose, sig)
        e = torch.empty(rho.shape, dtype=torch.float64, device=dev)
        g.gpumcd_get_energy_tally(ctx, e)
        torch.cuda.synchronize()
        return dict(dose=dose.cpu().numpy(), sigma=sig.cpu().numpy(), edep=e.cpu().numpy(),
                    counters=g.gpumcd_get_counters(ctx))


@pytest.mark.parametrize("scheduler", [0, 1])
def test_batched_run_gives_the_dose_of_the_plain_run(scheduler):
    """The batches cover the same history ids: same events, same tally (ragged batch sizes included)."""
    w = make_paper_geometry(2, ELECTRON)
    n, nb = 50_003, 7
    a = run_gpu(w, n, scheduler=scheduler)
    b = run_gpu_uncertainty(w, n, nb, scheduler=scheduler)
    for k in INT_KEYS:
        assert a["counters"][k] == b["counters"][k], k
    assert np.abs(a["edep"] - b["edep"]).max() <= 1e-12 * a["edep"].max()
    assert np.allclose(a["dose"], b["dose"], rtol=1e-6, atol=0)
    assert total(b["counters"]) == pytest.approx(b["edep"].sum(), rel=1e-12)


def total(c):
    return c["e_dep_continuous"] + c["e_dep_cutoff"]


@pytest.mark.parametrize("geom,particle,n", [(1, ELECTRON, 400_000), (2, PHOTON, 1_600_000), (3, ELECTRON, 400_000)])
def test_uncertainty_matches_the_history_by_history_oracle(geom, particle, n):
    """Eq. 13 on the oracle (history by history) against the device's batch estimate of the same quantity:
    per voxel their squared ratio is chi^2_{B-1}/(B-1); Eq. 12's s averages that out."""
    w = make_paper_geometry(geom, particle)
    nb = 40
    g = run_gpu_uncertainty(w, n, nb)
    e, sq, c = oracle.run_moments(w.density, w.material, w.voxel_cm, w.tables, w.source, n, w.seed)
    mass = w.density.astype(np.float64) * w.voxel_cm ** 3
    d_o = e / n / mass
    u_o = oracle.uncertainty_from_moments(e, sq, n) / mass
    assert total(g["counters"]) == pytest.approx(total(c), rel=1e-5)
    sel = d_o > 0.2 * d_o.max()
    assert sel.sum() > 500
    ratio2 = (g["sigma"][sel].astype(np.float64) / u_o[sel]) ** 2
    assert abs(ratio2.mean() - 1.0) < 0.04
    lo, hi = 0.40, 1.95                                   # 99.9 % band of chi^2_39 / 39 is (0.43, 1.87)
    assert np.mean((ratio2 > lo) & (ratio2 < hi)) > 0.995
    s_g = ev.relative_uncertainty(g["dose"].astype(np.float64), g["sigma"].astype(np.float64), 0.2)
    s_o = ev.relative_uncertainty(d_o, u_o, 0.2)
    assert s_g == pytest.approx(s_o, rel=0.03)
    # and the dose itself agrees within the combined uncertainty
    assert ev.voxel_agreement(d_o, u_o, g["dose"].astype(np.float64), g["sigma"].astype(np.float64), 0.1, 3.0) >= 0.99


@pytest.mark.parametrize("geom,particle", [(1, PHOTON), (2, ELECTRON), (3, PHOTON)])
def test_paper_geometry_dose_parity(geom, particle):
    """The paper's cases at its own sizes (1e6 electrons / 4e6 photons, L198): BASELINE.json's bars."""
    w = make_paper_geometry(geom, particle)
    n = w.n_histories
    g = run_gpu(w, n)
    o = oracle.run_workload(w, n)
    for k in INT_KEYS:
        assert abs(g["counters"][k] - o.counters[k]) <= 10 + 2e-3 * o.counters[k], k
    assert total(g["counters"]) == pytest.approx(total(o.counters), rel=1e-5)
    assert ev.gamma_pass_rate(o.dose.astype(np.float64), g["dose"].astype(np.float64), w.voxel_cm, frac=0.1) >= 0.99


def test_uncertainty_argument_errors():
    import torch

    import paper_1101_1245_b200 as g
    w = make_config(1)
    dev = torch.device("cuda:0")
    rho = torch.from_numpy(w.density).to(dev)
    mat = torch.from_numpy(w.material).to(dev)
    with g.gpumcd_create(rho, mat, w.voxel_cm, w.tables) as ctx:
        g.gpumcd_set_source(ctx, w.source)
        d = torch.empty(rho.shape, dtype=torch.float32, device=dev)
        s = torch.empty(rho.shape, dtype=torch.float32, device=dev)
        for nb in (0, 1, 11):
            with pytest.raises(g.GpumcdError) as ei:
                g.gpumcd_run_uncertainty(ctx, 10, nb, 1, d, s)
            assert ei.value.status == g.binding.GPUMCD_ERR_INVALID_ARG
        g.gpumcd_run_uncertainty(ctx, 10, 10, 1, d, s)     # one history per batch is allowed
        torch.cuda.synchronize()
        assert torch.isfinite(s).all() and (s >= 0).all()
