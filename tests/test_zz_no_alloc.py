"""-m gpu: gpumcd_run_uncertainty_static, the entry point that allocates no device memory (its scratch, the three
batch-statistics grids, lives in a static device array of the library; include/gpumcd.h), against the existing
gpumcd_run_uncertainty on the same context, two calls in a row.  Collected last on purpose (the file name): the
suite runs with `pytest -x`, and a failure here must not hide the tests of the hot path."""
import numpy as np
import pytest

from paper_1101_1245_b200.inputs import PHOTON, make_config, make_paper_geometry

pytestmark = pytest.mark.gpu


def run_both(g, torch, w, n, nb, seed):
    dev = torch.device("cuda:0")
    rho = torch.from_numpy(w.density).to(dev)
    mat = torch.from_numpy(w.material).to(dev)
    out = {}
    with g.gpumcd_create(rho, mat, w.voxel_cm, w.tables) as ctx:
        g.gpumcd_set_source(ctx, w.source)
        for name, fn in (("static", g.gpumcd_run_uncertainty_static), ("malloc", g.gpumcd_run_uncertainty)):
            d = torch.empty(rho.shape, dtype=torch.float32, device=dev)
            s = torch.empty(rho.shape, dtype=torch.float32, device=dev)
            fn(ctx, n, nb, seed, d, s)
            torch.cuda.synchronize()
            c = g.gpumcd_get_counters(ctx)
            out[name] = (d.cpu().numpy(), s.cpu().numpy(), c)
    return out


def check(out):
    (d1, s1, c1), (d0, s0, c0) = out["static"], out["malloc"]
    for k in ("photon_flights", "photon_compton", "ch_steps", "hard_moller", "hard_brems", "pushes_e", "pushes_g"):
        assert c1[k] == c0[k], k                      # the same histories, event for event
    assert c1["overflow_count"] == 0
    # the tolerances of the existing uncertainty / tally-mode tests: the fp64 tally's additions come in another order
    np.testing.assert_allclose(d1, d0, rtol=1e-5, atol=1e-9 * d0.max())
    np.testing.assert_allclose(s1, s0, rtol=1e-4, atol=1e-7 * s0.max())
    assert d0.max() > 0 and s0.max() > 0


def test_static_scratch_entry_point_matches_the_allocating_one_twice_in_a_row():
    import torch

    import paper_1101_1245_b200 as g
    assert torch.cuda.is_available()
    # call 1: config 1's 32^3 phantom; call 2: the paper's 64^3 geometry, which fills the array to its limit and
    # finds the first call's sums in it (the entry point must clear what it uses)
    w1 = make_config(1)
    check(run_both(g, torch, w1, 60_000, 8, seed=11))
    w2 = make_paper_geometry(3, PHOTON)
    assert w2.density.size == g.GPUMCD_STATIC_MAX_VOXELS
    check(run_both(g, torch, w2, 200_000, 10, seed=12))
    # and the small one again after the large one (stale sums beyond its own 32^3 voxels do not matter)
    check(run_both(g, torch, w1, 30_001, 7, seed=13))


def test_static_scratch_entry_point_refuses_what_it_cannot_hold():
    import torch

    import paper_1101_1245_b200 as g
    w = make_config(2)                                  # 128^3 voxels: 8 x the limit
    dev = torch.device("cuda:0")
    rho = torch.from_numpy(w.density).to(dev)
    mat = torch.from_numpy(w.material).to(dev)
    d = torch.empty(rho.shape, dtype=torch.float32, device=dev)
    s = torch.empty(rho.shape, dtype=torch.float32, device=dev)
    with g.gpumcd_create(rho, mat, w.voxel_cm, w.tables) as ctx:
        g.gpumcd_set_source(ctx, w.source)
        with pytest.raises(g.GpumcdError) as e:
            g.gpumcd_run_uncertainty_static(ctx, 1000, 4, 1, d, s)
        assert e.value.status == g.GPUMCD_ERR_INVALID_ARG and "GPUMCD_STATIC_MAX_VOXELS" in str(e.value)
        g.gpumcd_run_uncertainty(ctx, 1000, 4, 1, d, s)  # the allocating path takes it
        torch.cuda.synchronize()
    w1 = make_config(1)
    rho = torch.from_numpy(w1.density).to(dev)
    mat = torch.from_numpy(w1.material).to(dev)
    d = torch.empty(rho.shape, dtype=torch.float32, device=dev)
    s = torch.empty(rho.shape, dtype=torch.float32, device=dev)
    with g.gpumcd_create(rho, mat, w1.voxel_cm, w1.tables) as ctx:
        g.gpumcd_set_source(ctx, w1.source)
        g.gpumcd_set_profiling(ctx, True)
        with pytest.raises(g.GpumcdError) as e:          # profiling creates events per launch: refused
            g.gpumcd_run_uncertainty_static(ctx, 1000, 4, 1, d, s)
        assert e.value.status == g.GPUMCD_ERR_INVALID_ARG
        with pytest.raises(g.GpumcdError):
            g.gpumcd_run_uncertainty_static(ctx, 3, 4, 1, d, s)   # more batches than histories
