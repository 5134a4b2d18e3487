"""Helpers for the -m gpu parity tests: run a workload through the C ABI (via the thin binding)."""
import numpy as np


def run_gpu(w, n=None, seed=None, want_trace=False, want_edep=True, **opts):
    import torch

    import paper_1101_1245_b200 as g

    n = w.n_histories if n is None else int(n)
    seed = w.seed if seed is None else int(seed)
    dev = torch.device("cuda:0")
    rho = torch.from_numpy(np.ascontiguousarray(w.density)).to(dev)
    mat = torch.from_numpy(np.ascontiguousarray(w.material)).to(dev)
    out = {}
    with g.gpumcd_create(rho, mat, w.voxel_cm, w.tables, g.gpumcd_default_options(**opts)) as ctx:
        g.gpumcd_set_source(ctx, w.source)
        if want_trace:
            tr = torch.zeros(n, dtype=torch.int64, device=dev)
            g.gpumcd_run_trace(ctx, n, seed, tr)
            torch.cuda.synchronize()
            out["trace"] = tr.cpu().numpy().view(np.uint64)
        else:
            dose = torch.empty(rho.shape, dtype=torch.float32, device=dev)
            g.gpumcd_run(ctx, n, seed, dose)
            torch.cuda.synchronize()
            out["dose"] = dose.cpu().numpy()
        out["counters"] = g.gpumcd_get_counters(ctx)
        if want_edep:
            e = torch.empty(rho.shape, dtype=torch.float64, device=dev)
            g.gpumcd_get_energy_tally(ctx, e)
            torch.cuda.synchronize()
            out["edep"] = e.cpu().numpy()
    return out
