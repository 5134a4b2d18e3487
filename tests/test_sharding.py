"""N > 1 path on CPU (gloo, world size 2): disjoint history ranges plus one all-reduce reproduce the
single-process tally.  The transport on each rank is the oracle (test infrastructure)."""
import os

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1101_1245_b200.sharding import combine_dose, history_range


def test_history_ranges_partition_the_run():
    for n, world in ((10, 1), (10, 3), (1_000_003, 8), (5, 8)):
        spans = [history_range(n, r, world) for r in range(world)]
        assert spans[0][0] == 0
        for (a, ca), (b, _) in zip(spans, spans[1:]):
            assert a + ca == b
        assert sum(c for _, c in spans) == n
        assert max(c for _, c in spans) - min(c for _, c in spans) <= 1
    with pytest.raises(ValueError):
        history_range(10, 2, 2)


def _worker(rank, world, port, n_total, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    from paper_1101_1245_b200.inputs import make_config
    w = make_config(1)
    first, count = history_range(n_total, rank, world)
    r = oracle.run_workload(w, count, hist_begin=first, n_threads=1)
    dose = torch.from_numpy(r.dose.astype(np.float64))
    combine_dose(dose, count, n_total, dist)
    steps = torch.tensor([r.counters["ch_steps"]], dtype=torch.int64)
    dist.all_reduce(steps)
    if rank == 0:
        np.save(os.path.join(out_dir, "dose.npy"), dose.numpy())
        np.save(os.path.join(out_dir, "steps.npy"), steps.numpy())
    dist.destroy_process_group()


def test_two_ranks_reproduce_the_single_process_dose(tmp_path):
    import oracle
    from paper_1101_1245_b200.inputs import make_config
    n_total = 6001
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, n_total, str(tmp_path)), nprocs=2, join=True)
    w = make_config(1)
    ref = oracle.run_workload(w, n_total, n_threads=1)
    dose = np.load(tmp_path / "dose.npy")
    steps = np.load(tmp_path / "steps.npy")
    assert int(steps[0]) == ref.counters["ch_steps"]
    np.testing.assert_allclose(dose, ref.dose.astype(np.float64), rtol=2e-6, atol=1e-12 * ref.dose.max())
