"""Multi-GPU host logic: histories are independent, so every rank simulates its own
disjoint range of history ids and the resulting dose arrays are summed.  The counter-based RNG needs
no stream splitting: a history's draws depend only on (seed, history id).

The only exchange step of the method is the final sum, done with one all-reduce (NCCL on GPUs,
gloo in the CPU tests).  Dose is normalised per history, so the sum of per-rank doses over equal
shares is divided by the number of ranks."""
from __future__ import annotations

from typing import Tuple


def history_range(n_total: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous, disjoint, exhaustive split of [0, n_total): returns (first_history, count)."""
    if not (0 <= rank < world) or n_total < 0:
        raise ValueError("bad rank / world / n_total")
    base, rem = divmod(n_total, world)
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)


def combine_dose(dose, count: int, n_total: int, dist=None):
    """Turn a per-rank dose (normalised by ``count`` histories) into the global dose: weight by the
    rank's share, then all-reduce(sum).  Works on any torch tensor; ``dist`` = torch.distributed."""
    dose.mul_(count / max(n_total, 1))
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(dose)
    return dose
