"""Host-side logic of the multi-GPU path: bands are independent units, so H|psi> shards by
bands (or by k-point, the paper's `-NPOOL` pools, one MPI rank per GPU: PAPER.md:L236-238) with V, beta, D and the
maps replicated and NO data-path collective. The only communication is the benchmark's barrier and the
max-over-ranks reduction of the timed region. Pure Python + torch.distributed; no method arithmetic here.
"""
from __future__ import annotations

import torch


def split_bands(nbands_total: int, world: int) -> list[tuple[int, int]]:
    """Strong-scaling split: contiguous (band0, nb) per rank, sizes differ by at most one, empty shards allowed."""
    assert nbands_total >= 0 and world >= 1
    base, rem = divmod(nbands_total, world)
    out, b0 = [], 0
    for r in range(world):
        nb = base + (1 if r < rem else 0)
        out.append((b0, nb))
        b0 += nb
    return out


def weak_band_range(rank: int, nbands_per_rank: int) -> tuple[int, int]:
    """Weak-scaling shard (what bench.py times): every rank applies H to `nbands_per_rank` bands of its own,
    global band keys rank*nb .. (rank+1)*nb - 1, so no two ranks see the same psi."""
    assert rank >= 0 and nbands_per_rank >= 0
    return rank * nbands_per_rank, nbands_per_rank


def batches(nb: int, batch: int) -> list[tuple[int, int]]:
    """(offset, count) of the qe_hpsi_apply calls that cover nb bands in batches of `batch` (ragged tail kept)."""
    assert batch >= 1
    return [(b0, min(batch, nb - b0)) for b0 in range(0, nb, batch)]


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """MAX all-reduce of a scalar (the timed region's milliseconds). `dist` = torch.distributed or None."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_bands_per_s(world: int, nbands_per_rank: int, ms_per_step_max: float) -> float:
    """Whole-job throughput: the bands all ranks processed in one step / the slowest rank's step time."""
    return world * nbands_per_rank / (ms_per_step_max * 1e-3)
