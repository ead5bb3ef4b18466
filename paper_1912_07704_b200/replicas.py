"""Multi-GPU: replicas over time chunks ("parallel pipeline configuration/execution
on multiple GPUs").

The path shards with NO exchange step: chunks are independent given the S-sample overlap, so rank r of W owns chunks
r, r+W, r+2W, ... (``aa_strategy_shard``), reads only its own input span, keeps its own arena, and the candidate
lists are concatenated on the host. There is no collective on the data path; ``torch.distributed`` (NCCL on GPUs,
gloo in the CPU tests) is used only to gather the small candidate arrays and to take the max-over-ranks time.
Host logic only — nothing here computes any part of the search.
"""
from __future__ import annotations

import numpy as np


def chunks_of_rank(nchunks: int, rank: int, world: int) -> list[int]:
    """Chunk indices owned by ``rank`` (the rule ``aa_strategy_shard`` applies inside the library)."""
    if not (0 <= rank < world):
        raise ValueError(f"need 0 <= rank < world, got rank={rank}, world={world}")
    return list(range(rank, nchunks, world))


def input_span_of_rank(chunks, rank: int, world: int):
    """(first_sample, end_sample) of the input a rank touches, given ``chunks`` = [(start, len, n_out), ...] from
    ``aa_strategy_get_chunk``; None if the rank owns no chunk. A rank only needs these samples resident on its host."""
    mine = [chunks[j] for j in chunks_of_rank(len(chunks), rank, world)]
    if not mine:
        return None
    return int(min(c[0] for c in mine)), int(max(c[0] + c[1] for c in mine))


def canonical_order(cands: np.ndarray, n_out: int) -> np.ndarray:
    """Sort a structured candidate array into the library's canonical order (chunk, range, dm_index, sample), the chunk
    of a candidate being sample // n_out (chunk j covers output samples [j*n_out, (j+1)*n_out))."""
    if len(cands) == 0:
        return cands
    chunk = cands["sample"].astype(np.int64) // int(n_out)
    order = np.lexsort((cands["sample"], cands["dm_index"], cands["range"], chunk))
    return cands[order]


def gather_candidates(local: np.ndarray, n_out: int, group=None) -> np.ndarray:
    """All ranks' candidate arrays concatenated in canonical order, on every rank (object all-gather of small arrays)."""
    import torch.distributed as dist
    if not dist.is_available() or not dist.is_initialized() or dist.get_world_size(group) == 1:
        return canonical_order(local, n_out)
    parts = [None] * dist.get_world_size(group)
    dist.all_gather_object(parts, local, group=group)
    nonempty = [p for p in parts if len(p)]
    merged = np.concatenate(nonempty) if nonempty else local[:0]
    return canonical_order(merged, n_out)


def max_over_ranks(seconds: float, device=None, group=None) -> float:
    """The slowest rank's time: the figure every multi-GPU number is quoted on."""
    import torch
    import torch.distributed as dist
    if not dist.is_available() or not dist.is_initialized() or dist.get_world_size(group) == 1:
        return float(seconds)
    t = torch.tensor([seconds], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())
