"""Multi-GPU host logic: the path shards BY IMAGE.  RoI k reads and writes only
image batch_idx_k's pyramid, so rank r owns a contiguous block of images, their RoIs (batch index
re-based) and their output rows.  There is no exchange step and therefore no data-path collective;
torch.distributed is used only for the barrier and the max-over-ranks timing of bench.py."""
from typing import Tuple

import numpy as np


def image_range(n_img: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous, balanced block of images [lo, hi) owned by `rank`."""
    base, rem = divmod(n_img, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def shard_rois(rois: np.ndarray, n_img: int, rank: int, world: int):
    """Returns (local_rois, rows): the RoIs whose image this rank owns, with batch_idx re-based to
    the local pyramid, and their row indices in the global output.  RoIs with an invalid batch
    index are owned by nobody (their rows stay zero)."""
    lo, hi = image_range(n_img, rank, world)
    b = rois[:, 0]
    rows = np.nonzero((b >= lo) & (b < hi))[0]
    local = rois[rows].copy()
    local[:, 0] -= np.float32(lo)
    return local, rows


def max_over_ranks_ms(ms: float, dist=None, device=None) -> float:
    """Timing rule of bench.py: the job's time is the slowest rank's."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms)
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
