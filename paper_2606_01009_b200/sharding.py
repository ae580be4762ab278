"""Multi-GPU host logic: clips are independent units, so the path shards
over the batch with NO data-path collective.  One process per GPU; the basis (a pure function of nine scalars) is
rebuilt per rank.  The only communication is bookkeeping around the timed region: a barrier, and a MAX / SUM
reduction of the timing and the frame counts (NCCL on GPUs, gloo in the CPU tests).

No method arithmetic lives here: frames are counted by the library itself (melt_count_frames of include/melt.h, host-only
integer arithmetic that needs no GPU).
"""
import numpy as np

from . import binding as _mb


def rank_seed(base_seed, rank):
    """Weak scaling: every rank owns a full batch of the same recipe but a different random stream."""
    return int(base_seed) + 7919 * int(rank)


def frames_of(length, n_fft, hop, pad_reflect=False, drop_last=False):
    """Frame count of one clip: the library's own melt_count_frames (one copy of the formula)."""
    return _mb.melt_count_frames(length, n_fft, hop, _mb.MELT_PAD_REFLECT if pad_reflect else _mb.MELT_PAD_NONE, drop_last)


def partition_dense(n_clips, world):
    """Strong scaling of a dense batch: contiguous, near-equal clip ranges.  Returns [(lo, hi)] per rank."""
    base, rem = divmod(int(n_clips), int(world))
    out, lo = [], 0
    for r in range(world):
        hi = lo + base + (1 if r < rem else 0)
        out.append((lo, hi))
        lo = hi
    return out


def partition_ragged(lengths, world, n_fft, hop):
    """Strong scaling of a ragged batch: contiguous clip ranges balanced by FRAME count (the unit of work), so that a
    rank's packed samples stay one contiguous slice of the packed array.  Returns [(lo, hi)] per rank."""
    frames = np.array([frames_of(v, n_fft, hop) for v in lengths], dtype=np.int64)
    csum = np.concatenate([[0], np.cumsum(frames)])
    total = int(csum[-1])
    cuts = [0]
    for r in range(1, world):
        target = total * r / world
        i = int(np.searchsorted(csum, target, side="left"))
        if i > 0 and abs(csum[i - 1] - target) <= abs(csum[min(i, len(csum) - 1)] - target):
            i -= 1
        cuts.append(max(cuts[-1], min(i, len(lengths))))
    cuts.append(len(lengths))
    return [(cuts[r], cuts[r + 1]) for r in range(world)]


def reduce_step_time(dist, ms, device=None):
    """MAX over ranks of a per-rank duration (ms).  dist is torch.distributed or None (single process)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms)
    import torch
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def reduce_count(dist, n, device=None):
    """SUM over ranks of a per-rank unit count (frames)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return int(n)
    import torch
    t = torch.tensor([int(n)], dtype=torch.int64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return int(t.item())
