"""CPU, world_size 2 over gloo: the N > 1 host path of bench.py -- rank-distinct shards, no data-path collective,
MAX-over-ranks timing, SUM-over-ranks frame counts -- and the frame-balanced partition of ragged batches."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from paper_2606_01009_b200 import sharding, workloads as wl
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        c = wl.CONFIGS["cfg3"]
        # strong scaling of a ragged batch: both ranks generate the same batch and take their frame-balanced slice
        x, off = wl.speaker_ragged(16, c["seed"], c["fs"], 4000, 30000)
        lens = np.diff(off)
        parts = sharding.partition_ragged(lens, world, c["n_fft"], c["hop"])
        lo, hi = parts[rank]
        my_frames = sum(sharding.frames_of(v, c["n_fft"], c["hop"]) for v in lens[lo:hi])
        total = sharding.reduce_count(dist, my_frames)
        # weak scaling seeds differ per rank
        seed = sharding.rank_seed(c["seed"], rank)
        # timing: MAX over ranks
        t = sharding.reduce_step_time(dist, 1.0 + rank)
        dist.barrier()
        q.put((rank, lo, hi, my_frames, total, seed, t, float(x[off[lo]:off[hi]].sum())))
    finally:
        dist.destroy_process_group()


def test_two_rank_shards_cover_the_batch_once_and_reduce():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, lo0, hi0, f0, tot0, s0, t0, _), (r1, lo1, hi1, f1, tot1, s1, t1, _) = res
    assert (lo0, hi1) == (0, 16) and hi0 == lo1                       # contiguous cover, no overlap
    assert tot0 == tot1 == f0 + f1                                    # SUM of frames
    assert abs(f0 - f1) <= 0.25 * (f0 + f1)                           # balanced by frames
    assert s0 != s1                                                   # rank-distinct weak-scaling streams
    assert t0 == t1 == 2.0                                            # MAX over ranks


def test_partitions_are_exact_covers():
    from paper_2606_01009_b200 import sharding
    for n, w in [(32, 1), (32, 8), (5, 8), (0, 2), (1024, 3)]:
        parts = sharding.partition_dense(n, w)
        assert parts[0][0] == 0 and parts[-1][1] == n
        assert all(a[1] == b[0] for a, b in zip(parts, parts[1:]))
        assert max(h - l for l, h in parts) - min(h - l for l, h in parts) <= 1
    rng = np.random.default_rng(1)
    lens = rng.integers(0, 200000, 300)
    for w in (1, 2, 4, 8):
        parts = sharding.partition_ragged(lens, w, 400, 160)
        assert parts[0][0] == 0 and parts[-1][1] == 300
        assert all(a[1] == b[0] for a, b in zip(parts, parts[1:]))
        fr = [sum(sharding.frames_of(v, 400, 160) for v in lens[l:h]) for l, h in parts]
        assert max(fr) <= 1.15 * (sum(fr) / w) + 1300


def test_frames_of_matches_the_oracle_count():
    from oracle import melt_oracle as orc
    from paper_2606_01009_b200 import sharding
    for L in (0, 1, 199, 200, 201, 399, 400, 401, 559, 560, 16000, 480000, 480400):
        for pad in (False, True):
            for drop in (False, True):
                assert sharding.frames_of(L, 400, 160, pad, drop) == orc.num_frames(L, 400, 160, int(pad), drop)
