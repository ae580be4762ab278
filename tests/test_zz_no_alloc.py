"""melt_forward_ragged_noalloc (include/melt.h): the ragged forward whose only per-call scratch -- the device-side chunk prefix --
lives in a file-scope device array of the library, against melt_forward_ragged (scratch from the plan's stream-ordered pool) on
the same inputs.  Collected last on purpose (the run is `pytest -x`); passes alone in a fresh process (the first call
looks the array's address up) and after every other test (whatever they left in the array)."""
import numpy as np
import pytest

import parity_util as pu
from paper_2606_01009_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _batch(rng, n_clips, lo, hi):
    """Packed clips of arbitrary lengths (clip starts at any sample: all four misalignments occur)."""
    lens = rng.integers(lo, hi + 1, size=n_clips).astype(np.int64)
    offs = np.zeros(n_clips + 1, np.int64)
    offs[1:] = np.cumsum(lens)
    x = rng.normal(0.0, 0.1, int(offs[-1])).astype(np.float32)
    return x, offs


def _run(mb, torch, plan, fn, x, offs, stream):
    n = len(offs) - 1
    total = int(sum(mb.melt_num_frames(plan, int(v)) for v in np.diff(offs)))
    C = mb.melt_num_channels(plan)
    xd = torch.from_numpy(x).cuda()
    od = torch.from_numpy(offs).cuda()
    out = torch.full((max(total, 1), C), float("nan"), device="cuda")
    fo = torch.full((n + 1,), -1, dtype=torch.int64, device="cuda")
    fn(plan, xd, od, n, out, fo, stream)
    return xd, od, out, fo, total


@pytest.mark.parametrize("n_mfcc", [0, 13])
def test_noalloc_matches_pool_path_two_calls_in_a_row(n_mfcc):
    import torch
    from paper_2606_01009_b200 import binding as mb
    c = dict(wl.CONFIGS["cfg3"])   # speaker-style ragged batch: 16 kHz, 400 / 160, 40 Mel bins
    c["n_mfcc"] = n_mfcc
    plan = pu.plan_for(c, "compensated", layout="frame_major")
    try:
        rng = np.random.default_rng(20260601 + n_mfcc)
        # call 1: 37 clips spanning several 256-frame tiles with ragged tails; call 2: FEWER and shorter clips, so that the array still
        # holds entries of call 1 beyond the ones call 2 rewrites (lengths from 100 samples: shorter than a frame = no frames)
        xa, oa = _batch(rng, 37, 3000, 40000)
        xb, ob = _batch(rng, 5, 100, 9000)
        st = torch.cuda.current_stream().cuda_stream
        ref = [_run(mb, torch, plan, mb.melt_forward_ragged, x, o, st) for x, o in ((xa, oa), (xb, ob))]
        torch.cuda.synchronize()
        # the two allocation-free calls back to back in one stream, no synchronisation in between
        got = [_run(mb, torch, plan, mb.melt_forward_ragged_noalloc, x, o, st) for x, o in ((xa, oa), (xb, ob))]
        torch.cuda.synchronize()
        for (_, _, out_r, fo_r, total), (_, _, out_g, fo_g, _) in zip(ref, got):
            assert np.array_equal(fo_g.cpu().numpy(), fo_r.cpu().numpy())          # frame offsets: integers, bit-exact
            assert int(fo_g[-1]) == total
            a, b = out_g.cpu().numpy()[:total].astype(np.float64), out_r.cpu().numpy()[:total].astype(np.float64)
            assert np.isfinite(a).all() and np.isfinite(b).all()
            # same kernels on the same inputs: the bar is the one the log-domain parity tests use (ACC_LOG_BAR; cepstra: an
            # orthonormal DCT of such values does not grow the error)
            assert float(np.abs(a - b).max()) <= pu.ACC_LOG_BAR
    finally:
        mb.melt_plan_destroy(plan)


def test_noalloc_rejects_more_clips_than_the_array_holds():
    import torch
    from paper_2606_01009_b200 import binding as mb
    c = dict(wl.CONFIGS["cfg3"])
    plan = pu.plan_for(c, "compensated", layout="frame_major")
    try:
        n = mb.MELT_NOALLOC_MAX_CLIPS + 1
        x = torch.zeros(16, device="cuda")
        od = torch.zeros(n + 1, dtype=torch.int64, device="cuda")
        out = torch.zeros((1, mb.melt_num_channels(plan)), device="cuda")
        fo = torch.zeros(n + 1, dtype=torch.int64, device="cuda")
        with pytest.raises(mb.MeltError) as ei:
            mb.melt_forward_ragged_noalloc(plan, x, od, n, out, fo, torch.cuda.current_stream().cuda_stream)
        assert "MELT_NOALLOC_MAX_CLIPS" in str(ei.value)
        # the limit itself is accepted: MELT_NOALLOC_MAX_CLIPS clips, all empty but the last (800 samples = 3 frames)
        n = mb.MELT_NOALLOC_MAX_CLIPS
        st = torch.cuda.current_stream().cuda_stream
        x = 0.1 * torch.randn(800, device="cuda")
        od = torch.zeros(n + 1, dtype=torch.int64, device="cuda")
        od[n] = 800
        C = mb.melt_num_channels(plan)
        outs, fos = [], []
        for fn in (mb.melt_forward_ragged, mb.melt_forward_ragged_noalloc):
            out = torch.full((3, C), float("nan"), device="cuda")
            fo = torch.full((n + 1,), -1, dtype=torch.int64, device="cuda")
            fn(plan, x, od, n, out, fo, st)
            outs.append(out)
            fos.append(fo)
        torch.cuda.synchronize()
        assert torch.equal(fos[0], fos[1]) and int(fos[1][n]) == 3 and int(fos[1][n - 1]) == 0
        assert bool(torch.isfinite(outs[1]).all())
        assert float((outs[0] - outs[1]).abs().max()) <= pu.ACC_LOG_BAR
    finally:
        mb.melt_plan_destroy(plan)
