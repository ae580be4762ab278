"""GPU: no forward writes outside its output buffers.  compute-sanitizer is closed on this GPU pool (profiles/r02_sanitizer.md), so
the out-of-bounds check is done by hand: every output (features, tapped log-Mel, frame offsets) sits between two guard bands
filled with a sentinel bit pattern, and the bands must be untouched after dense, ragged, reflect-padded, 16-bit and MFCCT
forwards at shapes with partial tiles and partial chunks."""
import numpy as np
import pytest

import parity_util as pu

pytestmark = pytest.mark.gpu

GUARD = 4096          # elements on each side
SENTINEL = -777.0      # exact in fp32, fp16 and bf16; no output of the path comes near it


def _guarded(n, dtype, torch):
    buf = torch.full((n + 2 * GUARD,), SENTINEL if dtype != torch.int64 else -77, dtype=dtype, device="cuda")
    return buf, buf[GUARD:GUARD + n]


def _check(buf, n, torch, what):
    s = SENTINEL if buf.dtype != torch.int64 else -77
    ref = torch.full((GUARD,), s, dtype=buf.dtype, device="cuda")
    assert torch.equal(buf[:GUARD], ref), what + ": wrote before the buffer"
    assert torch.equal(buf[GUARD + n:], ref), what + ": wrote past the buffer"


@pytest.mark.parametrize("case", ["cfg1-feature", "cfg1-frame-reflect", "cfg1-f16", "cfg4b-kblock", "mfcct-tap", "odd-general"])
def test_dense_forwards_stay_inside_their_buffers(case):
    import torch
    from paper_2606_01009_b200 import binding as mb, workloads as wl
    rng = np.random.default_rng(len(case))
    c = dict(wl.CONFIGS["cfg4b" if case.startswith("cfg4b") else ("cfg3" if case == "mfcct-tap" else "cfg1")])
    layout, pad, dt, tap = c["layout"], False, torch.float32, False
    B, L = 3, 400 + 160 * 333 + 4
    if case == "cfg1-frame-reflect":
        layout, pad, c["drop_last"] = "frame_major", True, False
    if case == "cfg1-f16":
        dt = torch.float16
    if case == "cfg4b-kblock":
        B, L = 2, 2048 + 512 * 300
    if case == "mfcct-tap":
        layout, tap, c["ragged"] = "frame_major", True, False
    if case == "odd-general":      # hop % 4 != 0: the general kernel
        c.update(n_fft=401, hop=161, n_mels=23)
        layout = "frame_major"
    x = torch.from_numpy(rng.normal(0, 0.1, (B, L)).astype(np.float32)).cuda()
    plan = pu.plan_for(c, "compensated", layout=layout, pad=pad)
    try:
        if dt == torch.float16:
            mb.melt_plan_set_option(plan, mb.MELT_OPT_OUTPUT_DTYPE, mb.MELT_DTYPE_F16)
        T, C = mb.melt_num_frames(plan, L), mb.melt_num_channels(plan)
        n = B * T * C
        buf, out = _guarded(n, dt, torch)
        st = torch.cuda.current_stream().cuda_stream
        if tap:
            tbuf, tp = _guarded(B * T * c["n_mels"], torch.float32, torch)
            mb.melt_forward_tap(plan, x, None, B, L, out, tp, None, st)
        else:
            mb.melt_forward(plan, x, B, L, out, st)
        torch.cuda.synchronize()
        _check(buf, n, torch, case)
        assert torch.isfinite(out.float()).all() and not (out.float() == SENTINEL).any()
        if tap:
            _check(tbuf, B * T * c["n_mels"], torch, case + " tap")
    finally:
        mb.melt_plan_destroy(plan)


@pytest.mark.parametrize("pad", [False, True])
def test_ragged_forwards_stay_inside_their_buffers(pad):
    import torch
    from paper_2606_01009_b200 import binding as mb, workloads as wl
    c = dict(wl.CONFIGS["cfg3"])
    rng = np.random.default_rng(9)
    lens = [7001, 0, 399, 48003, 560, 400 + 31 * 160, 400 + 32 * 160, 90001, 123]
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    x = torch.from_numpy(rng.normal(0, 0.1, int(off[-1])).astype(np.float32)).cuda()
    plan = pu.plan_for(c, "compensated", layout="frame_major", pad=pad)
    try:
        total = int(sum(mb.melt_num_frames(plan, int(v)) for v in lens))
        buf, out = _guarded(total * 13, torch.float32, torch)
        tbuf, tp = _guarded(total * 40, torch.float32, torch)
        fbuf, fo = _guarded(len(lens) + 1, torch.int64, torch)
        mb.melt_forward_tap(plan, x, torch.from_numpy(off).cuda(), len(lens), 0, out, tp, fo, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        _check(buf, total * 13, torch, "cepstra")
        _check(tbuf, total * 40, torch, "tap")
        _check(fbuf, len(lens) + 1, torch, "frame offsets")
        assert int(fo[-1]) == total and torch.isfinite(out).all() and not (out == SENTINEL).any()
    finally:
        mb.melt_plan_destroy(plan)
