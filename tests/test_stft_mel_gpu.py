"""GPU parity of the conventional front end (melt_plan_create_stft_mel: STFT -> power -> triangular Mel filterbank -> log10; SURVEY.md
8(f) NEXT-4) against oracle/stft_mel_oracle.py, element by element, through the C ABI.  Bars: those of BASELINE.json's north_star,
applied to the Mel energies S -- |dS| <= 1e-3 max_m S_ref(frame) and |d log10| <= 5e-3 where S_ref >= 1e-6 frame max -- plus the
tighter regression bars the compensated operands reach."""
import numpy as np
import pytest

import parity_util as pu
from oracle import stft_mel_oracle as so
from paper_2606_01009_b200 import workloads as wl

pytestmark = pytest.mark.gpu

# what the fp16x3 DFT product + bf16x3 filterbank product reach on these inputs (measured r02: 6e-6 / 2e-4), with head-room
S_REG_BAR, L_REG_BAR = 5e-5, 1.5e-3


def _gpu(c, x_host, pad=False, drop_last=False, layout="frame_major", shift=0, host=False):
    """x_host [B, len] -> [B, T, M] float64 through melt_plan_create_stft_mel + melt_forward (or melt_forward_host)."""
    import torch
    from paper_2606_01009_b200 import binding as mb
    plan = mb.melt_plan_create_stft_mel(c["fs"], c["n_fft"], c["hop"], c["window"], c["n_mels"], c["fmin"], c["fmax"])
    try:
        mb.melt_plan_set_option(plan, mb.MELT_OPT_LAYOUT, int(layout == "feature_major"))
        mb.melt_plan_set_option(plan, mb.MELT_OPT_PAD, int(pad))
        mb.melt_plan_set_option(plan, mb.MELT_OPT_DROP_LAST, int(drop_last))
        B, L = x_host.shape
        T, C = mb.melt_num_frames(plan, L), mb.melt_num_channels(plan)
        assert C == c["n_mels"]
        shape = (B, C, T) if layout == "feature_major" else (B, T, C)
        st = torch.cuda.current_stream().cuda_stream
        if host:
            xp = torch.from_numpy(np.ascontiguousarray(x_host, np.float32)).pin_memory()
            op = torch.full(shape, float("nan")).pin_memory()
            mb.melt_forward_host(plan, xp, B, L, op, st)
            torch.cuda.synchronize()
            res = op.numpy().copy()
        else:
            buf = torch.zeros(B * L + 8, device="cuda")
            x = buf[shift:shift + B * L].view(B, L)
            x.copy_(torch.from_numpy(np.ascontiguousarray(x_host, np.float32)))
            out = torch.full(shape, float("nan"), device="cuda")
            mb.melt_selftest_poison_smem(st)
            mb.melt_forward(plan, x, B, L, out, st)
            torch.cuda.synchronize()
            res = out.cpu().numpy()
        if layout == "feature_major":
            res = res.transpose(0, 2, 1)
        return res.astype(np.float64)
    finally:
        mb.melt_plan_destroy(plan)


def _check(c, x, **kw):
    pad, drop_last = kw.get("pad", False), kw.get("drop_last", False)
    L = _gpu(c, x, **kw)
    ref = so.forward_batch(x, want=("S", "L"), fs=c["fs"], n_fft=c["n_fft"], hop=c["hop"], window_kind=c["window"], n_mels=c["n_mels"],
                           fmin=c["fmin"], fmax=c["fmax"], pad=int(pad), drop_last=drop_last)
    assert L.shape == ref["L"].shape and np.isfinite(L).all()
    serr = pu.power_error(10.0 ** L, ref["S"])
    lerr = pu.log_error(L, ref["L"], ref["S"])
    assert serr <= pu.P_BAR["compensated"] and lerr <= pu.LOG_BAR, (serr, lerr)       # the north_star bars
    assert serr <= S_REG_BAR and lerr <= L_REG_BAR, (serr, lerr)                        # what this kernel reaches
    return serr, lerr


def _cfg(name, **over):
    c = dict(wl.CONFIGS[name])
    c.update(over)
    return c


def test_single_clip_frame_major():
    c = _cfg("cfg0")
    _check(c, wl.make_inputs("cfg0")["x"])


def test_whisper_shape_reflect_drop_last_feature_major_several_tiles():
    # three 30 s clips (3000 frames each: 11.7 tiles per clip, a ragged last tile), Whisper options: reflect padding, last frame dropped
    c = _cfg("cfg1")
    x = wl.make_inputs("cfg1", 3)["x_unpadded"]
    _check(c, x, pad=True, drop_last=True, layout="feature_major")


def test_speaker_shape_unaligned_buffer_and_odd_length():
    # 40 filters 20-7600 Hz; clip length not a multiple of 4 and a buffer one float past a 16-byte boundary: the realigning copy runs first
    c = _cfg("cfg3")
    rng = np.random.default_rng(7)
    x = wl.make_inputs("cfg1", 2)["x_unpadded"][:, :70001] + rng.normal(0, 0.01, (2, 70001)).astype(np.float32)
    _check(c, np.ascontiguousarray(x, np.float32), shift=1)


def test_symmetric_window_other_geometry_and_tones():
    # 256-point symmetric Hann, hop 64 (129 bins, 9 K-steps of the filterbank product), 64 filters; pure tones + noise floor: bins that
    # hold 1e-6 of the frame maximum must still meet the log bar
    c = dict(fs=8000.0, n_fft=256, hop=64, window=wl.WINDOW_HANN_SYMMETRIC, n_mels=64, fmin=50.0, fmax=3900.0)
    rng = np.random.default_rng(11)
    n = np.arange(40000)
    x = np.stack([0.4 * np.sin(2 * np.pi * 440.0 * n / 8000.0) + 0.05 * np.sin(2 * np.pi * 2500.0 * n / 8000.0) + rng.normal(0, 1e-3, n.size),
                  rng.normal(0, 0.2, n.size)]).astype(np.float32)
    _check(c, x)


def test_all_zero_input_hits_the_clamp_and_short_clips_are_noops():
    import torch
    from paper_2606_01009_b200 import binding as mb
    c = _cfg("cfg0")
    L = _gpu(c, np.zeros((2, 4000), np.float32))
    assert np.all(L == -10.0)
    plan = mb.melt_plan_create_stft_mel(c["fs"], c["n_fft"], c["hop"], c["window"], c["n_mels"], c["fmin"], c["fmax"])
    try:
        out = torch.full((8,), 7.0, device="cuda")
        mb.melt_forward(plan, torch.zeros(800, device="cuda"), 2, 399, out)     # shorter than a frame: T = 0
        mb.melt_forward(plan, torch.zeros(800, device="cuda"), 0, 400, out)     # empty batch
        torch.cuda.synchronize()
        assert torch.all(out == 7.0)
    finally:
        mb.melt_plan_destroy(plan)


def test_host_buffer_entry_point():
    c = _cfg("cfg0")
    x = wl.make_inputs("cfg1", 4)["x_unpadded"][:, :160000]
    a = _gpu(c, x, host=True)
    b = _gpu(c, x)
    assert np.array_equal(a, b)


def test_what_the_plan_does_not_cover_fails_loudly():
    import torch
    from paper_2606_01009_b200 import binding as mb
    with pytest.raises(mb.MeltError):
        mb.melt_plan_create_stft_mel(16000.0, 512, 160, 0, 80, 0.0, 8000.0)        # 257 bins: beyond tensor memory
    with pytest.raises(mb.MeltError):
        mb.melt_plan_create_stft_mel(16000.0, 400, 161, 0, 80, 0.0, 8000.0)        # hop % 4 != 0
    with pytest.raises(mb.MeltError):
        mb.melt_plan_create_stft_mel(16000.0, 400, 160, 0, 200, 0.0, 8000.0)       # more than 128 filters
    plan = mb.melt_plan_create_stft_mel(16000.0, 400, 160, 0, 80, 0.0, 8000.0)
    try:
        for key, val in ((mb.MELT_OPT_PRECISION, mb.MELT_PREC_TF32), (mb.MELT_OPT_OUTPUT, mb.MELT_OUTPUT_POWER),
                         (mb.MELT_OPT_OUTPUT_DTYPE, mb.MELT_DTYPE_F16)):
            with pytest.raises(mb.MeltError):
                mb.melt_plan_set_option(plan, key, val)
        x = torch.zeros(2000, device="cuda")
        off = torch.tensor([0, 1000, 2000], dtype=torch.int64, device="cuda")
        out = torch.zeros((16, 80), device="cuda")
        fo = torch.zeros(3, dtype=torch.int64, device="cuda")
        with pytest.raises(mb.MeltError):
            mb.melt_forward_ragged(plan, x, off, 2, out, fo)
        with pytest.raises(mb.MeltError):
            mb.melt_forward_ragged_noalloc(plan, x, off, 2, out, fo)
    finally:
        mb.melt_plan_destroy(plan)
