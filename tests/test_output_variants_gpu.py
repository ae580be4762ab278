"""GPU parity of the output variants of SURVEY.md section 8(f) NEXT-3: 16-bit feature output (fp16 / bf16) and the paper's own
log form ln(S + eps) (Eq. 8), with and without the DCT, against the fp64 oracle."""
import numpy as np
import pytest

import parity_util as pu

pytestmark = pytest.mark.gpu


def _wl():
    from paper_2606_01009_b200 import workloads
    return workloads


def _orc():
    from oracle import melt_oracle
    return melt_oracle


def _run16(c, x, dtype, layout, offsets=None):
    """log-Mel of a dense batch (or a packed one) with a 16-bit output buffer -> float64 [B, T, C] / [sum T, C]."""
    import torch
    from paper_2606_01009_b200 import binding as mb
    tdt = torch.float16 if dtype == "f16" else torch.bfloat16
    plan = pu.plan_for(c, "compensated", layout=layout)
    try:
        mb.melt_plan_set_option(plan, mb.MELT_OPT_OUTPUT_DTYPE, mb.MELT_DTYPE_F16 if dtype == "f16" else mb.MELT_DTYPE_BF16)
        xd = torch.from_numpy(np.ascontiguousarray(x, np.float32)).cuda()
        C = mb.melt_num_channels(plan)
        st = torch.cuda.current_stream().cuda_stream
        if offsets is None:
            B, L = x.shape
            T = mb.melt_num_frames(plan, L)
            out = torch.full((B, C, T) if layout == "feature_major" else (B, T, C), float("nan"), dtype=tdt, device="cuda")
            mb.melt_forward(plan, xd, B, L, out, st)
            torch.cuda.synchronize()
            res = out.float().cpu().numpy().astype(np.float64)
            return res.transpose(0, 2, 1) if layout == "feature_major" else res
        n = len(offsets) - 1
        total = int(sum(mb.melt_num_frames(plan, int(v)) for v in np.diff(offsets)))
        out = torch.full((total, C), float("nan"), dtype=tdt, device="cuda")
        fo = torch.empty(n + 1, dtype=torch.int64, device="cuda")
        mb.melt_forward_ragged(plan, xd, torch.from_numpy(np.ascontiguousarray(offsets, np.int64)).cuda(), n, out, fo, st)
        torch.cuda.synchronize()
        return out.float().cpu().numpy().astype(np.float64)
    finally:
        mb.melt_plan_destroy(plan)


@pytest.mark.parametrize("dtype", ["f16", "bf16"])
@pytest.mark.parametrize("layout", ["feature_major", "frame_major"])
def test_sixteen_bit_log_mel_output_on_the_whisper_shape(dtype, layout):
    """The stored value is the fp32 log-Mel rounded once to the 16-bit type: against the oracle |dL| <= north-star bar (5e-3) + half an
    ulp of the type at |L| (fp16: 2^-11 |L| <= 3.9e-3 for |L| < 16, so fp16 output meets the 5e-3 bar on its own up to |L| ~ 2)."""
    c = dict(_wl().CONFIGS["cfg1"]); c["name"] = "cfg1"
    x = _wl().make_inputs("cfg1", 3)["x"]
    L16 = _run16(c, x, dtype, layout)
    ref = _orc().forward_batch(x, want=("P", "L"), **pu.oracle_kwargs(c))
    assert L16.shape == ref["L"].shape and np.isfinite(L16).all()
    half_ulp = 2.0 ** (-11 if dtype == "f16" else -8)
    fmax = ref["P"].max(axis=-1, keepdims=True)
    mask = ref["P"] >= pu.MASK_FLOOR * fmax
    excess = np.abs(L16 - ref["L"]) - half_ulp * np.abs(ref["L"]) * 1.001
    assert excess[mask].max() <= pu.LOG_BAR
    assert np.all(L16[ref["L"] == -10.0] == -10.0)             # the clamp value is exact in both types
    # and it is exactly the fp32 output rounded to the type
    import torch
    L32 = pu.gpu_dense(c, x, "compensated", layout=layout)
    t = torch.from_numpy(L32.astype(np.float32))
    want = t.to(torch.float16 if dtype == "f16" else torch.bfloat16).float().numpy().astype(np.float64)
    np.testing.assert_array_equal(L16, want)


def test_sixteen_bit_output_on_a_packed_batch_and_its_restrictions():
    import torch
    from paper_2606_01009_b200 import binding as mb
    c = dict(name="ragged16", fs=16000.0, n_fft=400, hop=160, window=0, n_mels=80, fmin=0.0, fmax=8000.0, n_mfcc=0, layout="frame_major")
    rng = np.random.default_rng(3)
    lens = [5000, 399, 48001, 16000, 70003]
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    x = rng.normal(0, 0.1, int(off[-1])).astype(np.float32)
    got = _run16(c, x, "f16", "frame_major", offsets=off)
    L32, _ = pu.gpu_ragged(c, x, off)
    want = torch.from_numpy(L32.astype(np.float32)).to(torch.float16).float().numpy().astype(np.float64)
    np.testing.assert_array_equal(got, want)
    # MFCCT / power / tap outputs stay fp32: the combination is refused, not silently ignored
    c3 = dict(_wl().CONFIGS["cfg3"])
    plan = pu.plan_for(c3, layout="frame_major")
    try:
        mb.melt_plan_set_option(plan, mb.MELT_OPT_OUTPUT_DTYPE, mb.MELT_DTYPE_F16)
        xd = torch.zeros(16000, device="cuda")
        out = torch.zeros(98 * 13, dtype=torch.float16, device="cuda")
        with pytest.raises(mb.MeltError) as ei:
            mb.melt_forward(plan, xd, 1, 16000, out)
        assert ei.value.status == mb.MELT_ERR_UNSUPPORTED
    finally:
        mb.melt_plan_destroy(plan)


@pytest.mark.parametrize("cfg", ["cfg0", "cfg1"])
def test_paper_form_ln_s_plus_eps(cfg):
    """Eq. (8) as printed: ln(S + eps), eps = 1e-10.  Error model: d ln(S + eps) = dS / (S + eps); inside the mask the north-star log
    bar in nats is 5e-3 ln 10 = 1.15e-2 (compensated mode measures ~3e-4)."""
    c = dict(_wl().CONFIGS[cfg]); c["name"] = cfg
    x = _wl().make_inputs(cfg, 2 if cfg == "cfg1" else None)["x"]
    got = pu.gpu_dense(c, x, "compensated", output="ln")
    ref = _orc().forward_batch(x, want=("P",), **pu.oracle_kwargs(c))
    want = _orc().ln_eps(ref["P"], 1e-10)
    assert got.shape == want.shape and np.isfinite(got).all()
    fmax = ref["P"].max(axis=-1, keepdims=True)
    mask = ref["P"] >= pu.MASK_FLOOR * fmax
    assert np.abs(got - want)[mask].max() <= pu.LOG_BAR * np.log(10.0)
    silent = ref["P"] == 0.0
    if silent.any():
        np.testing.assert_allclose(got[silent], np.log(1e-10), atol=1e-5)


def test_paper_form_mfcct_is_the_dct_of_ln():
    """MFCCT as the paper prints it (Eq. 9 on Eq. 8): C = ln(S + eps) D^T -- two-stage bars of DESIGN.md reading R9 with the tap in nats."""
    orc = _orc()
    c = dict(_wl().CONFIGS["cfg3"]); c["name"] = "cfg3-ln"
    rng = np.random.default_rng(11)
    x = rng.normal(0, 0.1, (2, 400 + 300 * 160)).astype(np.float32)
    C_gpu, L_gpu = pu.gpu_dense(c, x, "compensated", layout="frame_major", output="ln", tap=True)
    ref = orc.forward_batch(x, want=("P",), **pu.oracle_kwargs(c))
    Lref = orc.ln_eps(ref["P"], 1e-10)
    fmax = ref["P"].max(axis=-1, keepdims=True)
    mask = ref["P"] >= pu.MASK_FLOOR * fmax
    assert np.abs(L_gpu - Lref)[mask].max() <= pu.LOG_BAR * np.log(10.0)
    for b in range(2):
        assert np.abs(C_gpu[b] - orc.dct_apply(L_gpu[b], 13)).max() <= 2e-4


@pytest.mark.parametrize("layout", ["feature_major", "frame_major"])
def test_whisper_dynamic_range_normalisation(layout):
    """MELT_OUTPUT_LOG_WHISPER: per clip L <- (max(L, max_clip(L) - 8) + 4) / 4 on top of the contract log10 form.  The clip maximum is a
    loud bin (error ~1e-4), so inside the log mask the error is the log error / 4; below the clamp both sides sit on the floor."""
    orc = _orc()
    c = dict(_wl().CONFIGS["cfg1"]); c["name"] = "cfg1"
    x = _wl().make_inputs("cfg1", 3)["x"]
    x[1] *= 1e-3                                            # a quiet clip: its own maximum sets its own floor
    got = pu.gpu_dense(c, x, "compensated", layout=layout, output="whisper")
    ref = orc.forward_batch(x, want=("P", "L"), **pu.oracle_kwargs(c))
    want = np.stack([orc.whisper_norm(ref["L"][b]) for b in range(3)])
    assert got.shape == want.shape and np.isfinite(got).all()
    fmax = ref["P"].max(axis=-1, keepdims=True)
    mask = ref["P"] >= pu.MASK_FLOOR * fmax
    assert np.abs(got - want)[mask].max() <= pu.LOG_BAR / 4 + 1e-6
    for b in range(3):                                      # the floor itself: (max(max_clip - 8, -10) + 4) / 4 (-10: the log10 clamp)
        floor = (max(ref["L"][b].max() - 8.0, -10.0) + 4.0) / 4.0
        assert abs(got[b].min() - floor) <= 1e-3 and got[b].max() <= (ref["L"][b].max() + 4.0) / 4.0 + 1e-3
