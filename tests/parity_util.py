"""Shared helpers of the GPU parity tests: run the CUDA path through the C ABI, run the fp64 oracle on the same
bytes, and evaluate the north-star criteria (BASELINE.json north_star):

    P bar    max |P_gpu - P_ref| / max_k P_ref(frame)      <= 1e-3 (TF32 path), 3e-2 (bf16 path)
    log bar  max |L_gpu - L_ref| where P_ref >= 1e-6 * max_k P_ref(frame)      <= 5e-3
"""
import numpy as np

P_BAR = {"compensated": 1e-3, "tf32": 1e-3, "bf16": 3e-2}
LOG_BAR = 5e-3
MASK_FLOOR = 1e-6

# CUDA result against the CPU emulation of ITS OWN operand scheme (oracle/melt_emul.py: operands rounded exactly as the
# kernel rounds them, products summed in fp64): what is left is the tensor cores' fp32 accumulation in tensor memory.  That
# accumulation is not a correctly rounded sum: the 16 (8 for tf32) products of one tcgen05.mma are aligned to the largest
# exponent and TRUNCATED, and so is every addition into the accumulator, so the error is biased and grows with the number n of
# MMAs that feed one accumulator (n = K-steps x 3 products in COMPENSATED mode).  Measured on B200 over every config, mode
# and odd geometry of this suite (r02): max |dS| / S_max 1.1e-6 .. 1.6e-5 for n <= 48 (all 400-sample windows), 1.3e-5 .. 1.1e-4
# for n up to 384 (1024 .. 4096-sample windows); |dlog10| inside the mask <= 7.1e-4 everywhere.  The bars sit just above that
# and 5x .. 50x below the north-star bars; a dropped K-step or swapped Mel rows move S by >= 1e-2 S_max.
ACC_LOG_BAR = 1.5e-3  # max |L_gpu - log10(max(S_emul, 1e-10))| where S_ref >= 1e-6 frame max


def acc_p_bar(c, precision):
    """max |S_gpu - S_emul| / frame max allowed for the fp32 accumulation of config c in mode `precision` (see above)."""
    c2 = c["n_fft"] if c["window"] == 0 else c["n_fft"] - 1
    kf = c["n_fft"] - (c2 + 1) // 2
    kstep = 8 if precision == "tf32" else 16
    n_acc = -(-kf // kstep) * (3 if precision == "compensated" else 1)
    return 2e-5 if n_acc <= 48 else 2e-4


EMUL_SCHEME = {"compensated": "f16x3", "tf32": "tf32", "bf16": "bf16"}


def plan_for(c, precision="compensated", layout=None, pad=None, drop_last=None, output="log", n_mfcc=None, input_ready=False):
    """Create a plan for config dict c (workloads.CONFIGS entry or look-alike) with the given options."""
    from paper_2606_01009_b200 import binding as mb
    prec = {"compensated": mb.MELT_PREC_COMPENSATED, "tf32": mb.MELT_PREC_TF32, "bf16": mb.MELT_PREC_BF16}[precision]
    k = c["n_mfcc"] if n_mfcc is None else n_mfcc
    plan = mb.melt_plan_create(c["fs"], c["n_fft"], c["hop"], c["window"], c["n_mels"], c["fmin"], c["fmax"], 0, k)
    mb.melt_plan_set_option(plan, mb.MELT_OPT_PRECISION, prec)
    lay = c.get("layout", "frame_major") if layout is None else layout
    mb.melt_plan_set_option(plan, mb.MELT_OPT_LAYOUT, int(lay == "feature_major"))
    mb.melt_plan_set_option(plan, mb.MELT_OPT_DROP_LAST, int(c.get("drop_last", False) if drop_last is None else drop_last))
    mb.melt_plan_set_option(plan, mb.MELT_OPT_PAD, int(bool(pad)))
    if output == "power":
        mb.melt_plan_set_option(plan, mb.MELT_OPT_OUTPUT, mb.MELT_OUTPUT_POWER)
    if output == "whisper":
        mb.melt_plan_set_option(plan, mb.MELT_OPT_OUTPUT, mb.MELT_OUTPUT_LOG_WHISPER)
    if output == "ln":
        mb.melt_plan_set_option(plan, mb.MELT_OPT_OUTPUT, mb.MELT_OUTPUT_LN_EPS)
    if input_ready:
        mb.melt_plan_set_option(plan, mb.MELT_OPT_INPUT_READY, 1)
    return plan


def gpu_dense(c, x_host, precision="compensated", layout=None, pad=None, drop_last=None, output="log", n_mfcc=None,
              tap=False, input_ready=False):
    """x_host [B, len] float32 -> numpy [B, T, C] (always returned frame-major, whatever layout was computed).
    With tap=True (MFCCT plans) returns (cepstra, logmel)."""
    import torch
    from paper_2606_01009_b200 import binding as mb
    plan = plan_for(c, precision, layout, pad, drop_last, output, n_mfcc, input_ready)
    try:
        lay = c.get("layout", "frame_major") if layout is None else layout
        x = torch.from_numpy(np.ascontiguousarray(x_host, np.float32)).cuda()
        B, L = x.shape
        T, C, M = mb.melt_num_frames(plan, L), mb.melt_num_channels(plan), c["n_mels"]
        shape = (B, C, T) if lay == "feature_major" else (B, T, C)
        out = torch.full(shape, float("nan"), device="cuda")
        stream = torch.cuda.current_stream().cuda_stream
        mb.melt_selftest_poison_smem(stream)   # the forward must not depend on what is left in shared memory
        if tap:
            tshape = (B, M, T) if lay == "feature_major" else (B, T, M)
            lm = torch.full(tshape, float("nan"), device="cuda")
            mb.melt_forward_tap(plan, x, None, B, L, out, lm, None, stream)
        else:
            mb.melt_forward(plan, x, B, L, out, stream)
        torch.cuda.synchronize()
        res = out.cpu().numpy()
        if lay == "feature_major":
            res = res.transpose(0, 2, 1)
        if tap:
            lmh = lm.cpu().numpy()
            if lay == "feature_major":
                lmh = lmh.transpose(0, 2, 1)
            return res.astype(np.float64), lmh.astype(np.float64)
        return res.astype(np.float64)
    finally:
        mb.melt_plan_destroy(plan)


def gpu_ragged(c, x_host, offsets, precision="compensated", tap=False, pad=None, shift=0):
    """Packed clips -> (out [sum T_i, C], frame_offsets [n+1]) (+ logmel with tap=True).  shift: the device buffer starts
    `shift` floats past a 16-byte boundary (an unaligned packed batch)."""
    import torch
    from paper_2606_01009_b200 import binding as mb
    plan = plan_for(c, precision, layout="frame_major", pad=pad)
    try:
        n = len(offsets) - 1
        lens = np.diff(offsets)
        total = int(sum(mb.melt_num_frames(plan, int(v)) for v in lens))
        C, M = mb.melt_num_channels(plan), c["n_mels"]
        xbuf = torch.zeros(len(x_host) + 8, device="cuda")
        x = xbuf[shift:shift + len(x_host)]
        x.copy_(torch.from_numpy(np.ascontiguousarray(x_host, np.float32)))
        assert x.data_ptr() % 16 == 4 * (shift % 4)
        off = torch.from_numpy(np.ascontiguousarray(offsets, np.int64)).cuda()
        out = torch.full((max(total, 1), C), float("nan"), device="cuda")
        fo = torch.full((n + 1,), -1, dtype=torch.int64, device="cuda")
        stream = torch.cuda.current_stream().cuda_stream
        mb.melt_selftest_poison_smem(stream)   # the forward must not depend on what is left in shared memory
        lm = None
        if tap:
            lm = torch.full((max(total, 1), M), float("nan"), device="cuda")
            mb.melt_forward_tap(plan, x, off, n, 0, out, lm, fo, stream)
        else:
            mb.melt_forward_ragged(plan, x, off, n, out, fo, stream)
        torch.cuda.synchronize()
        res = (out.cpu().numpy()[:total].astype(np.float64), fo.cpu().numpy())
        if tap:
            res = res + (lm.cpu().numpy()[:total].astype(np.float64),)
        return res
    finally:
        mb.melt_plan_destroy(plan)


def oracle_kwargs(c, pad=None, drop_last=None, n_mfcc=None):  # noqa: D103
    return dict(fs=c["fs"], n_fft=c["n_fft"], hop=c["hop"], window_kind=c["window"], n_mels=c["n_mels"], fmin=c["fmin"],
                fmax=c["fmax"], n_mfcc=c["n_mfcc"] if n_mfcc is None else n_mfcc, pad=int(bool(pad)),
                drop_last=bool(c.get("drop_last", False) if drop_last is None else drop_last))


def power_error(P_gpu, P_ref):
    """max over elements of |dP| / frame max of P_ref (frames whose reference is all zero compare absolutely)."""
    fmax = P_ref.max(axis=-1, keepdims=True)
    denom = np.where(fmax > 0, fmax, 1.0)
    return float((np.abs(P_gpu - P_ref) / denom).max()) if P_ref.size else 0.0


def log_error(L_gpu, L_ref, P_ref):
    """max |dL| over the elements with P_ref >= 1e-6 * frame max (all elements of an all-zero frame)."""
    fmax = P_ref.max(axis=-1, keepdims=True)
    mask = P_ref >= MASK_FLOOR * fmax
    if not mask.any():
        return 0.0
    return float(np.abs(L_gpu - L_ref)[mask].max())


def emulated_power(c, x, precision, pad=None, drop_last=None):
    """S [B, T, M] of the dense batch x under the operand scheme of `precision` in the kernels' folded operand layout, products
    summed in fp64 on the CPU (oracle/melt_emul.py)."""
    from oracle import melt_emul as em
    return em.emulate_power_batch(x, fs=c["fs"], n_fft=c["n_fft"], hop=c["hop"], window_kind=c["window"], n_mels=c["n_mels"],
                                  fmin=c["fmin"], fmax=c["fmax"], scheme=EMUL_SCHEME[precision], layout="folded",
                                  pad=int(bool(pad)), drop_last=bool(c.get("drop_last", False) if drop_last is None else drop_last))


def single_pass_bars(precision, perr_emul, lerr_emul):
    """Bars of a CUDA result against the ORACLE for a mode whose operand rounding alone (emulated error perr_emul /
    lerr_emul against the oracle, exact summation) may exceed the north-star bar: the north-star bar where the arithmetic
    meets it, otherwise 1.25 x what the arithmetic gives plus the accumulation allowance -- never unbounded."""
    return max(P_BAR[precision], 1.25 * perr_emul + 2e-4), max(LOG_BAR, 1.25 * lerr_emul + ACC_LOG_BAR)
