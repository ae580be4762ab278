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
# kernel rounds them, products summed in fp64): what is left is the tensor cores' fp32 accumulation, ~2^-24 of the larger
# terms of a sum.  Derivation: |dR| <~ 2^-23 sum_j |a_j b_j| <~ 1e-6 R_max, so |dS| / S_max <~ 4e-6 on
# the loudest bins; a bin at the mask floor (S = 1e-6 S_max, |R| = 1e-3 R_max) then has |dS| / S <~ 2e-3, |dlog10| <~ 1e-3.
ACC_P_BAR = 1e-5      # max |S_gpu - S_emul| / frame max
ACC_LOG_BAR = 1.5e-3  # max |L_gpu - log10(max(S_emul, 1e-10))| where S_ref >= 1e-6 frame max
EMUL_SCHEME = {"compensated": "f16x3", "tf32": "tf32", "bf16": "bf16"}


def plan_for(c, precision="compensated", layout=None, pad=None, drop_last=None, output="log", n_mfcc=None):
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
    return plan


def gpu_dense(c, x_host, precision="compensated", layout=None, pad=None, drop_last=None, output="log", n_mfcc=None,
              tap=False):
    """x_host [B, len] float32 -> numpy [B, T, C] (always returned frame-major, whatever layout was computed).
    With tap=True (MFCCT plans) returns (cepstra, logmel)."""
    import torch
    from paper_2606_01009_b200 import binding as mb
    plan = plan_for(c, precision, layout, pad, drop_last, output, n_mfcc)
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


def gpu_ragged(c, x_host, offsets, precision="compensated", tap=False):
    """Packed clips -> (out [sum T_i, C], frame_offsets [n+1]) (+ logmel with tap=True)."""
    import torch
    from paper_2606_01009_b200 import binding as mb
    plan = plan_for(c, precision, layout="frame_major")
    try:
        n = len(offsets) - 1
        lens = np.diff(offsets)
        total = int(sum(mb.melt_num_frames(plan, int(v)) for v in lens))
        C, M = mb.melt_num_channels(plan), c["n_mels"]
        x = torch.from_numpy(np.ascontiguousarray(x_host, np.float32)).cuda()
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


def oracle_kwargs(c, pad=None, drop_last=None, n_mfcc=None):
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
    return max(P_BAR[precision], 1.25 * perr_emul + ACC_P_BAR), max(LOG_BAR, 1.25 * lerr_emul + ACC_LOG_BAR)
