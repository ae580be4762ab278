"""Precision-emulation harness -- TEST INFRASTRUCTURE ONLY, like everything under oracle/.

What it answers: "what would the projection R, I (Eq. 3) and the power S (Eq. 4) come out as if the two
GEMM operands of Eq. (6) were first rounded to a tensor-core operand format and the products were then
summed EXACTLY?"  The operands are rounded on the CPU with numpy, the products are summed in fp64 (a BLAS dgemm: error
~1e-16 relative), so the result carries the operand-rounding error of a scheme and nothing else.  Two uses:

  * which scheme can meet which north-star bar at all (the table of SURVEY.md section 7 "hard part 1", reproduced by
    tests/test_precision_emulation.py) -- compare emulate(...) with the fp64 oracle;
  * an ASSERTING parity test for the single-pass TF32 / bf16 kernels: the CUDA result must equal the emulation of ITS OWN
    operand scheme up to fp32-accumulation noise, which is orders of magnitude below the operand-rounding noise, so a kernel
    that dropped a K-step or swapped two Mel rows cannot hide behind the loose north-star bar.

Two operand layouts are emulated:

  layout="direct"   the paper's Eq. (3)/(5) operands literally: frame samples x_t[n] and basis rows w[n] cos / sin(2 pi f_m n / fs),
                    n = 0..N-1, each rounded to the format.
  layout="folded"   the operands the CUDA kernels feed the tensor cores: the window is symmetric about
                    c = c2/2 (c2 = N periodic Hann, N-1 symmetric Hann / rectangle) and S does not depend on the phase origin,
                    so with the phase referred to c
                        R' = sum_j wc[m][j] (x[a0+j] + x[b0-j]),   I' = sum_j ws[m][j] (x[a0+j] - x[b0-j]),   j = 0..kf-1,
                        a0 = ceil(c2/2), b0 = floor(c2/2), kf = N - a0,
                        wc[m][j] = g_j w[a0+j] cos(w_m (a0+j-c)),  ws[m][j] = w[a0+j] sin(w_m (a0+j-c)),  g_j = 1/2 when a0+j == b0-j,
                    and R'^2 + I'^2 = R^2 + I^2.  The sums / differences are formed in fp32 (one rounding, as an fp32 add
                    does), THEN rounded to the operand format; the coefficients are rounded from fp64 in one step.

Schemes (operand formats):
  "exact"    no operand rounding at all (fp64 products of the fp32 samples): pins the algebra of the layout itself
  "tf32"     both operands to 10 explicit mantissa bits; samples round-to-nearest ties AWAY (cvt.rna.tf32.f32), basis ties-to-even
  "tf32_rz"  samples truncated to tf32 (what a raw fp32 feed of kind::tf32 does), basis ties-to-even
  "bf16"     both operands to bf16, ties-to-even
  "f16x3"    COMPENSATED: a = 2^s_in * sample term, b = 2^14 * coefficient; a_hi = f16(a), a_lo = f16(fl32(a - a_hi)),
             b_hi = f16(b), b_lo = f16(b - b_hi); R = (a_hi.b_hi + a_lo.b_hi + a_hi.b_lo) * 2^-(s_in+14)   (3 products)
  "bf16x3"   the same with bf16 parts and no scaling

Mel centres and the window come from the pinned fp64 oracle (oracle/melt_oracle.c); nothing here touches the CUDA package.
"""
import numpy as np

from . import melt_oracle as orc

SCHEMES = ("exact", "tf32", "tf32_rz", "bf16", "f16x3", "bf16x3")
BASIS_SCALE_LOG2 = 14   # COMPENSATED stores the basis as 2^14 * value


# ------------------------------------------------------------------------------------------------ rounding primitives
def round_f64_to_format(v, mant, emin):
    """Round float64 array v to a binary format with `mant` explicit mantissa bits and minimum normal exponent `emin`
    (gradual underflow), round-to-nearest-even, no overflow handling (callers stay in range).  One rounding, in fp64."""
    v = np.asarray(v, np.float64)
    m, e = np.frexp(v)                      # v = m * 2^e, 0.5 <= |m| < 1  ->  exponent of the leading bit is e - 1
    ex = np.maximum(e - 1, emin)
    q = np.ldexp(v, mant - ex)              # in units of the quantum 2^(ex - mant); exact
    return np.ldexp(np.rint(q), ex - mant)  # rint: ties to even


def f64_to_f16(v):
    return round_f64_to_format(v, 10, -14)


def f64_to_bf16(v):
    return round_f64_to_format(v, 7, -126)


def f64_to_tf32(v):
    return round_f64_to_format(v, 10, -126)


def f32_to_tf32_rna(x):
    """cvt.rna.tf32.f32: round an fp32 array to 10 explicit mantissa bits, nearest, ties away from zero (bit arithmetic on
    the sign-magnitude pattern)."""
    b = np.ascontiguousarray(x, np.float32).view(np.uint32)
    return ((b + np.uint32(0x1000)) & np.uint32(0xFFFFE000)).view(np.float32)


def f32_to_tf32_rz(x):
    b = np.ascontiguousarray(x, np.float32).view(np.uint32)
    return (b & np.uint32(0xFFFFE000)).view(np.float32)


def f32_to_bf16_rne(x):
    b = np.ascontiguousarray(x, np.float32).view(np.uint32)
    r = b + np.uint32(0x7FFF) + ((b >> np.uint32(16)) & np.uint32(1))
    return (r & np.uint32(0xFFFF0000)).view(np.float32)


def f32_to_f16_rne(x):
    return np.ascontiguousarray(x, np.float32).astype(np.float16).astype(np.float32)


# ------------------------------------------------------------------------------------------------ operand construction
def fold_geometry(n_fft, window_kind):
    c2 = n_fft if window_kind == orc.HANN_PERIODIC else n_fft - 1   # w[n] = w[c2 - n]
    a0, b0 = (c2 + 1) // 2, c2 // 2
    return c2, a0, b0, n_fft - a0


def basis_operands(fs, n_fft, window_kind, n_mels, fmin, fmax, layout):
    """fp64 coefficient matrices (Wc [M, K], Ws [M, K]) of the chosen layout (K = N direct, kf folded)."""
    f = orc.centres(fmin, fmax, n_mels)
    w = orc.window(window_kind, n_fft)
    if layout == "direct":
        n = np.arange(n_fft, dtype=np.float64)
        arg = 2.0 * np.pi * np.outer(f, n) / fs
        return w * np.cos(arg), w * np.sin(arg)
    c2, a0, b0, kf = fold_geometry(n_fft, window_kind)
    na = a0 + np.arange(kf)
    nb = b0 - np.arange(kf)
    g = np.where(na == nb, 0.5, 1.0)
    arg = 2.0 * np.pi * np.outer(f, na - 0.5 * c2) / fs
    return g * w[na] * np.cos(arg), w[na] * np.sin(arg)


def frame_operands(x, n_fft, hop, window_kind, layout, t0, t1, fold_dtype=np.float32):
    """Sample-side operands of frames [t0, t1) of the (already padded) clip x: direct -> (X, X) with X [T, N] fp32;
    folded -> (S, D) with S = x[a0+j] + x[b0-j], D = x[a0+j] - x[b0-j], formed in `fold_dtype`: fp32 = ONE fp32 rounding, as
    the kernels' fp32 add does; fp64 = exact (scheme "exact", which pins the algebra alone)."""
    x = np.ascontiguousarray(x, np.float32)
    t = np.arange(t0, t1)[:, None] * hop
    if layout == "direct":
        X = x[t + np.arange(n_fft)[None, :]]
        return X, X
    c2, a0, b0, kf = fold_geometry(n_fft, window_kind)
    j = np.arange(kf)[None, :]
    fw = x[t + a0 + j].astype(fold_dtype)
    nb = b0 - j
    bw = np.where(nb >= 0, x[t + np.maximum(nb, 0)], np.float32(0.0)).astype(fold_dtype)
    return fw + bw, fw - bw                      # float32 + float32: correctly rounded fp32 add / subtract


def _products(A, Bm, scheme, in_scale_log2):
    """Sum over K of the operand-rounded products, in fp64.  A [T, K] fp32 sample-side operand, Bm [M, K] fp64 coefficients."""
    if scheme == "exact":
        return A.astype(np.float64) @ Bm.T
    if scheme in ("tf32", "tf32_rz"):
        a = (f32_to_tf32_rna if scheme == "tf32" else f32_to_tf32_rz)(A).astype(np.float64)
        return a @ f64_to_tf32(Bm).T
    if scheme == "bf16":
        return f32_to_bf16_rne(A).astype(np.float64) @ f64_to_bf16(Bm).T
    if scheme == "f16x3":
        a = A * np.float32(2.0 ** in_scale_log2)                      # exact (power of two), stays fp32
        a_hi = f32_to_f16_rne(a)
        a_lo = f32_to_f16_rne(a - a_hi)                               # fp32 subtraction: exact here, then one rounding to f16
        b = Bm * 2.0 ** BASIS_SCALE_LOG2
        b_hi = f64_to_f16(b)
        b_lo = f64_to_f16(b - b_hi)
        a_hi, a_lo = a_hi.astype(np.float64), a_lo.astype(np.float64)
        return (a_hi @ b_hi.T + a_lo @ b_hi.T + a_hi @ b_lo.T) * 2.0 ** -(in_scale_log2 + BASIS_SCALE_LOG2)
    if scheme == "bf16x3":
        a_hi = f32_to_bf16_rne(A)
        a_lo = f32_to_bf16_rne(A - a_hi)
        b_hi = f64_to_bf16(Bm)
        b_lo = f64_to_bf16(Bm - b_hi)
        a_hi, a_lo = a_hi.astype(np.float64), a_lo.astype(np.float64)
        return a_hi @ b_hi.T + a_lo @ b_hi.T + a_hi @ b_lo.T
    raise ValueError(scheme)


def emulate_power(x, fs, n_fft, hop, window_kind, n_mels, fmin, fmax, scheme, layout="folded", pad=orc.PAD_NONE,
                  drop_last=False, in_scale_log2=12, block=8192):
    """One clip x (1-D fp32) -> S [T, M] float64 under operand scheme `scheme` and operand layout `layout`, products
    summed in fp64.  Framing / padding follow the oracle (oracle.num_frames; numpy reflect semantics)."""
    x = np.ascontiguousarray(x, np.float32)
    T = orc.num_frames(x.shape[0], n_fft, hop, pad, drop_last)
    if pad == orc.PAD_REFLECT and T > 0:
        x = np.pad(x, n_fft // 2, mode="reflect")
    Wc, Ws = basis_operands(fs, n_fft, window_kind, n_mels, fmin, fmax, layout)
    out = np.empty((T, n_mels), np.float64)
    for t0 in range(0, T, block):
        t1 = min(T, t0 + block)
        Ac, As = frame_operands(x, n_fft, hop, window_kind, layout, t0, t1, np.float64 if scheme == "exact" else np.float32)
        R = _products(Ac, Wc, scheme, in_scale_log2)
        I = _products(As, Ws, scheme, in_scale_log2)
        out[t0:t1] = R * R + I * I
    return out


def emulate_power_batch(x, **kw):
    """Dense batch [B, len] -> [B, T, M]."""
    x = np.ascontiguousarray(x, np.float32)
    return np.stack([emulate_power(x[b], **kw) for b in range(x.shape[0])])


def log_mel(S):
    """Contract form of Eq. (8): log10(max(S, 1e-10)) (BASELINE.json north_star; reading R2)."""
    return np.log10(np.maximum(S, 1e-10))
