"""ctypes front end to oracle/melt_oracle.c (fp64 CPU oracle) -- TEST INFRASTRUCTURE ONLY.

Argument marshalling and layout only: every number comes out of melt_oracle.c, which states the
method's definition (Eq. 1-9) in double precision.  Nothing here imports the CUDA package.
"""
import ctypes as C
import numpy as np

from . import build as _build

HANN_PERIODIC, HANN_SYMMETRIC, RECT = 0, 1, 2
PAD_NONE, PAD_REFLECT = 0, 1

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        dp = C.POINTER(C.c_double)
        L.melt_oracle_num_threads.restype = C.c_int
        L.melt_oracle_hz_to_mel.restype = C.c_double
        L.melt_oracle_hz_to_mel.argtypes = [C.c_double]
        L.melt_oracle_mel_to_hz.restype = C.c_double
        L.melt_oracle_mel_to_hz.argtypes = [C.c_double]
        L.melt_oracle_centres.argtypes = [C.c_double, C.c_double, C.c_int, dp]
        L.melt_oracle_window.argtypes = [C.c_int, C.c_int, dp]
        L.melt_oracle_basis.argtypes = [C.c_double, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, dp, dp]
        L.melt_oracle_dct.argtypes = [C.c_int, C.c_int, dp]
        L.melt_oracle_num_frames.restype = C.c_longlong
        L.melt_oracle_num_frames.argtypes = [C.c_longlong, C.c_int, C.c_int, C.c_int, C.c_int]
        L.melt_oracle_forward.argtypes = [C.POINTER(C.c_float), C.c_longlong, C.c_double, C.c_int, C.c_int,
                                          C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, C.c_int, C.c_int,
                                          dp, dp, dp, dp, dp]
        L.melt_oracle_dct_apply.argtypes = [dp, C.c_longlong, C.c_int, C.c_int, dp]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def num_threads():
    return int(lib().melt_oracle_num_threads())


def hz_to_mel(f):
    return float(lib().melt_oracle_hz_to_mel(float(f)))


def mel_to_hz(mu):
    return float(lib().melt_oracle_mel_to_hz(float(mu)))


def centres(fmin, fmax, n_mels):
    f = np.empty(n_mels, np.float64)
    rc = lib().melt_oracle_centres(float(fmin), float(fmax), int(n_mels), _dp(f))
    if rc:
        raise ValueError("melt_oracle_centres rc=%d" % rc)
    return f


def window(kind, n_fft):
    w = np.empty(n_fft, np.float64)
    rc = lib().melt_oracle_window(int(kind), int(n_fft), _dp(w))
    if rc:
        raise ValueError("melt_oracle_window rc=%d" % rc)
    return w


def basis(fs, n_fft, window_kind, n_mels, fmin, fmax):
    Wr = np.empty((n_mels, n_fft), np.float64)
    Wi = np.empty((n_mels, n_fft), np.float64)
    rc = lib().melt_oracle_basis(float(fs), int(n_fft), int(window_kind), int(n_mels), float(fmin), float(fmax),
                                 _dp(Wr), _dp(Wi))
    if rc:
        raise ValueError("melt_oracle_basis rc=%d" % rc)
    return Wr, Wi


def dct_matrix(n_mfcc, n_mels):
    D = np.empty((n_mfcc, n_mels), np.float64)
    rc = lib().melt_oracle_dct(int(n_mfcc), int(n_mels), _dp(D))
    if rc:
        raise ValueError("melt_oracle_dct rc=%d" % rc)
    return D


def num_frames(length, n_fft, hop, pad=PAD_NONE, drop_last=False):
    return int(lib().melt_oracle_num_frames(int(length), int(n_fft), int(hop), int(pad), int(bool(drop_last))))


def forward(x, fs, n_fft, hop, window_kind, n_mels, fmin, fmax, n_mfcc=0, pad=PAD_NONE, drop_last=False,
            want=("P", "L", "C")):
    """One clip.  x: 1-D float32.  Returns dict of frame-major float64 arrays among R, I, P, L [T, M], C [T, K]."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    assert x.ndim == 1
    T = num_frames(x.shape[0], n_fft, hop, pad, drop_last)
    out = {}
    for k in ("R", "I", "P", "L"):
        out[k] = np.empty((T, n_mels), np.float64) if k in want else None
    out["C"] = np.empty((T, n_mfcc), np.float64) if (n_mfcc and "C" in want) else None
    rc = lib().melt_oracle_forward(x.ctypes.data_as(C.POINTER(C.c_float)), x.shape[0], float(fs), int(n_fft),
                                   int(hop), int(window_kind), int(n_mels), float(fmin), float(fmax), int(n_mfcc),
                                   int(pad), int(bool(drop_last)),
                                   _dp(out["R"]), _dp(out["I"]), _dp(out["P"]), _dp(out["L"]), _dp(out["C"]))
    if rc:
        raise ValueError("melt_oracle_forward rc=%d" % rc)
    return {k: v for k, v in out.items() if v is not None}


def forward_batch(x, **kw):
    """Dense batch x [B, len] -> dict of [B, T, .] arrays (frame-major per clip)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    assert x.ndim == 2
    outs = [forward(x[b], **kw) for b in range(x.shape[0])]
    return {k: np.stack([o[k] for o in outs]) for k in outs[0]} if outs else {}


def forward_ragged(x, offsets, **kw):
    """Packed clips x [sum len_i] with offsets [n+1] -> dict of packed [sum T_i, .] arrays + 'frame_offsets'."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    offsets = np.asarray(offsets, dtype=np.int64)
    outs = [forward(x[offsets[i]:offsets[i + 1]], **kw) for i in range(len(offsets) - 1)]
    keys = outs[0].keys() if outs else ()
    res = {k: np.concatenate([o[k] for o in outs], axis=0) for k in keys}
    fo = np.zeros(len(offsets), np.int64)
    if outs:
        k0 = next(iter(keys))
        fo[1:] = np.cumsum([o[k0].shape[0] for o in outs])
    res["frame_offsets"] = fo
    return res


def dct_apply(Lmat, n_mfcc):
    """Eq. (9) alone: Lmat [T, M] float64 -> [T, K]."""
    Lmat = np.ascontiguousarray(Lmat, dtype=np.float64)
    T, M = Lmat.shape
    Cout = np.empty((T, n_mfcc), np.float64)
    rc = lib().melt_oracle_dct_apply(_dp(Lmat), T, M, int(n_mfcc), _dp(Cout))
    if rc:
        raise ValueError("melt_oracle_dct_apply rc=%d" % rc)
    return Cout


def ln_eps(P, eps=1e-10):
    """Eq. (8) as printed: ln(S + eps), natural logarithm (PAPER.md:343 measures in nats), from the oracle's fp64
    S.  The paper does not state eps (reading R2); the CUDA path's default is 1e-10."""
    return np.log(np.asarray(P, np.float64) + float(eps))


def whisper_norm(L):
    """Whisper's dynamic-range normalisation of one clip's log10-Mel matrix L [T, M] (any layout: only the clip maximum enters):
    L <- max(L, max(L) - 8), then (L + 4) / 4 (PAPER.md:424 configures MelT to Whisper's log-Mel specification)."""
    L = np.asarray(L, np.float64)
    return (np.maximum(L, L.max() - 8.0) + 4.0) / 4.0
