"""Thin ctypes binding over libmelt_b200.so -- same names as the C calls in include/melt.h.

Argument marshalling only: every step of the path (framing, projection, power, log, DCT, store) runs in the
CUDA kernels behind the C ABI.  PyTorch is used by callers for device memory and streams only; this module
takes raw device pointers (ints) or torch tensors (``.data_ptr()``).  There is no CPU fallback: if the library
cannot be loaded the import of a symbol raises.
"""
import ctypes as C
import os

from . import build as _build

MELT_OK, MELT_ERR_INVALID_ARG, MELT_ERR_UNSUPPORTED, MELT_ERR_ALIGNMENT, MELT_ERR_CUDA, MELT_ERR_ALLOC = range(6)
MELT_WINDOW_HANN_PERIODIC, MELT_WINDOW_HANN_SYMMETRIC, MELT_WINDOW_RECT = 0, 1, 2
MELT_MEL_HTK, MELT_MEL_SLANEY = 0, 1
MELT_OPT_LAYOUT, MELT_OPT_PRECISION, MELT_OPT_DROP_LAST, MELT_OPT_PAD, MELT_OPT_INPUT_SCALE_LOG2, MELT_OPT_OUTPUT, \
    MELT_OPT_INPUT_READY, MELT_OPT_OUTPUT_DTYPE, MELT_OPT_LOG_EPS_EXP10 = range(9)
MELT_LAYOUT_FRAME_MAJOR, MELT_LAYOUT_FEATURE_MAJOR = 0, 1
MELT_PREC_COMPENSATED, MELT_PREC_TF32, MELT_PREC_BF16 = 0, 1, 2
MELT_PAD_NONE, MELT_PAD_REFLECT = 0, 1
MELT_OUTPUT_LOG, MELT_OUTPUT_POWER, MELT_OUTPUT_LN_EPS, MELT_OUTPUT_LOG_WHISPER = 0, 1, 2, 3
MELT_DTYPE_F32, MELT_DTYPE_F16, MELT_DTYPE_BF16 = 0, 1, 2

# every symbol include/melt.h declares (tests/test_abi.py checks the header against this list and the .so) ...
SYMBOLS = [
    "melt_plan_create", "melt_plan_create_stft_mel", "melt_plan_destroy", "melt_plan_set_option", "melt_num_frames", "melt_count_frames", "melt_num_channels",
    "melt_plan_reserve", "melt_plan_get_centres", "melt_forward", "melt_forward_host", "melt_forward_ragged",
    "melt_forward_ragged_noalloc", "melt_forward_tap", "melt_last_error", "melt_plan_describe",
]
# ... and the test aids of include/melt_test.h (not part of the product API)
TEST_SYMBOLS = ["melt_selftest_umma", "melt_selftest_umma2", "melt_selftest_poison_smem"]

_lib = None


class MeltError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("melt status %d: %s" % (status, msg))
        self.status = status


def library_path():
    return _build.LIB


def lib():
    """Load (building first if the sources are newer) libmelt_b200.so.  Raises if it cannot be had."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if not os.path.exists(path) or _build._stale():
        path = _build.build()
    _lib = load(path)
    return _lib


def load(path):
    """ctypes handle of a library build at `path` with every prototype declared (lib() uses it for the product library; tests
    load variant builds next to it)."""
    L = C.CDLL(path)
    vp, ip, ll, dbl = C.c_void_p, C.c_int, C.c_longlong, C.c_double
    L.melt_plan_create.restype = vp
    L.melt_plan_create.argtypes = [dbl, ip, ip, ip, ip, dbl, dbl, ip, ip]
    L.melt_plan_create_stft_mel.restype = vp
    L.melt_plan_create_stft_mel.argtypes = [dbl, ip, ip, ip, ip, dbl, dbl]
    L.melt_plan_destroy.restype = None
    L.melt_plan_destroy.argtypes = [vp]
    L.melt_plan_set_option.argtypes = [vp, ip, ip]
    L.melt_num_frames.restype = ll
    L.melt_num_frames.argtypes = [vp, ll]
    L.melt_count_frames.restype = ll
    L.melt_count_frames.argtypes = [ll, ip, ip, ip, ip]
    L.melt_plan_reserve.argtypes = [vp, C.c_ulonglong]
    L.melt_num_channels.argtypes = [vp]
    L.melt_plan_get_centres.argtypes = [vp, C.POINTER(dbl)]
    L.melt_forward.argtypes = [vp, vp, ip, ll, vp, vp]
    L.melt_forward_ragged.argtypes = [vp, vp, vp, ip, vp, vp, vp]
    L.melt_forward_ragged_noalloc.argtypes = [vp, vp, vp, ip, vp, vp, vp]
    L.melt_forward_host.argtypes = [vp, vp, ip, ll, vp, vp]
    L.melt_forward_tap.argtypes = [vp, vp, vp, ip, ll, vp, vp, vp, vp]
    L.melt_last_error.restype = C.c_char_p
    L.melt_plan_describe.restype = C.c_char_p
    L.melt_plan_describe.argtypes = [vp]
    L.melt_selftest_umma.argtypes = [ip, ip, ip, vp, vp, vp]
    L.melt_selftest_umma2.argtypes = [ip, ip, ip, vp, vp, vp]
    L.melt_selftest_poison_smem.argtypes = [vp]
    return L


def _ptr(t):
    if t is None:
        return None
    if isinstance(t, int):
        return t
    return int(t.data_ptr())


def _check(rc):
    if rc != MELT_OK:
        raise MeltError(rc, melt_last_error())


def melt_last_error():
    return lib().melt_last_error().decode()


def melt_plan_create(fs, n_fft, hop, window, n_mels, fmin, fmax, mel_scale=MELT_MEL_HTK, n_mfcc=0):
    h = lib().melt_plan_create(float(fs), int(n_fft), int(hop), int(window), int(n_mels), float(fmin), float(fmax),
                               int(mel_scale), int(n_mfcc))
    if not h:
        raise MeltError(-1, melt_last_error())
    return h


def melt_plan_create_stft_mel(fs, n_fft, hop, window, n_mels, fmin, fmax):
    """Plan of the conventional STFT -> power -> triangular Mel filterbank -> log10 front end (include/melt.h)."""
    h = lib().melt_plan_create_stft_mel(float(fs), int(n_fft), int(hop), int(window), int(n_mels), float(fmin), float(fmax))
    if not h:
        raise MeltError(-1, melt_last_error())
    return h


def melt_plan_destroy(plan):
    lib().melt_plan_destroy(plan)


def melt_plan_set_option(plan, key, value):
    _check(lib().melt_plan_set_option(plan, int(key), int(value)))


def melt_num_frames(plan, length):
    return int(lib().melt_num_frames(plan, int(length)))


def melt_count_frames(length, n_fft, hop, pad=MELT_PAD_NONE, drop_last=False):
    """Frames of a clip from the framing parameters alone (host-only integer arithmetic inside the library; no plan, no GPU)."""
    return int(lib().melt_count_frames(int(length), int(n_fft), int(hop), int(pad), int(bool(drop_last))))


def melt_plan_reserve(plan, nbytes):
    _check(lib().melt_plan_reserve(plan, int(nbytes)))


def melt_num_channels(plan):
    return int(lib().melt_num_channels(plan))


def melt_plan_get_centres(plan, n_mels):
    buf = (C.c_double * n_mels)()
    _check(lib().melt_plan_get_centres(plan, buf))
    return list(buf)


def melt_plan_describe(plan):
    return lib().melt_plan_describe(plan).decode()


def melt_forward(plan, x, batch, length, out, stream=0):
    _check(lib().melt_forward(plan, _ptr(x), int(batch), int(length), _ptr(out), stream or None))


def melt_forward_host(plan, x_host, batch, length, out_host, stream=0):
    """x_host / out_host: host pointers (ints), pinned torch CPU tensors or numpy arrays; asynchronous on `stream`."""
    def hp(t):
        if isinstance(t, int):
            return t
        return int(t.data_ptr()) if hasattr(t, "data_ptr") else int(t.ctypes.data)
    _check(lib().melt_forward_host(plan, hp(x_host), int(batch), int(length), hp(out_host), stream or None))


def melt_forward_ragged(plan, x, offsets, n_clips, out, out_frame_offsets, stream=0):
    _check(lib().melt_forward_ragged(plan, _ptr(x), _ptr(offsets), int(n_clips), _ptr(out), _ptr(out_frame_offsets),
                                     stream or None))


MELT_NOALLOC_MAX_CLIPS = 65536


def melt_forward_ragged_noalloc(plan, x, offsets, n_clips, out, out_frame_offsets, stream=0):
    """melt_forward_ragged without any allocation: scratch in a fixed device array (n_clips <= MELT_NOALLOC_MAX_CLIPS;
    calls that overlap on the GPU race on it -- see include/melt.h)."""
    _check(lib().melt_forward_ragged_noalloc(plan, _ptr(x), _ptr(offsets), int(n_clips), _ptr(out), _ptr(out_frame_offsets),
                                             stream or None))


def melt_forward_tap(plan, x, offsets, n_clips, length, out, logmel, out_frame_offsets, stream=0):
    _check(lib().melt_forward_tap(plan, _ptr(x), _ptr(offsets), int(n_clips), int(length), _ptr(out), _ptr(logmel),
                                  _ptr(out_frame_offsets), stream or None))


def melt_selftest_umma(kind, a, b):
    """a [128, k], b [n, k] numpy float32 (host) -> d [128, n] numpy float32."""
    import numpy as np
    a = np.ascontiguousarray(a, np.float32)
    b = np.ascontiguousarray(b, np.float32)
    n, k = b.shape
    assert a.shape == (128, k)
    d = np.empty((128, n), np.float32)
    _check(lib().melt_selftest_umma(int(kind), n, k, a.ctypes.data, b.ctypes.data, d.ctypes.data))
    return d


def melt_selftest_umma2(kind, a, b):
    """CTA-pair form: a [256, k], b [n, k] numpy float32 (host) -> d [256, n] numpy float32."""
    import numpy as np
    a = np.ascontiguousarray(a, np.float32)
    b = np.ascontiguousarray(b, np.float32)
    n, k = b.shape
    assert a.shape == (256, k)
    d = np.empty((256, n), np.float32)
    _check(lib().melt_selftest_umma2(int(kind), n, k, a.ctypes.data, b.ctypes.data, d.ctypes.data))
    return d


def melt_selftest_poison_smem(stream=0):
    """Fill every SM's shared memory with NaN bit patterns (test aid: forwards must not depend on stale shared memory)."""
    _check(lib().melt_selftest_poison_smem(stream or None))
