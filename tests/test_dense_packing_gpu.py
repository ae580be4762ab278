"""GPU: dense batches whose tiles pack 32-frame chunks ACROSS clip boundaries (csrc/melt_forward2_kernel.cuh, ChunkCursor).

A tile of the CTA-pair kernel is any 8 consecutive chunks of the batch, so the four lane quarters of a CTA may belong to
different clips, a CTA's chunk advances by a fixed stride with a carry from tile to tile, and the last tile of a batch may be
partly empty.  The geometries below are chosen to hit what the five configs do not: clips of ONE chunk (every lane quarter of a
tile another clip), chunk counts per clip that do not divide the per-tile stride, more tiles than CTA pairs (several rounds, so
the carry runs), several passes over the Mel bins, reflect padding at every clip edge inside a tile, the K-block staging form of
long windows, and a last tile with empty quarters.  Every output element is compared with the fp64 oracle (Eq. 1-8) under
the compensated-mode bars of test_parity_gpu.py and with the CPU emulation of the kernel's operand scheme; outputs are pre-filled
with NaN, so an unwritten row fails too."""
import numpy as np
import pytest

import parity_util as pu

pytestmark = pytest.mark.gpu

COMP_P_BAR = 2e-4


def _clips(n_clips, length, seed):
    """Noise plus one tone per clip (another frequency and level each), float32 [n_clips, length]."""
    rng = np.random.default_rng(seed)
    n = np.arange(length)
    f = rng.uniform(100.0, 7000.0, n_clips)[:, None]
    a = rng.uniform(0.05, 0.5, n_clips)[:, None]
    x = a * np.sin(2 * np.pi * f * n[None, :] / 16000.0 + rng.uniform(0, 6.28, n_clips)[:, None])
    x += rng.normal(0.0, 0.02, (n_clips, length))
    return x.astype(np.float32)


def _check(c, x, layout, pad=None, n_frames=None, p_bar=COMP_P_BAR):
    from oracle import melt_oracle as orc
    L = pu.gpu_dense(c, x, "compensated", layout=layout, pad=pad)
    P = pu.gpu_dense(c, x, "compensated", layout=layout, pad=pad, output="power", n_mfcc=0)
    assert np.isfinite(L).all() and np.isfinite(P).all()
    if n_frames is not None:
        assert L.shape[1] == n_frames
    ref = orc.forward_batch(x, want=("P", "L"), **pu.oracle_kwargs(c, pad=pad, n_mfcc=0))
    assert ref["L"].shape == L.shape
    perr, lerr = pu.power_error(P, ref["P"]), pu.log_error(L, ref["L"], ref["P"])
    # and against the CPU emulation of the kernel's own operand scheme (exact summation): what is left is the accumulation in tensor memory
    S_em = pu.emulated_power(c, x, "compensated", pad=pad)
    acc_p = pu.power_error(P, S_em)
    acc_l = pu.log_error(L, np.log10(np.maximum(S_em, 1e-10)), ref["P"])
    print("\n[packing] %d clips x %d frames, %d bins, %s: vs oracle |dP|/Pmax=%.2e |dlog10|=%.2e, vs own-scheme emulation %.2e / %.2e" % (
        x.shape[0], L.shape[1], c["n_mels"], layout, perr, lerr, acc_p, acc_l))
    # One loud tone per clip is the worst case of the truncating accumulation in tensor memory (coherent products of one sign): up to
    # 2.6e-5 of the frame maximum for 400-sample windows and 2.9e-4 for 2048-sample ones, where the noisier signals of the configs stay
    # below 1.6e-5 / 1.1e-4 (parity_util.acc_p_bar).  A chunk mapped to the wrong clip or row moves S by >= 1e-2 of the frame maximum.
    assert acc_p <= 2.5 * pu.acc_p_bar(c, "compensated") and acc_l <= pu.ACC_LOG_BAR
    assert perr <= p_bar and lerr <= pu.LOG_BAR


def _cfg(n_fft=400, hop=160, n_mels=80, fs=16000.0, fmax=8000.0):
    return dict(fs=fs, n_fft=n_fft, hop=hop, window=0, n_mels=n_mels, fmin=0.0, fmax=fmax, n_mfcc=0, name="packing")


@pytest.mark.parametrize("layout", ["feature_major", "frame_major"])
def test_two_chunks_per_clip_many_rounds(layout):
    # 700 clips x 40 frames: 1400 chunks = 175 tiles on 74 CTA pairs; every tile holds four clips
    _check(_cfg(), _clips(700, 400 + 39 * 160, 1), layout, n_frames=40)


def test_one_chunk_per_clip():
    # 1001 clips x 20 frames: every lane quarter of a tile is another clip; the last tile has one chunk and seven empty quarters
    _check(_cfg(), _clips(1001, 400 + 19 * 160, 2), "feature_major", n_frames=20)


def test_three_chunks_per_clip_two_bin_passes():
    # 200 bins = two passes over the bins (a tile is visited once per pass); 300 clips x 70 frames = 900 chunks = 113 tiles
    _check(_cfg(n_mels=200), _clips(300, 400 + 69 * 160, 3), "feature_major", n_frames=70)


def test_reflect_padding_at_every_clip_edge_inside_a_tile():
    # 150 clips of 0.5 s with in-library reflect padding: 51 frames = 2 chunks per clip, clip edges (mirrored samples) inside every tile
    _check(_cfg(), _clips(150, 8000, 4), "frame_major", pad=True, n_frames=51)


def test_long_window_k_block_staging():
    # 2048-sample windows (K-block staging): 90 clips x 45 frames = 180 chunks = 23 tiles, 128 bins
    c = _cfg(n_fft=2048, hop=512, n_mels=128, fs=22050.0, fmax=11025.0)
    # (a loud tone in a 2048-sample window: 192 truncating accumulations per bin leave up to 3e-4 of the frame maximum against the
    # oracle -- asserted against the north-star bar here, 2e-4 everywhere else)
    _check(c, _clips(90, 2048 + 44 * 512, 5), "feature_major", n_frames=45, p_bar=pu.P_BAR["compensated"])


def test_mfcct_rows_of_packed_tiles():
    # MFCCT (frame-major cepstra staged through shared memory per warp): 333 clips x 50 frames, two-stage check against the oracle's DCT
    from oracle import melt_oracle as orc
    c = dict(_cfg(n_mels=40, fmax=7600.0), n_mfcc=13)
    x = _clips(333, 400 + 49 * 160, 6)
    C, L = pu.gpu_dense(c, x, "compensated", layout="frame_major", tap=True)
    assert np.isfinite(C).all() and np.isfinite(L).all() and C.shape == (333, 50, 13)
    ref = orc.forward_batch(x, want=("P", "L"), **pu.oracle_kwargs(c, n_mfcc=0))
    assert pu.log_error(L, ref["L"], ref["P"]) <= pu.LOG_BAR
    for b in (0, 1, 166, 332):
        assert np.abs(C[b] - orc.dct_apply(L[b], 13)).max() <= 1e-4   # cepstra of the GPU's own log-Mel rows (DESIGN R9)
