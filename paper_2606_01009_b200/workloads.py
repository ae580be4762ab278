"""Seeded synthetic inputs shaped like BASELINE.json's five configs (recipe: DESIGN.md "Input recipe").

This module serves BOTH the fp64 oracle (tests) and the CUDA path (tests, bench.py).  It holds none of
the method's arithmetic -- only signal synthesis (sinusoids, harmonics, chirps, noise, silent spans,
numpy's own reflect padding) and the table of configurations.  It imports neither ``oracle`` nor the
CUDA binding.  The synthetic signals stand in for the paper's LibriSpeech / Libri6000 / VoxCeleb1
material, which is not available and is not reconstructed.

RNG: numpy PCG64, seed = BASE_SEED + config index (+ sweep index for config 4); one independent child
stream per clip (SeedSequence.spawn), so the result does not depend on generation order or threading.
Signals are synthesised in float64 and cast once to float32; the same bytes go to both sides.
"""
from concurrent.futures import ThreadPoolExecutor
import os

import numpy as np

BASE_SEED = 20260601

WINDOW_HANN_PERIODIC, WINDOW_HANN_SYMMETRIC, WINDOW_RECT = 0, 1, 2

# Plan parameters and shapes of BASELINE.json configs[0..4] (config 4 has four settings a-d).
CONFIGS = {
    "cfg0": dict(fs=16000.0, n_fft=400, hop=160, window=WINDOW_HANN_PERIODIC, n_mels=80, fmin=0.0, fmax=8000.0,
                 n_mfcc=0, n_clips=1, clip_len=16000, pad_reflect=False, drop_last=False, layout="frame_major",
                 seed=BASE_SEED + 0),
    "cfg1": dict(fs=16000.0, n_fft=400, hop=160, window=WINDOW_HANN_PERIODIC, n_mels=80, fmin=0.0, fmax=8000.0,
                 n_mfcc=0, n_clips=32, clip_len=480000, pad_reflect=True, drop_last=True, layout="feature_major",
                 seed=BASE_SEED + 1),
    "cfg2": dict(fs=16000.0, n_fft=400, hop=160, window=WINDOW_HANN_PERIODIC, n_mels=128, fmin=0.0, fmax=8000.0,
                 n_mfcc=0, n_clips=256, clip_len=480000, pad_reflect=True, drop_last=True, layout="feature_major",
                 seed=BASE_SEED + 2),
    "cfg3": dict(fs=16000.0, n_fft=400, hop=160, window=WINDOW_HANN_PERIODIC, n_mels=40, fmin=20.0, fmax=7600.0,
                 n_mfcc=13, n_clips=1024, min_len=64000, max_len=192000, ragged=True, pad_reflect=False,
                 drop_last=False, layout="frame_major", seed=BASE_SEED + 3),
    "cfg4a": dict(fs=22050.0, n_fft=1024, hop=256, window=WINDOW_HANN_PERIODIC, n_mels=128, fmin=0.0, fmax=11025.0,
                  n_mfcc=0, n_clips=64, clip_len=220500, pad_reflect=False, drop_last=False, layout="feature_major",
                  seed=BASE_SEED + 4),
    "cfg4b": dict(fs=22050.0, n_fft=2048, hop=512, window=WINDOW_HANN_PERIODIC, n_mels=128, fmin=0.0, fmax=11025.0,
                  n_mfcc=0, n_clips=64, clip_len=220500, pad_reflect=False, drop_last=False, layout="feature_major",
                  seed=BASE_SEED + 5),
    "cfg4c": dict(fs=44100.0, n_fft=2048, hop=512, window=WINDOW_HANN_PERIODIC, n_mels=256, fmin=0.0, fmax=22050.0,
                  n_mfcc=0, n_clips=64, clip_len=441000, pad_reflect=False, drop_last=False, layout="feature_major",
                  seed=BASE_SEED + 6),
    "cfg4d": dict(fs=44100.0, n_fft=4096, hop=1024, window=WINDOW_HANN_PERIODIC, n_mels=256, fmin=0.0, fmax=22050.0,
                  n_mfcc=0, n_clips=64, clip_len=441000, pad_reflect=False, drop_last=False, layout="feature_major",
                  seed=BASE_SEED + 7),
}


def plan_args(cfg):
    """The nine melt_plan_create scalars of a config, in call order."""
    c = CONFIGS[cfg] if isinstance(cfg, str) else cfg
    return (c["fs"], c["n_fft"], c["hop"], c["window"], c["n_mels"], c["fmin"], c["fmax"], 0, c["n_mfcc"])


def _pool_map(fn, items):
    nthr = min(len(items), max(1, (os.cpu_count() or 1)))
    if nthr <= 1:
        return [fn(i) for i in items]
    with ThreadPoolExecutor(nthr) as ex:
        return list(ex.map(fn, items))


def _sinusoid_mix(rng, n, fs, n_sin, f_rng=(50.0, 7200.0), a_rng=(0.05, 0.5)):
    t = np.arange(n, dtype=np.float64) / fs
    x = np.zeros(n, np.float64)
    for _ in range(n_sin):
        f = rng.uniform(*f_rng)
        a = rng.uniform(*a_rng)
        ph = rng.uniform(0.0, 2.0 * np.pi)
        x += a * np.sin(2.0 * np.pi * f * t + ph)
    return x


def single_clip(seed=BASE_SEED, n=16000, fs=16000.0, sigma=0.01):
    """configs[0]: sum of 3 sinusoids (f ~ U[50,7200] Hz, a ~ U[0.05,0.5], random phase) + N(0, sigma^2)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    x = _sinusoid_mix(rng, n, fs, 3)
    x += rng.normal(0.0, sigma, n)
    return x.astype(np.float32)


def whisper_batch(n_clips, seed, clip_len=480000, fs=16000.0, sigma=0.01):
    """configs[1]/[2]: per clip 1-8 sinusoids (laws of config 0) + noise, then 0-3 spans of U[0.2,2] s set to
    exactly 0.0 AFTER the noise is added (reading R11).  Returns the UNPADDED batch [n_clips, clip_len]."""
    children = np.random.SeedSequence(seed).spawn(n_clips)
    out = np.empty((n_clips, clip_len), np.float32)

    def one(b):
        rng = np.random.Generator(np.random.PCG64(children[b]))
        x = _sinusoid_mix(rng, clip_len, fs, int(rng.integers(1, 9)))
        x += rng.normal(0.0, sigma, clip_len)
        for _ in range(int(rng.integers(0, 4))):
            span = int(rng.uniform(0.2, 2.0) * fs)
            start = int(rng.integers(0, max(1, clip_len - span)))
            x[start:start + span] = 0.0
        out[b] = x.astype(np.float32)

    _pool_map(one, list(range(n_clips)))
    return out


def reflect_pad(x, p):
    """numpy 'reflect' padding by p samples per side along the last axis (edge sample not repeated)."""
    pad = [(0, 0)] * (x.ndim - 1) + [(p, p)]
    return np.ascontiguousarray(np.pad(x, pad, mode="reflect"))


def speaker_ragged(n_clips, seed, fs=16000.0, min_len=64000, max_len=192000, sigma=0.02):
    """configs[3]: ragged clips, lengths ~ U{min_len..max_len}, packed contiguously + int64 offsets.  Each clip:
    2-6 harmonic tones (f0 ~ U[80,300] Hz, 10 harmonics, harmonic k amplitude a/k with a ~ U[0.05,0.3],
    independent uniform phases; reading R12) + N(0, sigma^2)."""
    root = np.random.SeedSequence(seed)
    len_rng = np.random.Generator(np.random.PCG64(root.spawn(1)[0]))
    lengths = len_rng.integers(min_len, max_len + 1, size=n_clips).astype(np.int64)
    offsets = np.zeros(n_clips + 1, np.int64)
    offsets[1:] = np.cumsum(lengths)
    children = np.random.SeedSequence(seed + 1000003).spawn(n_clips)
    out = np.empty(int(offsets[-1]), np.float32)

    def one(i):
        rng = np.random.Generator(np.random.PCG64(children[i]))
        n = int(lengths[i])
        t = np.arange(n, dtype=np.float64) / fs
        x = rng.normal(0.0, sigma, n)
        for _ in range(int(rng.integers(2, 7))):
            f0 = rng.uniform(80.0, 300.0)
            a = rng.uniform(0.05, 0.3)
            for k in range(1, 11):
                ph = rng.uniform(0.0, 2.0 * np.pi)
                x += (a / k) * np.sin(2.0 * np.pi * (k * f0) * t + ph)
        out[offsets[i]:offsets[i + 1]] = x.astype(np.float32)

    _pool_map(one, list(range(n_clips)))
    return out, offsets


def hires_batch(n_clips, seed, fs, clip_len, sigma=0.01, amp=0.3):
    """configs[4]: linear chirp 100 Hz -> 0.45 fs over the clip (amplitude 0.3, random start phase) + N(0, sigma^2)."""
    children = np.random.SeedSequence(seed).spawn(n_clips)
    out = np.empty((n_clips, clip_len), np.float32)
    t = np.arange(clip_len, dtype=np.float64) / fs
    dur = clip_len / fs
    f0, f1 = 100.0, 0.45 * fs
    base_phase = 2.0 * np.pi * (f0 * t + 0.5 * (f1 - f0) / dur * t * t)

    def one(b):
        rng = np.random.Generator(np.random.PCG64(children[b]))
        x = amp * np.sin(base_phase + rng.uniform(0.0, 2.0 * np.pi))
        x += rng.normal(0.0, sigma, clip_len)
        out[b] = x.astype(np.float32)

    _pool_map(one, list(range(n_clips)))
    return out


def make_inputs(cfg, n_clips=None, seed=None):
    """Inputs of a named config (optionally with fewer clips, same per-clip streams; optionally another seed).
    Returns dict(x=..., offsets=None|int64[n+1], x_unpadded=... for the reflect-padded configs)."""
    c = dict(CONFIGS[cfg])
    if seed is not None:
        c["seed"] = int(seed)
    n = c["n_clips"] if n_clips is None else int(n_clips)
    if cfg == "cfg0":
        return dict(x=single_clip(c["seed"], c["clip_len"], c["fs"])[None, :], offsets=None)
    if cfg in ("cfg1", "cfg2"):
        raw = whisper_batch(n, c["seed"], c["clip_len"], c["fs"])
        return dict(x=reflect_pad(raw, c["n_fft"] // 2), x_unpadded=raw, offsets=None)
    if cfg == "cfg3":
        x, off = speaker_ragged(n, c["seed"], c["fs"], c["min_len"], c["max_len"])
        return dict(x=x, offsets=off)
    if cfg.startswith("cfg4"):
        return dict(x=hires_batch(n, c["seed"], c["fs"], c["clip_len"]), offsets=None)
    raise KeyError(cfg)


# ------------------------------------------------------------------------------------------------ the paper's own shapes
# Table 4 of the paper -- spectral front end 16 kHz / N = 400 / H = 160 /
# M = 80 / 80-7600 Hz, cepstral front end N = 1200 / H = 160 / M = 128 / K = 40 / 0-8000 Hz, "symmetric Hann" --
# on what the paper sweeps: one clip of 1 .. 160 s (Table 5), the number of Mel bins 40 .. 512 at 160 s
# (Fig. 6) and batches of 1 .. 256 utterances of 4 s (Fig. 7).  The paper measures on LibriSpeech /
# Libri6000 speech; these clips are the seeded harmonic-tone mixes of speaker_ragged (a voiced-speech-like spectrum), which
# stand in for that material.  No padding, frame-major output (the paper states neither; readings R3 / R5).
_SPEC = dict(fs=16000.0, n_fft=400, hop=160, window=WINDOW_HANN_SYMMETRIC, n_mels=80, fmin=80.0, fmax=7600.0, n_mfcc=0,
             pad_reflect=False, drop_last=False, layout="frame_major")
_CEP = dict(fs=16000.0, n_fft=1200, hop=160, window=WINDOW_HANN_SYMMETRIC, n_mels=128, fmin=0.0, fmax=8000.0, n_mfcc=40,
            pad_reflect=False, drop_last=False, layout="frame_major")
PAPER_CONFIGS = {}
for _d in (1, 10, 40, 160):
    PAPER_CONFIGS["paper_spec_%ds" % _d] = dict(_SPEC, n_clips=1, clip_len=16000 * _d, seed=BASE_SEED + 100 + _d)
    PAPER_CONFIGS["paper_cep_%ds" % _d] = dict(_CEP, n_clips=1, clip_len=16000 * _d, seed=BASE_SEED + 300 + _d)
for _m in (40, 128, 256, 512):
    PAPER_CONFIGS["paper_mel%d_160s" % _m] = dict(_SPEC, n_mels=_m, n_clips=1, clip_len=16000 * 160, seed=BASE_SEED + 500 + _m)
for _b in (1, 16, 256):
    PAPER_CONFIGS["paper_batch%d_4s" % _b] = dict(_SPEC, n_clips=_b, clip_len=64000, seed=BASE_SEED + 700 + _b)


def make_paper_inputs(name, n_clips=None):
    """Dense batch [n_clips, clip_len] float32 of a PAPER_CONFIGS entry: per clip 2-6 harmonic tones + noise (speaker_ragged's law)."""
    c = PAPER_CONFIGS[name]
    n = c["n_clips"] if n_clips is None else int(n_clips)
    x, off = speaker_ragged(n, c["seed"], c["fs"], c["clip_len"], c["clip_len"])
    return dict(x=x.reshape(n, c["clip_len"]), offsets=None)
