"""Randomised (seeded) geometries through the C ABI against the fp64 oracle: frame lengths, hops, Mel counts, windows,
layouts, dense / ragged batches, log-Mel / MFCCT.  Every case must meet the compensated-mode bars; the sweep exists to
exercise the kernel-selection logic (CTA-pair kernel in its resident / streamed / direct / several-pass / ragged forms and
the general kernel) on shapes nobody wrote a dedicated test for."""
import numpy as np
import pytest

import parity_util as pu

pytestmark = pytest.mark.gpu


def _case(rng):
    hop = int(rng.choice([4, 8, 40, 64, 100, 128, 160, 200, 256, 320, 512]))
    n_fft = int(float(rng.choice([1, 2, 2.5, 3, 4, 4.5, 7.5])) * hop) if rng.random() < 0.7 else int(rng.integers(hop, 6 * hop + 1))
    n_fft = min(max(n_fft, 8), 4096)
    n_mels = int(rng.choice([1, 5, 16, 23, 40, 64, 80, 96, 128, 130, 160, 200, 256]))
    fs = float(rng.choice([8000, 16000, 22050, 44100]))
    n_mfcc = int(rng.choice([0, 0, 0, min(13, n_mels)]))
    ragged = bool(rng.random() < 0.3)
    layout = "frame_major" if (ragged or n_mfcc) else str(rng.choice(["frame_major", "feature_major"]))
    return dict(name="rnd", fs=fs, n_fft=n_fft, hop=hop, window=int(rng.choice([0, 0, 1, 2])), n_mels=n_mels, fmin=0.0,
                fmax=fs / 2, n_mfcc=n_mfcc, layout=layout), ragged


@pytest.mark.parametrize("seed", [101, 102, 103])
def test_random_geometries_against_the_oracle(seed):
    from oracle import melt_oracle as orc
    rng = np.random.default_rng(seed)
    for _ in range(12):
        c, ragged = _case(rng)
        hop, n_fft = c["hop"], c["n_fft"]
        if ragged:
            lens = rng.integers(0, 40 * hop + n_fft, 7)
            lens[2] = n_fft
            off = np.zeros(8, np.int64)
            off[1:] = np.cumsum(lens)
            x = rng.normal(0, 0.1, int(off[-1])).astype(np.float32)
            res = pu.gpu_ragged(c, x, off, "compensated")
            ref = orc.forward_ragged(x, off, want=("P", "L", "C"), **pu.oracle_kwargs(c))
            np.testing.assert_array_equal(res[1], ref["frame_offsets"], err_msg=str(c))
            got = res[0]
        else:
            B = int(rng.integers(1, 4))
            L = n_fft + int(rng.integers(0, 600)) * hop + (0 if rng.random() < 0.7 else int(rng.integers(1, 4)))
            x = rng.normal(0, 0.1, (B, L)).astype(np.float32)
            got = pu.gpu_dense(c, x, "compensated")
            ref = orc.forward_batch(x, want=("P", "L", "C"), **pu.oracle_kwargs(c))
        assert np.isfinite(got).all(), c
        if got.size == 0:
            continue
        if c["n_mfcc"]:
            assert float(np.abs(got - ref["C"]).max()) <= 3.5e-2, c      # DESIGN.md reading R9: end-to-end cepstral bound
        else:
            assert pu.log_error(got, ref["L"], ref["P"]) <= pu.LOG_BAR, c
