"""fp64 CPU oracle of the CONVENTIONAL front end -- TEST INFRASTRUCTURE ONLY.

The comparator the paper measures MelT against ("short-time Fourier transform followed by triangular Mel filterbank
aggregation"; "power values are first computed on uniformly spaced FFT bins and subsequently aggregated through
nonnegative triangular weights"; Eq. (10): FFT + sparse Mel aggregation, nnz(F_Mel) <= M (N/2 + 1);
PAPER.md:246 "configured to the identical DSP specification (Table 4)"; PAPER.md:545 calls a hand-fused version future work).

Plain numpy in double precision, written out step by step; numpy's FFT serves as the DFT step (pinned against a brute-force
DFT in tests/test_stft_mel_oracle_pins.py).  Nothing here imports the CUDA package or shares code with it.

Where the paper is silent (readings of NEXT-4):
  * filter edges: the (M + 2)-point grid uniform in HTK mel between fmin and fmax, so that the filter centres ARE the MelT analysis
    frequencies ("placed at the center frequencies of the triangular Mel filterbank ... HTK Mel convention");
  * filter height: peak 1, no area normalisation (HTK; the paper names no normalisation);
  * framing, window, padding, drop-last and the log form log10(max(S, 1e-10)): those of the MelT contract (BASELINE.json north_star),
    "identical DSP specification".
"""
import numpy as np

HANN_PERIODIC, HANN_SYMMETRIC, RECT = 0, 1, 2
PAD_NONE, PAD_REFLECT = 0, 1


def hz_to_mel(f):
    """HTK mel map, Eq. (1)."""
    return 2595.0 * np.log10(1.0 + np.asarray(f, np.float64) / 700.0)


def mel_to_hz(mu):
    """Inverse map, Eq. (2)."""
    return 700.0 * (10.0 ** (np.asarray(mu, np.float64) / 2595.0) - 1.0)


def window(kind, n_fft):
    n = np.arange(n_fft, dtype=np.float64)
    if kind == HANN_PERIODIC:
        return 0.5 - 0.5 * np.cos(2.0 * np.pi * n / n_fft)
    if kind == HANN_SYMMETRIC:
        return 0.5 - 0.5 * np.cos(2.0 * np.pi * n / (n_fft - 1))
    return np.ones(n_fft, np.float64)


def filter_edges(fmin, fmax, n_mels):
    """The M + 2 edge / centre frequencies in Hz: uniform in mel, endpoints included; edges[1:-1] are the filter centres."""
    mu = np.linspace(float(hz_to_mel(fmin)), float(hz_to_mel(fmax)), n_mels + 2)
    return mel_to_hz(mu)


def mel_filterbank(fs, n_fft, n_mels, fmin, fmax):
    """F[m, k], m < M, k <= N/2: triangle rising from edges[m] to 1 at edges[m + 1] and falling to 0 at edges[m + 2], evaluated at
    the DFT bin frequencies k fs / N."""
    e = filter_edges(fmin, fmax, n_mels)
    fk = np.arange(n_fft // 2 + 1, dtype=np.float64) * fs / n_fft
    F = np.zeros((n_mels, n_fft // 2 + 1), np.float64)
    for m in range(n_mels):
        lo, ce, hi = e[m], e[m + 1], e[m + 2]
        up = (fk - lo) / (ce - lo)
        down = (hi - fk) / (hi - ce)
        F[m] = np.maximum(0.0, np.minimum(up, down))
    return F


def num_frames(length, n_fft, hop, pad=PAD_NONE, drop_last=False):
    if pad == PAD_REFLECT:
        if length < n_fft // 2 + 1:
            return 0
        length = length + 2 * (n_fft // 2)
    if length < n_fft:
        return 0
    return max(0, (length - n_fft) // hop + 1 - (1 if drop_last else 0))


def frames_of(x, n_fft, hop, pad=PAD_NONE, drop_last=False):
    """[T, N] frames of one clip (fp64), frame t = samples t hop .. t hop + N - 1 of the (optionally reflect-padded) clip."""
    x = np.asarray(x, np.float64)
    T = num_frames(len(x), n_fft, hop, pad, drop_last)
    if T == 0:
        return np.zeros((0, n_fft), np.float64)
    if pad == PAD_REFLECT:
        x = np.pad(x, n_fft // 2, mode="reflect")
    idx = np.arange(T)[:, None] * hop + np.arange(n_fft)[None, :]
    return x[idx]


def stft_power(x, n_fft, hop, window_kind, pad=PAD_NONE, drop_last=False):
    """P[t, k] = |sum_n w[n] x_t[n] exp(-2 pi i k n / N)|^2, k = 0 .. N/2."""
    fr = frames_of(x, n_fft, hop, pad, drop_last) * window(window_kind, n_fft)[None, :]
    X = np.fft.rfft(fr, n=n_fft, axis=1)
    return X.real ** 2 + X.imag ** 2


def forward(x, fs, n_fft, hop, window_kind, n_mels, fmin, fmax, pad=PAD_NONE, drop_last=False, want=("L",)):
    """One clip -> dict with any of "P" (STFT power [T, N/2+1]), "S" (Mel energies [T, M]), "L" (log10(max(S, 1e-10)))."""
    P = stft_power(x, n_fft, hop, window_kind, pad, drop_last)
    F = mel_filterbank(fs, n_fft, n_mels, fmin, fmax)
    S = P @ F.T
    out = {}
    if "P" in want:
        out["P"] = P
    if "S" in want:
        out["S"] = S
    if "L" in want:
        out["L"] = np.log10(np.maximum(S, 1e-10))
    return out


def forward_batch(x, want=("L",), **kw):
    """[B, len] -> dict of [B, T, .] arrays."""
    res = [forward(row, want=want, **kw) for row in np.asarray(x)]
    return {k: np.stack([r[k] for r in res]) for k in want}
