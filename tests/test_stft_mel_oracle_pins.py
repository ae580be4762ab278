"""Pins of oracle/stft_mel_oracle.py (the conventional STFT + triangular Mel filterbank front end) against
what the mathematics fixes: a brute-force DFT, closed forms of windowed tones, Parseval, the partition of unity of adjacent
triangles, the filter centres = the MelT analysis frequencies.  CPU only."""
import math

import numpy as np

from oracle import stft_mel_oracle as so


def test_dft_step_against_brute_force_loops():
    # tiny case, every sum written out: catches a wrong sign, a wrong bin range, a window applied to the wrong axis
    rng = np.random.default_rng(1)
    N, H = 16, 4
    x = rng.normal(size=40)
    for kind in (so.HANN_PERIODIC, so.HANN_SYMMETRIC, so.RECT):
        w = so.window(kind, N)
        P = so.stft_power(x, N, H, kind)
        T = (len(x) - N) // H + 1
        assert P.shape == (T, N // 2 + 1)
        for t in range(T):
            for k in range(N // 2 + 1):
                re = sum(w[n] * x[t * H + n] * math.cos(2 * math.pi * k * n / N) for n in range(N))
                im = -sum(w[n] * x[t * H + n] * math.sin(2 * math.pi * k * n / N) for n in range(N))
                assert abs(P[t, k] - (re * re + im * im)) <= 1e-12 * max(1.0, P[t].max())


def test_window_definitions():
    N = 400
    wp, ws = so.window(so.HANN_PERIODIC, N), so.window(so.HANN_SYMMETRIC, N)
    assert wp[0] == 0.0 and abs(wp[N // 2] - 1.0) < 1e-15 and abs(wp[1] - wp[N - 1]) < 1e-15      # periodic: w[n] = w[N - n]
    assert ws[0] == 0.0 and abs(ws[N - 1]) < 1e-15 and abs(ws[1] - ws[N - 2]) < 1e-15               # symmetric: w[n] = w[N - 1 - n]
    assert abs(wp.sum() - N / 2) < 1e-10                                                             # sum of a periodic Hann window


def test_tone_at_a_bin_centre_closed_forms():
    # x[n] = A cos(2 pi k0 n / N + phi): rectangular window -> P[k0] = (A N / 2)^2 and nothing elsewhere;
    # periodic Hann -> exactly three bins: P[k0] = (A N / 4)^2, P[k0 +- 1] = (A N / 8)^2
    N, H, A, k0, phi = 64, 16, 0.7, 9, 0.4
    n = np.arange(N + 3 * H)
    x = A * np.cos(2 * np.pi * k0 * n / N + phi)
    P = so.stft_power(x, N, H, so.RECT)
    assert np.allclose(P[:, k0], (A * N / 2) ** 2, rtol=1e-12)
    assert np.abs(np.delete(P, k0, axis=1)).max() < 1e-18 * (A * N) ** 2 * 1e6
    P = so.stft_power(x, N, H, so.HANN_PERIODIC)
    assert np.allclose(P[:, k0], (A * N / 4) ** 2, rtol=1e-12)
    assert np.allclose(P[:, k0 - 1], (A * N / 8) ** 2, rtol=1e-10) and np.allclose(P[:, k0 + 1], (A * N / 8) ** 2, rtol=1e-10)
    assert np.abs(np.delete(P, [k0 - 1, k0, k0 + 1], axis=1)).max() < 1e-20 * (A * N) ** 2 * 1e6


def test_parseval():
    rng = np.random.default_rng(2)
    N, H = 400, 160
    x = rng.normal(size=2000)
    w = so.window(so.HANN_PERIODIC, N)
    P = so.stft_power(x, N, H, so.HANN_PERIODIC)
    c = np.full(N // 2 + 1, 2.0)
    c[0] = c[-1] = 1.0
    for t in range(P.shape[0]):
        assert abs((P[t] * c).sum() - N * ((w * x[t * H:t * H + N]) ** 2).sum()) <= 1e-10 * (P[t] * c).sum()


def test_filter_centres_are_the_melt_analysis_frequencies():
    # the filter centres are the frequencies the MelT oracle projects on (written in C, from Eq. (1)-(2), independently)
    from oracle import melt_oracle as mo
    for fmin, fmax, M in ((0.0, 8000.0, 80), (20.0, 7600.0, 40), (80.0, 7600.0, 80), (0.0, 22050.0, 128)):
        e = so.filter_edges(fmin, fmax, M)
        assert abs(e[0] - fmin) < 1e-9 and abs(e[-1] - fmax) < 1e-8 and np.all(np.diff(e) > 0)
        assert np.allclose(e[1:-1], mo.centres(fmin, fmax, M), rtol=1e-13, atol=1e-10)
    # Eq. (1)-(2) at a value one can do by hand: mel(700) = 2595 log10(2), mel(6300) = 2595
    assert abs(float(so.hz_to_mel(700.0)) - 2595.0 * math.log10(2.0)) < 1e-12
    assert abs(float(so.hz_to_mel(6300.0)) - 2595.0) < 1e-12 and abs(float(so.mel_to_hz(2595.0)) - 6300.0) < 1e-9


def test_filterbank_shape_support_and_partition_of_unity():
    fs, N, M, fmin, fmax = 16000.0, 400, 80, 0.0, 8000.0
    F = so.mel_filterbank(fs, N, M, fmin, fmax)
    e = so.filter_edges(fmin, fmax, M)
    fk = np.arange(N // 2 + 1) * fs / N
    assert F.shape == (M, N // 2 + 1) and F.min() >= 0.0 and F.max() <= 1.0
    for m in (0, 1, 17, 79):
        inside = (fk > e[m]) & (fk < e[m + 2])
        assert np.all(F[m][inside] > 0) and np.all(F[m][~inside] == 0)              # support = the open interval between the outer edges
        k = np.nonzero(inside & (fk <= e[m + 1]))[0]
        assert np.allclose(F[m][k], (fk[k] - e[m]) / (e[m + 1] - e[m]), rtol=1e-13)  # rising flank, written the other way round
    # adjacent triangles sum to one between the first and the last centre (linear interpolation weights)
    mid = (fk >= e[1]) & (fk <= e[M])
    assert np.allclose(F.sum(axis=0)[mid], 1.0, rtol=1e-12)
    # a triangle is 1 at its own centre: choose fmax so that a centre falls exactly on a bin (M = 1: the centre is the mel midpoint)
    ce = float(so.mel_to_hz(0.5 * float(so.hz_to_mel(4000.0))))
    F1 = so.mel_filterbank(2.0 * ce * 8, 16, 1, 0.0, 4000.0)          # bin spacing = ce: bin 1 sits on the centre
    assert abs(F1[0, 1] - 1.0) < 1e-12 and F1[0, 0] == 0.0


def test_forward_scaling_and_clamp():
    rng = np.random.default_rng(3)
    kw = dict(fs=16000.0, n_fft=400, hop=160, window_kind=so.HANN_PERIODIC, n_mels=80, fmin=0.0, fmax=8000.0)
    x = rng.normal(0, 0.1, 4000)
    a = so.forward(x, want=("S", "L", "P"), **kw)
    b = so.forward(2.0 * x, want=("S", "L"), **kw)
    assert np.allclose(b["S"], 4.0 * a["S"], rtol=1e-12)                               # power is quadratic in the signal
    assert np.allclose(b["L"], a["L"] + math.log10(4.0), atol=1e-12)
    assert a["S"].shape == (23, 80) and np.allclose(a["S"], a["P"] @ so.mel_filterbank(16000.0, 400, 80, 0.0, 8000.0).T)
    z = so.forward(np.zeros(1000), want=("L",), **kw)["L"]
    assert np.all(z == -10.0)                                                          # log10(max(0, 1e-10))


def test_framing_padding_and_drop_last():
    x = np.arange(1000, dtype=np.float64)
    fr = so.frames_of(x, 400, 160)
    assert fr.shape == (4, 400) and fr[3, 0] == 480 and fr[3, -1] == 879
    frp = so.frames_of(x, 400, 160, pad=so.PAD_REFLECT)
    assert frp.shape == (7, 400) and frp[0, 200] == 0 and frp[0, 199] == 1 and frp[0, 0] == 200   # numpy 'reflect': edge not repeated
    assert so.num_frames(1000, 400, 160, so.PAD_REFLECT, drop_last=True) == 6
    assert so.num_frames(399, 400, 160) == 0 and so.num_frames(400, 400, 160) == 1
    assert so.num_frames(200, 400, 160, so.PAD_REFLECT) == 0 and so.num_frames(201, 400, 160, so.PAD_REFLECT) == 2   # 601 padded samples


def test_tone_energy_lands_in_the_filters_around_it():
    # a tone between two centres: its three Hann bins are shared by the two neighbouring filters with weights that sum to one,
    # so the two Mel energies add up to the tone's total STFT power (a transposed or shifted filterbank fails this)
    fs, N, H, M = 16000.0, 400, 160, 80
    e = so.filter_edges(0.0, 8000.0, M)
    k0 = 60                                            # 2400 Hz
    m = int(np.searchsorted(e, k0 * fs / N)) - 1       # e[m] < f <= e[m + 1]
    assert e[m] < k0 * fs / N <= e[m + 1]
    n = np.arange(N)
    x = 0.5 * np.cos(2 * np.pi * k0 * n / N)
    r = so.forward(x, fs, N, H, so.HANN_PERIODIC, M, 0.0, 8000.0, want=("S", "P"))
    assert abs(r["S"].sum() - r["P"].sum()) <= 1e-9 * r["P"].sum()      # all three bins lie between the first and last centre
    top2 = np.sort(np.argsort(r["S"][0])[-2:])
    assert top2[1] - top2[0] == 1 and e[top2[0] + 1] <= k0 * fs / N <= e[top2[1] + 1]
