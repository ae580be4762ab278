"""Pins for the fp64 oracle (oracle/melt_oracle.c): what the paper and the mathematics fix.

None of these tests retypes the oracle's own formula and compares it with itself: each checks against a
closed form, a library routine (numpy FFT, SciPy DCT), an invariant, a value stored under tests/golden/
or a pure-Python brute force.  Pin numbers follow SURVEY.md section 8(c).  CPU only.
"""
import math
import os

import numpy as np
import pytest

from oracle import melt_oracle as orc

GOLD = os.path.join(os.path.dirname(__file__), "golden")
W16 = dict(fs=16000.0, n_fft=400, hop=160, window_kind=orc.HANN_PERIODIC, n_mels=80, fmin=0.0, fmax=8000.0)


def _rows(name):
    with open(os.path.join(GOLD, name)) as fh:
        return [ln.split() for ln in fh if ln.strip() and not ln.startswith("#")]


# ---------------------------------------------------------------- P1: Mel centres (Eq. 1-2)
def test_p1_centres_golden():
    for M, fmin, fmax, m, val in _rows("mel_centres.txt"):
        f = orc.centres(float(fmin), float(fmax), int(M))
        assert f[int(m)] == pytest.approx(float(val), rel=1e-11)
    assert orc.hz_to_mel(8000.0) == pytest.approx(2840.023046708319, rel=1e-13)


@pytest.mark.parametrize("M,fmin,fmax", [(80, 0.0, 8000.0), (40, 20.0, 7600.0), (256, 0.0, 22050.0), (1, 0.0, 5600.0)])
def test_p1_centres_geometric_closed_form(M, fmin, fmax):
    """Uniform spacing in mu = 2595 log10(1+f/700) <=> (700+f_m) is a geometric sequence whose (M+2)-point
    extension starts at 700+fmin and ends at 700+fmax.  No log/pow needed to state it."""
    f = orc.centres(fmin, fmax, M)
    g = np.concatenate([[700.0 + fmin], 700.0 + f, [700.0 + fmax]])
    assert np.all(np.diff(g) > 0)
    np.testing.assert_allclose(g[1:-1] ** 2, g[:-2] * g[2:], rtol=1e-12)
    # inverse map really inverts the forward map
    for fm in f[:: max(1, M // 7)]:
        assert orc.mel_to_hz(orc.hz_to_mel(fm)) == pytest.approx(fm, rel=1e-12)


# ---------------------------------------------------------------- P7a: window sums (closed forms)
@pytest.mark.parametrize("N", [8, 400, 401, 1024])
def test_p7_window_sums(N):
    wp = orc.window(orc.HANN_PERIODIC, N)
    ws = orc.window(orc.HANN_SYMMETRIC, N)
    assert wp.sum() == pytest.approx(N / 2, rel=1e-12) and (wp ** 2).sum() == pytest.approx(3 * N / 8, rel=1e-12)
    assert ws.sum() == pytest.approx((N - 1) / 2, rel=1e-12) and (ws ** 2).sum() == pytest.approx(3 * (N - 1) / 8, rel=1e-12)
    assert wp[0] == 0.0 and ws[0] == 0.0 and abs(ws[-1]) < 1e-15
    np.testing.assert_allclose(wp[1:], wp[1:][::-1], atol=1e-15)      # periodic: symmetric about N/2
    np.testing.assert_allclose(ws, ws[::-1], atol=1e-15)              # symmetric about (N-1)/2
    np.testing.assert_array_equal(orc.window(orc.RECT, N), np.ones(N))


# ---------------------------------------------------------------- P2: integer-bin centres -> naive DFT / numpy FFT
@pytest.mark.parametrize("fs,fmax,M,bins", [(16000.0, 5600.0, 1, [35]), (28000.0, 10500.0, 3, [10, 30, 70])])
@pytest.mark.parametrize("win", [orc.HANN_PERIODIC, orc.HANN_SYMMETRIC, orc.RECT])
def test_p2_integer_bin_equals_dft(fs, fmax, M, bins, win):
    N, H = 400, 160
    f = orc.centres(0.0, fmax, M)
    np.testing.assert_allclose(f, np.array(bins) * fs / N, rtol=1e-12)
    rng = np.random.default_rng(7)
    x = rng.normal(0, 0.3, N + 3 * H).astype(np.float32)
    out = orc.forward(x, fs=fs, n_fft=N, hop=H, window_kind=win, n_mels=M, fmin=0.0, fmax=fmax, want=("R", "I", "P"))
    w = orc.window(win, N)
    n = np.arange(N)
    for t in range(out["P"].shape[0]):
        fr = x[t * H:t * H + N].astype(np.float64) * w
        X = np.fft.fft(fr)                                             # library routine: sum fr[n] e^{-2 pi i k n/N}
        naive = np.array([np.sum(fr * np.exp(-2j * np.pi * k * n / N)) for k in bins])
        np.testing.assert_allclose(out["P"][t], np.abs(X[bins]) ** 2, rtol=1e-9, atol=1e-12)
        np.testing.assert_allclose(out["P"][t], np.abs(naive) ** 2, rtol=1e-9, atol=1e-12)
        # Eq. (3) uses +sin: R + iI = conj(DFT bin)
        np.testing.assert_allclose(out["R"][t], X[bins].real, rtol=1e-9, atol=1e-9)
        np.testing.assert_allclose(out["I"][t], -X[bins].imag, rtol=1e-9, atol=1e-9)


# ---------------------------------------------------------------- P3: on-bin tone, periodic Hann: P = (A N / 4)^2
@pytest.mark.parametrize("phi", [0.0, 0.7, 2.9, -1.3])
def test_p3_on_bin_tone(phi):
    N, fs, A, k = 400, 16000.0, 0.5, 35
    n = np.arange(N + 320)
    x = (A * np.cos(2 * np.pi * k * n / N + phi)).astype(np.float64)
    # use float32-exact input so the widening in the oracle is exact: compare with the value for that input
    x32 = x.astype(np.float32)
    out = orc.forward(x32, fs=fs, n_fft=N, hop=160, window_kind=orc.HANN_PERIODIC, n_mels=1, fmin=0.0, fmax=5600.0)
    assert out["P"].shape == (3, 1)
    np.testing.assert_allclose(out["P"][:, 0], (A * N / 4) ** 2, rtol=2e-6)       # fp32 input rounding only
    np.testing.assert_allclose(out["L"][:, 0], 3.397940008672, atol=2e-6)


# ---------------------------------------------------------------- P4: closed form for any tone / any centre
def _dirichlet(theta, N):
    theta = np.asarray(theta, dtype=np.float64)
    s = np.sin(theta / 2)
    small = np.abs(s) < 1e-14
    val = np.exp(1j * theta * (N - 1) / 2) * np.sin(N * theta / 2) / np.where(small, 1.0, s)
    return np.where(small, N + 0j, val)


def _hann_response(theta, N, Lw):
    return 0.5 * _dirichlet(theta, N) - 0.25 * _dirichlet(theta + 2 * np.pi / Lw, N) - 0.25 * _dirichlet(theta - 2 * np.pi / Lw, N)


@pytest.mark.parametrize("win,Lw", [(orc.HANN_PERIODIC, 400), (orc.HANN_SYMMETRIC, 399)])
def test_p4_closed_form_hann_tone(win, Lw):
    N, H, fs, M = 400, 160, 16000.0, 80
    f = orc.centres(0.0, 8000.0, M)
    wm = 2 * np.pi * f / fs
    rng = np.random.default_rng(11)
    for _ in range(4):
        f0, A, phi = rng.uniform(60, 7900), rng.uniform(0.1, 0.9), rng.uniform(0, 2 * np.pi)
        w0 = 2 * np.pi * f0 / fs
        L = N + 2 * H
        x = A * np.cos(w0 * np.arange(L) + phi)
        # oracle takes float32: make the test signal exactly float32-representable and use it on both sides
        x32 = x.astype(np.float32)
        out = orc.forward(x32, fs=fs, n_fft=N, hop=H, window_kind=win, n_mels=M, fmin=0.0, fmax=8000.0,
                          want=("R", "I", "P"))
        for t in range(3):
            ph_t = phi + w0 * t * H
            Z = (A / 2) * (np.exp(1j * ph_t) * _hann_response(wm + w0, N, Lw) + np.exp(-1j * ph_t) * _hann_response(wm - w0, N, Lw))
            # tolerance: float32 rounding of the input (rel 6e-8 per sample) on sums of magnitude <= A N / 2
            np.testing.assert_allclose(out["R"][t], Z.real, atol=2e-5)
            np.testing.assert_allclose(out["I"][t], Z.imag, atol=2e-5)
            np.testing.assert_allclose(out["P"][t], np.abs(Z) ** 2, rtol=1e-4, atol=1e-6)


def test_p4_closed_form_exact_float32_tone():
    """Same closed form with a signal that IS exact in float32 (amplitude 1, frequencies fs/4 and fs/2 give
    samples in {0, +-1}), so the comparison is at fp64 level, 1e-10."""
    N, H, fs, M = 400, 160, 16000.0, 80
    f = orc.centres(0.0, 8000.0, M)
    wm = 2 * np.pi * f / fs
    n = np.arange(N + H)
    x = np.round(np.cos(np.pi / 2 * n)).astype(np.float32)           # cos(pi n / 2): 1,0,-1,0,...
    out = orc.forward(x, fs=fs, n_fft=N, hop=H, window_kind=orc.HANN_PERIODIC, n_mels=M, fmin=0.0, fmax=8000.0,
                      want=("R", "I", "P"))
    w0 = np.pi / 2
    for t in range(2):
        ph_t = w0 * t * H
        Z = 0.5 * (np.exp(1j * ph_t) * _hann_response(wm + w0, N, N) + np.exp(-1j * ph_t) * _hann_response(wm - w0, N, N))
        np.testing.assert_allclose(out["R"][t], Z.real, atol=1e-10)
        np.testing.assert_allclose(out["I"][t], Z.imag, atol=1e-10)
        np.testing.assert_allclose(out["P"][t], np.abs(Z) ** 2, rtol=1e-9, atol=1e-12)


# ---------------------------------------------------------------- P5: impulse -> flat spectrum; MFCCT of flat log-Mel
def test_p5_impulse_flat_and_dct_of_flat():
    N, H, fs, M, K = 400, 160, 16000.0, 40, 13
    x = np.zeros(N + 2 * H, np.float32)
    pos = 417
    x[pos] = 1.0
    out = orc.forward(x, fs=fs, n_fft=N, hop=H, window_kind=orc.HANN_PERIODIC, n_mels=M, fmin=20.0, fmax=7600.0, n_mfcc=K)
    w = orc.window(orc.HANN_PERIODIC, N)
    for t in range(3):
        n0 = pos - t * H
        expect = w[n0] ** 2 if 0 <= n0 < N else 0.0
        np.testing.assert_allclose(out["P"][t], expect, rtol=1e-10, atol=1e-18)
        c = math.log10(max(expect, 1e-10))
        assert out["C"][t, 0] == pytest.approx(math.sqrt(M) * c, rel=1e-10)
        np.testing.assert_allclose(out["C"][t, 1:], 0.0, atol=1e-10)


# ---------------------------------------------------------------- P6: linearity / quadratic identities
def test_p6_linearity_and_parallelogram():
    rng = np.random.default_rng(3)
    L = 400 + 5 * 160
    # dyadic-grid inputs (multiples of 2^-12 below 2) so x+y, x-y, 0.5x are exact in float32
    x = (rng.integers(-4096, 4096, L) / 4096.0).astype(np.float32)
    y = (rng.integers(-4096, 4096, L) / 4096.0).astype(np.float32)
    kw = dict(W16, want=("R", "I", "P"))
    ox, oy = orc.forward(x, **kw), orc.forward(y, **kw)
    os_, od = orc.forward((x + y).astype(np.float32), **kw), orc.forward((x - y).astype(np.float32), **kw)
    oh = orc.forward((0.5 * x).astype(np.float32), **kw)
    scale = np.abs(ox["R"]).max()
    np.testing.assert_allclose(os_["R"], ox["R"] + oy["R"], atol=1e-11 * scale)
    np.testing.assert_allclose(os_["I"], ox["I"] + oy["I"], atol=1e-11 * scale)
    np.testing.assert_allclose(oh["P"], 0.25 * ox["P"], rtol=1e-12)
    np.testing.assert_allclose(os_["P"] + od["P"], 2 * ox["P"] + 2 * oy["P"], rtol=1e-10, atol=1e-12 * scale ** 2)


# ---------------------------------------------------------------- P7b: white noise, E[P_m] = sigma^2 sum w^2
def test_p7_white_noise_mean_power():
    rng = np.random.default_rng(5)
    sigma, T = 0.01, 4000
    x = rng.normal(0, sigma, 400 + (T - 1) * 400).astype(np.float32)
    out = orc.forward(x, fs=16000.0, n_fft=400, hop=400, window_kind=orc.HANN_PERIODIC, n_mels=80, fmin=0.0, fmax=8000.0)
    mean = out["P"].mean(axis=0)                                       # independent frames (hop = N)
    # E = sigma^2 * 150 = 0.015; P_m ~ exponential -> std of the mean = E/sqrt(T) = 1.6%; allow 6 sigma
    np.testing.assert_allclose(mean, sigma ** 2 * 150.0, rtol=0.10)
    assert mean.mean() == pytest.approx(0.015, rel=0.02)


# ---------------------------------------------------------------- P8: structural invariants from the paper
def test_p8_stacked_gemm_and_window_in_basis():
    """PAPER.md:162 (window absorbed in the basis == windowing the frame) and PAPER.md:173 (one GEMM against the
    stacked basis == two GEMMs): the oracle's direct sums equal the matrix products with its Eq. (5) matrices."""
    rng = np.random.default_rng(9)
    N, H = 400, 160
    x = rng.normal(0, 0.2, N + 6 * H).astype(np.float32)
    out = orc.forward(x, **dict(W16, want=("R", "I")))
    Wr, Wi = orc.basis(16000.0, N, orc.HANN_PERIODIC, 80, 0.0, 8000.0)
    X = np.stack([x[t * H:t * H + N] for t in range(7)]).astype(np.float64)      # UNwindowed frames
    RI = X @ np.concatenate([Wr, Wi]).T                                          # stacked [W^(r); W^(i)]
    np.testing.assert_allclose(out["R"], RI[:, :80], atol=1e-11)
    np.testing.assert_allclose(out["I"], RI[:, 80:], atol=1e-11)
    np.testing.assert_allclose(out["R"], X @ Wr.T, atol=1e-11)
    # basis rows: w[n] cos(2 pi f_m n / fs) -- check a few entries with python math
    f = orc.centres(0.0, 8000.0, 80)
    w = orc.window(orc.HANN_PERIODIC, N)
    for m, n in [(0, 1), (17, 123), (79, 399), (40, 200)]:
        assert Wr[m, n] == pytest.approx(w[n] * math.cos(2 * math.pi * f[m] * n / 16000.0), abs=1e-13)
        assert Wi[m, n] == pytest.approx(w[n] * math.sin(2 * math.pi * f[m] * n / 16000.0), abs=1e-13)


def test_p8_shift_by_one_hop():
    rng = np.random.default_rng(13)
    x = rng.normal(0, 0.2, 400 + 9 * 160).astype(np.float32)
    a = orc.forward(x, **W16)["P"]
    b = orc.forward(x[160:], **W16)["P"]
    np.testing.assert_array_equal(a[1:], b)


def test_p8_reflect_reading_a_equals_reading_b():
    """DESIGN.md reading R5: library-side reflect padding (PAD_REFLECT on the raw clip) == harness-side
    numpy reflect padding followed by unpadded framing, bit for bit in fp64."""
    rng = np.random.default_rng(17)
    raw = rng.normal(0, 0.2, 16000).astype(np.float32)
    padded = np.pad(raw, (200, 200), mode="reflect")
    a = orc.forward(padded, **dict(W16, drop_last=True))
    b = orc.forward(raw, **dict(W16, pad=orc.PAD_REFLECT, drop_last=True))
    assert a["P"].shape == (100, 80)
    np.testing.assert_array_equal(a["P"], b["P"])
    np.testing.assert_array_equal(a["L"], b["L"])


# ---------------------------------------------------------------- frame counts (BASELINE.json configs)
def test_frame_counts():
    assert orc.num_frames(16000, 400, 160) == 98                                  # configs[0]
    assert orc.num_frames(480400, 400, 160) == 3001                               # configs[1], pre-padded
    assert orc.num_frames(480400, 400, 160, drop_last=True) == 3000
    assert orc.num_frames(480000, 400, 160, pad=orc.PAD_REFLECT, drop_last=True) == 3000
    assert orc.num_frames(220500, 1024, 256) == 858 and orc.num_frames(220500, 2048, 512) == 427
    assert orc.num_frames(441000, 2048, 512) == 858 and orc.num_frames(441000, 4096, 1024) == 427
    assert orc.num_frames(399, 400, 160) == 0 and orc.num_frames(400, 400, 160) == 1
    assert orc.num_frames(400, 400, 160, drop_last=True) == 0


# ---------------------------------------------------------------- P9: the paper's op/byte count
def test_p9_arithmetic_intensity_from_paper():
    rows = dict((r[0], r[1:]) for r in _rows("paper_constants.txt"))
    N, M = 400, 80
    assert 2 * N * 2 * M / (4 * N + 4 * 2 * M) == pytest.approx(float(rows["ai_flop_per_byte"][0]), abs=5e-3)
    nat, db = map(float, rows["nat_to_db_example"])
    assert nat * 10 / math.log(10) == pytest.approx(db, abs=5e-3)


# ---------------------------------------------------------------- P10: DCT-II
@pytest.mark.parametrize("K,M", [(13, 40), (40, 128), (5, 5)])
def test_p10_dct_orthonormal_and_scipy(K, M):
    from scipy.fft import dct
    D = orc.dct_matrix(K, M)
    np.testing.assert_allclose(D @ D.T, np.eye(K), atol=1e-14)
    ref = dct(np.eye(M), type=2, norm="ortho", axis=0)[:K]                        # library special case
    np.testing.assert_allclose(D, ref, atol=1e-14)
    rng = np.random.default_rng(1)
    Lm = rng.normal(0, 3, (6, M))
    np.testing.assert_allclose(orc.dct_apply(Lm, K), dct(Lm, type=2, norm="ortho", axis=1)[:, :K], atol=1e-12)


def test_p10_dct_golden():
    D = orc.dct_matrix(13, 40)
    for k, m, val in _rows("dct_values.txt"):
        assert D[int(k), int(m)] == pytest.approx(float(val), abs=1e-11)


# ---------------------------------------------------------------- P11: brute force on a tiny problem
def test_p11_brute_force_tiny():
    N, H, M, L, fs, fmin, fmax, K = 8, 3, 3, 20, 100.0, 5.0, 45.0, 2
    rng = np.random.default_rng(23)
    x = rng.normal(0, 1, L).astype(np.float32)
    for win in (orc.HANN_PERIODIC, orc.HANN_SYMMETRIC):
        out = orc.forward(x, fs=fs, n_fft=N, hop=H, window_kind=win, n_mels=M, fmin=fmin, fmax=fmax, n_mfcc=K,
                          want=("R", "I", "P", "L", "C"))
        T = (L - N) // H + 1
        assert out["P"].shape == (T, M)
        mu = lambda f: 2595.0 * math.log10(1.0 + f / 700.0)
        for t in range(T):
            Ls = []
            for m in range(M):
                mu_m = mu(fmin) + (m + 1) * (mu(fmax) - mu(fmin)) / (M + 1)
                fm = 700.0 * (10.0 ** (mu_m / 2595.0) - 1.0)
                r = i = 0.0
                for n in range(N):
                    den = N if win == orc.HANN_PERIODIC else N - 1
                    wn = 0.5 - 0.5 * math.cos(2 * math.pi * n / den)
                    r += wn * float(x[t * H + n]) * math.cos(2 * math.pi * fm * n / fs)
                    i += wn * float(x[t * H + n]) * math.sin(2 * math.pi * fm * n / fs)
                assert out["R"][t, m] == pytest.approx(r, abs=1e-13)
                assert out["I"][t, m] == pytest.approx(i, abs=1e-13)
                assert out["P"][t, m] == pytest.approx(r * r + i * i, rel=1e-12, abs=1e-15)
                Ls.append(math.log10(max(r * r + i * i, 1e-10)))
                assert out["L"][t, m] == pytest.approx(Ls[-1], abs=1e-12)
            for k in range(K):
                c = sum((math.sqrt(1.0 / M) if k == 0 else math.sqrt(2.0 / M) * math.cos(math.pi * k * (2 * m + 1) / (2 * M))) * Ls[m]
                        for m in range(M))
                assert out["C"][t, k] == pytest.approx(c, abs=1e-12)


# ---------------------------------------------------------------- P12: clamp
def test_p12_all_zero_clamp():
    x = np.zeros(2000, np.float32)
    out = orc.forward(x, fs=16000.0, n_fft=400, hop=160, window_kind=orc.HANN_PERIODIC, n_mels=40, fmin=20.0, fmax=7600.0, n_mfcc=13)
    assert np.all(out["L"] == -10.0)
    np.testing.assert_allclose(out["C"][:, 0], -10.0 * math.sqrt(40), rtol=1e-14)
    np.testing.assert_allclose(out["C"][:, 1:], 0.0, atol=1e-13)


# ---------------------------------------------------------------- batch / ragged wrappers
def test_batch_and_ragged_wrappers():
    rng = np.random.default_rng(29)
    xs = [rng.normal(0, 0.1, n).astype(np.float32) for n in (900, 400, 1500, 399)]
    off = np.concatenate([[0], np.cumsum([len(v) for v in xs])])
    packed = np.concatenate(xs)
    kw = dict(fs=16000.0, n_fft=400, hop=160, window_kind=orc.HANN_PERIODIC, n_mels=40, fmin=20.0, fmax=7600.0, n_mfcc=13)
    rag = orc.forward_ragged(packed, off, **kw)
    np.testing.assert_array_equal(rag["frame_offsets"], [0, 4, 5, 12, 12])
    single = orc.forward(xs[2], **kw)
    np.testing.assert_array_equal(rag["C"][5:12], single["C"])
    dense = orc.forward_batch(np.stack([xs[0], xs[0][::-1].copy()]), **kw)
    assert dense["P"].shape == (2, 4, 40)


def test_ln_eps_form_closed_values():
    """Eq. (8) as printed, ln(S + eps): an on-bin tone of amplitude 0.5 gives S = (A N / 4)^2 = 2500 (pin P3) -> ln(2500 + eps);
    silence gives ln(eps); and the two log forms are tied by ln(S) = ln(10) log10(S) wherever eps is negligible."""
    from oracle import melt_oracle as orc
    np.testing.assert_allclose(orc.ln_eps(np.array([2500.0, 0.0]), 1e-10), [np.log(2500.0 + 1e-10), np.log(1e-10)], rtol=0, atol=1e-15)
    x = (0.5 * np.cos(2 * np.pi * 35 * np.arange(400) / 400.0 + 0.3)).astype(np.float32)
    ref = orc.forward(x, fs=16000.0, n_fft=400, hop=160, window_kind=0, n_mels=1, fmin=0.0, fmax=5600.0, want=("P", "L"))
    np.testing.assert_allclose(orc.ln_eps(ref["P"])[0, 0], np.log(2500.0), atol=1e-6)
    np.testing.assert_allclose(orc.ln_eps(ref["P"]), np.log(10.0) * ref["L"], atol=1e-9)


def test_whisper_norm_closed_values():
    from oracle import melt_oracle as orc
    L = np.array([[2.0, -10.0, -5.9], [-6.0, -6.1, 1.0]])
    # max = 2 -> floor -6: values below -6 are raised to it; then (L + 4) / 4
    np.testing.assert_allclose(orc.whisper_norm(L), [[1.5, -0.5, -0.475], [-0.5, -0.5, 1.25]], rtol=0, atol=1e-15)
