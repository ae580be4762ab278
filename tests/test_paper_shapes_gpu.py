"""GPU parity on the paper's own shapes (SURVEY.md section 8(f) NEXT-1; PAPER.md:275-285 Table 4, :299 durations, :448-450 Mel-bin
sweep, :458 batch sweep): spectral front end (N = 400, H = 160, M = 80, 80-7600 Hz) and cepstral front end (N = 1200, H = 160,
M = 128, K = 40), symmetric Hann, against the fp64 oracle -- same bars as tests/test_parity_gpu.py."""
import numpy as np
import pytest

import parity_util as pu

pytestmark = pytest.mark.gpu


def _wl():
    from paper_2606_01009_b200 import workloads
    return workloads


def _orc():
    from oracle import melt_oracle
    return melt_oracle


def _cfg(name):
    c = dict(_wl().PAPER_CONFIGS[name])
    c["name"] = name
    return c


def _check_logmel(c, x, chunk=32):
    orc = _orc()
    L_gpu = pu.gpu_dense(c, x, "compensated")
    P_gpu = pu.gpu_dense(c, x, "compensated", output="power", n_mfcc=0)
    perr = lerr = 0.0
    for b0 in range(0, x.shape[0], chunk):
        ref = orc.forward_batch(x[b0:b0 + chunk], want=("P", "L"), **pu.oracle_kwargs(c, n_mfcc=0))
        assert ref["L"].shape == L_gpu[b0:b0 + chunk].shape
        perr = max(perr, pu.power_error(P_gpu[b0:b0 + chunk], ref["P"]))
        lerr = max(lerr, pu.log_error(L_gpu[b0:b0 + chunk], ref["L"], ref["P"]))
    print("\n[parity] %s frames=%d  |dP|/Pmax=%.3e  |dlog10|(masked)=%.3e" % (c["name"], L_gpu.shape[0] * L_gpu.shape[1], perr, lerr))
    assert np.isfinite(L_gpu).all()
    assert perr <= 2e-4 and lerr <= pu.LOG_BAR


@pytest.mark.parametrize("name", ["paper_spec_1s", "paper_spec_10s", "paper_spec_40s", "paper_spec_160s"])
def test_spectral_config_single_clips(name):
    c = _cfg(name)
    x = _wl().make_paper_inputs(name)["x"]
    assert x.shape == (1, c["clip_len"])
    _check_logmel(c, x)


@pytest.mark.parametrize("name", ["paper_mel40_160s", "paper_mel128_160s", "paper_mel256_160s", "paper_mel512_160s"])
def test_mel_bin_sweep_at_160s(name):
    c = _cfg(name)
    _check_logmel(c, _wl().make_paper_inputs(name)["x"])


@pytest.mark.parametrize("name", ["paper_batch1_4s", "paper_batch16_4s", "paper_batch256_4s"])
def test_batch_sweep_of_4s_utterances(name):
    c = _cfg(name)
    x = _wl().make_paper_inputs(name)["x"]
    assert x.shape == (c["n_clips"], 64000)
    _check_logmel(c, x)


@pytest.mark.parametrize("name", ["paper_cep_1s", "paper_cep_10s", "paper_cep_160s"])
def test_cepstral_config_n1200_m128_k40(name):
    """MFCCT with the paper's cepstral front end: 40 cepstra from 128 bins of a 75 ms window.  Two-stage bars of DESIGN.md reading
    R9: the tapped log-Mel against the oracle's, the cepstra against the oracle DCT of the GPU's own log-Mel, end to end bounded."""
    orc = _orc()
    c = _cfg(name)
    x = _wl().make_paper_inputs(name)["x"]
    C_gpu, L_gpu = pu.gpu_dense(c, x, "compensated", tap=True)
    ref = orc.forward_batch(x, want=("P", "L", "C"), **pu.oracle_kwargs(c))
    assert C_gpu.shape == ref["C"].shape and C_gpu.shape[2] == 40 and np.isfinite(C_gpu).all()
    lerr = pu.log_error(L_gpu, ref["L"], ref["P"])
    stage2 = max(float(np.abs(C_gpu[b] - orc.dct_apply(L_gpu[b], 40)).max()) for b in range(x.shape[0]))
    e2e = float(np.abs(C_gpu - ref["C"]).max())
    print("\n[parity] %s frames=%d  log-Mel err=%.3e  DCT-stage err=%.3e  end-to-end |dC|=%.3e" % (name, C_gpu.shape[1], lerr, stage2, e2e))
    assert lerr <= pu.LOG_BAR
    assert stage2 <= 1e-4
    D = orc.dct_matrix(40, 128)
    assert e2e <= float(np.abs(D).sum(axis=1).max()) * pu.LOG_BAR + 1e-4
