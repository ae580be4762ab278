"""GPU: the relaxed cluster synchronisation of the forward kernel against a build with full cluster barriers.

The product kernel uses execution-only cluster barriers at set-up and exit (barrier.cluster.arrive.relaxed: what they publish is
fenced separately, see melt_forward2_kernel.cuh) and overlaps consecutive launches (programmatic dependent launch).  A variant of
the library compiled with -DMELT_STRICT_CLUSTER_SYNC (barrier.cluster.arrive.release / wait.acquire everywhere) must give
BIT-IDENTICAL results: 1000 back-to-back forwards of alternating inputs into ONE output buffer, dense and ragged.  (SURVEY.md
section 4-iv; the compute-sanitizer logs are under profiles/.)"""
import ctypes as C
import os
import tempfile

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _run(L, c, xa, xb, n, offs=None):
    """n alternating forwards (xa, xb, xa, ...) into one buffer through library handle L; returns the final output."""
    import torch
    vp = C.c_void_p
    plan = L.melt_plan_create(c["fs"], c["n_fft"], c["hop"], c["window"], c["n_mels"], c["fmin"], c["fmax"], 0, c["n_mfcc"])
    assert plan
    try:
        assert L.melt_plan_set_option(plan, 0, int(c["layout"] == "feature_major")) == 0
        assert L.melt_plan_set_option(plan, 2, int(c.get("drop_last", False))) == 0
        assert L.melt_plan_set_option(plan, 6, 1) == 0                     # MELT_OPT_INPUT_READY: the overlapping form
        ta, tb = torch.from_numpy(xa).cuda(), torch.from_numpy(xb).cuda()
        st = torch.cuda.current_stream().cuda_stream
        if offs is None:
            B, Lc = xa.shape
            T, Cn = L.melt_num_frames(plan, Lc), L.melt_num_channels(plan)
            out = torch.zeros(B * T * Cn, device="cuda")
            for i in range(n):
                assert L.melt_forward(plan, vp((ta if i % 2 == 0 else tb).data_ptr()), B, Lc, vp(out.data_ptr()), vp(st)) == 0
        else:
            nclip = len(offs) - 1
            od = torch.from_numpy(offs).cuda()
            total = int(sum(L.melt_num_frames(plan, int(v)) for v in np.diff(offs)))
            out = torch.zeros(total * L.melt_num_channels(plan), device="cuda")
            fo = torch.zeros(nclip + 1, dtype=torch.int64, device="cuda")
            for i in range(n):
                assert L.melt_forward_ragged(plan, vp((ta if i % 2 == 0 else tb).data_ptr()), vp(od.data_ptr()), nclip, vp(out.data_ptr()),
                                             vp(fo.data_ptr()), vp(st)) == 0
        torch.cuda.synchronize()
        return out.cpu().numpy()
    finally:
        L.melt_plan_destroy(plan)


def test_strict_cluster_barriers_give_bit_identical_results():
    from paper_2606_01009_b200 import binding as mb, build, workloads as wl
    with tempfile.TemporaryDirectory() as tmp:
        strict = build.build(extra=["-DMELT_STRICT_CLUSTER_SYNC"], out_path=os.path.join(tmp, "libmelt_strict.so"), objdir=os.path.join(tmp, "obj"))
        Ls, Lp = mb.load(strict), mb.lib()
        c1 = wl.CONFIGS["cfg1"]
        d = wl.make_inputs("cfg1", 16)["x"]
        a = _run(Lp, c1, d[:8], d[8:], 1000)
        b = _run(Ls, c1, d[:8], d[8:], 1000)
        np.testing.assert_array_equal(a, b)
        assert np.isfinite(a).all()
        c3 = wl.CONFIGS["cfg3"]
        x, off = wl.speaker_ragged(48, 5, c3["fs"], 4000, 60000)
        rng = np.random.default_rng(0)
        x2 = (x + rng.normal(0, 0.01, x.shape)).astype(np.float32)
        a = _run(Lp, c3, x, x2, 300, off)
        b = _run(Ls, c3, x, x2, 300, off)
        np.testing.assert_array_equal(a, b)
