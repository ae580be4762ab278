"""GPU: the tensor-core building block (tcgen05.mma, A from tensor memory, B from shared memory in the
no-swizzle canonical layout) against a float64 matrix product of the operands rounded to the MMA's input type."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _round(v, kind):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(v, np.float32))
    if kind == 0:
        return t.to(torch.float16).to(torch.float64).numpy()
    if kind == 1:
        return t.to(torch.bfloat16).to(torch.float64).numpy()
    # tf32, round to nearest, ties away (cvt.rna) on A; B is rounded to nearest even on the host: use values on a
    # 2^-8 grid so both roundings are exact
    return v.astype(np.float64)


@pytest.mark.parametrize("kind", [0, 1, 2])
@pytest.mark.parametrize("n,k", [(16, 16), (80, 48), (128, 208), (256, 64), (48, 256)])
def test_umma_ts_matches_float64(kind, n, k):
    from paper_2606_01009_b200 import binding as mb
    rng = np.random.default_rng(100 * kind + n + k)
    if kind == 2:
        k = max(8, k // 2)
    # values on a coarse dyadic grid: exactly representable in fp16 / bf16 / tf32, products and sums exact in fp32
    a = rng.integers(-32, 33, (128, k)).astype(np.float32) / 16.0
    b = rng.integers(-32, 33, (n, k)).astype(np.float32) / 16.0
    d = mb.melt_selftest_umma(kind, a, b)
    ref = _round(a, kind) @ _round(b, kind).T
    np.testing.assert_array_equal(d.astype(np.float64), ref)


def test_umma_ts_random_fp16():
    from paper_2606_01009_b200 import binding as mb
    rng = np.random.default_rng(5)
    a = rng.normal(0, 1, (128, 208)).astype(np.float32)
    b = rng.normal(0, 1, (80, 208)).astype(np.float32)
    d = mb.melt_selftest_umma(0, a, b)
    ref = _round(a, 0) @ _round(b, 0).T
    np.testing.assert_allclose(d, ref, rtol=0, atol=2e-5 * np.abs(ref).max())


@pytest.mark.parametrize("kind", [0, 1, 2])
@pytest.mark.parametrize("n,k", [(32, 16), (80, 48), (128, 208), (256, 64), (48, 256)])
def test_umma2_cta_pair_matches_float64(kind, n, k):
    """tcgen05.mma.cta_group::2: 256 rows over a CTA pair, B split by rows between the two CTAs' shared memories."""
    from paper_2606_01009_b200 import binding as mb
    rng = np.random.default_rng(1000 + 100 * kind + n + k)
    if kind == 2:
        k = max(8, k // 2)
    a = rng.integers(-32, 33, (256, k)).astype(np.float32) / 16.0
    b = rng.integers(-32, 33, (n, k)).astype(np.float32) / 16.0
    d = mb.melt_selftest_umma2(kind, a, b)
    ref = _round(a, kind) @ _round(b, kind).T
    np.testing.assert_array_equal(d.astype(np.float64), ref)
