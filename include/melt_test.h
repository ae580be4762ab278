/*
 * melt_test.h -- test aids of libmelt_b200.so.  NOT part of the product API (include/melt.h): these entry points exist so
 * that tests/ can exercise the tensor-core building block of the forward kernels in isolation and can make sure that no forward
 * depends on what an earlier kernel left in shared memory.
 */
#ifndef MELT_TEST_H_
#define MELT_TEST_H_

#ifdef __cplusplus
extern "C" {
#endif

/*
 * Self-test of the tensor-core building block used by the forward kernels: D[128, n] = A[128, k] . B[n, k]^T
 * with A written to tensor memory by threads and B read from shared memory (tcgen05.mma, A-from-TMEM form).
 *   kind: 0 = fp16, 1 = bf16, 2 = tf32;  a, b host fp32 row-major (values are rounded to `kind` inside);
 *   d host fp32 [128, n] result.  n % 16 == 0, 16 <= n <= 256; k % 16 == 0 (fp16/bf16) or k % 8 == 0 (tf32), k <= 256.
 * Synchronous.  Returns a melt_status.
 */
int melt_selftest_umma(int kind, int n, int k, const float *a, const float *b, float *d);

/*
 * Self-test of the CTA-pair form of the same building block (tcgen05.mma.cta_group::2 on a cluster of two CTAs):
 * D[256, n] = A[256, k] . B[n, k]^T, CTA r of the pair holding rows [128 r, 128 r + 128) of A in its tensor memory
 * and rows [r n/2, (r+1) n/2) of B in its shared memory.  a host fp32 [256, k]; b host fp32 [n, k]; d host fp32
 * [256, n].  n % 16 == 0, 32 <= n <= 256; k as for melt_selftest_umma.  Synchronous.  Returns a melt_status.
 */
int melt_selftest_umma2(int kind, int n, int k, const float *a, const float *b, float *d);

/*
 * Test aid: fills the shared memory of every SM of the current device with NaN bit patterns (one resident block per SM
 * with the largest opt-in dynamic allocation), on `stream` (a cudaStream_t; NULL = default stream), asynchronously.
 * The forward kernels must not depend on what earlier kernels left in shared memory (staging
 * ring); tests call this before a forward.  Returns a melt_status.
 */
int melt_selftest_poison_smem(void *stream);

#ifdef __cplusplus
}
#endif
#endif /* MELT_TEST_H_ */
