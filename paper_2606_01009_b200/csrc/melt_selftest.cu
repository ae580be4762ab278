// melt_selftest.cu -- self-test of the tensor-core building block of the forward kernels:
// D[128, n] = A[128, k] . B[n, k]^T with A written to tensor memory by threads (thread = row, tcgen05.st),
// B brought to shared memory by the bulk-copy engine in the no-swizzle canonical layout, one tcgen05.mma
// (A-from-TMEM form) per K-step issued by a single thread, completion through tcgen05.commit -> mbarrier,
// and the accumulator read back with tcgen05.ld.  Exactly the mechanisms melt_fwd_kernel relies on.
#include "melt_internal.h"
#include "../../include/melt_test.h"
#include "sm100_ptx.cuh"

#include <cuda_bf16.h>
#include <cuda_fp16.h>

namespace melt {

struct SelftestParams {
    int kind, n, k;
    const float *a;      // device [128, k] fp32
    const uint8_t *bimg; // device, K-step slabs of n*32 bytes
    float *d;            // device [128, n]
};

__global__ void __launch_bounds__(128, 1) selftest_umma_kernel(const SelftestParams p) {
    extern __shared__ __align__(128) uint8_t smem[];
    __shared__ __align__(8) uint64_t bar_b, bar_mma;
    __shared__ uint32_t tmem_base_s;

    const int tid = threadIdx.x, warp = tid >> 5;
    const int kstep = p.kind == OP_TF32 ? 8 : 16;
    const int nsteps = p.k / kstep;
    const uint32_t slab = (uint32_t)p.n * 32u;

    if (tid == 0) {
        mbar_init(smem_u32(&bar_b), 1);
        mbar_init(smem_u32(&bar_mma), 1);
        fence_barrier_init();
    }
    if (warp == 0) {
        tmem_alloc(smem_u32(&tmem_base_s), 512);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = tmem_base_s;

    if (tid == 0) {
        mbar_arrive_expect_tx(smem_u32(&bar_b), slab * (uint32_t)nsteps);
        for (int s = 0; s < nsteps; ++s)
            bulk_g2s(smem_u32(smem) + (uint32_t)s * slab, p.bimg + (size_t)s * slab, slab, smem_u32(&bar_b));
    }

    // A: row `tid` -> TMEM lane `tid`, columns [256, ...): 16-bit kinds pack two K elements per column (even k low).
    const uint32_t a_col0 = 256;
    const uint32_t lane_addr = tmem_base + ((uint32_t)(warp * 32) << 16);
    const float *arow = p.a + (size_t)tid * p.k;
    for (int s = 0; s < nsteps; ++s) {
        uint32_t v[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            if (p.kind == OP_TF32) {
                v[c] = cvt_tf32_rna(arow[s * 8 + c]);
            } else if (p.kind == OP_F16) {
                __half2 h = __floats2half2_rn(arow[s * 16 + 2 * c], arow[s * 16 + 2 * c + 1]);
                v[c] = *reinterpret_cast<uint32_t *>(&h);
            } else {
                __nv_bfloat162 h = __floats2bfloat162_rn(arow[s * 16 + 2 * c], arow[s * 16 + 2 * c + 1]);
                v[c] = *reinterpret_cast<uint32_t *>(&h);
            }
        }
        tmem_st8(lane_addr + a_col0 + (uint32_t)s * 8u, v);
    }
    tmem_wait_st();
    tc_fence_before();
    __syncthreads();

    if (tid == 0) {
        tc_fence_after();
        mbar_wait(smem_u32(&bar_b), 0);
        const uint32_t idesc = umma_idesc(p.kind == OP_F16 ? UMMA_F16 : (p.kind == OP_BF16 ? UMMA_BF16 : UMMA_TF32), (uint32_t)p.n);
        for (int s = 0; s < nsteps; ++s) {
            uint64_t bdesc = umma_smem_desc_kmajor_noswz(smem_u32(smem) + (uint32_t)s * slab, 128, 256);
            if (p.kind == OP_TF32) umma_ts_tf32(tmem_base, tmem_base + a_col0 + (uint32_t)s * 8u, bdesc, idesc, s > 0);
            else umma_ts_f16(tmem_base, tmem_base + a_col0 + (uint32_t)s * 8u, bdesc, idesc, s > 0);
        }
        tc_commit(smem_u32(&bar_mma));
    }
    mbar_wait(smem_u32(&bar_mma), 0);
    tc_fence_after();

    for (int c0 = 0; c0 < p.n; c0 += 16) {
        uint32_t v[16];
        tmem_ld16(lane_addr + (uint32_t)c0, v);
        tmem_wait_ld();
#pragma unroll
        for (int c = 0; c < 16; ++c) p.d[(size_t)tid * p.n + c0 + c] = __uint_as_float(v[c]);
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem_base, 512);
}


// ---------------------------------------------------------------------------------------------- CTA-pair variant
// D[256, n] = A[256, k] . B[n, k]^T on a cluster of two CTAs (tcgen05.mma.cta_group::2): CTA r holds rows
// [128 r, 128 r + 128) of A in ITS tensor memory and rows [r n/2, (r+1) n/2) of B in ITS shared memory; the leader
// (rank 0) issues every MMA; completion is multicast to one mbarrier per CTA.  This is the building block of
// melt_fwd2_kernel.
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(128, 1) selftest_umma2_kernel(const SelftestParams p) {
    extern __shared__ __align__(128) uint8_t smem[];
    __shared__ __align__(8) uint64_t bar_b, bar_mma, bar_afull;
    __shared__ uint32_t tmem_base_s;

    const int tid = threadIdx.x, warp = tid >> 5;
    const uint32_t rank = cluster_ctarank();
    const int kstep = p.kind == OP_TF32 ? 8 : 16;
    const int nsteps = p.k / kstep;
    const uint32_t slab = (uint32_t)(p.n / 2) * 32u;

    if (tid == 0) {
        mbar_init(smem_u32(&bar_b), 1);
        mbar_init(smem_u32(&bar_mma), 1);
        mbar_init(smem_u32(&bar_afull), 8);  // one elected lane per warp, 4 warps, 2 CTAs
        fence_barrier_init();
    }
    if (warp == 0) {
        tmem_alloc2(smem_u32(&tmem_base_s), 512);
        tmem_relinquish2();
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem_base = tmem_base_s;

    if (tid == 0) {
        mbar_arrive_expect_tx(smem_u32(&bar_b), slab * (uint32_t)nsteps);
        const uint8_t *src = p.bimg + (size_t)rank * slab * nsteps;
        for (int s = 0; s < nsteps; ++s)
            bulk_g2s(smem_u32(smem) + (uint32_t)s * slab, src + (size_t)s * slab, slab, smem_u32(&bar_b));
    }

    const uint32_t a_col0 = 256;
    const uint32_t lane_addr = tmem_base + ((uint32_t)(warp * 32) << 16);
    const float *arow = p.a + ((size_t)rank * 128 + tid) * p.k;
    for (int s = 0; s < nsteps; ++s) {
        uint32_t v[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            if (p.kind == OP_TF32) {
                v[c] = cvt_tf32_rna(arow[s * 8 + c]);
            } else if (p.kind == OP_F16) {
                __half2 h = __floats2half2_rn(arow[s * 16 + 2 * c], arow[s * 16 + 2 * c + 1]);
                v[c] = *reinterpret_cast<uint32_t *>(&h);
            } else {
                __nv_bfloat162 h = __floats2bfloat162_rn(arow[s * 16 + 2 * c], arow[s * 16 + 2 * c + 1]);
                v[c] = *reinterpret_cast<uint32_t *>(&h);
            }
        }
        tmem_st8(lane_addr + a_col0 + (uint32_t)s * 8u, v);
    }
    tmem_wait_st();
    tc_fence_before();
    mbar_wait(smem_u32(&bar_b), 0);  // every thread: this CTA's half of B has landed
    __syncwarp();
    if ((tid & 31) == 0) mbar_arrive_cluster_release(mapa_cluster(smem_u32(&bar_afull), 0));  // tell the leader: A rows + B half ready

    if (rank == 0 && tid == 0) {
        mbar_wait_cluster(smem_u32(&bar_afull), 0);
        tc_fence_after();
        const uint32_t idesc = umma_idesc(p.kind == OP_F16 ? UMMA_F16 : (p.kind == OP_BF16 ? UMMA_BF16 : UMMA_TF32), (uint32_t)p.n, 256u);
        for (int s = 0; s < nsteps; ++s) {
            uint64_t bdesc = umma_smem_desc_kmajor_noswz(smem_u32(smem) + (uint32_t)s * slab, 128, 256);
            if (p.kind == OP_TF32) umma2_ts_tf32(tmem_base, tmem_base + a_col0 + (uint32_t)s * 8u, bdesc, idesc, s > 0);
            else umma2_ts_f16(tmem_base, tmem_base + a_col0 + (uint32_t)s * 8u, bdesc, idesc, s > 0);
        }
        tc_commit2(smem_u32(&bar_mma), 3);
    }
    mbar_wait(smem_u32(&bar_mma), 0);
    tc_fence_after();

    float *drow = p.d + ((size_t)rank * 128 + tid) * p.n;
    for (int c0 = 0; c0 < p.n; c0 += 16) {
        uint32_t v[16];
        tmem_ld16(lane_addr + (uint32_t)c0, v);
        tmem_wait_ld();
#pragma unroll
        for (int c = 0; c < 16; ++c) drow[c0 + c] = __uint_as_float(v[c]);
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    if (warp == 0) tmem_dealloc2(tmem_base, 512);
}

}  // namespace melt

extern "C" int melt_selftest_umma(int kind, int n, int k, const float *a, const float *b, float *d) {
    using namespace melt;
    if (kind < 0 || kind > 2 || !a || !b || !d) return fail(MELT_ERR_INVALID_ARG, "melt_selftest_umma: bad argument");
    const int kstep = operand_kstep(kind);
    if (n < 16 || n > 256 || n % 16 || k < kstep || k > 256 || k % kstep)
        return fail(MELT_ERR_INVALID_ARG, "melt_selftest_umma: n=%d k=%d out of range", n, k);
    int dev = 0;
    cudaDeviceProp prop;
    MELT_CUDA(cudaGetDevice(&dev));
    MELT_CUDA(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10) return fail(MELT_ERR_UNSUPPORTED, "device is sm_%d%d, need sm_100", prop.major, prop.minor);

    const int nsteps = k / kstep;
    const size_t slab = (size_t)n * 32, img_bytes = slab * nsteps;
    if (img_bytes > 200 * 1024) return fail(MELT_ERR_INVALID_ARG, "melt_selftest_umma: B image too large");
    std::vector<uint8_t> img(img_bytes);
    for (int s = 0; s < nsteps; ++s)
        pack_b_slab(kind, n, [&](int r, int kk) { return (double)b[(size_t)r * k + s * kstep + kk]; }, img.data() + s * slab);

    float *da = nullptr, *dd = nullptr;
    uint8_t *dimg = nullptr;
    MELT_CUDA(cudaMalloc(&da, sizeof(float) * 128 * k));
    MELT_CUDA(cudaMalloc(&dd, sizeof(float) * 128 * n));
    MELT_CUDA(cudaMalloc(&dimg, img_bytes));
    MELT_CUDA(cudaMemcpy(da, a, sizeof(float) * 128 * k, cudaMemcpyHostToDevice));
    MELT_CUDA(cudaMemcpy(dimg, img.data(), img_bytes, cudaMemcpyHostToDevice));
    MELT_CUDA(cudaFuncSetAttribute(selftest_umma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)img_bytes));
    SelftestParams p{kind, n, k, da, dimg, dd};
    selftest_umma_kernel<<<1, 128, img_bytes>>>(p);
    MELT_CUDA(cudaGetLastError());
    MELT_CUDA(cudaDeviceSynchronize());
    MELT_CUDA(cudaMemcpy(d, dd, sizeof(float) * 128 * n, cudaMemcpyDeviceToHost));
    cudaFree(da);
    cudaFree(dd);
    cudaFree(dimg);
    return MELT_OK;
}


extern "C" int melt_selftest_umma2(int kind, int n, int k, const float *a, const float *b, float *d) {
    using namespace melt;
    if (kind < 0 || kind > 2 || !a || !b || !d) return fail(MELT_ERR_INVALID_ARG, "melt_selftest_umma2: bad argument");
    const int kstep = operand_kstep(kind);
    if (n < 32 || n > 256 || n % 16 || k < kstep || k > 256 || k % kstep)
        return fail(MELT_ERR_INVALID_ARG, "melt_selftest_umma2: n=%d k=%d out of range", n, k);
    int dev = 0;
    cudaDeviceProp prop;
    MELT_CUDA(cudaGetDevice(&dev));
    MELT_CUDA(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10) return fail(MELT_ERR_UNSUPPORTED, "device is sm_%d%d, need sm_100", prop.major, prop.minor);

    const int nsteps = k / kstep, nh = n / 2;
    const size_t slab = (size_t)nh * 32, half_bytes = slab * nsteps, img_bytes = 2 * half_bytes;
    if (half_bytes > 200 * 1024) return fail(MELT_ERR_INVALID_ARG, "melt_selftest_umma2: B image too large");
    std::vector<uint8_t> img(img_bytes);
    for (int r = 0; r < 2; ++r)
        for (int s = 0; s < nsteps; ++s)
            pack_b_slab(kind, nh, [&](int row, int kk) { return (double)b[(size_t)(r * nh + row) * k + s * kstep + kk]; },
                        img.data() + r * half_bytes + s * slab);

    float *da = nullptr, *dd = nullptr;
    uint8_t *dimg = nullptr;
    MELT_CUDA(cudaMalloc(&da, sizeof(float) * 256 * k));
    MELT_CUDA(cudaMalloc(&dd, sizeof(float) * 256 * n));
    MELT_CUDA(cudaMalloc(&dimg, img_bytes));
    MELT_CUDA(cudaMemcpy(da, a, sizeof(float) * 256 * k, cudaMemcpyHostToDevice));
    MELT_CUDA(cudaMemcpy(dimg, img.data(), img_bytes, cudaMemcpyHostToDevice));
    MELT_CUDA(cudaFuncSetAttribute(selftest_umma2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)half_bytes));
    SelftestParams p{kind, n, k, da, dimg, dd};
    selftest_umma2_kernel<<<2, 128, half_bytes>>>(p);
    MELT_CUDA(cudaGetLastError());
    MELT_CUDA(cudaDeviceSynchronize());
    MELT_CUDA(cudaMemcpy(d, dd, sizeof(float) * 256 * n, cudaMemcpyDeviceToHost));
    cudaFree(da);
    cudaFree(dd);
    cudaFree(dimg);
    return MELT_OK;
}

// ---------------------------------------------------------------------------------------------- shared-memory poison
__global__ void __launch_bounds__(256, 1) poison_smem_kernel(int n16) {
    extern __shared__ __align__(16) unsigned char ps[];
    uint4 *z = reinterpret_cast<uint4 *>(ps);
    for (int i = threadIdx.x; i < n16; i += 256) z[i] = make_uint4(0x7fc00000u, 0xffc00000u, 0x7f800001u, 0x7fc00000u);
}

extern "C" int melt_selftest_poison_smem(void *stream) {
    int dev = 0, sms = 0, smem = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess)
        return melt::fail(MELT_ERR_CUDA, "melt_selftest_poison_smem: device query failed");
    if (cudaFuncSetAttribute(poison_smem_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess)
        return melt::fail(MELT_ERR_CUDA, "melt_selftest_poison_smem: cannot opt in to %d bytes of shared memory", smem);
    poison_smem_kernel<<<4 * sms, 256, smem, (cudaStream_t)stream>>>(smem / 16);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return melt::fail(MELT_ERR_CUDA, "melt_selftest_poison_smem: %s", cudaGetErrorString(e));
    return MELT_OK;
}
