#pragma once
// melt_forward2_kernel.cuh -- the hot path (steps S1-S6 of SURVEY.md 8(a)) as ONE persistent, warp-specialised kernel on CTA
// PAIRS (thread-block clusters of two SMs, tcgen05.mma.cta_group::2).  A tile is 256 consecutive frames of one clip:
// CTA r of the pair owns frames [128 r, 128 r + 128) of it (its 128 tensor-memory lanes).
//
//   loader warp       raw fp32 signal (global) -> shared-memory staging ring, implicit im2col by the tensor-map engine: one
//                     cp.async.bulk.tensor box per chunk of 32 frames over a 3-D map of the signal whose row stride (hop) is
//                     smaller than its row extent, so overlapping frames are never materialised; the chunk is prefetched
//                     into L2 while the loader waits for a free slot.  Clip tails fall back to one bulk copy per hop-row.
//   converter warps   2 groups x 4 warps, thread = frame; the groups take K-steps round-robin.  128-bit conflict-free shared
//                     loads (row pitch = 4 * odd words), fold of the frame about the window centre (x[c+j] +- x[c-j]), split
//                     into tensor-core operands (fp16 hi + lo, or bf16, or tf32) with packed fp32 arithmetic and tcgen05.st
//                     straight into TENSOR MEMORY: the A operand never exists in shared or global memory.
//   basis             each CTA keeps HALF of the folded cos/sin basis (nb/2 Mel rows per operand kind) resident in shared
//                     memory, one barrier per K-step slab; the pair's tensor cores read both halves (cta_group::2).
//   MMA issuers       two warps of the leader CTA on different schedulers: one accumulates R (cos rows), the other I (sin
//                     rows); tcgen05.mma.cta_group::2 kind::f16 / kind::tf32, M = 256 over the pair, A from tensor memory,
//                     B from shared memory, fp32 accumulators in tensor memory (R in columns [0, nb), I in [nb, 2 nb)),
//                     double-buffered when they fit.  An iteration covers two K-steps.
//   epilogue warps    tcgen05.ld -> R^2 + I^2 -> log10(max(., 1e-10)) -> optional DCT-II (fp32 FMA) -> coalesced stores.
//
// Hand-offs are mbarriers; cross-CTA ones are remote arrivals (mapa) and multicast tcgen05.commit.  Consecutive forwards on a
// stream overlap through programmatic dependent launch (see launch_one).
#include "melt_plan.h"
#include "sm100_ptx.cuh"

#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include <algorithm>
#include <atomic>
#include <cstdlib>

namespace melt {

enum { P2_COMP = 0, P2_TF32 = 1, P2_BF16 = 2 };
// barrier indices (8 bytes each)
enum {
    V_STG_FULL = 0, V_STG_EMPTY = V2_MAX_STG, V_A_FULL = 2 * V2_MAX_STG, V_A_EMPTY = V_A_FULL + 16, V_ACC_FULL = V_A_EMPTY + 16,
    V_ACC_EMPTY = V_ACC_FULL + 2, V_B_FULL = V_ACC_EMPTY + 2, V_B_PEER = V_B_FULL + V2_MAX_UNITS, V_DONE = V_B_PEER + V2_MAX_UNITS, V_STG_READY = V_DONE + 1, V_B_EMPTY = V_STG_READY + V2_MAX_STG, V_INFO = V_B_EMPTY + 8, V_KFULL = V_INFO + 32, V_KEMPTY = V_KFULL + 24,
    V_P_READY = V_KEMPTY + 24, V_D2_FULL = V_P_READY + 1, V_FB_FULL = V_D2_FULL + 1, V_FB_PEER = V_FB_FULL + 1,   // MODE 4 (filterbank product)
    V_NBARS = V_FB_PEER + 1
};
constexpr int V2_MAX_A_SLOTS = 16;
constexpr int W_LOAD = 0, W_MMA = 1, W_BASIS = 2, W_MMA2 = 3, W_EPI0 = 4, W_CONV0 = 8;

__device__ __forceinline__ float4 lds128(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ float4 ldg128(const char *p) {   // read-only path, 16-byte aligned
    float4 v;
    asm volatile("ld.global.nc.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ float ldg32(const char *p) {
    float v;
    asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ float lds32(uint32_t addr) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
// packed fp32 pairs in one 64-bit register (sm_100 FADD2 / FMUL2: two lanes per issue slot)
__device__ __forceinline__ uint64_t f2_pack(float lo, float hi) {
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ uint64_t f2_add(uint64_t a, uint64_t b) {
    uint64_t r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ uint64_t f2_sub(uint64_t a, uint64_t b) {
    uint64_t r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ uint64_t f2_fma(uint64_t a, uint64_t b, uint64_t c) {
    uint64_t r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ void f2_unpack(uint64_t a, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a)); }
__device__ __forceinline__ uint64_t f2_mul(uint64_t a, uint64_t b) {
    uint64_t r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ __half2 f2_to_half2(uint64_t a) {   // round to nearest even, lane 0 -> low half
    float lo, hi;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a));
    return __floats2half2_rn(lo, hi);
}
__device__ __forceinline__ uint64_t half2_to_f2(__half2 h) {
    const float2 f = __half22float2(h);
    return f2_pack(f.x, f.y);
}
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// Optional event trace (development builds only, -DMELT_TRACE): lane 0 of every warp of cluster 0 appends (tag, clock) pairs.
#ifdef MELT_TRACE
static __device__ long long *g_melt_trace = nullptr;   // [2 ranks][16 warps][1024] events; one copy per translation unit (set by melt_debug_set_trace in melt_forward2_comp.cu)
#define TRACE_WORDS (2 * 16 * 1024 + 592 + 148 * 8 + 64)   // one region per traced launch (K2Params::trace_slot)
#define TRACE_BASE (g_melt_trace + (size_t)p.trace_slot * TRACE_WORDS)
#define TRACE_PT(i) do { if (g_melt_trace && threadIdx.x == 0) TRACE_BASE[2 * 16 * 1024 + 592 + blockIdx.x * 8 + (i)] = clock64(); } while (0)
#define TRACE_DECL int tr_n = 0; long long *tr_buf = (g_melt_trace && cluster_id_x() == 0 && (threadIdx.x & 31) == 0 && threadIdx.x < 512) ? TRACE_BASE + ((size_t)cluster_ctarank() * 16 + (threadIdx.x >> 5)) * 1024 : nullptr;
#define TRACE(tag) do { if (tr_buf && tr_n < 1023) tr_buf[++tr_n] = ((long long)(tag) << 48) | (clock64() & 0xFFFFFFFFFFFFll); if (tr_buf) tr_buf[0] = tr_n; } while (0)
#define TRACE_CTA(which) do { if (g_melt_trace && threadIdx.x == 0) { TRACE_BASE[2 * 16 * 1024 + blockIdx.x * 2 + (which)] = (long long)globaltimer_ns(); TRACE_BASE[2 * 16 * 1024 + 296 + blockIdx.x * 2 + (which)] = clock64(); } } while (0)
#else
#define TRACE_CTA(which) do { } while (0)
#define TRACE_PT(i) do { } while (0)
#define TRACE_DECL
#define TRACE(tag) do { } while (0)
#endif

// Log-Mel epilogue of the 16-bin blocks blk0, blk0 + step, ... of one tile for one thread (= frame).  Used when a tile's
// accumulator is drained by several warps per lane quarter (single accumulator stage: the MMAs of the next tile cannot
// start before the drain, so the converter warps take their share of it instead of waiting).
__device__ __forceinline__ void epi_fast_share(uint32_t t_r, uint32_t t_i, int nb, int n_mels, float *optr, long long cstride,
                                               bool valid, float off, int blk0, int step, int ot = 0) {
    const float kLog10_2 = 0.30102999566398120f;
    const bool vec4 = cstride == 1 && ((reinterpret_cast<uintptr_t>(optr) & 15) == 0) && ot == 0;   // (warp-uniform: rows are n_ch * 4 bytes apart)
    if (ot != 0) {
        // 16-bit output (MELT_OPT_OUTPUT_DTYPE): optr / cstride count 2-byte elements; fp16 or bf16, round to nearest even
        unsigned short *o16 = reinterpret_cast<unsigned short *>(optr);
        for (int c0 = 16 * blk0; c0 < nb; c0 += 16 * step) {
            uint32_t vr[16], vi[16];
            tmem_ld16(t_r + (uint32_t)c0, vr);
            tmem_ld16(t_i + (uint32_t)c0, vi);
            tmem_wait_ld();
            const int nrem = n_mels - c0;
            unsigned short *o = o16 + (long long)c0 * cstride;
            unsigned short bits[16];
#pragma unroll
            for (int c = 0; c < 16; ++c) {
                const float r = __uint_as_float(vr[c]), im = __uint_as_float(vi[c]);
                const float v = fmaxf(fmaf(lg2_ftz(fmaf(r, r, im * im)), kLog10_2, off), -10.f);
                bits[c] = ot == 1 ? __half_as_ushort(__float2half_rn(v)) : __bfloat16_as_ushort(__float2bfloat16_rn(v));
            }
            if (nrem >= 16 && cstride == 1 && (reinterpret_cast<uintptr_t>(o) & 15) == 0) {   // frame-major rows: two 128-bit stores
                if (valid) {
                    uint32_t w[8];
#pragma unroll
                    for (int c = 0; c < 8; ++c) w[c] = (uint32_t)bits[2 * c] | ((uint32_t)bits[2 * c + 1] << 16);
                    reinterpret_cast<uint4 *>(o)[0] = make_uint4(w[0], w[1], w[2], w[3]);
                    reinterpret_cast<uint4 *>(o)[1] = make_uint4(w[4], w[5], w[6], w[7]);
                }
            } else {
#pragma unroll
                for (int c = 0; c < 16; ++c) {
                    if (valid && c < nrem) *o = bits[c];
                    o += cstride;
                }
            }
        }
        return;
    }
    for (int c0 = 16 * blk0; c0 < nb; c0 += 16 * step) {
        uint32_t vr[16], vi[16];
        tmem_ld16(t_r + (uint32_t)c0, vr);
        tmem_ld16(t_i + (uint32_t)c0, vi);
        tmem_wait_ld();
        const int nrem = n_mels - c0;   // bins of this block that exist
        float *o = optr + (long long)c0 * cstride;
        if (nrem >= 16 && vec4) {
            // frame-major rows (cstride == 1, 16-byte aligned): the block is 64 contiguous bytes of this thread's row -- four 128-bit
            // stores fill whole 32-byte sectors (one 4-byte store per bin touches 32 sectors per instruction for 128 useful bytes)
            if (valid) {
                float v[16];
#pragma unroll
                for (int c = 0; c < 16; ++c) {
                    const float r = __uint_as_float(vr[c]), im = __uint_as_float(vi[c]);
                    v[c] = fmaxf(fmaf(lg2_ftz(fmaf(r, r, im * im)), kLog10_2, off), -10.f);
                }
#pragma unroll
                for (int c = 0; c < 16; c += 4) *reinterpret_cast<float4 *>(o + c) = make_float4(v[c], v[c + 1], v[c + 2], v[c + 3]);
            }
        } else if (nrem >= 16) {
            if (valid) {
#pragma unroll
                for (int c = 0; c < 16; ++c) {
                    const float r = __uint_as_float(vr[c]), im = __uint_as_float(vi[c]);
                    *o = fmaxf(fmaf(lg2_ftz(fmaf(r, r, im * im)), kLog10_2, off), -10.f);   // Eq. (4), Eq. (8) in contract form
                    o += cstride;
                }
            }
        } else {
#pragma unroll
            for (int c = 0; c < 16; ++c) {
                const float r = __uint_as_float(vr[c]), im = __uint_as_float(vi[c]);
                if (valid && c < nrem) *o = fmaxf(fmaf(lg2_ftz(fmaf(r, r, im * im)), kLog10_2, off), -10.f);
                o += cstride;
            }
        }
    }
}

// Epilogue of one tile for one thread (= frame) in the general case: power or log output, optional tap of the log-Mel
// matrix, optional DCT-II.  The DCT keeps 16 accumulators: more than 16 cepstra are produced in blocks of 16, the log-Mel
// values being re-formed from tensor memory for every block (the paper's K = 40 costs three passes over the bins; keeping 40
// .. 64 accumulators per thread instead pushed the whole kernel to 128 registers with spills).  Returns after handing the
// accumulator stage back.
template <bool HAS_DCT>
__device__ __forceinline__ void epi_generic(const K2Params &p, uint32_t t_r, uint32_t t_i, const float *dct_s, float *optr, float *tptr,
                                            long long cstride, bool valid, int lane, uint32_t acc_empty_bar, int nm,
                                            float *stage, float *warp_out, int nvalid) {
    const bool ln_form = p.output_power == 2;
    const float la = ln_form ? p.out_scale : 1.f, lb = ln_form ? p.ln_eps : 0.f;
    const float lc = ln_form ? 0.69314718055994531f : 0.30102999566398120f, ld = ln_form ? 0.f : p.out_log10_offset;
    const float lmin = ln_form ? -3.0e38f : -10.f;
    const int K = p.n_mfcc;
    for (int q0 = 0; q0 < (HAS_DCT ? K : 1); q0 += 16) {
        float cacc[HAS_DCT ? 16 : 1];
#pragma unroll
        for (int k = 0; k < (HAS_DCT ? 16 : 1); ++k) cacc[k] = 0.f;
        for (int c0 = 0; c0 < p.nb; c0 += 16) {
            uint32_t vr[16], vi[16];
            tmem_ld16(t_r + (uint32_t)c0, vr);
            tmem_ld16(t_i + (uint32_t)c0, vi);
            tmem_wait_ld();
            // The 16 values of the block first, all independent (power, one MUFU.LG2, FMA, max each), THEN the DCT / the stores: with
            // the per-bin guard `m < nm` around everything, every bin was a branch target of its own and its latency chain (FMA ->
            // LG2 -> FMA -> max -> 16 FMAs) ran alone -- the four epilogue warps took ~7000 of every ~8000 cycles of a tile of the
            // speaker-style batch and the MMA issuers waited 3300 of them for an accumulator stage (r02 trace).  Bins beyond the
            // plan's (the block is padded to 16) carry zero basis rows, hence finite values, and meet ZERO rows of the DCT table
            // (cleared at set-up), so the DCT needs no guard; the stores keep theirs as a predicate.
            const int nfull = nm - c0;   // bins of this block that exist (>= 16: all of them)
            float v[16];
            const bool is_power = p.output_power == 1;
#pragma unroll
            for (int c = 0; c < 16; ++c) {
                const float r = __uint_as_float(vr[c]), im = __uint_as_float(vi[c]);
                const float praw = fmaf(r, r, im * im);                                          // Eq. (4)
                // one formula for both log forms (two branches inside the unrolled bin loop cost the ragged MFCCT batch 35 %):
                //   contract form (Eq. 8, DESIGN R2): log10(max(S, 1e-10)) = max(lg2(1 * praw + 0) * log10(2) + offset, -10)
                //   printed form:                     ln(S + eps)          = max(lg2(scale * praw + eps) * ln(2) + 0, -inf)
                const float lv = fmaxf(fmaf(lg2_ftz(fmaf(praw, la, lb)), lc, ld), lmin);
                v[c] = is_power ? praw * p.out_scale : lv;
            }
            if (HAS_DCT) {
                if (q0 == 0 && tptr && valid) {
#pragma unroll
                    for (int c = 0; c < 16; ++c)
                        if (c < nfull) tptr[(c0 + c) * cstride] = v[c];
                }
                const float *drow = dct_s + c0 * p.dct_pitch + q0;
                // (scalar FMAs on purpose: packed FFMA2 pairs measured 6.5 % SLOWER on the ragged MFCCT batch, 226.7 vs 212.8 us)
#pragma unroll
                for (int c = 0; c < 16; ++c) {
#pragma unroll
                    for (int q4 = 0; q4 < 4; ++q4) {   // the table's rows are zero padded to whole blocks of 16 cepstra
                        const float4 d = *reinterpret_cast<const float4 *>(drow + c * p.dct_pitch + 4 * q4);   // D[q0 + 4 q4 .. + 3][c0 + c]
                        cacc[4 * q4 + 0] = fmaf(d.x, v[c], cacc[4 * q4 + 0]);
                        cacc[4 * q4 + 1] = fmaf(d.y, v[c], cacc[4 * q4 + 1]);
                        cacc[4 * q4 + 2] = fmaf(d.z, v[c], cacc[4 * q4 + 2]);
                        cacc[4 * q4 + 3] = fmaf(d.w, v[c], cacc[4 * q4 + 3]);
                    }
                }
            } else if (valid) {
#pragma unroll
                for (int c = 0; c < 16; ++c)
                    if (c < nfull) optr[(c0 + c) * cstride] = v[c];
            }
        }
        if (!HAS_DCT || q0 + 16 >= K) {   // last pass over the accumulators: the MMAs of the tile after next may overwrite them
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_remote(acc_empty_bar);
        }
        if (HAS_DCT && stage != nullptr) {                                                           // Eq. (9)
            // frame-major cepstra: the 32 frames of this warp are 32 * n_mfcc consecutive floats of the output.  Every thread
            // parks its row in shared memory, then the warp writes the block with consecutive lanes on consecutive addresses
            // (a thread storing its own row touches n_mfcc scattered 4-byte pieces: 13x the sector traffic for 13 cepstra).
#pragma unroll
            for (int k = 0; k < 16; ++k)
                if (q0 + k < K) stage[lane * K + q0 + k] = cacc[k];
        } else if (HAS_DCT && valid) {
#pragma unroll
            for (int k = 0; k < 16; ++k)
                if (q0 + k < K) optr[(q0 + k) * cstride] = cacc[k];
        }
    }
    if (HAS_DCT && stage != nullptr) {
        __syncwarp();
        const int n_out = nvalid * K;
        for (int w = lane; w < n_out; w += 32) warp_out[w] = stage[w];
        __syncwarp();
    }
}

// MODE 4, the conventional front end: the accumulators hold R | I of the N/2 + 1 DFT
// bins of this thread's frame.  (1) power per bin, split into a bf16 "hi" and a bf16 "mid" part (P = hi + mid to ~2^-17) and written
// back IN PLACE over R as the A operand of a second tensor-core product: the 16 bins of a block become 8 columns of hi pairs and 8
// columns of mid pairs -- K-step s of that product reads columns [16 s, 16 s + 8) and [16 s + 8, 16 s + 16); (2) hand-off to the
// issuer warp, which multiplies by the triangular filterbank (bf16 hi + mid slabs in shared memory; hi.hi + mid.hi + hi.mid) into
// the columns of I, no longer needed; (3) log10(max(., 1e-10)) of the Mel energies, stored like a log-Mel row.
__device__ __forceinline__ void epi_fbank(const K2Params &p, uint32_t t_r, uint32_t t_i, float *optr, long long cstride, bool valid,
                                          int lane, uint32_t p_ready_remote, uint32_t d2_full_bar, uint32_t d2_parity, uint32_t acc_empty_bar) {
    const float kLog10_2 = 0.30102999566398120f;
    for (int c0 = 0; c0 < p.nb; c0 += 16) {
        uint32_t vr[16], vi[16], w[16];
        tmem_ld16(t_r + (uint32_t)c0, vr);
        tmem_ld16(t_i + (uint32_t)c0, vi);
        tmem_wait_ld();
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const float r0 = __uint_as_float(vr[2 * j]), i0 = __uint_as_float(vi[2 * j]);
            const float r1 = __uint_as_float(vr[2 * j + 1]), i1 = __uint_as_float(vi[2 * j + 1]);
            const float p0 = fmaf(r0, r0, i0 * i0), p1 = fmaf(r1, r1, i1 * i1);            // |X[k]|^2 (scaled by the operand scales)
            const __nv_bfloat162 h = __floats2bfloat162_rn(p0, p1);
            const float2 hf = __bfloat1622float2(h);
            const __nv_bfloat162 m = __floats2bfloat162_rn(p0 - hf.x, p1 - hf.y);
            w[j] = *reinterpret_cast<const uint32_t *>(&h);                                 // K elements (2 j, 2 j + 1): low half first
            w[8 + j] = *reinterpret_cast<const uint32_t *>(&m);
        }
        tmem_st16(t_r + (uint32_t)c0, w);
    }
    tmem_wait_st();
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive_remote(p_ready_remote);
    mbar_wait(d2_full_bar, d2_parity);
    tc_fence_after();
    const bool vec4 = cstride == 1 && ((reinterpret_cast<uintptr_t>(optr) & 15) == 0);   // warp-uniform (rows are n_ch * 4 bytes apart)
    for (int c0 = 0; c0 < p.fb_nb; c0 += 16) {
        uint32_t d[16];
        tmem_ld16(t_i + (uint32_t)c0, d);
        tmem_wait_ld();
        float v[16];
#pragma unroll
        for (int c = 0; c < 16; ++c) v[c] = fmaxf(fmaf(lg2_ftz(__uint_as_float(d[c])), kLog10_2, p.out_log10_offset), -10.f);
        const int nrem = p.fb_mels - c0;
        float *o = optr + (long long)c0 * cstride;
        if (nrem >= 16 && vec4) {
            if (valid) {
#pragma unroll
                for (int c = 0; c < 16; c += 4) *reinterpret_cast<float4 *>(o + c) = make_float4(v[c], v[c + 1], v[c + 2], v[c + 3]);
            }
        } else {
#pragma unroll
            for (int c = 0; c < 16; ++c) {
                if (valid && c < nrem) *o = v[c];
                o += cstride;
            }
        }
    }
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive_remote(acc_empty_bar);
}

// Address of output element `idx` (elements of 4 bytes, or of 2 bytes with a 16-bit MELT_OPT_OUTPUT_DTYPE).
__device__ __forceinline__ float *out_at(const K2Params &p, long long idx) {
    return p.out_dtype == 0 ? p.out + idx : reinterpret_cast<float *>(reinterpret_cast<unsigned short *>(p.out) + idx);
}

// Where the 32-frame chunk of one lane quarter of a tile lives.
struct Tile2 {
    int clip, t0;      // clip index, first frame of the chunk within the clip
    long long T;       // frames of the clip
    long long s0;      // index of the clip's first sample in x
    long long f0;      // index of the clip's first frame in the (packed or dense) frame order
    int pass;          // pass over the Mel bins (more than 128 bins: every tile is visited once per pass)
};
// The clips are cut into 32-frame CHUNKS (the unit one converter / epilogue warp works on) and a tile is any 8 consecutive chunks
// of the packed chunk order -- the four lane quarters of a CTA may belong to different clips, so the tail of a clip wastes at most
// 31 rows instead of up to 255.  Ragged batches: only the loader looks chunks up (chunk_prefix, written by the scan kernel, is the
// exclusive prefix of chunks per clip); it hands what the other warps need to them in shared memory (ChunkInfo).  Dense batches:
// every warp finds its chunk by arithmetic (ChunkCursor).
struct ChunkInfo {
    long long row0;   // index of the chunk's first frame in the packed output
    int nvalid;       // frames of the chunk that exist (0 .. 32)
    int dlt;          // words by which the staged chunk sits further into its rows than the load table says (clip offset & 3)
};
// Dense batches: the clips are cut into 32-frame chunks and a tile is any 8 consecutive chunks of the batch (chunks_per_clip per
// clip, clip after clip), as in a ragged batch: the tail of a clip wastes at most 31 rows instead of up to 255 -- 376 instead of 384
// tiles on the Whisper-shaped batch, 216 instead of 256 on 64 x 858 frames.  Chunk g = 8 tile + 4 rank + q is chunk g % chunks_per_clip
// of clip g / chunks_per_clip; Tile2::t0 = first frame of THAT chunk within its clip.
// The order in which the loader issues the four chunks of a tile.  The staging ring holds less than two tiles, so the chunk issued LAST
// only starts when a chunk of the current tile is released, and its converter warps wait for it at every tile boundary (~1000 cycles
// in the r02 trace).  Dense batches give that wait to lane quarter 2 -- whose converter warps share their scheduler with no MMA issuer
// and run a K-step ~230 cycles faster than those of quarters 1 and 3 -- instead of quarter 3, the slowest.  Ragged batches keep the
// natural order (the loader's clip search only moves forward).
#ifndef MELT_CHUNK_ORDER
#define MELT_CHUNK_ORDER 0x2013   /* nibble qi: quarter issued qi-th = 3, 1, 0, 2 */
#define MELT_CHUNK_POS 0x0312     /* nibble q: position of quarter q in that order */
#endif
template <bool RAGGED>
__device__ __forceinline__ int chunk_order(int qi) { return RAGGED ? qi : (MELT_CHUNK_ORDER >> (4 * qi)) & 3; }
template <bool RAGGED>
__device__ __forceinline__ int chunk_pos(int q) { return RAGGED ? q : (MELT_CHUNK_POS >> (4 * q)) & 3; }

// The mapping without a division per tile: a CTA's visits are tile_step apart, so the chunk of a fixed lane quarter advances by
// a fixed number of chunks from one visit to the next -- (adv_b clips, adv_c chunks) with one carry; with several passes over the
// bins (a tile is visited once per pass, visit = tile * passes + pass) the pass advances too, and its carry moves one tile (8 chunks)
// further.  (Four divisions per tile in the loader warp, the pacemaker of the kernel, cost 2-4 % on the workloads whose tile count
// the packing does not change.)
struct ChunkCursor {
    int b, c, pass, adv_b, adv_c, adv_p, cpc, passes;
    __device__ __forceinline__ void init(const K2Params &p, int first_visit, int visit_step, int rank, int q) {
        cpc = p.chunks_per_clip;
        passes = p.passes;
        const int tile0 = first_visit / passes, dt = visit_step / passes;
        pass = first_visit - tile0 * passes;
        adv_p = visit_step - dt * passes;
        const int g0 = tile0 * 8 + rank * 4 + q;
        b = g0 / cpc;
        c = g0 - b * cpc;
        const int adv = 8 * dt;
        adv_b = adv / cpc;
        adv_c = adv - adv_b * cpc;
    }
    __device__ __forceinline__ void next() {
        b += adv_b;
        c += adv_c;
        pass += adv_p;
        if (pass >= passes) { pass -= passes; c += 8; }
        while (c >= cpc) { c -= cpc; ++b; }
    }
    // the chunk dq lane quarters further on (dq < 4)
    __device__ __forceinline__ void get(const K2Params &p, int dq, Tile2 &ti) const {
        int bb = b, cc = c + dq;
        while (cc >= cpc) { cc -= cpc; ++bb; }
        if (bb >= p.n_clips) { bb = 0; cc = cpc; }   // beyond the last chunk of the batch: t0 >= T, no frames
        ti.pass = pass;
        ti.clip = bb;
        ti.t0 = cc * 32;
        ti.T = p.frames_per_clip;
        ti.s0 = (long long)bb * p.len;
        ti.f0 = (long long)bb * p.frames_per_clip;
    }
};

// Ragged batches: a clip starts at any sample of the packed buffer, but the copy engines want 16-byte aligned sources, so a
// chunk is fetched from the aligned sample below its start: frame sample n then sits dlt = (clip offset & 3) words further
// into the staged rows than the load table says.  The converter reads the aligned quads around it (one more per direction)
// and picks its 2 KS samples with offsets that are compile-time constants of the instantiation <DLT>: no pass over the chunk
// in shared memory (an earlier version shifted every chunk down by dlt words first: ~2600 cycles per tile).
//   forward run  : table quads tb[0 .. NQ) (samples n0 + 4 i ..) and the quad after them, tb[9]
//   mirrored run : table quads tb[4 .. 4 + NQ) (samples run - SIGMA + 4 i ..) and the quad after them, tb[10]
// Rows overlap by their padding words (a staged row is hop + 4 samples of the signal), so the words after a quad that ends a
// row are the first samples of the next row: reading dlt words past a table quad never leaves the signal.
template <int KS, int SIGMA, int DLT>
__device__ __forceinline__ void load_shifted(uint32_t fb, const short *tb, float (&fw)[KS], float (&bw)[KS]) {
    constexpr int NQ = KS / 4, BS = SIGMA + DLT;
    float wf[KS + 4], wb[KS + 4];
#pragma unroll
    for (int i = 0; i <= NQ; ++i) {
        const float4 f = lds128(fb + (uint32_t)(int)tb[i < NQ ? i : 9]);
        wf[4 * i + 0] = f.x; wf[4 * i + 1] = f.y; wf[4 * i + 2] = f.z; wf[4 * i + 3] = f.w;
        const float4 g = lds128(fb + (uint32_t)(int)tb[i < NQ ? 4 + i : 10]);
        wb[4 * i + 0] = g.x; wb[4 * i + 1] = g.y; wb[4 * i + 2] = g.z; wb[4 * i + 3] = g.w;
    }
#pragma unroll
    for (int e = 0; e < KS; ++e) {
        fw[e] = wf[e + DLT];
        bw[KS - 1 - e] = wb[BS + e];   // sample `run + e` of the descending run is the partner of pair KS - 1 - e
    }
}

// K-block staging (very long windows): kb points at samples n0 .. of the thread's frame (forward run of the K-step, n0 = a0 + KS u)
// and kb + half at run - SIGMA .. (its mirrored run from the aligned sample below it), both 16-byte aligned, KS + 4 samples each.
template <int KS, int SIGMA>
__device__ __forceinline__ void load_kstaged(uint32_t kb, uint32_t half, float (&fw)[KS], float (&bw)[KS]) {
    constexpr int NQ = KS / 4, NB = NQ + (SIGMA > 0 ? 1 : 0);
    float wb[KS + 4];
#pragma unroll
    for (int i = 0; i < NQ; ++i) {
        const float4 f = lds128(kb + 16u * (uint32_t)i);
        fw[4 * i + 0] = f.x; fw[4 * i + 1] = f.y; fw[4 * i + 2] = f.z; fw[4 * i + 3] = f.w;
    }
#pragma unroll
    for (int i = 0; i < NB; ++i) {
        const float4 g = lds128(kb + half + 16u * (uint32_t)i);
        wb[4 * i + 0] = g.x; wb[4 * i + 1] = g.y; wb[4 * i + 2] = g.z; wb[4 * i + 3] = g.w;
    }
#pragma unroll
    for (int e = 0; e < KS; ++e) bw[KS - 1 - e] = wb[SIGMA + e];   // sample `run + e` of the descending run is the partner of pair KS - 1 - e
}

template <int PREC, int SIGMA, bool RAGGED, int MODE, bool STREAM, bool DIRECT>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(v2_threads(MODE), 1) melt_fwd2_kernel(const __grid_constant__ K2Params p) {
    extern __shared__ __align__(128) uint8_t smem[];
    // Who drains the accumulators: MODE 0 the four epilogue warps alone (next to two converter groups); MODE 1 (single accumulator
    // stage, log-Mel) the epilogue warps and the converter warps together; MODE 2 (log-Mel) there are no epilogue warps -- they
    // form a third converter group and every converter warp drains a third of the bins of the previous tile; MODE 3 (log-Mel):
    // four drain warps AND three converter groups, 640 threads; MODE 5: MODE 3 with a second set of four drain warps (warps 20-23,
    // the odd 16-bin blocks), 768 threads (launch_one says which is used when).
    constexpr bool SHARE = MODE == 1 || MODE == 2;
    constexpr bool FB = MODE == 4;                                        // conventional front end: filterbank product after the power (see epi_fbank)
    static_assert(!FB || (STREAM && !DIRECT && !RAGGED && PREC == P2_COMP), "MODE 4: dense batches, streamed basis, compensated operands");
    constexpr int NG = (MODE == 2 || MODE == 3 || MODE == 5) ? V2_CONV_GROUPS : V2_CONV_GROUPS - 1;   // converter groups: 3 without epilogue warps, 2 next to them
    constexpr int NT = v2_threads(MODE);                                  // threads of the block
    // Dense batches: the four chunks of a CTA's FIRST tile are requested by its four epilogue / drain warps (idle until the first
    // accumulator is full), one each and all at once, not one after the other by the loader warp, whose per-chunk bookkeeping (~700
    // cycles) spread them over the first ~5000 cycles of every launch (r02 trace: first MMA 7300 cycles after the CTA's entry).
    constexpr bool HELPED = !RAGGED && !DIRECT && MODE != 2;
    constexpr int CONV0 = MODE == 2 ? W_EPI0 : W_CONV0;                   // first converter warp
    constexpr int DRAINERS = MODE == 2 ? NG : 1 + NG;                     // warps per lane quarter that drain (SHARE)
    constexpr int DRAIN0 = MODE == 2 ? 0 : 1;                             // block index of converter group 0's share
    TRACE_CTA(0);
    constexpr int KS = (PREC == P2_TF32) ? 8 : 16;  // folded pairs per K-step
    constexpr int NQ = KS / 4;                      // 128-bit loads per direction per K-step
    const uint32_t sbase = smem_u32(smem);
    const uint32_t bar0 = sbase + p.off_bar;
    auto BAR = [&](int idx) -> uint32_t { return bar0 + (uint32_t)idx * 8u; };
    uint32_t *tmem_ptr_s = reinterpret_cast<uint32_t *>(smem + p.off_bar + V_NBARS * 8);
    // ragged batches: what the loader found out about each chunk (a ring over the last 8 tiles x 4 lane quarters, entry
    // [q + 4 (tl & 7)] for the chunk of quarter q of this CTA's tl-th tile): the converter warps need its misalignment, whoever
    // drains the accumulators its first output row and its number of valid frames -- nobody else has to search the clip table
    ChunkInfo *chunk_info = reinterpret_cast<ChunkInfo *>(smem + p.off_bar + V_NBARS * 8 + 16);
    float *dct_s = reinterpret_cast<float *>(smem + p.off_dct);

    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);   // provably warp-uniform: role branches stay non-divergent
    const uint32_t rank = cluster_ctarank();
    const int S = p.stg_slots;

    // ------------------------------------------------------------------ one-time setup
    // Who does what, so that nothing waits for anything it does not need (set-up used to cost ~3000 cycles per launch, now the
    // ~1000 of the tensor-memory allocation): the basis warp allocates tensor memory first thing; warps 4.. clear the margins of
    // the staging ring; the loader warp sets up the staging barriers itself and -- after a named barrier with the clearing warps
    // only -- goes straight to its loop, so the first tile's chunks are in flight while the rest of the block is still setting
    // up; the two issuer warps set up all other barriers.  The loader joins the cluster barrier by arriving early and waiting
    // at its very end (it needs nothing the barrier publishes).
    constexpr bool EARLY_LOADER = !DIRECT;                       // direct-load form: the loader warp has no work
    constexpr int SETUP_THREADS = EARLY_LOADER ? NT - 32 : NT;
    if (warp == W_BASIS) {
        tmem_alloc2(smem_u32(tmem_ptr_s), 512);
        tmem_relinquish2();
    }
    if (tid >= 128) {
        // What a frame of zero-weighted (padded) folded pairs may read must be finite, never a stale NaN / Inf bit pattern: up to
        // 128 bytes before its chunk's slot and after it (the load table is checked against that).  A full-chunk box writes
        // its whole slot, the clipped form below clears its slot first; what is left to clear at start-up is the 128 bytes
        // on either side of every slot boundary, plus the slot tails (< 128 bytes) no copy writes.  (Clearing the whole ring
        // cost ~1300 cycles per launch, shared-memory store bandwidth.)
        const int s = (tid - 128) / 24, j = (tid - 128) - s * 24;
        if (s <= S && (s > 0 || j >= 8))
            *reinterpret_cast<float4 *>(smem + p.off_stg + (size_t)s * p.slot_bytes - 256 + 16 * j) = make_float4(0.f, 0.f, 0.f, 0.f);
        fence_proxy_async_smem();  // the zero fill (generic proxy) is ordered before the bulk copies (async proxy) that follow
    }
    static_assert(13 * 24 <= NT - 128, "one thread per 16 bytes of margin");
    if (warp == W_LOAD) {
        // staging barriers: FULL (one arrival + transaction bytes), EMPTY (one arrival per converter group), READY (ragged)
        if (lane < V2_MAX_STG) {
            mbar_init(BAR(V_STG_FULL + lane), 1u);
            mbar_init(BAR(V_STG_EMPTY + lane), (uint32_t)NG);
            mbar_init(BAR(V_STG_READY + lane), 1u);
        }
        mbar_init(BAR(V_INFO + lane), 1u);   // 32 = 8 tile phases x 4 lane quarters: chunk info published (ragged batches)
        if (lane < 24) {                      // K-step staging: two slots per converter warp (4 quarters x up to 3 groups)
            mbar_init(BAR(V_KFULL + lane), 1u);
            mbar_init(BAR(V_KEMPTY + lane), (uint32_t)NG);   // every converter group of the quarter releases every block
        }
        fence_barrier_init();
    } else if (warp == W_MMA || warp == W_MMA2) {
        const int n_b = STREAM ? 8 : (p.units < V2_MAX_UNITS ? p.units : V2_MAX_UNITS);   // basis barriers in use
        const int t64 = (warp == W_MMA ? 0 : 32) + lane;
        for (int i = t64; i < 16; i += 64) { mbar_init(BAR(V_A_FULL + i), 8u); mbar_init(BAR(V_A_EMPTY + i), 2u); }   // A_EMPTY: both issuers commit
        if (t64 < 2) { mbar_init(BAR(V_ACC_FULL + t64), 2u); mbar_init(BAR(V_ACC_EMPTY + t64), (uint32_t)(SHARE ? 8 * DRAINERS : (MODE == 5 ? 16 : 8))); }
        for (int i = t64; i < n_b; i += 64) { mbar_init(BAR(V_B_FULL + i), 1u); mbar_init(BAR(V_B_PEER + i), 1u); }
        if (t64 < 8) mbar_init(BAR(V_B_EMPTY + t64), 2u);                                // both issuers release a slab
        if (t64 == 8) mbar_init(BAR(V_DONE), 2u);                                        // both MMA issuers
        if (FB && t64 == 9) mbar_init(BAR(V_P_READY), 8u);                               // the four epilogue warps of both CTAs
        if (FB && t64 >= 10 && t64 < 13) mbar_init(BAR(V_D2_FULL + (t64 - 10)), 1u);     // D2_FULL, FB_FULL, FB_PEER
        fence_barrier_init();
    }
    if (p.n_mfcc > 0)   // the DCT table, with zero rows for the bins that pad the last 16-bin block (see epi_generic)
        for (int i = tid; i < p.nb * p.dct_pitch; i += NT) dct_s[i] = i < p.n_mels * p.dct_pitch ? __ldg(p.dct + i) : 0.f;
    TRACE_PT(1);
    uint32_t tmem_base = 0;
    if (EARLY_LOADER && warp == W_LOAD) {
        // the loader: margins cleared (named barrier with the clearing warps), its own barriers set up -> start copying
        asm volatile("bar.sync 1, %0;" ::"n"(NT - 96) : "memory");
        cluster_arrive_relaxed();
    } else {
        if (EARLY_LOADER && tid >= 128) {
            // (the warps that issue the first tile's copies wait like the loader: margins cleared, staging barriers set up)
            if (HELPED && warp >= W_EPI0 && warp < W_EPI0 + 4) asm volatile("bar.sync 1, %0;" ::"n"(NT - 96) : "memory");
            else asm volatile("bar.arrive 1, %0;" ::"n"(NT - 96) : "memory");
        }
        TRACE_PT(2);
        tc_fence_before();
        asm volatile("bar.sync 2, %0;" ::"n"(SETUP_THREADS) : "memory");   // tensor memory allocated, barriers set up (this CTA)
        TRACE_PT(3);
#ifdef MELT_STRICT_CLUSTER_SYNC
        cluster_sync_all();
#else
        cluster_arrive_relaxed();   // barrier set-up is published by fence.mbarrier_init; everything else set up here is CTA-local
        cluster_wait();
#endif
        TRACE_PT(4);
        tc_fence_after();
        tmem_base = *tmem_ptr_s;
    }
    if (tid == 32) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");   // the next forward may start filling freed SMs

    // Programmatic dependent launch: this grid may have started while the previous kernel of the stream is still running.
    // Everything above touched only this block's shared / tensor memory and the plan's own tables.  Unless the caller vouches
    // for the input (MELT_OPT_INPUT_READY), wait here -- before the first read of x / offsets -- for the predecessor to complete
    // and its writes to be visible; otherwise the wait is taken just before the first global store (dep_done below).
    if (!p.input_ready) asm volatile("griddepcontrol.wait;" ::: "memory");
    const int first_tile = (int)cluster_id_x(), tile_step = (int)cluster_nid_x();
    const int n_tiles = (RAGGED ? (p.tile_prefix[p.n_clips] + 7) / 8 : p.n_tiles) * p.passes;   // ragged: 8 chunks per tile, counted by the scan kernel; one visit per pass over the bins
    TRACE_DECL
    TRACE(1);
    if (warp == W_LOAD && DIRECT) {
        // K-block staging (windows too long for staged 32-frame chunks): lane q of this warp feeds the converter warps of lane
        // quarter q: per block of four K-steps one box with the forward runs and one with the mirrored runs -- (4 KS + 4)
        // consecutive samples of the quarter's 32 frames each, rows one hop apart in the signal -- into the quarter's two-slot
        // ring.  Four K-steps per box because the tensor-map engine pays per ROW: boxes of a single K-step (80-byte rows) held
        // the kernel at ~1000 cycles per K-step.  Every converter group has a K-step in every block (four consecutive K-steps
        // cover all residues mod 2 and mod 3), so every warp of the quarter waits for -- and releases -- every block.
        if constexpr (!RAGGED) {
            const bool active = lane < 4;
            if (lane == 0) tma_prefetch_desc(p.tmap);
            int kslot = 0;
            uint32_t kph = 0;
            const uint32_t ring0 = sbase + p.off_stg + (uint32_t)(lane * 2) * (uint32_t)p.kslot_bytes;
            const uint32_t half = (uint32_t)p.kslot_bytes >> 1;
            const int nblk = (p.units + 3) >> 2;
            ChunkCursor cur;
            cur.init(p, first_tile, tile_step, (int)rank, lane & 3);
            for (int tile = first_tile; tile < n_tiles; tile += tile_step) {
                Tile2 ti;
                cur.get(p, 0, ti);
                cur.next();
                const int r0 = ti.t0;   // first frame of the quarter's chunk (rows beyond the clip are zero-filled)
                for (int kb = 0; kb < nblk; ++kb) {
                    if (active) {
                        mbar_wait(BAR(V_KEMPTY + 2 * lane + kslot), kph ^ 1u);
                        const uint32_t full = BAR(V_KFULL + 2 * lane + kslot), dst = ring0 + (uint32_t)kslot * (uint32_t)p.kslot_bytes;
                        mbar_arrive_expect_tx(full, (uint32_t)p.kslot_bytes);
                        tma_load_3d(dst, p.tmap, p.a0 + KS * 4 * kb, r0, ti.clip, full);                                       // samples a0 + KS (4 kb) ..
                        tma_load_3d(dst + half, p.tmap, p.b0 - KS * (4 * kb + 3) - (KS - 1) - SIGMA, r0, ti.clip, full);    // the mirrored runs of K-steps 4 kb + 3 .. 4 kb
                        if (++kslot == 2) { kslot = 0; kph ^= 1u; }
                    }
                }
            }
        }
    } else if (warp == W_LOAD) {
        // ============================================================== signal loader (bulk-copy engine)
        // The whole warp runs the (uniform) loop; one elected lane issues the copies.
        // The chunk of lane quarter q of this CTA's tl-th tile lands in memory slot (4 tl + q) mod S, but its barriers are
        // FULL / EMPTY / READY [q + 4 (tl mod P)], P = ceil(S / 4): every waiter then waits for EVERY phase of the barriers it
        // uses (a converter warp of quarter q waits on [q + 4 (tl mod P)] at every tile; this loader waits, in chunk order, for
        // the release of chunk c - S before it overwrites that chunk's slot with chunk c).  Indexing the barriers by memory slot
        // would let a warp meet a barrier whose previous phase belongs to another quarter's chunk and which it never
        // waited for: if that phase has not completed yet, a parity wait for the following phase succeeds at once (found with
        // single-pass modes whose operand ring holds a whole tile: a quarter without valid frames ran a tile ahead and read
        // a slot that still held, or was still receiving, the previous chunk).
        int slot = 0, cq = 0, ctp = 0;        // memory slot, lane quarter and tile phase of the next chunk
        uint32_t cph = 0;
        int eq = 0, etp = 0;                  // the same for chunk c - S (whose release frees the slot), valid once c >= S
        uint32_t eph = 0;
        int chunk_count = 0;
        const int P = p.stg_phases;
        const long long len = p.len;
        if (p.tma_rows > 0 && lane == 0) tma_prefetch_desc(p.tmap);
        constexpr bool ragged = RAGGED;
        const long long total = ragged ? p.offsets[p.n_clips] : 0;   // samples in the packed buffer
        // ragged: the clip the last chunk belonged to.  Chunk indices only grow, so the next clip is found by probing the 32
        // prefix entries after the current one at once (one load latency; a tile step is ~25 clips on the speaker-style batch)
        const int total_chunks = ragged ? p.tile_prefix[p.n_clips] : 0;
        int rg_clip = 0, rg_lo = 0, rg_hi = ragged ? p.tile_prefix[1] : 0;
        long long rg_f0 = 0, rg_T = 0, rg_s0 = 0, rg_len = 0;
        bool rg_have = false;
        int tl = 0;   // tiles of this CTA so far
        // This warp's loop is the pacemaker of the whole kernel (one chunk per ~quarter tile), and a 64-bit division costs it
        // hundreds of cycles: per chunk there is none.  Reflect padding moves a chunk's start vpad samples down = r_pad hop-rows
        // up and c0_pad columns in; a ragged clip's start in the 2-D map (row, column) is divided out once per clip.
        const int vq = p.vpad > 0 ? p.vpad / p.hop : 0, vr = p.vpad - vq * p.hop;
        const int c0_pad = vr ? p.hop - vr : 0, r_pad = vq + (vr ? 1 : 0);
        long long rg_rclip = 0;
        int rg_cclip = 0;
        ChunkCursor cur;   // dense: the chunk of lane quarter 0 of the current tile
        if constexpr (!ragged) cur.init(p, first_tile, tile_step, (int)rank, 0);
        for (int tile = first_tile; tile < n_tiles; tile += tile_step) {
            for (int qi = 0; qi < 4; ++qi) {
                const int q = chunk_order<ragged>(qi);   // the lane quarter whose chunk is issued qi-th
                Tile2 ti;
                long long row0;
                if constexpr (!ragged) {
                    cur.get(p, q, ti);
                    row0 = (long long)ti.t0;
                } else {
                    const int g = (p.passes > 1 ? tile / p.passes : tile) * 8 + (int)rank * 4 + q;   // chunk index in the packed chunk order
                    ti.pass = 0;
                    if (g >= total_chunks) {          // beyond the last chunk: no frames
                        ti.clip = 0; ti.T = 0; ti.s0 = 0; ti.f0 = 0;
                        row0 = 0;
                    } else {
                        while (g >= rg_hi) {          // warp-uniform: the largest clip whose first chunk is <= g
                            const int idx = rg_clip + 1 + lane;
                            const int v = idx <= p.n_clips ? __ldg(p.tile_prefix + idx) : 0x7fffffff;
                            const int cnt = __popc(__ballot_sync(0xffffffffu, v <= g));
                            if (cnt == 32) { rg_clip += 32; rg_lo = __shfl_sync(0xffffffffu, v, 31); continue; }
                            if (cnt > 0) { rg_lo = __shfl_sync(0xffffffffu, v, cnt - 1); rg_clip += cnt; }
                            rg_hi = __shfl_sync(0xffffffffu, v, cnt);
                            rg_have = false;
                        }
                        if (!rg_have) {
                            rg_f0 = p.frame_offsets[rg_clip];
                            rg_T = p.frame_offsets[rg_clip + 1] - rg_f0;
                            rg_s0 = __ldg(p.offsets + rg_clip);
                            rg_len = __ldg(p.offsets + rg_clip + 1) - rg_s0;
                            rg_have = true;
                            const long long sc = (rg_s0 & ~3ll) - p.vpad;    // where the clip's frame 0 starts (aligned down; may be < 0)
                            rg_rclip = sc / p.hop;
                            rg_cclip = (int)(sc - rg_rclip * p.hop);
                            if (rg_cclip < 0) { rg_cclip += p.hop; --rg_rclip; }
                        }
                        ti.clip = rg_clip; ti.T = rg_T; ti.s0 = rg_s0; ti.f0 = rg_f0;
                        row0 = (long long)(g - rg_lo) * 32;
                    }
                }
                const int b = ti.clip;
                const float *xb = p.x + ti.s0;
                const long long clip_len = ragged ? rg_len : len;
                const int n_rows = row0 < ti.T ? p.rows_per_chunk : 0;
                const uint32_t dst0 = sbase + p.off_stg + (uint32_t)slot * (uint32_t)p.slot_bytes;
                // ragged: the chunk starts at sample s of the packed buffer = column s % hop of hop-row s / hop of the 2-D map
                // The tensor-map engine wants the box to start on a 16-byte boundary: it is fetched from the aligned sample below
                // (clip starts are arbitrary; hop % 4 == 0, so every chunk of a clip has the same misalignment) and the
                // converter warp that owns the chunk shifts it down by (s0 & 3) words in shared memory.
                // Virtual reflect padding (MELT_PAD_REFLECT): frame t of a clip starts vpad samples before sample t * hop, so the
                // chunk's first row starts at clip-relative sample st (negative at the head of a clip).  The box is addressed by its
                // start sample: column st % hop of hop-row st / hop (both maps are hop + pitch samples wide for that).
                const long long st = row0 * p.hop - p.vpad;
                long long s = 0;
                int c0 = 0, c1 = (int)row0, c2 = b;
                bool by_tma;
                if (!ragged) {
                    if (p.vpad == 0) {
                        by_tma = n_rows > 0 && row0 + n_rows <= (long long)p.tma_rows;
                        if (HELPED && tl == 0 && by_tma) {   // requested by the epilogue warp of this lane quarter (same predicate there)
                            if (++slot == S) slot = 0;
                            ++chunk_count;
                            if (++cq == 4) { cq = 0; if (++ctp == P) { ctp = 0; cph ^= 1u; } }
                            continue;
                        }
                    } else {
                        c0 = c0_pad; c1 = (int)row0 - r_pad;    // st = c1 * hop + c0 (st >= 0)
                        by_tma = n_rows > 0 && st >= 0 && (long long)c1 + n_rows <= (long long)p.tma_rows;   // every row of the box inside the clip
                    }
                } else {
                    s = (ti.s0 & ~3ll) + st;                    // = (rg_rclip + row0) * hop + rg_cclip
                    c0 = rg_cclip; c1 = (int)(rg_rclip + row0); c2 = 0;
                    by_tma = n_rows > 0 && s >= 0 && s + (long long)(p.rows_per_chunk - 1) * p.hop + (p.pitch_bytes >> 2) <= total;
                    if (p.vpad > 0) {   // and every valid frame of the chunk inside its clip (what lies beyond is mirrored, not the next clip)
                        const long long tlast = row0 + 31 < ti.T - 1 ? row0 + 31 : ti.T - 1;
                        by_tma = by_tma && st >= 0 && tlast * p.hop - p.vpad + p.n_fft <= clip_len;
                    }
                }
                // The staging ring holds less than two tiles, so the loader usually sits here waiting for a slot: pull the
                // chunk into L2 meanwhile -- when the slot frees, the copy into shared memory costs an L2 hit, not a DRAM access
                if (by_tma && elect_one()) tma_prefetch_l2_3d(p.tmap, c0, c1, c2);
                __syncwarp();
                TRACE(10);
                if (chunk_count >= S) {      // the slot's previous tenant, chunk c - S, has been read by every converter group
                    mbar_wait(BAR(V_STG_EMPTY + chunk_order<ragged>(eq) + 4 * etp), eph);
                    if (++eq == 4) { eq = 0; if (++etp == P) { etp = 0; eph ^= 1u; } }
                }
                const uint32_t full = BAR(V_STG_FULL + q + 4 * ctp);
                // ragged: the chunk's misalignment travels with it (read by the converters after their wait on `full`; the
                // thread that writes it is the one that arrives on `full`, so the arrival publishes it)
                ChunkInfo *const info = chunk_info + q + 4 * (tl & 7);
                ChunkInfo info_v;
                info_v.row0 = ti.f0 + row0;
                info_v.nvalid = (int)(ti.T - row0 <= 0 ? 0 : (ti.T - row0 < 32 ? ti.T - row0 : 32));
                info_v.dlt = (int)(ti.s0 & 3ll);
                const uint32_t info_bar = BAR(V_INFO + q + 4 * (tl & 7));   // for the epilogue warps, which wait on nothing else the loader signals
                TRACE(11);
                if (p.vpad > 0 && !by_tma && n_rows > 0) {
                    // Edge chunk of a reflect-padded clip (its first chunk and its last one or two): hop-rows that lie inside the
                    // clip are bulk-copied as they are; the two or three rows that reach before the first or beyond the last
                    // sample are filled element by element with the mirrored samples x[-j] / x[2 (len - 1) - j] (numpy 'reflect':
                    // the edge sample is not repeated).  Ragged batches: in the layout the realignment pass expects (the chunk as
                    // fetched from the aligned sample below its start).
                    const int pw = p.pitch_bytes >> 2;
                    const long long jbase = st - (ragged ? (ti.s0 & 3ll) : 0ll);
                    float *dstp = reinterpret_cast<float *>(smem + p.off_stg + (size_t)slot * p.slot_bytes);
                    // Only the rows a VALID frame of the chunk can read are brought in (its window, the K padding of the last K-step,
                    // the alignment slack of ragged chunks): the last chunk of a clip has up to ~10 rows beyond that, and filling
                    // them element by element held this warp -- the pacemaker of the kernel -- for tens of thousands of cycles
                    // (the Whisper-shaped batch with MELT_OPT_PAD: 35.6 us against 23.7 us on a pre-padded batch; now 25.5).
                    const int n_need = min(n_rows, info_v.nvalid + (p.n_fft + 34) / p.hop + 1);
                    uint32_t bulk_bytes = 0;
                    for (int r = 0; r < n_need; ++r) {
                        const long long jlo = jbase + (long long)r * p.hop;
                        if (jlo >= 0 && jlo + pw <= clip_len) { bulk_bytes += (uint32_t)p.pitch_bytes; continue; }
                        for (int col0 = lane; col0 < pw; col0 += 128) {   // four independent loads in flight per lane, then the stores
                            float v[4];
#pragma unroll
                            for (int u4 = 0; u4 < 4; ++u4) {
                                long long j = jlo + col0 + 32 * u4;
                                j = j < 0 ? -j : j;
                                j = j >= clip_len ? 2 * (clip_len - 1) - j : j;
                                j = j < 0 ? 0 : (j >= clip_len ? clip_len - 1 : j);   // (columns beyond the row, clips shorter than the padding: any sample)
                                v[u4] = __ldg(xb + j);
                            }
#pragma unroll
                            for (int u4 = 0; u4 < 4; ++u4)
                                if (col0 + 32 * u4 < pw) dstp[r * pw + col0 + 32 * u4] = v[u4];
                        }
                    }
                    __syncwarp();   // every lane's stores precede lane 0's arrival below
                    if (lane == 0) {
                        if (ragged) { *info = info_v; mbar_arrive(info_bar); }
                        if (bulk_bytes) mbar_arrive_expect_tx(full, bulk_bytes);
                        else mbar_arrive(full);
                    }
                    __syncwarp();
                    for (int r = lane; r < n_need; r += 32) {   // one bulk copy per row inside the clip, a row per lane (the phase cannot complete before lane 0's arrival above)
                        const long long jlo = jbase + (long long)r * p.hop;
                        if (jlo >= 0 && jlo + pw <= clip_len) bulk_g2s(dst0 + (uint32_t)r * (uint32_t)p.pitch_bytes, xb + jlo, (uint32_t)p.pitch_bytes, full);
                    }
                    __syncwarp();
                    TRACE(12);
                    if (++slot == S) slot = 0;
                    ++chunk_count;
                    if (++cq == 4) { cq = 0; if (++ctp == P) { ctp = 0; cph ^= 1u; } }
                    continue;
                }
                if (ragged && !by_tma) {
                    // The chunk that reaches beyond the packed buffer (the last one of the last clip; or a chunk without rows): hop-rows
                    // that lie inside the buffer as one bulk copy each (s, hop and the pitch are multiples of 4 samples), the one or
                    // two that straddle its end and those beyond it element by element, zeros past the end.  It is ONE chunk per
                    // call, but the LAST one: read element by element as a whole (180 dependent iterations of a global load and a
                    // shared store in this warp) it kept its CTA pair busy for ~20 us after every other pair had finished -- a
                    // tenth of the speaker-style batch (trace: the ragged kernel's tiles were as fast as the dense kernel's).
                    const int pw = p.pitch_bytes >> 2;
                    float *dstp = reinterpret_cast<float *>(smem + p.off_stg + (size_t)slot * p.slot_bytes);
                    uint32_t bulk_bytes = 0;
                    for (int r = 0; r < n_rows; ++r) {
                        const long long gl = s + (long long)r * p.hop;
                        if (gl >= 0 && gl + pw <= total) { bulk_bytes += (uint32_t)p.pitch_bytes; continue; }
                        for (int col = lane; col < pw; col += 32) {
                            const long long g = gl + col;
                            dstp[r * pw + col] = (g >= 0 && g < total) ? __ldg(p.x + g) : 0.f;
                        }
                    }
                    __syncwarp();   // every lane's stores precede lane 0's arrival below
                    if (lane == 0) {
                        *info = info_v;
                        mbar_arrive(info_bar);
                        if (bulk_bytes) mbar_arrive_expect_tx(full, bulk_bytes);
                        else mbar_arrive(full);
                    }
                    __syncwarp();
                    for (int r = lane; r < n_rows; r += 32) {   // a row per lane (the phase cannot complete before lane 0's arrival above)
                        const long long gl = s + (long long)r * p.hop;
                        if (gl >= 0 && gl + pw <= total) bulk_g2s(dst0 + (uint32_t)r * (uint32_t)p.pitch_bytes, p.x + gl, (uint32_t)p.pitch_bytes, full);
                    }
                    __syncwarp();
                    TRACE(12);
                    if (++slot == S) slot = 0;
                    ++chunk_count;
                    if (++cq == 4) { cq = 0; if (++ctp == P) { ctp = 0; cph ^= 1u; } }
                    continue;
                }
                if (!by_tma && n_rows > 0) {
                    // the clipped form writes only the samples the clip has: the rest of the slot is cleared first (see set-up)
                    float4 *z = reinterpret_cast<float4 *>(smem + p.off_stg + (size_t)slot * p.slot_bytes);
                    for (int i = lane; i < p.slot_bytes / 16; i += 32) z[i] = make_float4(0.f, 0.f, 0.f, 0.f);
                    fence_proxy_async_smem();   // generic-proxy stores before the bulk copies (async proxy) into the same slot
                    __syncwarp();
                }
                if (elect_one()) {
                    if (ragged) { *info = info_v; mbar_arrive(info_bar); }
                    if (by_tma) {
                        // one tensor-map box = the whole chunk: rows_per_chunk hop-rows of pitch width (implicit im2col)
                        mbar_arrive_expect_tx(full, (uint32_t)p.rows_per_chunk * (uint32_t)p.pitch_bytes);
                        tma_load_3d(dst0, p.tmap, c0, c1, c2, full);
                    } else {
                        // clip tail (or no tensor map): one bulk copy per hop-row, clipped to the clip
                        long long avail = clip_len - row0 * p.hop;                 // samples of the clip from the chunk's first row on
                        avail = avail < 0 ? 0 : avail;
                        const long long want = (long long)n_rows * p.hop;
                        const uint32_t total_b = (uint32_t)(avail < want ? avail : want) * 4u;
                        if (total_b) mbar_arrive_expect_tx(full, total_b);
                        else mbar_arrive(full);
                        uint32_t dst = dst0;
                        const float *src = xb + row0 * p.hop;
                        uint32_t left = total_b;
                        const uint32_t row_bytes = (uint32_t)p.hop * 4u;
                        while (left) {
                            const uint32_t nb = left < row_bytes ? left : row_bytes;
                            bulk_g2s(dst, src, nb, full);
                            dst += (uint32_t)p.pitch_bytes; src += p.hop; left -= nb;
                        }
                    }
                }
                __syncwarp();
                TRACE(12);
                if (++slot == S) slot = 0;
                ++chunk_count;
                if (++cq == 4) { cq = 0; if (++ctp == P) { ctp = 0; cph ^= 1u; } }
            }
            ++tl;
            if constexpr (!ragged) cur.next();
        }
        (void)cph;
        if (EARLY_LOADER) cluster_wait();   // the phase it arrived on at set-up, before the exit barrier below
    } else if (warp == W_BASIS) {
        // ============================================================== basis: this CTA's half, resident
        // One barrier per K-step slab, so that the first tile's MMAs start as soon as the first slabs have landed.
        if (first_tile < n_tiles) {
            const uint8_t *src = p.b_img + (size_t)rank * p.passes * p.units * p.unit_b_bytes;   // this CTA's half of the Mel rows
            if (!STREAM) {   // a template parameter: the resident instantiation carries no streaming code (0.7 us per cfg1 step)
                if (elect_one()) {
                    for (int u = 0; u < p.units; ++u) {
                        mbar_arrive_expect_tx(BAR(V_B_FULL + u), p.unit_b_bytes);
                        bulk_g2s(sbase + p.off_b + (uint32_t)u * p.unit_b_bytes, src + (size_t)u * p.unit_b_bytes, p.unit_b_bytes, BAR(V_B_FULL + u));
                    }
                }
                __syncwarp();
                if (rank == 1) {  // tell the leader, slab by slab, that the peer half has landed
                    for (int u = 0; u < p.units; ++u) {
                        mbar_wait(BAR(V_B_FULL + u), 0);
                        // complete_tx has made the slab visible in this CTA's shared memory; the tensor core of the pair reads
                        // it through the async proxy, so a plain remote arrival (no cluster-scope fence, which costs ~1000 cycles
                        // with bulk copies in flight) is the hand-off
                        if (lane == 0) mbar_arrive_remote(mapa_cluster(BAR(V_B_PEER + u), 0));
                    }
                }
            } else {
                // long windows: the K-step slabs of every tile stream from L2 through a ring of b_slots slabs; the issuers
                // release a slab (multicast tcgen05.commit to both CTAs) when its MMAs have completed
                if constexpr (FB) {   // the filterbank image of this CTA (its half of the filter rows): resident for the whole launch
                    const uint32_t fb_bytes = 2u * (uint32_t)p.fb_units * p.fb_kind_bytes;
                    if (elect_one()) {
                        mbar_arrive_expect_tx(BAR(V_FB_FULL), fb_bytes);
                        bulk_g2s(sbase + p.off_fb, p.fb_img + (size_t)rank * fb_bytes, fb_bytes, BAR(V_FB_FULL));
                    }
                    __syncwarp();
                }
                int slot = 0;
                uint32_t ph = 0;
                for (int tile = first_tile; tile < n_tiles; tile += tile_step) {
                    const uint8_t *psrc = src + (size_t)(tile % p.passes) * p.units * p.unit_b_bytes;   // this pass' rows of the basis
                    for (int u = 0; u < p.units; ++u) {
                        mbar_wait(BAR(V_B_EMPTY + slot), ph ^ 1u);
                        if (elect_one()) {
                            mbar_arrive_expect_tx(BAR(V_B_FULL + slot), p.unit_b_bytes);
                            bulk_g2s(sbase + p.off_b + (uint32_t)slot * p.unit_b_bytes, psrc + (size_t)u * p.unit_b_bytes, p.unit_b_bytes, BAR(V_B_FULL + slot));
                        }
                        __syncwarp();
                        if (++slot == p.b_slots) { slot = 0; ph ^= 1u; }
                    }
                }
            }
        }
    } else if (warp == W_MMA || warp == W_MMA2) {
        // ============================================================== MMA issuers (leader CTA)
        // Two issuer warps on different schedulers: W_MMA accumulates R (A = folded sums, B = cos rows), W_MMA2 accumulates I
        // (A = folded differences, B = sin rows).  Every accumulator has ONE issuing thread, so the summation order is fixed.
        // An iteration covers two K-steps: the fixed cost of a hand-off (barrier probe, fence, election, operand set-up) is
        // then paid once per ~480 cycles of tensor work instead of once per ~240, which a warp that shares its scheduler
        // with three busy converter / epilogue warps could not keep up with.
        if (STREAM && rank == 1 && warp == W_MMA && first_tile < n_tiles) {
            // streamed basis: this (otherwise idle) warp of the peer CTA tells the leader when a slab of the peer half has landed
            if constexpr (FB) {   // and, once, when the peer half of the filterbank image has
                mbar_wait(BAR(V_FB_FULL), 0);
                if (lane == 0) mbar_arrive_remote(mapa_cluster(BAR(V_FB_PEER), 0));
                __syncwarp();
            }
            int slot = 0;
            uint32_t ph = 0;
            for (int tile = first_tile; tile < n_tiles; tile += tile_step) {
                for (int u = 0; u < p.units; ++u) {
                    mbar_wait(BAR(V_B_FULL + slot), ph);
                    if (lane == 0) mbar_arrive_remote(mapa_cluster(BAR(V_B_PEER + slot), 0));
                    __syncwarp();
                    if (++slot == p.b_slots) { slot = 0; ph ^= 1u; }
                }
            }
        }
        if (rank == 0 && first_tile < n_tiles) {
            const int which = warp == W_MMA ? 0 : 1;
            const uint32_t idesc = umma_idesc(PREC == P2_COMP ? UMMA_F16 : (PREC == P2_BF16 ? UMMA_BF16 : UMMA_TF32), (uint32_t)p.nb, 256u);
            // shared-memory descriptors of K-step 0; K-step u adds u * unit_b_bytes (in 16-byte units) to the address field
            // B kinds: COMPENSATED [wc_hi, wc_lo, ws_hi, ws_lo]; single pass [wc, ws]
            const uint32_t b0 = sbase + p.off_b + (uint32_t)which * (PREC == P2_COMP ? 2u : 1u) * p.kind_bytes;
            const uint64_t dsc_hi = umma_smem_desc_kmajor_noswz(b0, 128, 256);
            const uint64_t dsc_lo = umma_smem_desc_kmajor_noswz(b0 + p.kind_bytes, 128, 256);
            const uint64_t dstep = (uint64_t)(p.unit_b_bytes >> 4);
            const int units = p.units, a_slots = p.a_slots, acc_stages = p.acc_stages;
            // A kinds: COMPENSATED s_hi @0, s_lo @8, d_hi @16, d_lo @24; single pass s @0, d @8
            const uint32_t a_base = tmem_base + (uint32_t)p.a_col0 + (uint32_t)which * (PREC == P2_COMP ? 16u : 8u);
            const uint32_t unit_cols = (uint32_t)p.unit_cols;
            const uint32_t acc_cols = (uint32_t)p.acc_cols;
            const uint32_t d_base = tmem_base + (uint32_t)which * (uint32_t)p.nb;
            int aslot = 0, stage = 0;
            uint32_t aph = 0, sph = 0;
            bool basis_pending = true;
            bool fb_pending = true;   // MODE 4
            uint32_t pph = 0;         // MODE 4: phase of P_READY
            constexpr bool b_res = !STREAM;
            const int b_slots = p.b_slots;
            int bslot = 0;          // streamed basis: ring slot of the next K-step's slab (resident basis: slot = K-step)
            uint32_t bph = 0;
            for (int tile = first_tile; tile < n_tiles; tile += tile_step) {
                TRACE(20);
                mbar_wait(BAR(V_ACC_EMPTY + stage), sph ^ 1u);
                TRACE(21);
                const uint32_t d = d_base + (uint32_t)stage * acc_cols;
                uint64_t du = 0;   // resident basis: descriptor offset of K-step u
                for (int u = 0; u < units; u += 2, du += 2 * dstep) {
                    const bool two = u + 1 < units;
                    int aslot1 = aslot + 1;
                    uint32_t aph1 = aph;
                    if (aslot1 == a_slots) { aslot1 = 0; aph1 ^= 1u; }
                    int bs0, bs1;
                    uint32_t bp0 = 0, bp1 = 0;
                    if (b_res) {
                        bs0 = u; bs1 = u + 1;
                    } else {
                        bs0 = bslot; bp0 = bph;
                        bs1 = bslot + 1; bp1 = bph;
                        if (bs1 == b_slots) { bs1 = 0; bp1 ^= 1u; }
                    }
                    if (basis_pending || !b_res) {
                        mbar_wait(BAR(V_B_FULL + bs0), bp0); mbar_wait_cluster(BAR(V_B_PEER + bs0), bp0);
                        if (two) { mbar_wait(BAR(V_B_FULL + bs1), bp1); mbar_wait_cluster(BAR(V_B_PEER + bs1), bp1); }
                    }
                    mbar_wait(BAR(V_A_FULL + aslot), aph);
                    if (two) mbar_wait(BAR(V_A_FULL + aslot1), aph1);
                    TRACE(22);
                    tc_fence_after();
                    if (elect_one()) {
                        const uint32_t a0 = a_base + (uint32_t)aslot * unit_cols, a1 = a_base + (uint32_t)aslot1 * unit_cols;
                        const uint64_t du0 = b_res ? du : (uint64_t)bs0 * dstep, du1 = b_res ? du + dstep : (uint64_t)bs1 * dstep;
                        const uint32_t acc = u > 0;
                        if (PREC == P2_COMP) {
                            umma2_ts_f16(d, a0, dsc_hi + du0, idesc, acc);          // hi . hi
                            umma2_ts_f16(d, a0 + 8, dsc_hi + du0, idesc, 1);        // lo . hi
                            umma2_ts_f16(d, a0, dsc_lo + du0, idesc, 1);            // hi . lo
                        } else if (PREC == P2_TF32) {
                            umma2_ts_tf32(d, a0, dsc_hi + du0, idesc, acc);
                        } else {
                            umma2_ts_f16(d, a0, dsc_hi + du0, idesc, acc);
                        }
                        tc_commit2(BAR(V_A_EMPTY + aslot), 3);
                        if (!b_res) tc_commit2(BAR(V_B_EMPTY + bs0), 3);
                        if (two) {
                            if (PREC == P2_COMP) {
                                umma2_ts_f16(d, a1, dsc_hi + du1, idesc, 1);
                                umma2_ts_f16(d, a1 + 8, dsc_hi + du1, idesc, 1);
                                umma2_ts_f16(d, a1, dsc_lo + du1, idesc, 1);
                            } else if (PREC == P2_TF32) {
                                umma2_ts_tf32(d, a1, dsc_hi + du1, idesc, 1);
                            } else {
                                umma2_ts_f16(d, a1, dsc_hi + du1, idesc, 1);
                            }
                            tc_commit2(BAR(V_A_EMPTY + aslot1), 3);
                            if (!b_res) tc_commit2(BAR(V_B_EMPTY + bs1), 3);
                        }
                        if (u + 2 >= units) tc_commit2(BAR(V_ACC_FULL + stage), 3);
                    }
                    __syncwarp();
                    TRACE(23);
                    if (!b_res) {
                        bslot = bs0; bph = bp0;
                        const int adv = two ? 2 : 1;
                        for (int k = 0; k < adv; ++k)
                            if (++bslot == b_slots) { bslot = 0; bph ^= 1u; }
                    }
                    if (two) { aslot = aslot1; aph = aph1; }
                    if (++aslot == a_slots) { aslot = 0; aph ^= 1u; }
                }
                basis_pending = false;
                if constexpr (FB) {
                    if (which == 0) {
                        // the filterbank product of this tile (issuer R only): A = the power the epilogue warps of both CTAs wrote over R
                        // (bf16 hi | mid column groups), B = the filterbank slabs, D2 = the columns of I (single accumulator stage)
                        if (fb_pending) { mbar_wait(BAR(V_FB_FULL), 0); mbar_wait_cluster(BAR(V_FB_PEER), 0); fb_pending = false; }
                        mbar_wait(BAR(V_P_READY), pph);
                        pph ^= 1u;
                        tc_fence_after();
                        if (elect_one()) {
                            const uint32_t idesc2 = umma_idesc(UMMA_BF16, (uint32_t)p.fb_nb, 256u);
                            const uint32_t fb0 = sbase + p.off_fb;
                            const uint64_t fd_hi = umma_smem_desc_kmajor_noswz(fb0, 128, 256);
                            const uint64_t fd_mid = umma_smem_desc_kmajor_noswz(fb0 + p.fb_kind_bytes, 128, 256);
                            const uint64_t fstep = (uint64_t)((2u * p.fb_kind_bytes) >> 4);
                            const uint32_t d2 = tmem_base + (uint32_t)p.nb;
                            for (int s2 = 0; s2 < p.fb_units; ++s2) {
                                const uint32_t a_hi = tmem_base + 16u * (uint32_t)s2;
                                umma2_ts_f16(d2, a_hi, fd_hi + (uint64_t)s2 * fstep, idesc2, s2 > 0);     // hi . hi
                                umma2_ts_f16(d2, a_hi + 8, fd_hi + (uint64_t)s2 * fstep, idesc2, 1);      // mid . hi
                                umma2_ts_f16(d2, a_hi, fd_mid + (uint64_t)s2 * fstep, idesc2, 1);         // hi . mid
                            }
                            tc_commit2(BAR(V_D2_FULL), 3);
                        }
                        __syncwarp();
                    }
                }
                if (++stage == acc_stages) { stage = 0; sph ^= 1u; }
            }
            // Nobody waits for the last operand-slot releases (tcgen05.commit arrivals, multicast to both CTAs).  They must not
            // land after a CTA has exited and the next grid -- which may start on this SM right away (programmatic dependent
            // launch) -- has re-initialised the barriers at the same shared-memory addresses: one more commit, behind all the
            // others, is awaited by both CTAs before they retire.
            if (elect_one()) tc_commit2(BAR(V_DONE), 3);
            __syncwarp();
            // Likewise the peer's last accumulator releases (remote arrivals on this CTA's barriers that no later tile waits
            // for): this CTA takes them before it retires, so that the exit barrier below needs no memory ordering.
            for (int k = 0; k < acc_stages; ++k) {
                mbar_wait(BAR(V_ACC_EMPTY + stage), sph ^ 1u);
                if (++stage == acc_stages) { stage = 0; sph ^= 1u; }
            }
        }
    } else if ((MODE != 2 && warp >= W_EPI0 && warp < W_EPI0 + 4) || (MODE == 5 && warp >= W_CONV0 + 4 * NG)) {
        // ============================================================== epilogue (thread = frame)
        const int q = warp & 3;
        const int row = q * 32 + lane;
        const uint32_t lane_taddr = tmem_base + ((uint32_t)(q * 32) << 16);
        const uint32_t acc_empty_remote = mapa_cluster(BAR(V_ACC_EMPTY), 0);
        const float kLog10_2 = 0.30102999566398120f;
        int stage = 0;
        uint32_t sph = 0;
        // (plain log-Mel output never comes here: it runs without epilogue warps, MODE 2)
        bool dep_done = false;
        int tl = 0;   // tiles of this CTA so far
        ChunkCursor cur;   // dense: this warp's chunk of the current tile
        if constexpr (!RAGGED) cur.init(p, first_tile, tile_step, (int)rank, q);
        if constexpr (HELPED) {
            // the chunk of this lane quarter of the CTA's first tile, if it is an ordinary one (one tensor-map box): see HELPED
            if (warp < W_EPI0 + 4 && first_tile < n_tiles && p.vpad == 0) {
                Tile2 ht;
                cur.get(p, 0, ht);
                if ((long long)ht.t0 < ht.T && ht.t0 + p.rows_per_chunk <= p.tma_rows) {
                    if (lane == 0) {
                        const uint32_t full = BAR(V_STG_FULL + q);   // tile phase 0
                        mbar_arrive_expect_tx(full, (uint32_t)p.rows_per_chunk * (uint32_t)p.pitch_bytes);
                        tma_load_3d(sbase + p.off_stg + (uint32_t)chunk_pos<RAGGED>(q) * (uint32_t)p.slot_bytes, p.tmap, 0, ht.t0, ht.clip, full);
                    }
                    __syncwarp();
                }
            }
        }
        for (int tile = first_tile; tile < n_tiles; tile += tile_step) {
            // where this warp's 32 rows go: dense batches by division; ragged ones from the loader's chunk record (acquired through
            // the INFO barrier of this ring entry: this warp is its only waiter and waits for each of its phases once, in order)
            long long out_row0;       // ragged: first output row of the chunk
            int nvalid32;             // ragged: frames of the chunk that exist
            Tile2 ti;
            if constexpr (RAGGED) {
                mbar_wait(BAR(V_INFO + q + 4 * (tl & 7)), (uint32_t)((tl >> 3) & 1));
                const ChunkInfo ci = chunk_info[q + 4 * (tl & 7)];
                out_row0 = ci.row0; nvalid32 = ci.nvalid;
                ti.clip = 0; ti.t0 = 0; ti.T = 0; ti.s0 = 0; ti.f0 = 0;
                ti.pass = p.passes > 1 ? tile % p.passes : 0;
            } else {
                cur.get(p, 0, ti);
                cur.next();
                out_row0 = 0; nvalid32 = 0;
            }
            ++tl;
            const int b = ti.clip;
            const int t0 = ti.t0 - q * 32;   // so that frame t0 + row is this thread's (row = 32 q + lane)
            const long long T = ti.T;
            const bool valid = RAGGED ? lane < nvalid32 : (long long)(t0 + row) < T;
            float *optr, *tptr;
            long long cstride;
            const int c_off = ti.pass * p.nb;                                   // first bin of this pass
            const int nm = p.n_mels - c_off < p.nb ? p.n_mels - c_off : p.nb;   // bins of this pass
            if (RAGGED) {        // packed, frame-major
                optr = p.out + (out_row0 + lane) * p.n_ch + c_off;
                tptr = p.tap ? p.tap + (out_row0 + lane) * p.n_mels + c_off : nullptr;
                cstride = 1;
            } else if (p.feature_major) {
                optr = p.out + ((long long)b * p.n_ch + c_off) * T + t0 + row;
                tptr = p.tap ? p.tap + ((long long)b * p.n_mels + c_off) * T + t0 + row : nullptr;
                cstride = T;
            } else {   // frame-major
                optr = p.out + (ti.f0 + t0 + row) * p.n_ch + c_off;
                tptr = p.tap ? p.tap + (ti.f0 + t0 + row) * p.n_mels + c_off : nullptr;
                cstride = 1;
            }
            TRACE(30);
            mbar_wait(BAR(V_ACC_FULL + stage), sph);
            if (!dep_done) { asm volatile("griddepcontrol.wait;" ::: "memory"); dep_done = true; }   // before the first global store
            TRACE(31);
            tc_fence_after();
            const uint32_t t_r = lane_taddr + (uint32_t)stage * (uint32_t)p.acc_cols, t_i = t_r + (uint32_t)p.nb;
            if constexpr (FB) {
                epi_fbank(p, t_r, t_i, optr, cstride, valid, lane, mapa_cluster(BAR(V_P_READY), 0), BAR(V_D2_FULL), (uint32_t)((tl - 1) & 1),
                          acc_empty_remote + (uint32_t)stage * 8u);
            } else if (SHARE || MODE == 3 || MODE == 5) {
                // single accumulator stage, log-Mel: this warp drains every third 16-bin block, the two converter warps of the
                // lane quarter the others (MODE 3: plain log-Mel, this warp drains every block)
                epi_fast_share(t_r, t_i, p.nb, nm, RAGGED ? out_at(p, (out_row0 + lane) * p.n_ch + c_off) : (p.feature_major ? out_at(p, ((long long)b * p.n_ch + c_off) * T + t0 + row) : out_at(p, (ti.f0 + t0 + row) * p.n_ch + c_off)),
                               cstride, valid, p.out_log10_offset, MODE == 5 && warp >= W_CONV0 ? 1 : 0, MODE == 3 ? 1 : (MODE == 5 ? 2 : DRAINERS), p.out_dtype);
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_remote(acc_empty_remote + (uint32_t)stage * 8u);
            } else {
                const uint32_t eb = acc_empty_remote + (uint32_t)stage * 8u;
                // frame-major MFCCT with a staging block: this warp's 32 frames start at row (t0 + 32 q) of the clip
                float *estage = (p.off_epi && !p.feature_major) ? reinterpret_cast<float *>(smem + p.off_epi) + q * 32 * p.n_mfcc : nullptr;
                float *ewout = RAGGED ? p.out + out_row0 * p.n_ch : p.out + (ti.f0 + t0 + q * 32) * p.n_ch;
                const long long erem = T - (long long)(t0 + q * 32);
                const int envalid = RAGGED ? nvalid32 : (erem <= 0 ? 0 : (erem < 32 ? (int)erem : 32));
                if (p.n_mfcc == 0) epi_generic<false>(p, t_r, t_i, dct_s, optr, tptr, cstride, valid, lane, eb, nm, estage, ewout, envalid);
                else epi_generic<true>(p, t_r, t_i, dct_s, optr, tptr, cstride, valid, lane, eb, nm, estage, ewout, envalid);
            }
            TRACE(32);
            if (++stage == p.acc_stages) { stage = 0; sph ^= 1u; }
        }
    } else if (warp >= CONV0) {
        // ============================================================== converters (thread = frame; the groups take K-step pairs round-robin)
        const int q = warp & 3, g = (warp - CONV0) >> 2;
        const uint32_t lane_taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)p.a_col0;
        const uint32_t a_full_remote = mapa_cluster(BAR(V_A_FULL), 0);
        const uint32_t row_off = sbase + p.off_stg + (uint32_t)lane * (uint32_t)p.pitch_bytes;
        const float S_in = p.in_scale;
        int sslot = chunk_pos<RAGGED>(q);        // memory slot of this warp's chunk: (4 tl + its position in the loader's issue order) mod S
        int sbar = q;                            // its barriers: q + 4 (tl mod P) (see the loader)
        uint32_t sph = 0;
        int aslot = g % p.a_slots;               // ring position of unit counter ug = it * units + u, first u = g
        uint32_t aph = (uint32_t)((g / p.a_slots) & 1);
        // SHARE (single accumulator stage, log-Mel): this warp also drains its share of the previous tile's accumulator --
        // after its second K-step of the next tile, so that the MMAs find operands waiting when the drain releases them.
        int pend_tile = -1, pend_tl = 0, dstage = 0;
        ChunkCursor dcur;   // dense: this warp's chunk of the tile to drain next
        if constexpr (!RAGGED) dcur.init(p, first_tile, tile_step, (int)rank, q);
        int tl = 0;   // tiles of this CTA so far
        // K-block staging (DIRECT): the two-slot ring of this lane quarter, fed by lane q of the loader warp; a row = 4 KS + 4 samples
        const int kidx = 2 * q;
        const uint32_t kring = sbase + p.off_stg + (uint32_t)kidx * (uint32_t)p.kslot_bytes + (uint32_t)lane * (uint32_t)((4 * KS + 4) * 4);
        int cur_blk = -1;
        int kslot = 0;
        uint32_t kph = 0;
        uint32_t dph = 0;
        bool dep_done = false;
        const uint32_t acc_empty_remote = mapa_cluster(BAR(V_ACC_EMPTY), 0);
#define DRAIN_PENDING()                                                                                          \
        do {                                                                                                     \
            Tile2 dt;                                                                                            \
            bool dvalid;                                                                                         \
            float *doptr;                                                                                        \
            int dc_off;                                                                                          \
            if constexpr (RAGGED) {   /* this warp converted the chunk of tile pend_tl itself: its record is in the ring */ \
                const ChunkInfo ci = chunk_info[q + 4 * (pend_tl & 7)];                                          \
                dt.T = 0;                                                                                        \
                dc_off = (p.passes > 1 ? pend_tile % p.passes : 0) * p.nb;                                       \
                dvalid = lane < ci.nvalid;                                                                       \
                doptr = out_at(p, (ci.row0 + lane) * p.n_ch + dc_off);                                           \
            } else {                                                                                             \
                dcur.get(p, 0, dt);   /* tiles are drained in order */                                           \
                dcur.next();                                                                                     \
                const int drow = q * 32 + lane, dt0 = dt.t0 - q * 32;                                            \
                dvalid = (long long)(dt0 + drow) < dt.T;                                                         \
                dc_off = dt.pass * p.nb;                                                                         \
                doptr = p.feature_major ? out_at(p, ((long long)dt.clip * p.n_ch + dc_off) * dt.T + dt0 + drow)  \
                                        : out_at(p, (dt.f0 + dt0 + drow) * p.n_ch + dc_off);                     \
            }                                                                                                    \
            const int dnm = p.n_mels - dc_off < p.nb ? p.n_mels - dc_off : p.nb;                                 \
            mbar_wait(BAR(V_ACC_FULL + dstage), dph);                                                            \
            if (!dep_done) { asm volatile("griddepcontrol.wait;" ::: "memory"); dep_done = true; }               \
            tc_fence_after();                                                                                    \
            const uint32_t dtr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)dstage * (uint32_t)p.acc_cols; \
            epi_fast_share(dtr, dtr + (uint32_t)p.nb, p.nb, dnm, doptr, p.feature_major ? dt.T : 1, dvalid,      \
                           p.out_log10_offset, DRAIN0 + g, DRAINERS, p.out_dtype);                               \
            tc_fence_before();                                                                                   \
            __syncwarp();                                                                                        \
            if (lane == 0) mbar_arrive_remote(acc_empty_remote + (uint32_t)dstage * 8u);                         \
            if (++dstage == p.acc_stages) { dstage = 0; dph ^= 1u; }                                             \
            pend_tile = -1;                                                                                      \
        } while (0)
        int u = g;
        for (int tile = first_tile; tile < n_tiles; tile += tile_step) {
            TRACE(40);
            if constexpr (DIRECT) {
                // K-step staging: this group takes K-steps g, g + NG, ... of every tile (the loader feeds them in that order);
                // ring position of the tile's first one from the running K-step count
                u = g;
                const int ug0 = tl * p.units + g;
                aslot = ug0 % p.a_slots;
                aph = (uint32_t)((ug0 / p.a_slots) & 1);
                cur_blk = -1;
            } else {
                mbar_wait(BAR(V_STG_FULL + sbar), sph);
            }
            // ragged: words by which this chunk sits further into its rows than the load table says (see load_shifted)
            const int dlt = RAGGED ? chunk_info[q + 4 * (tl & 7)].dlt : 0;
            TRACE(41);
            const uint32_t fb = row_off + (uint32_t)sslot * (uint32_t)p.slot_bytes;
            bool released = false;
            // The staged chunk is handed back to the loader as soon as this warp's last K-step of the tile has been read and
            // folded (its samples are in registers), not after the operand store and its hand-off.
#define STG_RELEASE_IF_LAST()                                                                       \
            do {                                                                                    \
                if (!DIRECT && u + NG >= p.units) {                                                 \
                    __syncwarp();                                                                   \
                    if (lane == 0) mbar_arrive(BAR(V_STG_EMPTY + sbar));                            \
                    released = true;                                                                \
                }                                                                                   \
            } while (0)
            // this group's K-steps: every NG-th of the running count over the CTA's tiles (u carries over from the previous
            // tile), so that a K-step count that NG does not divide is spread evenly over the groups
            const int u0 = u;
            while (u < p.units) {
                if (SHARE && pend_tile >= 0 && u >= u0 + 2 * NG) DRAIN_PENDING();
                // ---- loads: NQ forward quads, NQ mirrored quads (+ one single when the mirrored run starts at 1 mod 4)
                TRACE(42);
                const short *tb = p.tab[DIRECT ? 0 : u];
                // ---- fold, scale, split: the operand words of this K-step (COMPENSATED: s_hi | s_lo | d_hi | d_lo, 8 words each;
                // single pass: s | d).  The arithmetic sits INSIDE every load variant below (ragged batches have four: chunk
                // misalignment 0-3): joined behind a common set of loaded samples, the variants met in fixed registers and every
                // K-step paid ~45 register moves for it -- the ragged kernel issued 12.5 % more instructions than the dense one on
                // the SAME batch and, being issue-bound, ran 14 % longer (ncu: 134.3 M vs 119.3 M, 230 vs 201 us).
                constexpr int NW = PREC == P2_COMP ? 32 : 16;
                uint32_t vw[NW];
                auto split = [&](const float (&fw)[KS], const float (&bw)[KS]) {
                    if constexpr (PREC == P2_COMP) {
                        // packed fp32 arithmetic (FMUL2 / FADD2): two folded pairs per instruction.  The mirrored samples are
                        // scaled one by one, which also puts them in pair order at no cost; scaling by 2^s is exact, so
                        // t + b == fma(f, S, b).
                        const uint64_t S2 = f2_pack(S_in, S_in);
#pragma unroll
                        for (int c = 0; c < 8; ++c) {
                            const uint64_t t = f2_mul(f2_pack(fw[2 * c], fw[2 * c + 1]), S2);
                            const uint64_t b = f2_pack(bw[2 * c] * S_in, bw[2 * c + 1] * S_in);
                            const uint64_t s = f2_add(t, b), d = f2_sub(t, b);
                            const __half2 sh = f2_to_half2(s), dh = f2_to_half2(d);
                            const uint64_t sr = f2_sub(s, half2_to_f2(sh)), dr = f2_sub(d, half2_to_f2(dh));
                            const __half2 sl = f2_to_half2(sr), dl = f2_to_half2(dr);
                            vw[c] = *reinterpret_cast<const uint32_t *>(&sh);
                            vw[8 + c] = *reinterpret_cast<const uint32_t *>(&sl);
                            vw[16 + c] = *reinterpret_cast<const uint32_t *>(&dh);
                            vw[24 + c] = *reinterpret_cast<const uint32_t *>(&dl);
                        }
                    } else if constexpr (PREC == P2_BF16) {
#pragma unroll
                        for (int c = 0; c < 8; ++c) {
                            const __nv_bfloat162 sh = __floats2bfloat162_rn(fw[2 * c] + bw[2 * c], fw[2 * c + 1] + bw[2 * c + 1]);
                            const __nv_bfloat162 dh = __floats2bfloat162_rn(fw[2 * c] - bw[2 * c], fw[2 * c + 1] - bw[2 * c + 1]);
                            vw[c] = *reinterpret_cast<const uint32_t *>(&sh);
                            vw[8 + c] = *reinterpret_cast<const uint32_t *>(&dh);
                        }
                    } else {
#pragma unroll
                        for (int c = 0; c < 8; ++c) {
                            vw[c] = cvt_tf32_rna(fw[c] + bw[c]);
                            vw[8 + c] = cvt_tf32_rna(fw[c] - bw[c]);
                        }
                    }
                };
                if constexpr (DIRECT) {     // K-block staging: the runs of this K-step lie in the block's slot of the quarter's ring
                    const int kb = u >> 2;
                    while (cur_blk < kb) {   // warp-uniform: move on to the block of this K-step (every block is waited for and released)
                        if (cur_blk >= 0) {
                            __syncwarp();
                            if (lane == 0) mbar_arrive(BAR(V_KEMPTY + kidx + kslot));
                            if (++kslot == 2) { kslot = 0; kph ^= 1u; }
                        }
                        ++cur_blk;
                        mbar_wait(BAR(V_KFULL + kidx + kslot), kph);
                    }
                    const uint32_t kbase = kring + (uint32_t)kslot * (uint32_t)p.kslot_bytes;
                    const uint32_t off_f = (uint32_t)((u - 4 * kb) * KS * 4), off_b = ((uint32_t)p.kslot_bytes >> 1) + (uint32_t)((4 * kb + 3 - u) * KS * 4);
                    float fw[KS], bw[KS];
                    load_kstaged<KS, SIGMA>(kbase + off_f, off_b - off_f, fw, bw);
                    split(fw, bw);
                } else if (RAGGED && dlt != 0) {   // warp-uniform: one misalignment per chunk
                    float fw[KS], bw[KS];
                    if (dlt == 1) { load_shifted<KS, SIGMA, 1>(fb, tb, fw, bw); split(fw, bw); }
                    else if (dlt == 2) { load_shifted<KS, SIGMA, 2>(fb, tb, fw, bw); split(fw, bw); }
                    else { load_shifted<KS, SIGMA, 3>(fb, tb, fw, bw); split(fw, bw); }
                } else {
                    float fw[KS], bw[KS];
#pragma unroll
                    for (int i = 0; i < NQ; ++i) {
                        const float4 f = lds128(fb + (uint32_t)(int)tb[i]);
                        fw[4 * i + 0] = f.x; fw[4 * i + 1] = f.y; fw[4 * i + 2] = f.z; fw[4 * i + 3] = f.w;
                    }
                    // mirrored partner of pair e is the sample at position KS-1-e of the descending run
                    if (SIGMA == 0) {
#pragma unroll
                        for (int i = 0; i < NQ; ++i) {
                            const float4 f = lds128(fb + (uint32_t)(int)tb[4 + i]);     // samples rs+4i .. rs+4i+3
                            bw[KS - 1 - (4 * i + 0)] = f.x; bw[KS - 1 - (4 * i + 1)] = f.y;
                            bw[KS - 1 - (4 * i + 2)] = f.z; bw[KS - 1 - (4 * i + 3)] = f.w;
                        }
                    } else {
#pragma unroll
                        for (int i = 0; i < NQ; ++i) {
                            const float4 f = lds128(fb + (uint32_t)(int)tb[4 + i]);     // samples rs-1+4i .. rs+2+4i
                            if (i > 0) bw[KS - 1 - (4 * i - 1)] = f.x;                  // position 4i-1 of the run
                            bw[KS - 1 - (4 * i + 0)] = f.y; bw[KS - 1 - (4 * i + 1)] = f.z; bw[KS - 1 - (4 * i + 2)] = f.w;
                        }
                        bw[0] = lds32(fb + (uint32_t)(int)tb[8]);   // position KS-1 of the run
                    }
                    split(fw, bw);
                }
                const uint32_t dst = lane_taddr + (uint32_t)aslot * (uint32_t)p.unit_cols;
                TRACE(43);
                STG_RELEASE_IF_LAST();
                mbar_wait(BAR(V_A_EMPTY + aslot), aph ^ 1u);   // the operand is ready in registers before the slot is
                TRACE(44);
                tc_fence_after();
                if constexpr (PREC == P2_COMP) {
                    tmem_st8(dst, vw);
                    tmem_st8(dst + 8, vw + 8);
                    tmem_st8(dst + 16, vw + 16);
                    tmem_st8(dst + 24, vw + 24);
                } else {
                    tmem_st16(dst, vw);
                }
                // hand the slot to the MMA issuers right away: a slot is held only from its store to the end of its MMAs
                tmem_wait_st();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_remote(a_full_remote + (uint32_t)aslot * 8u);
                TRACE(45);
                // advance to this group's next K-step
                u += NG;
                aslot += NG;
                while (aslot >= p.a_slots) { aslot -= p.a_slots; aph ^= 1u; }
            }
            u -= p.units;   // position in the next tile
            if constexpr (DIRECT) {   // the blocks of this tile this warp had no K-step in (a partial last block), and the last one held
                const int nblk = (p.units + 3) >> 2;
                while (cur_blk < nblk) {
                    if (cur_blk >= 0) {
                        __syncwarp();
                        if (lane == 0) mbar_arrive(BAR(V_KEMPTY + kidx + kslot));
                        if (++kslot == 2) { kslot = 0; kph ^= 1u; }
                    }
                    if (++cur_blk < nblk) mbar_wait(BAR(V_KFULL + kidx + kslot), kph);
                }
            }
            if (!DIRECT && !released) {   // a group without K-steps in this geometry
                __syncwarp();
                if (lane == 0) mbar_arrive(BAR(V_STG_EMPTY + sbar));
            }
            sslot += 4;
            if (sslot >= S) sslot -= S;
            sbar += 4;
            if (sbar >= 4 * p.stg_phases) { sbar -= 4 * p.stg_phases; sph ^= 1u; }
            if (SHARE) {
                if (pend_tile >= 0) DRAIN_PENDING();   // short windows: fewer than three K-steps per group
                pend_tile = tile;
                pend_tl = tl;
            }
            ++tl;
        }
        if (SHARE && pend_tile >= 0) DRAIN_PENDING();   // the last tile
#undef STG_RELEASE_IF_LAST
#undef DRAIN_PENDING
    }

    // ------------------------------------------------------------------ teardown
    TRACE_PT(5);
    tc_fence_before();
    __syncthreads();
    // All tensor-core work of the pair, and the barrier arrivals it triggers, are done before a CTA retires: every warp takes the
    // issuers' final commit here, where it has (almost) always completed -- the basis warp used to probe this barrier for the
    // whole launch, on the scheduler it shares with the converter warps of lane quarter 2 (cfg4d tf32 217 -> 203 us).
    if (first_tile < n_tiles) mbar_wait(BAR(V_DONE), 0);
    TRACE_PT(6);
#ifdef MELT_STRICT_CLUSTER_SYNC
    cluster_sync_all();
#else
    // execution barrier only: every cross-CTA arrival has been waited for (the DONE commit, the accumulator releases above);
    // with release semantics the barrier would wait ~1500 cycles for this CTA's last output stores to be performed
    cluster_arrive_relaxed();
    cluster_wait();
#endif
    TRACE_PT(7);
    if (warp == W_BASIS) tmem_dealloc2(tmem_base, 512);
    TRACE_CTA(1);
}


// ---------------------------------------------------------------------------------------------- launch (per precision TU)
template <int PREC, int SIGMA, bool RAGGED, int MODE, bool STREAM, bool DIRECT>
static int launch_one_s(const K2Params &kp, int grid, cudaStream_t stream) {
    // the opt-in shared-memory size is a per-device attribute of the function: set once per device (bit d of the mask)
    static std::atomic<unsigned long long> attr_done{0};
    int dev = 0;
    MELT_CUDA(cudaGetDevice(&dev));
    const unsigned long long bit = 1ull << (dev & 63);
    if (dev >= 64 || !(attr_done.load(std::memory_order_acquire) & bit)) {
        MELT_CUDA(cudaFuncSetAttribute(melt_fwd2_kernel<PREC, SIGMA, RAGGED, MODE, STREAM, DIRECT>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BUDGET));
        attr_done.fetch_or(bit, std::memory_order_release);
    }
    // Programmatic dependent launch: the CTAs of this grid are dispatched as soon as SMs of the previous kernel in the stream
    // free up (its clusters finish at different times: 376 tiles on 74 pairs), instead of after its last CTA has retired and
    // a fresh launch has ramped up.  The kernel orders itself behind that kernel with griddepcontrol.wait: before its first read
    // of the caller's buffers by default, before its first global store only when the caller vouches for the input
    // (K2Params::input_ready, MELT_OPT_INPUT_READY).
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid, 1, 1);
    cfg.blockDim = dim3(v2_threads(MODE), 1, 1);
    cfg.dynamicSmemBytes = kp.smem_bytes;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
#ifdef MELT_TRACE
    static int trace_slot = 0;   // development builds: every launch records into its own region of the trace buffer (16 regions)
    K2Params kt = kp;
    kt.trace_slot = trace_slot++ & 15;
    MELT_CUDA(cudaLaunchKernelEx(&cfg, melt_fwd2_kernel<PREC, SIGMA, RAGGED, MODE, STREAM, DIRECT>, kt));
#else
    MELT_CUDA(cudaLaunchKernelEx(&cfg, melt_fwd2_kernel<PREC, SIGMA, RAGGED, MODE, STREAM, DIRECT>, kp));
#endif
    return MELT_OK;
}

template <int PREC, int SIGMA, bool RAGGED, int MODE>
static int launch_one_r(const K2Params &kp, int grid, cudaStream_t stream) {
    if (kp.direct) {   // dense, streamed basis only (plan_build_v2)
        if (RAGGED) return fail(MELT_ERR_UNSUPPORTED, "internal: direct mode is dense only");
        return launch_one_s<PREC, SIGMA, false, MODE, true, true>(kp, grid, stream);
    }
    return kp.b_resident ? launch_one_s<PREC, SIGMA, RAGGED, MODE, false, false>(kp, grid, stream)
                         : launch_one_s<PREC, SIGMA, RAGGED, MODE, true, false>(kp, grid, stream);
}

template <int PREC, int SIGMA>
static int launch_one(const K2Params &kp, int grid, cudaStream_t stream) {
    // Who drains the accumulators.  Power / tap / ln / MFCCT outputs: four epilogue warps next to two converter groups (MODE 0).
    // Plain log-Mel: three converter groups, and either four dedicated drain warps next to them (MODE 3, 640 threads) or -- when
    // the accumulator has a single stage, the basis is resident and the MMAs run at half rate (TF32): the tensor pipe is the
    // bound and idles while a tile is drained -- every converter warp drains a third of the previous tile's bins (MODE 2).
    // Measured (r02, B200, back to back): MODE 3 vs MODE 2  cfg1 -3.6 %, 256 x 4 s clips -13 %, cfg4a tf32 / bf16 -4.5 / -6.8 %,
    // cfg2 tf32 +5 % (hence the exception), everything else within +-2 %.  MODE 5 = MODE 3 with EIGHT drain warps (two per lane
    // quarter, alternate 16-bin blocks; 768 threads) where a single accumulator stage puts the drain between two tiles' MMAs and the
    // basis is resident: cfg2 compensated 256 -> 247 us; with a streamed basis or K-block staging it measured 0.5-1.5 % slower.
    const bool plain = kp.n_mfcc == 0 && !kp.output_power && kp.tap == nullptr;
    const int mode = !plain ? 0 : (PREC == P2_TF32 && kp.acc_stages == 1 && kp.b_resident && !kp.direct ? 2 : (kp.acc_stages == 1 && kp.b_resident && !kp.direct ? 5 : 3));
    if (kp.offsets) {
        if (mode == 5) return launch_one_s<PREC, SIGMA, true, 5, false, false>(kp, grid, stream);
        if (mode == 3) return launch_one_r<PREC, SIGMA, true, 3>(kp, grid, stream);
        return mode == 2 ? launch_one_r<PREC, SIGMA, true, 2>(kp, grid, stream) : launch_one_r<PREC, SIGMA, true, 0>(kp, grid, stream);
    }
    if (mode == 5) return launch_one_s<PREC, SIGMA, false, 5, false, false>(kp, grid, stream);
    if (mode == 3) return launch_one_r<PREC, SIGMA, false, 3>(kp, grid, stream);
    return mode == 2 ? launch_one_r<PREC, SIGMA, false, 2>(kp, grid, stream) : launch_one_r<PREC, SIGMA, false, 0>(kp, grid, stream);
}


}  // namespace melt
