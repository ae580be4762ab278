// melt_forward.cu -- the hot path as ONE persistent, warp-specialised sm_100a kernel (steps S1-S6 of SURVEY.md 8(a)):
//
//   loader warps      raw fp32 signal (global) -> shared-memory staging, TRANSPOSED ([sample-in-hop][hop-row]) so that
//                     a converter thread that owns one frame reads it without bank conflicts.  Implicit im2col: each
//                     sample is fetched from HBM/L2 once per tile; overlapping frames exist only on chip.  Reflect
//                     padding and clip bounds are resolved here.
//   converter warps   thread = frame.  Folds the frame about the window centre (sum / difference of mirrored samples),
//                     splits to the tensor-core operand format (fp16 hi + fp16 lo, or bf16, or tf32) and writes the
//                     A operand straight into TENSOR MEMORY (tcgen05.st) -- A never touches shared memory.
//   basis producer    bulk-copy engine (cp.async.bulk): K-step slabs of the folded cos/sin basis, resident in shared
//                     memory when they fit (Whisper shape), else a ring streamed from L2.
//   MMA issuer        one thread: tcgen05.mma kind::f16 / kind::tf32, A from tensor memory, B from shared memory,
//                     fp32 accumulators in tensor memory (R in columns [0, nb), I in [nb, 2 nb)), double-buffered.
//   epilogue warps    tcgen05.ld -> R^2 + I^2 -> log10(max(., 1e-10)) -> optional DCT-II (fp32 FMA) -> global stores.
//
// All hand-offs are mbarriers (full/empty pairs); tcgen05.commit releases A slots, basis slots and accumulators.
#include "melt_plan.h"
#include "sm100_ptx.cuh"

#include <cuda_bf16.h>
#include <cuda_fp16.h>

namespace melt {

enum { PREC_COMP = 0, PREC_TF32 = 1, PREC_BF16 = 2 };
// barrier indices (8 bytes each) inside the barrier block
enum { B_FULL = 0, B_EMPTY = 32, A_FULL = 64, A_EMPTY = 72, ACC_FULL = 80, ACC_EMPTY = 82, STG_FULL = 84, STG_EMPTY = 88, NBARS = 92 };

struct TileInfo {
    const float *xb;      // clip base
    long long clip_len;   // samples in the clip
    long long T;          // frames in the clip
    long long out_frame0; // global frame index (over all clips) of tile row 0
    int clip, t0, nvalid;
};

__device__ __forceinline__ long long frames_of(const KParams &p, long long len) {
    long long padded = len;
    if (p.pad) {
        if (len < (long long)(p.n_fft / 2) + 1) return 0;
        padded += 2LL * (p.n_fft / 2);
    }
    if (padded < p.n_fft) return 0;
    long long T = (padded - p.n_fft) / p.hop + 1 - (p.drop_last ? 1 : 0);
    return T < 0 ? 0 : T;
}

__device__ __forceinline__ void get_tile(const KParams &p, int tile, TileInfo &ti) {
    if (p.offsets == nullptr) {
        const int b = tile / p.tiles_per_clip;
        ti.clip = b;
        ti.t0 = (tile - b * p.tiles_per_clip) * TILE_M;
        ti.T = p.frames_per_clip;
        ti.xb = p.x + (long long)b * p.len;
        ti.clip_len = p.len;
        ti.out_frame0 = (long long)b * ti.T + ti.t0;
    } else {
        int lo = 0, hi = p.n_clips;  // largest i with tile_prefix[i] <= tile
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (__ldg(p.tile_prefix + mid) <= tile) lo = mid; else hi = mid;
        }
        const long long o0 = __ldg(p.offsets + lo), o1 = __ldg(p.offsets + lo + 1);
        ti.clip = lo;
        ti.t0 = (tile - __ldg(p.tile_prefix + lo)) * TILE_M;
        ti.clip_len = o1 - o0;
        ti.T = frames_of(p, ti.clip_len);
        ti.xb = p.x + o0;
        ti.out_frame0 = p.frame_offsets[lo] + ti.t0;
    }
    const long long rem = ti.T - ti.t0;
    ti.nvalid = rem < TILE_M ? (int)rem : TILE_M;
}

// Sample j (clip coordinates, may be outside [0, L)) of the virtually padded clip.
__device__ __forceinline__ float fetch_sample(const KParams &p, const TileInfo &ti, long long j) {
    if (p.pad) {
        if (j < 0) j = -j;
        if (j >= ti.clip_len) j = 2 * (ti.clip_len - 1) - j;
    }
    return (j >= 0 && j < ti.clip_len) ? __ldg(ti.xb + j) : 0.f;
}

template <int KQ>
__device__ __forceinline__ void dct_accumulate(float (&cacc)[MAX_MFCC], const float *drow, float v) {
#pragma unroll
    for (int q = 0; q < KQ; ++q) {
        const float4 d = *reinterpret_cast<const float4 *>(drow + 4 * q);
        cacc[4 * q + 0] = fmaf(d.x, v, cacc[4 * q + 0]);
        cacc[4 * q + 1] = fmaf(d.y, v, cacc[4 * q + 1]);
        cacc[4 * q + 2] = fmaf(d.z, v, cacc[4 * q + 2]);
        cacc[4 * q + 3] = fmaf(d.w, v, cacc[4 * q + 3]);
    }
}

template <int PREC>
__global__ void __launch_bounds__(NUM_THREADS, 1) melt_fwd_kernel(const __grid_constant__ KParams p) {
    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t sbase = smem_u32(smem);
    const uint32_t bar0 = sbase + p.off_bar;
    auto BAR = [&](int idx) -> uint32_t { return bar0 + (uint32_t)idx * 8u; };
    uint32_t *tmem_ptr_s = reinterpret_cast<uint32_t *>(smem + p.off_bar + NBARS * 8);
    float *stg = reinterpret_cast<float *>(smem + p.off_stg);
    uint32_t *tab_s = reinterpret_cast<uint32_t *>(smem + p.off_tab);
    float *dct_s = reinterpret_cast<float *>(smem + p.off_dct);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    // ------------------------------------------------------------------ one-time setup
    if (tid == 0) {
        for (int i = 0; i < MAX_B_SLOTS; ++i) { mbar_init(BAR(B_FULL + i), 1); mbar_init(BAR(B_EMPTY + i), 1); }
        for (int i = 0; i < MAX_A_SLOTS; ++i) { mbar_init(BAR(A_FULL + i), NUM_CONV_THREADS / 2); mbar_init(BAR(A_EMPTY + i), 1); }
        for (int i = 0; i < 2; ++i) { mbar_init(BAR(ACC_FULL + i), 1); mbar_init(BAR(ACC_EMPTY + i), NUM_EPI_THREADS); }
        for (int i = 0; i < MAX_STG_SLOTS; ++i) { mbar_init(BAR(STG_FULL + i), NUM_LOAD_THREADS); mbar_init(BAR(STG_EMPTY + i), NUM_CONV_THREADS); }
        fence_barrier_init();
    }
    if (warp == WARP_TMEM) {
        tmem_alloc(smem_u32(tmem_ptr_s), 512);
        tmem_relinquish();
    }
    for (int i = tid; i < p.units * p.kstep; i += NUM_THREADS) tab_s[i] = __ldg(p.tab + i);
    if (p.n_mfcc > 0)
        for (int i = tid; i < p.n_mels * p.dct_pitch; i += NUM_THREADS) dct_s[i] = __ldg(p.dct + i);
    for (int i = tid; i < p.stg_slots * TILE_M; i += NUM_THREADS)  // the zero row of every staging slot
        stg[(size_t)(i / TILE_M) * p.stg_slot_words + (p.stg_slot_words - TILE_M) + (i % TILE_M)] = 0.f;
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr_s;

    const int n_tiles = p.offsets ? __ldg(p.tile_prefix + p.n_clips) : p.n_tiles;
    const int first_tile = blockIdx.x, tile_step = gridDim.x;
    const int chunks_per_pass = (p.units + p.chunk_units - 1) / p.chunk_units;

    if (warp == WARP_BPROD) {
        // ============================================================== basis producer (bulk-copy engine)
        if (lane == 0 && first_tile < n_tiles) {
            if (p.b_resident) {
                for (int u = 0; u < p.units; ++u) {
                    mbar_arrive_expect_tx(BAR(B_FULL + u), p.unit_b_bytes);
                    bulk_g2s(sbase + p.off_b + (uint32_t)u * p.unit_b_bytes, p.b_img + (size_t)u * p.unit_b_bytes, p.unit_b_bytes,
                             BAR(B_FULL + u));
                }
            } else {
                uint32_t it = 0;
                for (int tile = first_tile; tile < n_tiles; tile += tile_step)
                    for (int ps = 0; ps < p.passes; ++ps)
                        for (int u = 0; u < p.units; ++u, ++it) {
                            const uint32_t slot = it % (uint32_t)p.b_slots, ph = (it / (uint32_t)p.b_slots) & 1u;
                            mbar_wait(BAR(B_EMPTY + slot), ph ^ 1u);
                            mbar_arrive_expect_tx(BAR(B_FULL + slot), p.unit_b_bytes);
                            bulk_g2s(sbase + p.off_b + slot * p.unit_b_bytes,
                                     p.b_img + ((size_t)ps * p.units + u) * p.unit_b_bytes, p.unit_b_bytes, BAR(B_FULL + slot));
                        }
            }
        }
    } else if (warp == WARP_MMA) {
        // ============================================================== MMA issuer (one thread)
        if (lane == 0) {
            const uint32_t idesc = umma_idesc(PREC == PREC_COMP ? UMMA_F16 : (PREC == PREC_BF16 ? UMMA_BF16 : UMMA_TF32), (uint32_t)p.nb);
            const uint32_t kind_bytes = (uint32_t)p.nb * 32u;
            uint32_t a_it = 0, b_it = 0, acc_it = 0;
            for (int tile = first_tile; tile < n_tiles; tile += tile_step)
                for (int ps = 0; ps < p.passes; ++ps, ++acc_it) {
                    const uint32_t stage = acc_it % (uint32_t)p.acc_stages, aph = (acc_it / (uint32_t)p.acc_stages) & 1u;
                    mbar_wait(BAR(ACC_EMPTY + stage), aph ^ 1u);
                    tc_fence_after();
                    const uint32_t d_r = tmem_base + stage * (uint32_t)p.acc_cols, d_i = d_r + (uint32_t)p.nb;
                    for (int u = 0; u < p.units; ++u, ++a_it, ++b_it) {
                        const uint32_t aslot = a_it % (uint32_t)p.a_slots;
                        uint32_t bslot;
                        if (p.b_resident) { bslot = (uint32_t)u; mbar_wait(BAR(B_FULL + bslot), 0); }
                        else { bslot = b_it % (uint32_t)p.b_slots; mbar_wait(BAR(B_FULL + bslot), (b_it / (uint32_t)p.b_slots) & 1u); }
                        mbar_wait(BAR(A_FULL + aslot), (a_it / (uint32_t)p.a_slots) & 1u);
                        tc_fence_after();
                        const uint32_t a = tmem_base + (uint32_t)p.a_col0 + aslot * (uint32_t)p.unit_cols;
                        const uint32_t b = sbase + p.off_b + bslot * p.unit_b_bytes;
                        const uint32_t acc = u > 0;
                        if (PREC == PREC_COMP) {
                            // A kinds: s_hi @0, s_lo @8, d_hi @16, d_lo @24;  B kinds: wc_hi, wc_lo, ws_hi, ws_lo
                            const uint64_t wc_hi = umma_smem_desc_kmajor_noswz(b, 128, 256);
                            const uint64_t wc_lo = umma_smem_desc_kmajor_noswz(b + kind_bytes, 128, 256);
                            const uint64_t ws_hi = umma_smem_desc_kmajor_noswz(b + 2 * kind_bytes, 128, 256);
                            const uint64_t ws_lo = umma_smem_desc_kmajor_noswz(b + 3 * kind_bytes, 128, 256);
                            umma_ts_f16(d_r, a + 0, wc_hi, idesc, acc);
                            umma_ts_f16(d_i, a + 16, ws_hi, idesc, acc);
                            umma_ts_f16(d_r, a + 8, wc_hi, idesc, 1);
                            umma_ts_f16(d_i, a + 24, ws_hi, idesc, 1);
                            umma_ts_f16(d_r, a + 0, wc_lo, idesc, 1);
                            umma_ts_f16(d_i, a + 16, ws_lo, idesc, 1);
                        } else {
                            const uint64_t wc = umma_smem_desc_kmajor_noswz(b, 128, 256);
                            const uint64_t ws = umma_smem_desc_kmajor_noswz(b + kind_bytes, 128, 256);
                            if (PREC == PREC_TF32) { umma_ts_tf32(d_r, a + 0, wc, idesc, acc); umma_ts_tf32(d_i, a + 8, ws, idesc, acc); }
                            else { umma_ts_f16(d_r, a + 0, wc, idesc, acc); umma_ts_f16(d_i, a + 8, ws, idesc, acc); }
                        }
                        tc_commit(BAR(A_EMPTY + aslot));
                        if (!p.b_resident) tc_commit(BAR(B_EMPTY + bslot));
                    }
                    tc_commit(BAR(ACC_FULL + stage));
                }
        }
    } else if (warp >= WARP_EPI0 && warp < WARP_EPI0 + 4) {
        // ============================================================== epilogue (thread = frame)
        const int row = (warp & 3) * 32 + lane;
        const uint32_t lane_taddr = tmem_base + ((uint32_t)((warp & 3) * 32) << 16);
        const float kLog10_2 = 0.30102999566398120f;
        uint32_t acc_it = 0;
        for (int tile = first_tile; tile < n_tiles; tile += tile_step) {
            TileInfo ti;
            get_tile(p, tile, ti);
            const bool valid = row < ti.nvalid;
            float cacc[MAX_MFCC];
            if (p.n_mfcc > 0) {
#pragma unroll
                for (int q = 0; q < MAX_MFCC; ++q) cacc[q] = 0.f;
            }
            // element (frame, channel c) of a C-channel output lives at base + c * cstride
            long long fbase, tbase;
            long long cstride_out, cstride_tap;
            if (p.feature_major) {
                fbase = (long long)ti.clip * p.n_ch * ti.T + ti.t0 + row; cstride_out = ti.T;
                tbase = (long long)ti.clip * p.n_mels * ti.T + ti.t0 + row; cstride_tap = ti.T;
            } else {
                fbase = (ti.out_frame0 + row) * p.n_ch; cstride_out = 1;
                tbase = (ti.out_frame0 + row) * p.n_mels; cstride_tap = 1;
            }
            for (int ps = 0; ps < p.passes; ++ps, ++acc_it) {
                const uint32_t stage = acc_it % (uint32_t)p.acc_stages, aph = (acc_it / (uint32_t)p.acc_stages) & 1u;
                mbar_wait(BAR(ACC_FULL + stage), aph);
                tc_fence_after();
                const uint32_t t_r = lane_taddr + stage * (uint32_t)p.acc_cols, t_i = t_r + (uint32_t)p.nb;
                for (int c0 = 0; c0 < p.nb; c0 += 16) {
                    uint32_t vr[16], vi[16];
                    tmem_ld16(t_r + (uint32_t)c0, vr);
                    tmem_ld16(t_i + (uint32_t)c0, vi);
                    tmem_wait_ld();
#pragma unroll
                    for (int c = 0; c < 16; ++c) {
                        const int m = ps * p.nb + c0 + c;
                        if (m < p.n_mels) {
                            const float r = __uint_as_float(vr[c]), im = __uint_as_float(vi[c]);
                            const float praw = fmaf(r, r, im * im);                         // Eq. (4)
                            float v;
                            if (p.output_power == 1) v = praw * p.out_scale;
                            else if (p.output_power == 2) v = lg2_ftz(fmaf(praw, p.out_scale, p.ln_eps)) * 0.69314718055994531f;   // ln(S + eps)
                            else v = fmaxf(fmaf(__log2f(praw), kLog10_2, p.out_log10_offset), -10.f);  // Eq. (8), contract form
                            if (p.n_mfcc > 0) {
                                const float *drow = dct_s + m * p.dct_pitch;
                                if (p.dct_pitch <= 16) dct_accumulate<4>(cacc, drow, v);       // the table's rows are padded to 16 cepstra
                                else if (p.dct_pitch <= 32) dct_accumulate<8>(cacc, drow, v);
                                else if (p.dct_pitch <= 48) dct_accumulate<12>(cacc, drow, v);
                                else dct_accumulate<16>(cacc, drow, v);
                                if (p.tap && valid) p.tap[tbase + m * cstride_tap] = v;
                            } else if (valid) {
                                p.out[fbase + m * cstride_out] = v;
                            }
                        }
                    }
                }
                tc_fence_before();
                mbar_arrive(BAR(ACC_EMPTY + stage));
            }
            if (p.n_mfcc > 0 && valid) {                                                      // Eq. (9)
#pragma unroll
                for (int q = 0; q < MAX_MFCC; ++q)
                    if (q < p.n_mfcc) p.out[fbase + q * cstride_out] = cacc[q];
            }
        }
    } else if (warp >= WARP_CONV0 && warp < WARP_CONV0 + 8) {
        // ============================================================== converters (thread = frame, two groups alternate K-steps)
        const int grp = (warp - WARP_CONV0) >> 2;
        const int row = (warp & 3) * 32 + lane;
        const uint32_t lane_taddr = tmem_base + ((uint32_t)((warp & 3) * 32) << 16);
        uint32_t ug = 0, tile_it = 0;
        for (int tile = first_tile; tile < n_tiles; tile += tile_step, ++tile_it)
            for (int ps = 0; ps < p.passes; ++ps)
                for (int u = 0; u < p.units; ++u, ++ug) {
                    const int chunk = u / p.chunk_units;
                    const uint32_t cidx = p.stg_comb ? (tile_it * (uint32_t)p.passes + (uint32_t)ps) * (uint32_t)chunks_per_pass + (uint32_t)chunk
                                                     : tile_it;
                    const uint32_t sslot = cidx % (uint32_t)p.stg_slots, sph = (cidx / (uint32_t)p.stg_slots) & 1u;
                    if ((int)(ug & 1u) == grp) {
                        const uint32_t aslot = ug % (uint32_t)p.a_slots;
                        mbar_wait(BAR(STG_FULL + sslot), sph);
                        mbar_wait(BAR(A_EMPTY + aslot), ((ug / (uint32_t)p.a_slots) & 1u) ^ 1u);
                        tc_fence_after();
                        const float *sp = stg + (size_t)sslot * p.stg_slot_words + row;
                        const uint4 *tb = reinterpret_cast<const uint4 *>(tab_s + u * p.kstep);
                        const uint32_t dst = lane_taddr + (uint32_t)p.a_col0 + aslot * (uint32_t)p.unit_cols;
                        if (PREC == PREC_TF32) {
                            uint32_t vs[8], vd[8];
#pragma unroll
                            for (int g = 0; g < 2; ++g) {
                                const uint4 t = tb[g];
                                const uint32_t tt[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
                                for (int e = 0; e < 4; ++e) {
                                    const float a = sp[tt[e] & 0xFFFFu], b = sp[tt[e] >> 16];
                                    vs[4 * g + e] = cvt_tf32_rna(a + b);
                                    vd[4 * g + e] = cvt_tf32_rna(a - b);
                                }
                            }
                            tmem_st8(dst + 0, vs);
                            tmem_st8(dst + 8, vd);
                        } else {
                            uint32_t vsh[8], vsl[8], vdh[8], vdl[8];
#pragma unroll
                            for (int g = 0; g < 4; ++g) {
                                const uint4 t = tb[g];
                                const uint32_t tt[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
                                for (int e = 0; e < 4; e += 2) {
                                    const float a0 = sp[tt[e] & 0xFFFFu], b0 = sp[tt[e] >> 16];
                                    const float a1 = sp[tt[e + 1] & 0xFFFFu], b1 = sp[tt[e + 1] >> 16];
                                    const float s0 = a0 + b0, s1 = a1 + b1, d0 = a0 - b0, d1 = a1 - b1;
                                    const int c = 2 * g + (e >> 1);
                                    if (PREC == PREC_COMP) {
                                        const __half2 sh = __floats2half2_rn(s0, s1), dh = __floats2half2_rn(d0, d1);
                                        const float2 shf = __half22float2(sh), dhf = __half22float2(dh);
                                        const __half2 sl = __floats2half2_rn(s0 - shf.x, s1 - shf.y);
                                        const __half2 dl = __floats2half2_rn(d0 - dhf.x, d1 - dhf.y);
                                        vsh[c] = *reinterpret_cast<const uint32_t *>(&sh);
                                        vsl[c] = *reinterpret_cast<const uint32_t *>(&sl);
                                        vdh[c] = *reinterpret_cast<const uint32_t *>(&dh);
                                        vdl[c] = *reinterpret_cast<const uint32_t *>(&dl);
                                    } else {
                                        const __nv_bfloat162 sh = __floats2bfloat162_rn(s0, s1), dh = __floats2bfloat162_rn(d0, d1);
                                        vsh[c] = *reinterpret_cast<const uint32_t *>(&sh);
                                        vdh[c] = *reinterpret_cast<const uint32_t *>(&dh);
                                    }
                                }
                            }
                            if (PREC == PREC_COMP) {
                                tmem_st8(dst + 0, vsh);
                                tmem_st8(dst + 8, vsl);
                                tmem_st8(dst + 16, vdh);
                                tmem_st8(dst + 24, vdl);
                            } else {
                                tmem_st8(dst + 0, vsh);
                                tmem_st8(dst + 8, vdh);
                            }
                        }
                        tmem_wait_st();
                        tc_fence_before();
                        mbar_arrive(BAR(A_FULL + aslot));
                    }
                    // every converter thread releases the staging slot once, after its own last read of the chunk
                    const bool chunk_end = (u == p.units - 1) || ((u + 1) % p.chunk_units == 0);
                    if (chunk_end && (p.stg_comb || ps == p.passes - 1)) mbar_arrive(BAR(STG_EMPTY + sslot));
                }
    } else if (warp >= WARP_LOAD0) {
        // ============================================================== loaders (implicit im2col: global -> transposed staging)
        const int tl = tid - WARP_LOAD0 * 32, wl = warp - WARP_LOAD0;
        const long long padn = p.pad ? (long long)(p.n_fft / 2) : 0;
        uint32_t cit = 0;
        for (int tile = first_tile; tile < n_tiles; tile += tile_step) {
            TileInfo ti;
            get_tile(p, tile, ti);
            const long long src0 = (long long)ti.t0 * p.hop - padn;  // clip coordinate of the tile's first sample
            if (!p.stg_comb) {
                const uint32_t sslot = cit % (uint32_t)p.stg_slots, sph = (cit / (uint32_t)p.stg_slots) & 1u;
                mbar_wait(BAR(STG_EMPTY + sslot), sph ^ 1u);
                float *dst = stg + (size_t)sslot * p.stg_slot_words;
                const int span = (ti.nvalid - 1) * p.hop + p.n_fft;
                const float *base = ti.xb + src0;
                const bool vec_ok = ((reinterpret_cast<uintptr_t>(base) & 15) == 0) && ((p.hop & 3) == 0);
                for (int s = tl * 4; s < span; s += NUM_LOAD_THREADS * 4) {
                    const long long j = src0 + s;
                    float v[4];
                    if (vec_ok && j >= 0 && j + 3 < ti.clip_len) {
                        const float4 t = __ldg(reinterpret_cast<const float4 *>(base + s));
                        v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
                    } else {
#pragma unroll
                        for (int e = 0; e < 4; ++e) v[e] = fetch_sample(p, ti, j + e);
                    }
                    if ((p.hop & 3) == 0) {
                        const uint32_t hrow = (uint32_t)(((unsigned long long)(uint32_t)s * p.hop_inv40) >> 40);
                        const uint32_t phi = (uint32_t)s - hrow * (uint32_t)p.hop;
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            if (s + e < span) dst[(phi + e) * (uint32_t)p.stg_pitch + hrow] = v[e] * p.in_scale;
                    } else {
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const uint32_t se = (uint32_t)(s + e);
                            const uint32_t hrow = (uint32_t)(((unsigned long long)se * p.hop_inv40) >> 40);
                            const uint32_t phi = se - hrow * (uint32_t)p.hop;
                            if (s + e < span) dst[phi * (uint32_t)p.stg_pitch + hrow] = v[e] * p.in_scale;
                        }
                    }
                }
                mbar_arrive(BAR(STG_FULL + sslot));
                ++cit;
            } else {
                for (int ps = 0; ps < p.passes; ++ps)
                    for (int ch = 0; ch < chunks_per_pass; ++ch, ++cit) {
                        const uint32_t sslot = cit % (uint32_t)p.stg_slots, sph = (cit / (uint32_t)p.stg_slots) & 1u;
                        mbar_wait(BAR(STG_EMPTY + sslot), sph ^ 1u);
                        float *dst = stg + (size_t)sslot * p.stg_slot_words;
                        const int j0 = ch * 64;
                        for (int r = wl; r < ti.nvalid; r += NUM_LOAD_THREADS / 32)
                            for (int c = lane; c < 128; c += 32) {
                                const int j = j0 + (c & 63);
                                if (j < p.kf) {
                                    const int n = c < 64 ? p.a0 + j : p.b0 - j;
                                    dst[c * p.stg_pitch + r] = fetch_sample(p, ti, src0 + (long long)r * p.hop + n) * p.in_scale;
                                }
                            }
                        mbar_arrive(BAR(STG_FULL + sslot));
                    }
            }
        }
    }

    // ------------------------------------------------------------------ teardown
    tc_fence_before();
    __syncthreads();
    if (warp == WARP_TMEM) tmem_dealloc(tmem_base, 512);
}

// ---------------------------------------------------------------------------------------------- ragged prologue
// frame counts -> exclusive prefix sums of frames (int64, caller's array) and of 128-frame tiles (int32, plan workspace)
__global__ void __launch_bounds__(1024, 1) ragged_scan_kernel(const KParams p, const long long *offsets, int n_clips,
                                                             long long *frame_offsets, int *tile_prefix, int tile_m) {
    __shared__ long long wf[32];
    __shared__ int wt[32];
    __shared__ long long carry_f;
    __shared__ int carry_t;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // Programmatic dependent launch (see launch_ragged_scan): this block may have been scheduled while the previous kernel of the
    // stream is still running -- the forward kernel behind it may be scheduled now, and nothing is read or written before that
    // previous kernel (which may produce `offsets`, or still read the arrays written below) has completed.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (tid == 0) { carry_f = 0; carry_t = 0; }
    __syncthreads();
    for (int base = 0; base < n_clips; base += 1024) {
        const int i = base + tid;
        long long f = 0;
        int t = 0;
        if (i < n_clips) {
            f = frames_of(p, offsets[i + 1] - offsets[i]);
            t = (int)((f + tile_m - 1) / tile_m);
        }
        long long fi = f;
        int tii = t;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const long long a = __shfl_up_sync(0xffffffffu, fi, d);
            const int b = __shfl_up_sync(0xffffffffu, tii, d);
            if (lane >= d) { fi += a; tii += b; }
        }
        if (lane == 31) { wf[warp] = fi; wt[warp] = tii; }
        __syncthreads();
        if (warp == 0) {
            long long a = wf[lane];
            int b = wt[lane];
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const long long a2 = __shfl_up_sync(0xffffffffu, a, d);
                const int b2 = __shfl_up_sync(0xffffffffu, b, d);
                if (lane >= d) { a += a2; b += b2; }
            }
            wf[lane] = a; wt[lane] = b;
        }
        __syncthreads();
        const long long pf = carry_f + (warp ? wf[warp - 1] : 0) + fi - f;  // exclusive
        const int pt = carry_t + (warp ? wt[warp - 1] : 0) + tii - t;
        if (i < n_clips) { frame_offsets[i] = pf; tile_prefix[i] = pt; }
        __syncthreads();
        if (tid == 1023) { carry_f = pf + f; carry_t = pt + t; }
        __syncthreads();
    }
    if (tid == 0) { frame_offsets[n_clips] = carry_f; tile_prefix[n_clips] = carry_t; }
}

int launch_ragged_scan(const melt_plan *pl, const long long *offsets, int n_clips, long long *frame_offsets, int *tile_prefix, int tile_m, cudaStream_t stream) {
    // launched like the forward kernels (programmatic stream serialisation): the block is scheduled as soon as an SM of the previous
    // kernel frees up and orders itself behind that kernel with griddepcontrol.wait, instead of paying a full launch latency after
    // the previous forward has drained -- and the forward kernel behind it is scheduled early in turn
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(1, 1, 1);
    cfg.blockDim = dim3(1024, 1, 1);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    MELT_CUDA(cudaLaunchKernelEx(&cfg, ragged_scan_kernel, pl->kp, offsets, n_clips, frame_offsets, tile_prefix, tile_m));
    return MELT_OK;
}

int launch_forward(const melt_plan *pl, const KParams &kp, cudaStream_t stream) {
    // the opt-in shared-memory size is a per-device attribute of the function: set once per device (bit d of the mask)
    static std::atomic<unsigned long long> attr_done{0};
    const unsigned long long bit = 1ull << (pl->device & 63);
    if (pl->device >= 64 || !(attr_done.load(std::memory_order_acquire) & bit)) {
        MELT_CUDA(cudaFuncSetAttribute(melt_fwd_kernel<PREC_COMP>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BUDGET));
        MELT_CUDA(cudaFuncSetAttribute(melt_fwd_kernel<PREC_TF32>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BUDGET));
        MELT_CUDA(cudaFuncSetAttribute(melt_fwd_kernel<PREC_BF16>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BUDGET));
        attr_done.fetch_or(bit, std::memory_order_release);
    }
    int grid = pl->sm_count;
    if (kp.n_tiles >= 0 && kp.n_tiles < grid) grid = kp.n_tiles;
    if (grid < 1) return MELT_OK;
    switch (pl->precision) {
        case MELT_PREC_COMPENSATED: melt_fwd_kernel<PREC_COMP><<<grid, NUM_THREADS, kp.smem_bytes, stream>>>(kp); break;
        case MELT_PREC_TF32: melt_fwd_kernel<PREC_TF32><<<grid, NUM_THREADS, kp.smem_bytes, stream>>>(kp); break;
        default: melt_fwd_kernel<PREC_BF16><<<grid, NUM_THREADS, kp.smem_bytes, stream>>>(kp); break;
    }
    MELT_CUDA(cudaGetLastError());
    return MELT_OK;
}

}  // namespace melt
