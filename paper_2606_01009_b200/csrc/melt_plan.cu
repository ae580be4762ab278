// melt_plan.cu -- host side of the C ABI: plan construction (Eq. 1, 2, 5, 9 in double precision, conversion to
// tensor-core operand images), options, validation and the forward entry points.
//
// What the plan precomputes:
//   * f_m.
//   * The window w[n] and its symmetry centre c = (a0 + b0)/2.  Both Hann flavours and the
//     rectangular window satisfy w[a0 + j] = w[b0 - j]; P = R^2 + I^2 does not depend on the phase origin, so with
//     the phase referred to c the cos rows are even and the sin rows odd about c, and Eq. (3) folds to
//         R' = sum_j wc[m][j] (x[a0+j] + x[b0-j]),   I' = sum_j ws[m][j] (x[a0+j] - x[b0-j]),   j = 0..kf-1
//     with wc[m][j] = g_j w[a0+j] cos(w_m (a0 + j - c)), ws[m][j] = w[a0+j] sin(w_m (a0 + j - c)), g_j = 1/2 for
//     the self-paired centre sample, 1 otherwise.  R'^2 + I'^2 = R^2 + I^2 exactly; half the MMA work of Eq. (6).
//   * The basis images: for every pass over the Mel bins and every K-step, one contiguous slab per operand kind in
//     the no-swizzle canonical UMMA layout, so that the kernel moves a K-step of the basis with ONE bulk copy.
#include "melt_plan.h"

#include <algorithm>

namespace melt {

static const double kPi = 3.14159265358979323846264338327950288;
static const int kBasisScaleLog2 = 14;  // COMPENSATED: basis stored as 2^14 * value (keeps the fp16 lo part normal)

static double hz_to_mel(double f) { return 2595.0 * std::log10(1.0 + f / 700.0); }    // Eq. (1)
static double mel_to_hz(double m) { return 700.0 * (std::pow(10.0, m / 2595.0) - 1.0); }  // Eq. (2)

static long long frames_for(const melt_plan *p, long long len) {
    if (len < 0) return 0;
    long long padded = len;
    if (p->pad == MELT_PAD_REFLECT) {
        if (len < (long long)(p->n_fft / 2) + 1) return 0;
        padded += 2LL * (p->n_fft / 2);
    }
    if (padded < p->n_fft) return 0;
    long long T = (padded - p->n_fft) / p->hop + 1 - (p->drop_last ? 1 : 0);
    return T < 0 ? 0 : T;
}

static void free_device(melt_plan *p) {
    cudaFree(p->d_bimg);
    cudaFree(p->d_tab);
    cudaFree(p->d_dct);
    cudaFree(p->d_bimg2);
    cudaFree(p->d_fbimg);
    p->d_bimg2 = nullptr;
    p->d_fbimg = nullptr;
    p->v2_ok = false;
    p->d_bimg = nullptr;
    p->d_tab = nullptr;
    p->d_dct = nullptr;
}

static int round_up(int v, int m) { return (v + m - 1) / m * m; }

int plan_build_device(melt_plan *p) {
    KParams &k = p->kp;
    const int N = p->n_fft, H = p->hop, M = p->n_mels;
    const int kind = p->precision == MELT_PREC_COMPENSATED ? OP_F16 : (p->precision == MELT_PREC_BF16 ? OP_BF16 : OP_TF32);
    const bool comp = p->precision == MELT_PREC_COMPENSATED;

    // ---- fold geometry
    const int c2 = (p->window == MELT_WINDOW_HANN_PERIODIC) ? N : N - 1;  // w[n] = w[c2 - n]
    k.a0 = (c2 + 1) / 2;
    k.b0 = c2 / 2;
    k.kf = N - k.a0;
    if (k.kf < 1) return fail(MELT_ERR_UNSUPPORTED, "n_fft=%d too short for the folded projection", N);
    for (int j = 0; j < k.kf; ++j) {
        int na = k.a0 + j, nb = k.b0 - j;
        double wb = nb >= 0 ? p->win[nb] : 0.0;
        if (nb < 0 && std::fabs(p->win[na]) > 1e-14) return fail(MELT_ERR_UNSUPPORTED, "window is not symmetric");
        if (nb >= 0 && std::fabs(p->win[na] - wb) > 1e-13) return fail(MELT_ERR_UNSUPPORTED, "window is not symmetric");
    }
    const double centre = 0.5 * (double)c2;

    // ---- tiling of the contraction and of the Mel bins
    k.n_fft = N; k.hop = H; k.n_mels = M; k.n_mfcc = p->n_mfcc; k.n_ch = p->fb_mels > 0 ? p->fb_mels : (p->n_mfcc > 0 ? p->n_mfcc : M);   // (conventional plan: M DFT bins in, fb_mels filters out)
    k.kstep = operand_kstep(kind);
    k.units = (k.kf + k.kstep - 1) / k.kstep;
    k.nk = comp ? 4 : 2;
    k.passes = (M + 127) / 128;
    k.nb = round_up((M + k.passes - 1) / k.passes, 16);
    k.acc_cols = 2 * k.nb;
    k.unit_cols = k.nk * 8;
    k.acc_stages = (2 * k.acc_cols + 4 * k.unit_cols <= 512) ? 2 : 1;
    k.a_col0 = k.acc_stages * k.acc_cols;
    k.a_slots = std::min(MAX_A_SLOTS, (512 - k.a_col0) / k.unit_cols);
    if (k.a_slots < 2) return fail(MELT_ERR_UNSUPPORTED, "tensor-memory budget exceeded (nb=%d)", k.nb);
    k.unit_b_bytes = (uint32_t)(k.nk * k.nb * 32);
    k.dct_pitch = round_up(std::max(p->n_mfcc, 1), 16);   // floats per Mel bin: whole blocks of 16 cepstra (zero padded)

    // ---- shared-memory plan
    const uint32_t tab_bytes = (uint32_t)(k.units * k.kstep * 4);
    const uint32_t dct_bytes = p->n_mfcc > 0 ? (uint32_t)(M * k.dct_pitch * 4) : 0;
    const uint32_t bar_bytes = 1024;
    const uint32_t fixed = round_up((int)(tab_bytes + dct_bytes + bar_bytes), 128) + 128;
    const int rows_whole = TILE_M + (N - 1) / H;          // hop-rows touched by one tile
    const int pitch_whole = rows_whole | 1;               // odd: conflict-free transposed stores
    const long long whole_words = (long long)H * pitch_whole + TILE_M;
    const long long whole_bytes = whole_words * 4;
    k.hop_inv40 = ((1ull << 40) + (unsigned long long)H - 1) / (unsigned long long)H;
    const bool whole_ok = whole_words < 65536 && (long long)TILE_M * H + N < (1 << 24) && H < 65536 &&
                          whole_bytes + 2LL * k.unit_b_bytes + fixed <= SMEM_BUDGET;
    uint32_t stg_bytes;
    if (whole_ok) {
        k.stg_comb = 0; k.stg_slots = 1; k.chunk_units = k.units;
        k.stg_pitch = pitch_whole; k.stg_slot_words = (int)whole_words;
        stg_bytes = (uint32_t)whole_bytes;
    } else {
        k.stg_comb = 1; k.chunk_units = 64 / k.kstep;  // 64 folded samples per chunk
        k.stg_pitch = TILE_M + 1;
        k.stg_slot_words = 2 * 64 * k.stg_pitch + TILE_M;
        k.stg_slots = 3;
        while (k.stg_slots > 2 && (long long)SMEM_BUDGET - (long long)k.stg_slots * k.stg_slot_words * 4 - fixed < 4LL * k.unit_b_bytes)
            --k.stg_slots;  // wide bases (M = 128 per pass, fp16x3): trade one staging slot for a deeper basis ring
        stg_bytes = (uint32_t)(k.stg_slots * k.stg_slot_words * 4);
    }
    const long long b_room = (long long)SMEM_BUDGET - stg_bytes - fixed;
    int fit = (int)std::min<long long>(b_room / k.unit_b_bytes, MAX_B_SLOTS);
    if (fit < 2) return fail(MELT_ERR_UNSUPPORTED, "shared-memory budget exceeded (n_fft=%d hop=%d n_mels=%d)", N, H, M);
    k.b_resident = (k.passes == 1 && k.units <= fit) ? 1 : 0;
    k.b_slots = k.b_resident ? k.units : std::min(fit, 8);
    k.off_b = 0;
    k.off_stg = (uint32_t)round_up((int)(k.b_slots * k.unit_b_bytes), 128);
    k.off_tab = k.off_stg + (uint32_t)round_up((int)stg_bytes, 128);
    k.off_dct = k.off_tab + (uint32_t)round_up((int)tab_bytes, 16);
    k.off_bar = (uint32_t)round_up((int)(k.off_dct + dct_bytes), 16);
    k.smem_bytes = k.off_bar + bar_bytes;
    if (k.smem_bytes > (uint32_t)SMEM_BUDGET) return fail(MELT_ERR_UNSUPPORTED, "shared-memory budget exceeded");

    // ---- numerics
    const int s_in = comp ? p->in_scale_log2 : 0, s_b = comp ? kBasisScaleLog2 : 0;
    k.in_scale = (float)std::ldexp(1.0, s_in);
    k.out_scale = (float)std::ldexp(1.0, -2 * (s_in + s_b));
    k.out_log10_offset = (float)(-2.0 * (s_in + s_b) * std::log10(2.0));
    k.output_power = p->output == MELT_OUTPUT_LOG_WHISPER ? MELT_OUTPUT_LOG : p->output;   // melt_output of the forward kernel (the Whisper normalisation is a post-pass)
    k.ln_eps = (float)std::pow(10.0, (double)p->eps_exp10);
    k.pad = p->pad; k.drop_last = p->drop_last; k.feature_major = p->layout == MELT_LAYOUT_FEATURE_MAJOR;

    // ---- staging offset table: for folded index j, where samples a0 + j and b0 - j of a frame live in a staging slot
    //      (word offset of row 0; the converter adds its row).  j >= kf (K padding) points at the zero row.
    std::vector<uint32_t> tab((size_t)k.units * k.kstep);
    const uint32_t zero_off = (uint32_t)(k.stg_slot_words - TILE_M);
    for (int j = 0; j < k.units * k.kstep; ++j) {
        uint32_t oa = zero_off, ob = zero_off;
        if (j < k.kf) {
            if (!k.stg_comb) {
                int na = k.a0 + j, nb = k.b0 - j;
                oa = (uint32_t)((na % H) * k.stg_pitch + na / H);
                ob = nb >= 0 ? (uint32_t)((nb % H) * k.stg_pitch + nb / H) : zero_off;
            } else {
                int jc = j % 64;
                oa = (uint32_t)(jc * k.stg_pitch);
                ob = (k.b0 - j >= 0) ? (uint32_t)((64 + jc) * k.stg_pitch) : zero_off;
            }
        }
        tab[j] = oa | (ob << 16);
    }

    // ---- basis images (Eq. 5 folded), double -> operand format in one rounding
    const double bscale = std::ldexp(1.0, s_b);
    const size_t img_bytes = (size_t)k.passes * k.units * k.unit_b_bytes;
    std::vector<uint8_t> img(img_bytes, 0);
    auto coef = [&](int m, int j, bool sine) -> double {
        if (m >= M || j >= k.kf) return 0.0;
        const int na = k.a0 + j;
        const double g = (na == k.b0 - j) ? 0.5 : 1.0;
        const double arg = 2.0 * kPi * p->centres[m] * ((double)na - centre) / p->fs;
        return bscale * p->win[na] * (sine ? std::sin(arg) : g * std::cos(arg));
    };
    auto hi_of = [&](double v) -> double {
        if (kind == OP_F16) return f16_bits_to_f64(f64_to_f16_bits(v));
        if (kind == OP_BF16) return bf16_bits_to_f64(f64_to_bf16_bits(v));
        return tf32_bits_to_f64(f64_to_tf32_bits(v));
    };
    for (int ps = 0; ps < k.passes; ++ps)
        for (int u = 0; u < k.units; ++u) {
            uint8_t *slab = img.data() + ((size_t)ps * k.units + u) * k.unit_b_bytes;
            for (int kk = 0; kk < k.nk; ++kk) {
                // kinds: COMPENSATED [wc_hi, wc_lo, ws_hi, ws_lo]; single pass [wc, ws]
                const bool sine = comp ? (kk >= 2) : (kk == 1);
                const bool lo = comp && (kk & 1);
                pack_b_slab(kind, k.nb, [&](int r, int kq) {
                    double v = coef(ps * k.nb + r, u * k.kstep + kq, sine);
                    return lo ? v - hi_of(v) : v;
                }, slab + (size_t)kk * k.nb * 32);
            }
        }

    // ---- DCT table (Eq. 9), [m][k] so a thread reads all k of one bin as float4s
    std::vector<float> dct;
    if (p->n_mfcc > 0) {
        dct.assign((size_t)M * k.dct_pitch, 0.f);
        for (int m = 0; m < M; ++m)
            for (int q = 0; q < p->n_mfcc; ++q) {
                double d = q == 0 ? std::sqrt(1.0 / M) : std::sqrt(2.0 / M) * std::cos(kPi * q * (2 * m + 1) / (2.0 * M));
                dct[(size_t)m * k.dct_pitch + q] = (float)d;
            }
    }

    // ---- upload
    free_device(p);
    MELT_CUDA(cudaMalloc(&p->d_bimg, img_bytes));
    MELT_CUDA(cudaMemcpy(p->d_bimg, img.data(), img_bytes, cudaMemcpyHostToDevice));
    MELT_CUDA(cudaMalloc(&p->d_tab, tab.size() * 4));
    MELT_CUDA(cudaMemcpy(p->d_tab, tab.data(), tab.size() * 4, cudaMemcpyHostToDevice));
    if (!dct.empty()) {
        MELT_CUDA(cudaMalloc(&p->d_dct, dct.size() * 4));
        MELT_CUDA(cudaMemcpy(p->d_dct, dct.data(), dct.size() * 4, cudaMemcpyHostToDevice));
    }
    k.b_img = p->d_bimg; k.tab = p->d_tab; k.dct = p->d_dct;

    char buf[512];
    snprintf(buf, sizeof(buf),
             "melt_b200 prec=%s fold(a0=%d,b0=%d,kf=%d) kstep=%d units=%d nb=%d passes=%d tmem(acc=%dx%d,a_slots=%d) "
             "basis=%s(%d x %u B) staging=%s(%d x %d words) smem=%u B",
             comp ? "fp16x3" : (kind == OP_BF16 ? "bf16" : "tf32"), k.a0, k.b0, k.kf, k.kstep, k.units, k.nb, k.passes,
             k.acc_stages, k.acc_cols, k.a_slots, k.b_resident ? "resident" : "ring", k.b_slots, k.unit_b_bytes,
             k.stg_comb ? "comb" : "whole", k.stg_slots, k.stg_slot_words, k.smem_bytes);
    p->desc = buf;
    return plan_build_v2(p);   // the CTA-pair kernel takes the geometries it covers; this kernel stays the general path
}

static int validate_common(const melt_plan *p, const float *x, void *out) {
    if (!p) return fail(MELT_ERR_INVALID_ARG, "plan is NULL");
    if (!x || !out) return fail(MELT_ERR_INVALID_ARG, "x / out is NULL");
    const uintptr_t omask = p->out_dtype == MELT_DTYPE_F32 ? 3 : 1;
    if (((uintptr_t)x & 3) || ((uintptr_t)out & omask)) return fail(MELT_ERR_ALIGNMENT, "x must be 4-byte aligned, out aligned to its element size");
    int dev = -1;
    MELT_CUDA(cudaGetDevice(&dev));
    if (dev != p->device) return fail(MELT_ERR_INVALID_ARG, "plan was created on device %d, current device is %d", p->device, dev);
    return MELT_OK;
}

// Per-call device scratch from the plan's stream-ordered pool: usable by work submitted to `st` after this call, released
// (cudaFreeAsync on `st`) once everything that uses it has been submitted.  No host synchronisation, nothing stored in the plan.
static int scratch_alloc(const melt_plan *p, void **ptr, size_t bytes, cudaStream_t st) {
    *ptr = nullptr;
    if (cudaMallocFromPoolAsync(ptr, bytes, p->pool, st) != cudaSuccess) {
        (void)cudaGetLastError();
        return fail(MELT_ERR_ALLOC, "per-call scratch of %zu bytes (stream-ordered pool)", bytes);
    }
    return MELT_OK;
}

// ---- MELT_OUTPUT_LOG_WHISPER post-pass: per clip, L <- (max(L, max_clip(L) - 8) + 4) / 4 (any layout: a clip is `per_clip` contiguous floats)
__device__ __forceinline__ int float_order(float f) { const int i = __float_as_int(f); return i >= 0 ? i : i ^ 0x7fffffff; }   // monotone float -> int
__global__ void whisper_max_kernel(const float *__restrict__ out, long long per_clip, int *__restrict__ cmax) {
    const float *o = out + (long long)blockIdx.y * per_clip;
    float m = -3.0e38f;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < per_clip; i += (long long)gridDim.x * blockDim.x) m = fmaxf(m, __ldg(o + i));
    for (int d = 16; d > 0; d >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, d));
    if ((threadIdx.x & 31) == 0) atomicMax(cmax + blockIdx.y, float_order(m));
}
__global__ void whisper_apply_kernel(float *__restrict__ out, long long per_clip, const int *__restrict__ cmax) {
    float *o = out + (long long)blockIdx.y * per_clip;
    const int c = cmax[blockIdx.y];
    const float floor_v = __int_as_float(c >= 0 ? c : c ^ 0x7fffffff) - 8.0f;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < per_clip; i += (long long)gridDim.x * blockDim.x)
        o[i] = (fmaxf(o[i], floor_v) + 4.0f) * 0.25f;
}
static int scratch_alloc(const melt_plan *p, void **ptr, size_t bytes, cudaStream_t st);
static int whisper_normalise(const melt_plan *p, float *out, int n_clips, long long per_clip, cudaStream_t st) {
    int *cmax = nullptr;
    int rc = scratch_alloc(p, (void **)&cmax, sizeof(int) * (size_t)n_clips, st);
    if (rc) return rc;
    cudaError_t e = cudaMemsetAsync(cmax, 0x80, sizeof(int) * (size_t)n_clips, st);   // 0x80808080: below the order key of any log10 value
    const unsigned bx = (unsigned)std::max<long long>(1, std::min<long long>((per_clip + 2047) / 2048, 256));
    if (e == cudaSuccess) { whisper_max_kernel<<<dim3(bx, (unsigned)n_clips), 256, 0, st>>>(out, per_clip, cmax); e = cudaGetLastError(); }
    if (e == cudaSuccess) { whisper_apply_kernel<<<dim3(bx, (unsigned)n_clips), 256, 0, st>>>(out, per_clip, cmax); e = cudaGetLastError(); }
    cudaFreeAsync(cmax, st);
    return e == cudaSuccess ? MELT_OK : cuda_fail(e, "whisper normalisation");
}

static int forward_impl(const melt_plan *p, const float *x, const long long *offsets, int n_clips, long long len,
                        void *out_any, float *tap, long long *out_frame_offsets, void *stream, bool input_ready) {
    int rc = validate_common(p, x, out_any);
    if (rc) return rc;
    float *out = static_cast<float *>(out_any);   // 16-bit outputs: the CTA-pair kernel addresses it in bytes
    const bool out16 = p->out_dtype != MELT_DTYPE_F32;
    if (out16 && (p->n_mfcc > 0 || p->output != MELT_OUTPUT_LOG || tap))
        return fail(MELT_ERR_UNSUPPORTED, "16-bit output: log-Mel output (n_mfcc == 0, MELT_OUTPUT_LOG, no tap) only");
    if (p->fb_mels > 0 && (offsets || tap || !p->v2_ok))
        return fail(MELT_ERR_UNSUPPORTED, "conventional (STFT + Mel filterbank) plan: dense batches through melt_forward / melt_forward_host only");
    const bool whisper = p->output == MELT_OUTPUT_LOG_WHISPER;
    if (whisper && (offsets || tap)) return fail(MELT_ERR_UNSUPPORTED, "Whisper-normalised output: dense batches without tap only");
    if (n_clips < 0) return fail(MELT_ERR_INVALID_ARG, "negative clip count");
    if (tap && ((uintptr_t)tap & 3)) return fail(MELT_ERR_ALIGNMENT, "logmel must be 4-byte aligned");
    p->used.store(true, std::memory_order_relaxed);
    if (n_clips == 0) return MELT_OK;
    KParams kp = p->kp;
    kp.x = x; kp.out = out; kp.tap = tap; kp.n_clips = n_clips;
    cudaStream_t st = (cudaStream_t)stream;
    const bool reflect = p->pad == MELT_PAD_REFLECT;
    if (offsets) {
        if (n_clips > MAX_CLIPS) return fail(MELT_ERR_UNSUPPORTED, "n_clips=%d exceeds %d", n_clips, MAX_CLIPS);
        if (!out_frame_offsets) return fail(MELT_ERR_INVALID_ARG, "out_frame_offsets is NULL");
        if (kp.feature_major) return fail(MELT_ERR_UNSUPPORTED, "ragged batches are frame-major only");
        // the device-side tile index of this call (exclusive prefix of tiles per clip): per-call scratch, so that ragged
        // forwards of one plan may run concurrently on several streams
        int *tile_prefix = nullptr;
        rc = scratch_alloc(p, (void **)&tile_prefix, sizeof(int) * ((size_t)n_clips + 1), st);
        if (rc) return rc;
        const bool v2 = p->v2_ok && !p->k2.direct && (((uintptr_t)x & 15) == 0);
        if (v2) {
            // the CTA-pair kernel: tiles of 8 chunks of 32 frames, looked up on the device; chunks start at any sample of the packed buffer
            rc = launch_ragged_scan(p, offsets, n_clips, out_frame_offsets, tile_prefix, 32, st);   // exclusive prefix of 32-frame chunks per clip
            K2Params k2 = p->k2;
            k2.x = x; k2.out = out; k2.tap = tap; k2.n_clips = n_clips; k2.len = 0; k2.frames_per_clip = 0;
            k2.chunks_per_clip = 0; k2.n_tiles = -1;
            k2.offsets = offsets; k2.frame_offsets = out_frame_offsets; k2.tile_prefix = tile_prefix;
            k2.vpad = reflect ? p->n_fft / 2 : 0;
            k2.out_dtype = p->out_dtype;
            k2.input_ready = 0;   // the scan kernel just ahead in the stream produces what the kernel reads at its entry
            if (rc == MELT_OK && v2_encode_tmap_ragged(k2) == MELT_OK && k2.tma_rows > 0) {
                rc = launch_forward2(p, k2, st);
                cudaFreeAsync(tile_prefix, st);
                return rc;
            }
        }
        if (rc == MELT_OK && out16) rc = fail(MELT_ERR_UNSUPPORTED, "16-bit output needs the CTA-pair kernel (hop %% 4 == 0, 16-byte aligned x, staged window)");
        if (rc == MELT_OK) rc = launch_ragged_scan(p, offsets, n_clips, out_frame_offsets, tile_prefix, TILE_M, st);
        kp.offsets = offsets; kp.frame_offsets = out_frame_offsets; kp.tile_prefix = tile_prefix;
        kp.len = 0; kp.frames_per_clip = 0; kp.tiles_per_clip = 0; kp.n_tiles = -1;
        if (rc == MELT_OK) rc = launch_forward(p, kp, st);
        cudaFreeAsync(tile_prefix, st);
        return rc;
    }
    if (len < 0) return fail(MELT_ERR_INVALID_ARG, "negative len");
    const long long T = frames_for(p, len);
    if (T == 0) return MELT_OK;
    const long long tpc = (T + TILE_M - 1) / TILE_M;
    if (tpc * n_clips > 0x7fffffffLL) return fail(MELT_ERR_UNSUPPORTED, "too many tiles");
    const float *const x_caller = x;
    const long long len_caller = len;
    if (p->v2_ok && !(tap && ((uintptr_t)tap & 3))) {
        K2Params k2 = p->k2;
        const bool aligned = v2_accepts(p, x, len);
        // Reflect padding is virtual on the staged forms of the kernel (the loader's edge path mirrors the indices).  Two cases
        // still take ONE copy pass into pool scratch first: a batch whose clip starts are not 16-byte aligned (pointer or clip
        // length; copied at an aligned clip stride), and reflect padding on the direct-load form (very long windows, whose
        // converter threads read their frames from global memory and cannot mirror): the padded signal is written out.
        const bool copy_pad = reflect && (k2.direct || !aligned);
        const bool realign = !reflect && !aligned;
        float *scratch = nullptr;
        if (copy_pad || realign) {
            const int padn = copy_pad ? p->n_fft / 2 : 0;
            const long long plen = (len + 2LL * padn + 3) & ~3LL;   // up to 3 filler samples no frame reads
            rc = scratch_alloc(p, (void **)&scratch, (size_t)n_clips * (size_t)plen * sizeof(float), st);
            if (rc) return rc;
            rc = launch_reflect_pad(x, scratch, n_clips, len, padn, plen, st);
            if (rc) { cudaFreeAsync(scratch, st); return rc; }
            x = scratch;
            len = plen;
            k2.vpad = 0;
            k2.input_ready = 0;   // the copy kernel just ahead in the stream produces the kernel's input
        } else {
            k2.vpad = reflect ? p->n_fft / 2 : 0;
            k2.input_ready = input_ready ? 1 : 0;
        }
        const long long cpc2 = (T + 31) / 32;                          // 32-frame chunks per clip; a tile = 8 consecutive chunks of the batch
        const long long nt2 = (cpc2 * n_clips + 7) / 8;
        if (cpc2 * n_clips > 0x7fffffffLL || nt2 * std::max(1, p->k2.passes) > 0x7fffffffLL) { if (scratch) cudaFreeAsync(scratch, st); return fail(MELT_ERR_UNSUPPORTED, "too many tiles"); }
        k2.x = x; k2.out = out; k2.tap = tap; k2.n_clips = n_clips; k2.len = len; k2.frames_per_clip = T;
        k2.out_dtype = p->out_dtype;
        k2.chunks_per_clip = (int)std::max(1LL, cpc2); k2.n_tiles = (int)nt2;
        k2.offsets = nullptr; k2.frame_offsets = nullptr; k2.tile_prefix = nullptr;
        v2_encode_tmap(k2);
        if (!k2.direct || k2.tma_rows > 0) {   // (K-step staging needs its tensor map; without one the general kernel takes the batch)
            rc = launch_forward2(p, k2, st);
            if (scratch) cudaFreeAsync(scratch, st);
            if (rc == MELT_OK && whisper) rc = whisper_normalise(p, out, n_clips, (long long)T * p->kp.n_ch, st);
            return rc;
        }
        if (scratch) cudaFreeAsync(scratch, st);   // the general kernel pads / realigns on the fly: give it the caller's batch
        x = x_caller;
        len = len_caller;
    }
    if (out16) return fail(MELT_ERR_UNSUPPORTED, "16-bit output needs the CTA-pair kernel (hop %% 4 == 0, n_fft with an aligned fold)");
    kp.offsets = nullptr; kp.frame_offsets = nullptr; kp.tile_prefix = nullptr;
    kp.len = len; kp.frames_per_clip = T; kp.tiles_per_clip = (int)tpc; kp.n_tiles = (int)(tpc * n_clips);
    rc = launch_forward(p, kp, st);
    if (rc == MELT_OK && whisper) rc = whisper_normalise(p, out, n_clips, (long long)T * p->kp.n_ch, st);
    return rc;
}

}  // namespace melt

using namespace melt;

// fb_mels = 0: the MelT / MFCCT plan of the paper.  fb_mels > 0 (melt_plan_create_stft_mel): the conventional front end -- the
// projection runs on the N/2 + 1 DFT bins (n_mels = their number) and a triangular filterbank of fb_mels filters follows the power.
static melt_plan *create_impl(double fs, int n_fft, int hop, int window, int n_mels, double fmin, double fmax,
                              int mel_scale, int n_mfcc, int fb_mels) {
    if (!(fs > 0.0) || !std::isfinite(fs)) { set_error("fs must be positive"); return nullptr; }
    if (n_fft < 2 || n_fft > 65536) { set_error("n_fft=%d out of range [2, 65536]", n_fft); return nullptr; }
    if (hop < 1 || hop > 65535) { set_error("hop=%d out of range [1, 65535]", hop); return nullptr; }
    if (window < 0 || window > 2) { set_error("unknown window %d", window); return nullptr; }
    if (n_mels < 1 || n_mels > 1024) { set_error("n_mels=%d out of range [1, 1024]", n_mels); return nullptr; }
    if (!(fmin >= 0.0) || !(fmax > fmin) || !(fmax <= fs / 2.0 * (1.0 + 1e-12))) {
        set_error("need 0 <= fmin < fmax <= fs/2 (got %g, %g, fs=%g)", fmin, fmax, fs);
        return nullptr;
    }
    if (mel_scale != MELT_MEL_HTK) { set_error("mel_scale %d unsupported: the paper defines the HTK scale only", mel_scale); return nullptr; }
    if (n_mfcc < 0 || n_mfcc > n_mels || n_mfcc > MAX_MFCC) { set_error("n_mfcc=%d out of range [0, min(n_mels, %d)]", n_mfcc, MAX_MFCC); return nullptr; }
    int dev = 0;
    cudaDeviceProp prop;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) { cuda_fail(e, "cudaGetDeviceProperties"); return nullptr; }
    if (prop.major != 10) { set_error("device is sm_%d%d: this library is sm_100a only and has no fallback", prop.major, prop.minor); return nullptr; }

    melt_plan *p = new (std::nothrow) melt_plan();
    if (!p) { set_error("out of host memory"); return nullptr; }
    p->fs = fs; p->fmin = fmin; p->fmax = fmax; p->n_fft = n_fft; p->hop = hop; p->window = window; p->n_mels = n_mels;
    p->mel_scale = mel_scale; p->n_mfcc = n_mfcc;
    p->layout = MELT_LAYOUT_FRAME_MAJOR; p->precision = MELT_PREC_COMPENSATED; p->drop_last = 0; p->pad = MELT_PAD_NONE;
    p->in_scale_log2 = 12; p->output = MELT_OUTPUT_LOG; p->input_ready = 0; p->out_dtype = MELT_DTYPE_F32; p->eps_exp10 = -10; p->used.store(false); p->device = dev; p->sm_count = prop.multiProcessorCount;
    p->fb_mels = fb_mels; p->d_fbimg = nullptr;
    p->d_bimg = nullptr; p->d_bimg2 = nullptr; p->v2_ok = false; p->v2_sigma = 0; p->d_tab = nullptr; p->d_dct = nullptr;
    p->pool = nullptr; p->copy_in = nullptr; p->copy_out = nullptr;
    memset(&p->kp, 0, sizeof(p->kp));
    {   // the scratch pool: device memory of this device, kept (not returned to the driver) between calls
        cudaMemPoolProps props;
        memset(&props, 0, sizeof(props));
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        e = cudaMemPoolCreate(&p->pool, &props);
        if (e == cudaSuccess) {
            unsigned long long keep = ~0ull;
            e = cudaMemPoolSetAttribute(p->pool, cudaMemPoolAttrReleaseThreshold, &keep);
        }
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&p->copy_in, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&p->copy_out, cudaStreamNonBlocking);
        if (e != cudaSuccess) { cuda_fail(e, "scratch pool / copy streams"); melt_plan_destroy(p); return nullptr; }
    }
    // Eq. (1)-(2): M centres uniformly spaced in mel between fmin and fmax, endpoints excluded
    p->centres.resize(n_mels);
    const double mlo = hz_to_mel(fmin), mhi = hz_to_mel(fmax);
    for (int m = 0; m < n_mels; ++m) p->centres[m] = mel_to_hz(mlo + (double)(m + 1) * (mhi - mlo) / (double)(n_mels + 1));
    if (fb_mels > 0) {
        // conventional front end: analysis frequencies = the DFT bins k fs / N, k = 0 .. N/2, then
        // F[m][k] = max(0, min((f_k - e_m) / (e_{m+1} - e_m), (e_{m+2} - f_k) / (e_{m+2} - e_{m+1}))) with the M + 2 edges e uniform
        // in HTK mel between fmin and fmax (their interior points are the MelT centres); peak 1, no normalisation
        for (int k = 0; k < n_mels; ++k) p->centres[k] = (double)k * fs / (double)n_fft;
        std::vector<double> e((size_t)fb_mels + 2);
        for (int i = 0; i < fb_mels + 2; ++i) e[i] = mel_to_hz(mlo + (double)i * (mhi - mlo) / (double)(fb_mels + 1));
        p->fb.assign((size_t)fb_mels * n_mels, 0.0);
        for (int m = 0; m < fb_mels; ++m)
            for (int k = 0; k < n_mels; ++k) {
                const double f = p->centres[k];
                const double up = (f - e[m]) / (e[m + 1] - e[m]), down = (e[m + 2] - f) / (e[m + 2] - e[m + 1]);
                p->fb[(size_t)m * n_mels + k] = std::max(0.0, std::min(up, down));
            }
    }
    p->win.resize(n_fft);
    for (int n = 0; n < n_fft; ++n) {
        if (window == MELT_WINDOW_HANN_PERIODIC) p->win[n] = 0.5 - 0.5 * std::cos(2.0 * kPi * n / n_fft);
        else if (window == MELT_WINDOW_HANN_SYMMETRIC) p->win[n] = 0.5 - 0.5 * std::cos(2.0 * kPi * n / (n_fft - 1));
        else p->win[n] = 1.0;
    }
    if (plan_build_device(p) != MELT_OK) { melt_plan_destroy(p); return nullptr; }
    if (fb_mels > 0 && !p->v2_ok) {
        set_error("melt_plan_create_stft_mel: geometry not covered (needs hop %% 4 == 0, an aligned fold and n_fft / 2 + 1 <= 224 bins: n_fft=%d hop=%d)", n_fft, hop);
        melt_plan_destroy(p);
        return nullptr;
    }
    return p;
}

extern "C" melt_plan *melt_plan_create(double fs, int n_fft, int hop, int window, int n_mels, double fmin, double fmax,
                                       int mel_scale, int n_mfcc) {
    return create_impl(fs, n_fft, hop, window, n_mels, fmin, fmax, mel_scale, n_mfcc, 0);
}

extern "C" melt_plan *melt_plan_create_stft_mel(double fs, int n_fft, int hop, int window, int n_mels, double fmin, double fmax) {
    if (n_mels < 1 || n_mels > 128) { set_error("n_mels=%d out of range [1, 128] for the conventional front end", n_mels); return nullptr; }
    if (n_fft < 2 || (n_fft & 1) || n_fft / 2 + 1 > 224) { set_error("melt_plan_create_stft_mel: n_fft=%d must be even with n_fft / 2 + 1 <= 224 bins", n_fft); return nullptr; }
    if (!(fmin >= 0.0) || !(fmax > fmin)) { set_error("need 0 <= fmin < fmax"); return nullptr; }
    return create_impl(fs, n_fft, hop, window, n_fft / 2 + 1, fmin, fmax, MELT_MEL_HTK, 0, n_mels);
}

extern "C" void melt_plan_destroy(melt_plan *p) {
    if (!p) return;
    free_device(p);
    if (p->copy_in) cudaStreamDestroy(p->copy_in);
    if (p->copy_out) cudaStreamDestroy(p->copy_out);
    if (p->pool) cudaMemPoolDestroy(p->pool);
    delete p;
}

extern "C" int melt_plan_set_option(melt_plan *p, int key, int value) {
    if (!p) return fail(MELT_ERR_INVALID_ARG, "plan is NULL");
    if (p->used.load()) return fail(MELT_ERR_INVALID_ARG, "plan is immutable after its first forward call");
    if (p->fb_mels > 0 && ((key == MELT_OPT_PRECISION && value != MELT_PREC_COMPENSATED) || (key == MELT_OPT_OUTPUT && value != MELT_OUTPUT_LOG) ||
                           (key == MELT_OPT_OUTPUT_DTYPE && value != MELT_DTYPE_F32)))
        return fail(MELT_ERR_UNSUPPORTED, "conventional (STFT + Mel filterbank) plan: compensated precision, log10 output, fp32 only");
    switch (key) {
        case MELT_OPT_LAYOUT:
            if (value < 0 || value > 1) return fail(MELT_ERR_INVALID_ARG, "bad layout %d", value);
            p->layout = value; break;
        case MELT_OPT_PRECISION:
            if (value < 0 || value > 2) return fail(MELT_ERR_INVALID_ARG, "bad precision %d", value);
            p->precision = value; break;
        case MELT_OPT_DROP_LAST:
            if (value < 0 || value > 1) return fail(MELT_ERR_INVALID_ARG, "bad drop_last %d", value);
            p->drop_last = value; break;
        case MELT_OPT_PAD:
            if (value < 0 || value > 1) return fail(MELT_ERR_INVALID_ARG, "bad pad %d", value);
            p->pad = value; break;
        case MELT_OPT_INPUT_SCALE_LOG2:
            if (value < -24 || value > 24) return fail(MELT_ERR_INVALID_ARG, "bad input scale %d", value);
            p->in_scale_log2 = value; break;
        case MELT_OPT_OUTPUT:
            if (value < 0 || value > 3) return fail(MELT_ERR_INVALID_ARG, "bad output %d", value);
            if ((value == MELT_OUTPUT_POWER || value == MELT_OUTPUT_LOG_WHISPER) && p->n_mfcc > 0) return fail(MELT_ERR_INVALID_ARG, "power / Whisper-normalised output needs n_mfcc == 0");
            p->output = value; break;
        case MELT_OPT_OUTPUT_DTYPE:
            if (value < 0 || value > 2) return fail(MELT_ERR_INVALID_ARG, "bad output dtype %d", value);
            p->out_dtype = value;
            return MELT_OK;   // checked against the other options at the forward call
        case MELT_OPT_LOG_EPS_EXP10:
            if (value < -30 || value > 0) return fail(MELT_ERR_INVALID_ARG, "bad eps exponent %d", value);
            p->eps_exp10 = value; break;
        case MELT_OPT_INPUT_READY:
            if (value < 0 || value > 1) return fail(MELT_ERR_INVALID_ARG, "bad input_ready %d", value);
            p->input_ready = value;
            return MELT_OK;   // a launch-time flag: no operand image depends on it
        default:
            return fail(MELT_ERR_INVALID_ARG, "unknown option %d", key);
    }
    return plan_build_device(p);
}

extern "C" long long melt_num_frames(const melt_plan *p, long long len) { return p ? frames_for(p, len) : 0; }
extern "C" long long melt_count_frames(long long len, int n_fft, int hop, int pad, int drop_last) {
    if (len < 0 || n_fft < 1 || hop < 1) return 0;
    long long padded = len;
    if (pad == MELT_PAD_REFLECT) {
        if (len < (long long)(n_fft / 2) + 1) return 0;
        padded += 2LL * (n_fft / 2);
    }
    if (padded < n_fft) return 0;
    const long long T = (padded - n_fft) / hop + 1 - (drop_last ? 1 : 0);
    return T < 0 ? 0 : T;
}
extern "C" int melt_plan_reserve(melt_plan *p, unsigned long long bytes) {
    if (!p) return fail(MELT_ERR_INVALID_ARG, "plan is NULL");
    if (bytes == 0) return MELT_OK;
    void *q = nullptr;   // grow the pool once: the memory stays with it (release threshold = unlimited)
    if (cudaMallocFromPoolAsync(&q, (size_t)bytes, p->pool, nullptr) != cudaSuccess) { (void)cudaGetLastError(); return fail(MELT_ERR_ALLOC, "reserve of %llu bytes", bytes); }
    MELT_CUDA(cudaFreeAsync(q, nullptr));
    MELT_CUDA(cudaStreamSynchronize(nullptr));
    return MELT_OK;
}
extern "C" int melt_num_channels(const melt_plan *p) { return p ? p->kp.n_ch : 0; }

extern "C" int melt_plan_get_centres(const melt_plan *p, double *f_hz) {
    if (!p || !f_hz) return fail(MELT_ERR_INVALID_ARG, "NULL argument");
    std::copy(p->centres.begin(), p->centres.end(), f_hz);
    return MELT_OK;
}

extern "C" const char *melt_plan_describe(const melt_plan *p) { return p ? p->desc.c_str() : ""; }

extern "C" int melt_forward(const melt_plan *p, const float *x, int batch, long long len, void *out, void *stream) {
    return forward_impl(p, x, nullptr, batch, len, out, nullptr, nullptr, stream, p && p->input_ready);
}

// Host buffers: the batch is cut into groups of clips; upload of group k + 1 (copy_in stream), kernel of group k (the caller's
// stream) and download of group k - 1 (copy_out stream) overlap.  PCIe is full duplex, so the call costs about
// max(upload, download) + one group's worth of the other two stages instead of their sum.
extern "C" int melt_forward_host(const melt_plan *p, const float *x_host, int batch, long long len, void *out_host_any, void *stream) {
    if (!p) return fail(MELT_ERR_INVALID_ARG, "plan is NULL");
    if (batch < 0 || len < 0) return fail(MELT_ERR_INVALID_ARG, "negative batch / len");
    const long long T = frames_for(p, len);
    if (batch == 0 || T == 0) return MELT_OK;
    if (!x_host || !out_host_any) return fail(MELT_ERR_INVALID_ARG, "x_host / out_host is NULL");
    int dev = -1;
    MELT_CUDA(cudaGetDevice(&dev));
    if (dev != p->device) return fail(MELT_ERR_INVALID_ARG, "plan was created on device %d, current device is %d", p->device, dev);
    // device / host output copies are handled in units of 4 bytes: a clip of 16-bit outputs must be a whole number of them
    const size_t esize = p->out_dtype == MELT_DTYPE_F32 ? 4 : 2;
    if (((size_t)T * (size_t)p->kp.n_ch * esize) & 3) return fail(MELT_ERR_UNSUPPORTED, "melt_forward_host: 16-bit output needs an even number of elements per clip");
    float *out_host = static_cast<float *>(out_host_any);
    const size_t clip_in = (size_t)len, clip_out = (size_t)T * (size_t)p->kp.n_ch * esize / 4;
    cudaStream_t st = (cudaStream_t)stream;
    float *ws_in = nullptr, *ws_out = nullptr;
    int rc = scratch_alloc(p, (void **)&ws_in, (size_t)batch * clip_in * sizeof(float), st);
    if (rc) return rc;
    rc = scratch_alloc(p, (void **)&ws_out, (size_t)batch * clip_out * sizeof(float), st);
    if (rc) { cudaFreeAsync(ws_in, st); return rc; }
    // groups of clips: about 8 MB of input each, at most 16 groups.  The first upload and the last download are not overlapped, which
    // argues for small groups; every group costs ~8 runtime calls on the host, which argues against: 32 groups of 2 MB made the
    // Whisper-shaped batch host-bound (1.61 ms against 1.31 ms with 8 groups).
    constexpr int kMaxGroups = 16;
    int per = (int)std::max<size_t>(1, ((size_t)8 << 20) / (clip_in * sizeof(float)));
    if ((batch + per - 1) / per > kMaxGroups) per = (batch + kMaxGroups - 1) / kMaxGroups;
    const int groups = (batch + per - 1) / per;
    cudaEvent_t ev_start = nullptr, ev_in[kMaxGroups] = {}, ev_k[kMaxGroups] = {}, ev_done = nullptr;
    cudaError_t e = cudaEventCreateWithFlags(&ev_start, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ev_done, cudaEventDisableTiming);
    for (int g = 0; g < groups && e == cudaSuccess; ++g) {
        e = cudaEventCreateWithFlags(&ev_in[g], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ev_k[g], cudaEventDisableTiming);
    }
    auto cleanup = [&]() {   // destroying a recorded event is legal: its resources are released when it has completed
        if (ev_start) cudaEventDestroy(ev_start);
        if (ev_done) cudaEventDestroy(ev_done);
        for (int g = 0; g < kMaxGroups; ++g) { if (ev_in[g]) cudaEventDestroy(ev_in[g]); if (ev_k[g]) cudaEventDestroy(ev_k[g]); }
    };
    if (e != cudaSuccess) { cleanup(); cudaFreeAsync(ws_in, st); cudaFreeAsync(ws_out, st); return cuda_fail(e, "cudaEventCreate"); }
    // the copy streams start behind everything already in the caller's stream (which includes the scratch allocations)
    e = cudaEventRecord(ev_start, st);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(p->copy_in, ev_start, 0);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(p->copy_out, ev_start, 0);
    rc = MELT_OK;
    for (int g = 0; g < groups && e == cudaSuccess && rc == MELT_OK; ++g) {
        const int b0 = g * per, nb = std::min(per, batch - b0);
        e = cudaMemcpyAsync(ws_in + (size_t)b0 * clip_in, x_host + (size_t)b0 * clip_in, (size_t)nb * clip_in * sizeof(float), cudaMemcpyHostToDevice, p->copy_in);
        if (e == cudaSuccess) e = cudaEventRecord(ev_in[g], p->copy_in);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(st, ev_in[g], 0);
        if (e != cudaSuccess) break;
        // the kernel's input was produced by a copy it is fully ordered behind (event), never by the kernel ahead of it
        rc = forward_impl(p, ws_in + (size_t)b0 * clip_in, nullptr, nb, len, ws_out + (size_t)b0 * clip_out, nullptr, nullptr, stream, true);
        if (rc != MELT_OK) break;
        e = cudaEventRecord(ev_k[g], st);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(p->copy_out, ev_k[g], 0);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(out_host + (size_t)b0 * clip_out, ws_out + (size_t)b0 * clip_out, (size_t)nb * clip_out * sizeof(float),
                                cudaMemcpyDeviceToHost, p->copy_out);
    }
    // the caller's stream waits for the last download; the scratch goes back to the pool behind it
    if (e == cudaSuccess) e = cudaEventRecord(ev_done, p->copy_out);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(st, ev_done, 0);
    cudaFreeAsync(ws_in, st);
    cudaFreeAsync(ws_out, st);
    cleanup();
    if (rc != MELT_OK) return rc;
    if (e != cudaSuccess) return cuda_fail(e, "melt_forward_host pipeline");
    return MELT_OK;
}
extern "C" int melt_forward_ragged(const melt_plan *p, const float *x, const long long *offsets, int n_clips, void *out,
                                   long long *out_frame_offsets, void *stream) {
    if (!offsets) return fail(MELT_ERR_INVALID_ARG, "offsets is NULL");
    return forward_impl(p, x, offsets, n_clips, 0, out, nullptr, out_frame_offsets, stream, false);
}

// ---------------------------------------------------------------------------------------------- allocation-free ragged forward
// melt_forward_ragged for callers that must not allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc): the
// one piece of per-call scratch of the ragged path, the device-side chunk / tile prefix (n_clips + 1 ints), lives in this
// file-scope device array instead of the plan's stream-ordered pool.  Every GPU that loads the library holds its 256 KB until exit.
// In host code `g_noalloc_tile_prefix` is a host-side stand-in, not a device address: the kernels get the address that
// cudaGetSymbolAddress returns, looked up once per device with that device current.  All calls share the array: calls that
// overlap on the GPU (different streams) race on it; calls in one stream are ordered (the scan kernel that rewrites the array is
// a plain launch, so it starts only after the previous forward kernel has completed).  Nothing in it has to start at zero: the
// scan kernel writes entries 0 .. n_clips of every call before the forward kernel reads them, and no entry beyond n_clips is read.
static __device__ __align__(256) int g_noalloc_tile_prefix[MELT_NOALLOC_MAX_CLIPS + 1];

static int noalloc_tile_prefix(int device, int **ptr) {
    static std::atomic<int *> addr[64];   // per device; zero-initialised
    int *a = (device >= 0 && device < 64) ? addr[device].load(std::memory_order_acquire) : nullptr;
    if (!a) {
        MELT_CUDA(cudaGetSymbolAddress((void **)&a, g_noalloc_tile_prefix));   // the current device is `device` (validate_common)
        if (!a) return fail(MELT_ERR_CUDA, "cudaGetSymbolAddress returned a null address");
        if (device >= 0 && device < 64) addr[device].store(a, std::memory_order_release);
    }
    *ptr = a;
    return MELT_OK;
}

extern "C" int melt_forward_ragged_noalloc(const melt_plan *p, const float *x, const long long *offsets, int n_clips, void *out_any,
                                           long long *out_frame_offsets, void *stream) {
    if (!offsets) return fail(MELT_ERR_INVALID_ARG, "offsets is NULL");
    int rc = validate_common(p, x, out_any);
    if (rc) return rc;
    if (p->fb_mels > 0) return fail(MELT_ERR_UNSUPPORTED, "conventional (STFT + Mel filterbank) plan: dense batches only");
    float *out = static_cast<float *>(out_any);
    const bool out16 = p->out_dtype != MELT_DTYPE_F32;
    if (out16 && (p->n_mfcc > 0 || p->output != MELT_OUTPUT_LOG))
        return fail(MELT_ERR_UNSUPPORTED, "16-bit output: log-Mel output (n_mfcc == 0, MELT_OUTPUT_LOG) only");
    if (p->output == MELT_OUTPUT_LOG_WHISPER) return fail(MELT_ERR_UNSUPPORTED, "Whisper-normalised output: dense batches only");
    if (n_clips < 0) return fail(MELT_ERR_INVALID_ARG, "negative clip count");
    if (n_clips > MELT_NOALLOC_MAX_CLIPS)
        return fail(MELT_ERR_UNSUPPORTED, "melt_forward_ragged_noalloc: n_clips=%d exceeds MELT_NOALLOC_MAX_CLIPS=%d (use melt_forward_ragged)",
                    n_clips, MELT_NOALLOC_MAX_CLIPS);
    if (!out_frame_offsets) return fail(MELT_ERR_INVALID_ARG, "out_frame_offsets is NULL");
    if (p->kp.feature_major) return fail(MELT_ERR_UNSUPPORTED, "ragged batches are frame-major only");
    p->used.store(true, std::memory_order_relaxed);
    if (n_clips == 0) return MELT_OK;
    int *tile_prefix = nullptr;
    rc = noalloc_tile_prefix(p->device, &tile_prefix);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    // from here on: the ragged branch of forward_impl with the static array in place of pool scratch
    const bool v2 = p->v2_ok && !p->k2.direct && (((uintptr_t)x & 15) == 0);
    if (v2) {
        rc = launch_ragged_scan(p, offsets, n_clips, out_frame_offsets, tile_prefix, 32, st);   // exclusive prefix of 32-frame chunks per clip
        K2Params k2 = p->k2;
        k2.x = x; k2.out = out; k2.tap = nullptr; k2.n_clips = n_clips; k2.len = 0; k2.frames_per_clip = 0;
        k2.chunks_per_clip = 0; k2.n_tiles = -1;
        k2.offsets = offsets; k2.frame_offsets = out_frame_offsets; k2.tile_prefix = tile_prefix;
        k2.vpad = p->pad == MELT_PAD_REFLECT ? p->n_fft / 2 : 0;
        k2.out_dtype = p->out_dtype;
        k2.input_ready = 0;   // the scan kernel just ahead in the stream produces what the kernel reads at its entry
        if (rc == MELT_OK && v2_encode_tmap_ragged(k2) == MELT_OK && k2.tma_rows > 0) return launch_forward2(p, k2, st);
    }
    if (rc == MELT_OK && out16) rc = fail(MELT_ERR_UNSUPPORTED, "16-bit output needs the CTA-pair kernel (hop %% 4 == 0, 16-byte aligned x, staged window)");
    if (rc == MELT_OK) rc = launch_ragged_scan(p, offsets, n_clips, out_frame_offsets, tile_prefix, TILE_M, st);
    KParams kp = p->kp;
    kp.x = x; kp.out = out; kp.tap = nullptr; kp.n_clips = n_clips;
    kp.offsets = offsets; kp.frame_offsets = out_frame_offsets; kp.tile_prefix = tile_prefix;
    kp.len = 0; kp.frames_per_clip = 0; kp.tiles_per_clip = 0; kp.n_tiles = -1;
    if (rc == MELT_OK) rc = launch_forward(p, kp, st);
    return rc;
}

extern "C" int melt_forward_tap(const melt_plan *p, const float *x, const long long *offsets, int n_clips, long long len,
                                float *out, float *logmel, long long *out_frame_offsets, void *stream) {
    return forward_impl(p, x, offsets, n_clips, len, out, logmel, out_frame_offsets, stream, p && p->input_ready);
}
