// melt_forward2.cu -- host side of the CTA-pair forward kernel (melt_forward2_kernel.cuh): geometry and shared-memory plan,
// basis images, tensor maps and the launch dispatcher.  The kernel template is instantiated in melt_forward2_{comp,tf32,bf16}.cu.
#include "melt_forward2_kernel.cuh"

namespace melt {

int launch_forward2_comp(const K2Params &kp, int grid, int sigma, cudaStream_t stream);
int launch_forward2_tf32(const K2Params &kp, int grid, int sigma, cudaStream_t stream);
int launch_forward2_bf16(const K2Params &kp, int grid, int sigma, cudaStream_t stream);

// ---------------------------------------------------------------------------------------------- host side
static int round_up2(int v, int m) { return (v + m - 1) / m * m; }

int plan_build_v2(melt_plan *p) {
    p->v2_ok = false;
    K2Params &k = p->k2;
    const KParams &k1 = p->kp;
    memset(&k, 0, sizeof(k));
    const int N = p->n_fft, H = p->hop, M = p->n_mels;
    const bool comp = p->precision == MELT_PREC_COMPENSATED;
    const int kind = comp ? OP_F16 : (p->precision == MELT_PREC_BF16 ? OP_BF16 : OP_TF32);
    k.n_fft = N; k.hop = H; k.n_mels = M; k.n_mfcc = p->n_mfcc; k.n_ch = k1.n_ch;
    k.kstep = operand_kstep(kind);
    k.units = (k1.kf + k.kstep - 1) / k.kstep;
    k.nk = comp ? 4 : 2;
    k.unit_cols = k.nk * 8;
    k.passes = (M + 127) / 128;                                   // more than 128 bins: several passes, each tile visited once per pass
    k.nb = round_up2((M + k.passes - 1) / k.passes, 16);
    if (k.nb < 32) k.nb = 32;
    const bool fbank = p->fb_mels > 0;                            // conventional front end: all DFT bins of a frame in ONE pass (the
    if (fbank) {                                                  // filterbank product needs them together), compensated operands only
        if (!comp) return MELT_OK;
        k.passes = 1;
        k.nb = round_up2(M, 16);
        k.fb_mels = p->fb_mels;
        k.fb_nb = std::max(32, round_up2(p->fb_mels, 16));
        k.fb_units = k.nb / 16;
        k.fb_kind_bytes = (uint32_t)(k.fb_nb / 2) * 32u;
        if (k.fb_nb > k.nb) return MELT_OK;                       // the filterbank's accumulator reuses the columns of I
    }
    // ---- what the kernel covers (everything else stays on the general v1 kernel)
    k.a0 = k1.a0; k.b0 = k1.b0;
    if ((H & 3) || (k1.a0 & 3)) return MELT_OK;
    if (p->pad != MELT_PAD_NONE && (N & 7)) return MELT_OK;   // reflect padding: the padded copy keeps every clip start 16-byte aligned
    if (k.passes > 1 && p->n_mfcc > 0) return MELT_OK;             // the DCT needs all bins of a frame in one pass
    const int rs = k1.b0 - (k.kstep - 1);           // lowest sample of the mirrored run of unit 0
    const int sigma = ((rs % 4) + 4) % 4;
    if (sigma > 1) return MELT_OK;
    p->v2_sigma = sigma;
    k.acc_cols = 2 * k.nb;
    k.acc_stages = (2 * k.acc_cols + 4 * k.unit_cols <= 512) ? 2 : 1;
    k.a_col0 = k.acc_stages * k.acc_cols;
    k.a_slots = std::min(V2_MAX_A_SLOTS, (512 - k.a_col0) / k.unit_cols);
    if (k.a_slots < 2) return MELT_OK;
    const int pitch_words = ((H / 4) & 1) ? H : H + 4;   // pitch / 4 odd: 8 consecutive rows hit 8 distinct 16-byte bank groups
    // hop-rows a 32-frame chunk touches; one more when the rows carry no padding words: a ragged chunk is fetched from up to
    // three samples below its start and shifted down, which needs those samples at the end of the last row
    // (+3 samples: in a ragged batch a chunk sits up to three words further into its rows, see load_shifted in the kernel)
    k.rows_per_chunk = 32 + (N - 1 + 3) / H + (pitch_words == H ? 1 : 0);
    if (k.rows_per_chunk > 64) return MELT_OK;
    k.pitch_bytes = pitch_words * 4;
    k.slot_bytes = round_up2(k.rows_per_chunk * k.pitch_bytes, 128);   // tensor-map boxes land on 128-byte boundaries
    k.kind_bytes = (uint32_t)(k.nb / 2) * 32u;
    k.unit_b_bytes = (uint32_t)k.nk * k.kind_bytes;
    k.dct_pitch = k1.dct_pitch;
    const uint32_t b_bytes = (uint32_t)k.units * k.unit_b_bytes;
    const uint32_t dct_only = p->n_mfcc > 0 ? (uint32_t)(std::max(M, k.nb) * k.dct_pitch * 4) : 0;   // rows for the bins that pad the last block too (zero)
    // MFCCT, frame-major: 4 epilogue warps x 32 frames x n_mfcc floats behind the DCT table (cepstra transposed for coalesced stores)
    const uint32_t epi_bytes = (p->n_mfcc > 0 && p->layout == MELT_LAYOUT_FRAME_MAJOR) ? (uint32_t)(4 * 32 * p->n_mfcc * 4) : 0;
    const uint32_t fb_bytes = fbank ? (uint32_t)round_up2((int)(2u * (uint32_t)k.fb_units * k.fb_kind_bytes), 128) : 0;   // this CTA's half of the filterbank image
    const uint32_t dct_bytes = dct_only + epi_bytes + fb_bytes;
    const uint32_t bar_bytes = (uint32_t)round_up2(V_NBARS * 8 + 16 + 32 * 16, 128);   // barriers, tensor-memory address, chunk records of ragged batches (32 x 16 B)
    k.off_b = 0;
    // The basis half stays resident when that leaves room for at least five staging slots; otherwise (long windows, > 128 bins) its
    // K-step slabs are streamed from L2 through a ring of 8 slabs; when five chunk slots do not fit next to that: K-block staging.
    k.b_resident = 1; k.b_slots = k.units;
    if (k.passes > 1) { k.b_resident = 0; k.b_slots = std::min(8, k.units); }   // every pass needs other rows: streamed
    if (fbank) { k.b_resident = 0; k.b_slots = std::min(8, k.units); }          // the kernel's MODE 4 is instantiated for a streamed basis
    for (;;) {
        const uint32_t ring_bytes = (uint32_t)k.b_slots * k.unit_b_bytes;
        k.off_stg = (uint32_t)round_up2((int)ring_bytes, 128) + 128;  // 128-byte zero guard in front of the staging ring
        const long long room = (long long)SMEM_BUDGET - k.off_stg - 128 - dct_bytes - bar_bytes - 256;
        k.stg_slots = (int)std::min<long long>(room > 0 ? room / k.slot_bytes : 0, V2_MAX_STG);
        if (k.stg_slots >= 5) break;
        if (k.b_resident) { k.b_resident = 0; k.b_slots = std::min(8, k.units); continue; }
        if (fbank) {                     // a shallower basis ring until five chunks fit next to the filterbank image
            if (k.b_slots > 3) { --k.b_slots; continue; }
            return MELT_OK;
        }
        {
            // Not even a streamed basis with its full ring leaves room for five staged 32-frame chunks (long windows: a chunk is
            // 32 hops of the signal).  K-BLOCK STAGING instead: the loader brings, per lane quarter and block of four K-steps, just
            // the forward and the mirrored runs of its 32 frames -- one tensor-map box of (4 kstep + 4) x 32 samples each, rows one
            // hop apart -- into a two-slot ring per quarter.  (r01 let the converter threads read their frames from global memory:
            // every lane of a load touches another 128-byte line, and the L1 tag stage, not L2 or DRAM, bounded the kernel at
            // ~3000 cycles per K-step.  A shallower basis ring would buy the five chunk slots for 1024-sample windows -- cfg4a ran
            // that way until r02: 56 us against 46 us with K-block staging.)
            k.direct = 1; k.stg_slots = 0;
            k.kslot_bytes = 2 * 32 * (4 * k.kstep + 4) * 4;   // forward + mirrored block: 32 frames x (four K-steps + 4 samples)
            for (k.b_slots = std::min(8, k.units);; --k.b_slots) {
                k.off_stg = (uint32_t)round_up2((int)((uint32_t)k.b_slots * k.unit_b_bytes), 128) + 128;
                if ((long long)k.off_stg + 8LL * k.kslot_bytes + 128 + dct_bytes + bar_bytes + 256 <= SMEM_BUDGET) break;
                if (k.b_slots <= std::min(3, k.units)) return MELT_OK;
            }
            break;
        }
    }
    k.stg_phases = std::max(1, (k.stg_slots + 3) / 4);
    k.off_dct = (uint32_t)round_up2((int)(k.off_stg + (uint32_t)k.stg_slots * k.slot_bytes + (k.direct ? 8u * k.kslot_bytes : 0u) + 128), 128);
    k.off_epi = epi_bytes ? k.off_dct + dct_only : 0;
    k.off_fb = k.off_dct + dct_only + epi_bytes;   // (128-byte aligned: a filterbank plan has no DCT table)
    k.off_bar = (uint32_t)round_up2((int)(k.off_dct + dct_bytes), 128);
    k.smem_bytes = k.off_bar + bar_bytes;
    if (k.smem_bytes > (uint32_t)SMEM_BUDGET) return MELT_OK;
    k.in_scale = k1.in_scale; k.out_scale = k1.out_scale; k.out_log10_offset = k1.out_log10_offset;
    k.output_power = k1.output_power; k.feature_major = k1.feature_major; k.ln_eps = k1.ln_eps; k.out_dtype = 0;

    // ---- per-unit load table: byte offset of sample n of a frame = ((n div H) * pitch + n mod H) * 4 (floor division)
    auto off_of = [&](int n) -> int {
        if (k.direct) return 4 * n;   // byte offset within the frame in global memory
        int row = n >= 0 ? n / H : -((-n + H - 1) / H);
        return (row * pitch_words + (n - row * H)) * 4;
    };
    if (!k.direct && k.units > V2_MAX_UNITS) return MELT_OK;   // the staged forms look their offsets up per K-step
    // (K-step staging computes its box coordinates; what a box covers outside [0, N) of a frame row is zero-filled by the engine)
    for (int u = 0; u < (k.direct ? 0 : k.units); ++u) {
        const int nq = k.kstep / 4;
        for (int i = 0; i < nq; ++i) k.tab[u][i] = (short)off_of(k1.a0 + k.kstep * u + 4 * i);
        const int run = k1.b0 - k.kstep * u - (k.kstep - 1);   // lowest sample of the mirrored run
        for (int i = 0; i < nq; ++i) k.tab[u][4 + i] = (short)off_of(run - sigma + 4 * i);
        k.tab[u][8] = (short)off_of(run + k.kstep - 1);
        k.tab[u][9] = (short)off_of(k1.a0 + k.kstep * u + k.kstep);     // the quads after the two runs (ragged batches: shifted chunks)
        k.tab[u][10] = (short)off_of(run - sigma + k.kstep);
        for (int i = 0; i < V2_TAB; ++i)
            if (k.direct) {   // every read must stay inside the frame: [0, N) samples
                const bool quad = i < nq || (i >= 4 && i < 4 + nq), single = i == 8 && sigma == 1;
                if ((quad && (k.tab[u][i] < 0 || k.tab[u][i] + 16 > 4 * N)) || (single && (k.tab[u][i] < 0 || k.tab[u][i] + 4 > 4 * N))) return MELT_OK;
            } else if (k.tab[u][i] < -128 || k.tab[u][i] + 16 > k.slot_bytes + 128) return MELT_OK;   // stays inside ring + guards
    }

    // ---- basis image: [rank][unit][kind][nb/2 rows] slabs (same folded coefficients as v1, split by Mel row)
    const double kPi = 3.14159265358979323846264338327950288;
    const int c2 = (p->window == MELT_WINDOW_HANN_PERIODIC) ? N : N - 1;
    const double centre = 0.5 * (double)c2;
    const int s_b = comp ? 14 : 0;
    const double bscale = std::ldexp(1.0, s_b);
    auto coef = [&](int m, int j, bool sine) -> double {
        if (m >= M || j >= k1.kf) return 0.0;
        const int na = k1.a0 + j;
        const double gsc = (na == k1.b0 - j) ? 0.5 : 1.0;
        const double arg = 2.0 * kPi * p->centres[m] * ((double)na - centre) / p->fs;
        return bscale * p->win[na] * (sine ? std::sin(arg) : gsc * std::cos(arg));
    };
    auto hi_of = [&](double v) -> double {
        if (kind == OP_F16) return f16_bits_to_f64(f64_to_f16_bits(v));
        if (kind == OP_BF16) return bf16_bits_to_f64(f64_to_bf16_bits(v));
        return tf32_bits_to_f64(f64_to_tf32_bits(v));
    };
    // image: [rank][pass][unit] slabs; pass ps covers Mel rows [ps * nb, ps * nb + nb), CTA rank r the half [r * nb/2, ...) of them
    const size_t img_bytes = (size_t)2 * k.passes * b_bytes;
    std::vector<uint8_t> img(img_bytes, 0);
    const int nh = k.nb / 2;
    for (int r = 0; r < 2; ++r)
        for (int ps = 0; ps < k.passes; ++ps)
            for (int u = 0; u < k.units; ++u) {
                uint8_t *slab = img.data() + (((size_t)r * k.passes + ps) * k.units + u) * k.unit_b_bytes;
                for (int kk = 0; kk < k.nk; ++kk) {
                    const bool sine = comp ? (kk >= 2) : (kk == 1);
                    const bool lo = comp && (kk & 1);
                    pack_b_slab(kind, nh, [&](int row, int kq) {
                        const int m = ps * k.nb + r * nh + row;
                        double v = (r * nh + row < k.nb) ? coef(m, u * k.kstep + kq, sine) : 0.0;
                        return lo ? v - hi_of(v) : v;
                    }, slab + (size_t)kk * k.kind_bytes);
                }
            }
    cudaFree(p->d_bimg2);
    p->d_bimg2 = nullptr;
    MELT_CUDA(cudaMalloc(&p->d_bimg2, img_bytes));
    MELT_CUDA(cudaMemcpy(p->d_bimg2, img.data(), img_bytes, cudaMemcpyHostToDevice));
    k.b_img = p->d_bimg2;
    k.dct = p->d_dct;
    if (fbank) {
        // B operand of the second product, D2[frame][filter] = sum_k P[frame][k] F[filter][k]: per CTA rank r its half of the filter rows,
        // per K-step of 16 bins a bf16 "hi" slab and a bf16 "mid" slab (F = hi + mid to ~2^-17; the products hi.hi + mid.hi + hi.mid)
        const int fh = k.fb_nb / 2;
        const size_t fimg_bytes = (size_t)2 * k.fb_units * 2 * k.fb_kind_bytes;
        std::vector<uint8_t> fimg(fimg_bytes, 0);
        auto fval = [&](int row, int bin) -> double { return (row < p->fb_mels && bin < M) ? p->fb[(size_t)row * M + bin] : 0.0; };
        for (int r = 0; r < 2; ++r)
            for (int u = 0; u < k.fb_units; ++u)
                for (int kk = 0; kk < 2; ++kk)
                    pack_b_slab(OP_BF16, fh, [&](int row, int kq) {
                        const double v = fval(r * fh + row, u * 16 + kq);
                        return kk ? v - bf16_bits_to_f64(f64_to_bf16_bits(v)) : v;
                    }, fimg.data() + (((size_t)r * k.fb_units + u) * 2 + kk) * k.fb_kind_bytes);
        MELT_CUDA(cudaMalloc(&p->d_fbimg, fimg_bytes));
        MELT_CUDA(cudaMemcpy(p->d_fbimg, fimg.data(), fimg_bytes, cudaMemcpyHostToDevice));
        k.fb_img = p->d_fbimg;
    }
    p->v2_ok = true;
    char buf[512];
    snprintf(buf, sizeof(buf),
             "melt_b200 v2 (CTA pair, 256-frame tiles) prec=%s fold(a0=%d,b0=%d,kf=%d) kstep=%d units=%d nb=%d tmem(acc=%dx%d,"
             "a_slots=%d) basis=%s half (%d x %u B/CTA) staging=%d x %d B chunks of 32 frames (pitch %d B) smem=%u B",
             comp ? "fp16x3" : (kind == OP_BF16 ? "bf16" : "tf32"), k1.a0, k1.b0, k1.kf, k.kstep, k.units, k.nb, k.acc_stages,
             k.acc_cols, k.a_slots, k.b_resident ? "resident" : "streamed", k.b_slots, k.unit_b_bytes, k.stg_slots, k.slot_bytes, k.pitch_bytes, k.smem_bytes);
    p->desc = std::string(buf) + " | general path: " + p->desc;
    return MELT_OK;
}

// The tensor map depends on the call's buffer (x, len, batch), so it is encoded per call on the host (a few hundred
// nanoseconds of integer packing inside the driver; no allocation, no synchronisation) and travels as a kernel parameter.
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = []() -> EncodeTiledFn {
        void *f = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
            return nullptr;
        return (EncodeTiledFn)f;
    }();
    return fn;
}

int v2_encode_tmap(K2Params &k) {
    k.tma_rows = 0;
    if (k.direct) {
        // K-step staging: rows = frames (stride hop, extent n_fft: what a box covers beyond a frame's window is out of bounds and
        // zero-filled), one box = (kstep + 4) samples of 32 consecutive frames
        EncodeTiledFn encd = encode_tiled_fn();
        if (!encd || k.len < k.n_fft) return MELT_OK;
        const long long frows = (k.len - k.n_fft) / k.hop + 1;
        if (frows > 0x7fffffffLL) return MELT_OK;
        CUtensorMap tmd;
        const cuuint64_t gd[3] = {(cuuint64_t)k.n_fft, (cuuint64_t)frows, (cuuint64_t)k.n_clips};
        const cuuint64_t gs[2] = {(cuuint64_t)k.hop * 4u, (cuuint64_t)k.len * 4u};
        const cuuint32_t bx[3] = {(cuuint32_t)(4 * k.kstep + 4), 32u, 1u};
        const cuuint32_t es[3] = {1u, 1u, 1u};
        if ((gs[0] & 15) || (gs[1] & 15) || gs[1] >= (1ull << 40)) return MELT_OK;
        if (encd(&tmd, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float *>(k.x), gd, gs, bx, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                 CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return MELT_OK;
        memcpy(k.tmap, &tmd, 128);
        k.tma_rows = (int)frows;
        return MELT_OK;
    }
    EncodeTiledFn enc = encode_tiled_fn();
    const long long W = k.pitch_bytes / 4;
    // virtual reflect padding: a chunk starts at any multiple of 4 samples of the clip, i.e. at column (start % hop) of hop-row
    // (start / hop): the rows are declared hop + W samples wide for that (as in the ragged map below)
    const long long Wd = W + (k.vpad > 0 ? k.hop : 0);
    if (!enc || W > 256 || k.rows_per_chunk > 256 || k.len < Wd) return MELT_OK;
    const long long rows = (k.len - Wd) / k.hop + 1;   // rows whose whole declared extent stays inside a clip (hence inside the buffer)
    if (rows < k.rows_per_chunk || rows > 0x7fffffffLL) return MELT_OK;
    static_assert(sizeof(CUtensorMap) == 128, "CUtensorMap size");
    CUtensorMap tm;
    const cuuint64_t gdim[3] = {(cuuint64_t)Wd, (cuuint64_t)rows, (cuuint64_t)k.n_clips};
    const cuuint64_t gstr[2] = {(cuuint64_t)k.hop * 4u, (cuuint64_t)k.len * 4u};   // overlapping rows: stride (hop) < extent (pitch)
    const cuuint32_t box[3] = {(cuuint32_t)W, (cuuint32_t)k.rows_per_chunk, 1u};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    if ((gstr[1] & 15) || gstr[1] >= (1ull << 40)) return MELT_OK;
    const CUresult r = enc(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float *>(k.x), gdim, gstr, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return MELT_OK;   // the per-row bulk-copy loader covers everything
    memcpy(k.tmap, &tm, 128);
    k.tma_rows = (int)rows;
    return MELT_OK;
}

// Ragged batches: ONE 2-D map over the whole packed buffer, rows of `hop` samples that are (hop + pitch) samples wide, so a
// box of pitch x rows_per_chunk samples can start at any sample s: column s % hop of row s / hop.  The row count is not
// known on the host (the offsets live on the device): the map is declared far longer than any buffer and the kernel only
// requests boxes that lie inside [0, offsets[n_clips]).
int v2_encode_tmap_ragged(K2Params &k) {
    k.tma_rows = 0;
    EncodeTiledFn enc = encode_tiled_fn();
    const long long W = k.pitch_bytes / 4;
    if (!enc || W > 256 || k.rows_per_chunk > 256) return MELT_OK;
    CUtensorMap tm;
    const cuuint64_t rows = 1ull << 30;
    const cuuint64_t gdim[3] = {(cuuint64_t)(W + k.hop), rows, 1};
    const cuuint64_t gstr[2] = {(cuuint64_t)k.hop * 4u, (cuuint64_t)k.hop * 4u * rows};
    const cuuint32_t box[3] = {(cuuint32_t)W, (cuuint32_t)k.rows_per_chunk, 1u};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    if ((gstr[0] & 15) || gstr[1] >= (1ull << 40)) return MELT_OK;
    const CUresult r = enc(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float *>(k.x), gdim, gstr, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return MELT_OK;   // the general kernel takes the batch
    memcpy(k.tmap, &tm, 128);
    k.tma_rows = 1;
    return MELT_OK;
}

bool v2_accepts(const melt_plan *p, const float *x, long long len) {
    return p->v2_ok && (((uintptr_t)x & 15) == 0) && ((len & 3) == 0);
}

// Reflect padding for the CTA-pair kernel: xp[b][i] = x[b][rho(i - pad)], rho(j) = -j for j < 0, 2 (len - 1) - j for j >= len
// (edge sample not repeated), i in [0, len + 2 pad).  One pass over the signal into a plan-owned copy.
__global__ void reflect_pad_kernel(const float *__restrict__ x, float *__restrict__ xp, long long len, int pad, long long plen, int vec) {
    const long long b = blockIdx.y;
    const float *xb = x + b * len;
    float *pb = xp + b * plen;
    const long long stride = (long long)gridDim.x * blockDim.x, t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (vec) {   // interior as 16-byte copies (x, len and pad are all 16-byte aligned), the 2 * pad reflected samples one by one
        const float4 *src = reinterpret_cast<const float4 *>(xb);
        float4 *dst = reinterpret_cast<float4 *>(pb + pad);
        for (long long i = t0; i < len / 4; i += stride) dst[i] = __ldg(src + i);
        for (long long i = t0; i < plen - len; i += stride) {
            const long long ip = i < pad ? i : len + i;          // position in the padded clip
            long long j = ip - pad;
            if (j < 0) j = -j;
            if (j >= len) j = 2 * (len - 1) - j;
            if (j < 0) j = 0;   // filler samples of very short clips (never read by a frame)
            pb[ip] = xb[j];
        }
        return;
    }
    for (long long i = t0; i < plen; i += stride) {
        long long j = i - pad;
        if (j < 0) j = -j;
        if (j >= len) j = 2 * (len - 1) - j;
        if (j < 0) j = 0;
        pb[i] = xb[j];
    }
}

int launch_reflect_pad(const float *x, float *xp, int batch, long long len, int pad, long long plen, cudaStream_t stream) {   // plen >= len + 2 pad
    const int vec = (((uintptr_t)x & 15) == 0) && (len % 4 == 0) && (pad % 4 == 0);
    const long long work = vec ? len / 4 : plen;
    const int bx = (int)std::max<long long>(1, std::min<long long>((work + 511) / 512, 2048));
    reflect_pad_kernel<<<dim3((unsigned)bx, (unsigned)batch), 256, 0, stream>>>(x, xp, len, pad, plen, vec);
    MELT_CUDA(cudaGetLastError());
    return MELT_OK;
}

int launch_forward2(const melt_plan *pl, const K2Params &kp, cudaStream_t stream) {
    int pairs = pl->sm_count / 2;
    if (kp.n_tiles >= 0 && (long long)kp.n_tiles * kp.passes < pairs) pairs = kp.n_tiles * kp.passes;   // ragged (n_tiles < 0): counted on the device
    if (pairs < 1) return MELT_OK;
    const int grid = 2 * pairs;
    const int sg = pl->v2_sigma;
    if (kp.fb_mels > 0) return launch_forward2_fb(kp, grid, sg, stream);
    switch (pl->precision) {
        case MELT_PREC_COMPENSATED: return launch_forward2_comp(kp, grid, sg, stream);
        case MELT_PREC_TF32: return launch_forward2_tf32(kp, grid, sg, stream);
        default: return launch_forward2_bf16(kp, grid, sg, stream);
    }
}

}  // namespace melt
