// melt_plan.h -- the plan object and the kernel parameter block (host + device view).
#pragma once
#include "melt_internal.h"

#include <atomic>

namespace melt {

constexpr int TILE_M = 128;         // frames per tile = UMMA M
constexpr int MAX_B_SLOTS = 32;     // shared-memory slots (K-step slabs) of the basis ring / resident basis
constexpr int MAX_A_SLOTS = 8;      // tensor-memory slots (K-steps) of the A-operand ring
constexpr int MAX_STG_SLOTS = 4;    // signal staging slots
constexpr int MAX_CLIPS = 1 << 20;  // ragged batches: clips per call
constexpr int MAX_MFCC = 64;
constexpr int SMEM_BUDGET = 232448; // 227 KB: max dynamic shared memory per CTA on sm_100

// Warp roles of melt_fwd_kernel (20 warps).
constexpr int WARP_BPROD = 0, WARP_MMA = 1, WARP_TMEM = 2, WARP_EPI0 = 4, WARP_CONV0 = 8, WARP_LOAD0 = 16;
constexpr int NUM_WARPS = 20, NUM_THREADS = NUM_WARPS * 32;
constexpr int NUM_EPI_THREADS = 128, NUM_CONV_THREADS = 256, NUM_LOAD_THREADS = 128;

struct KParams {
    // ---- analysis geometry
    int n_fft, hop, n_mels, n_mfcc, n_ch;  // n_ch = output channels per frame
    int a0, b0, kf;                        // folded pairs: (a0 + j, b0 - j), j = 0..kf-1
    int kstep, units;                      // K elements per MMA, K-steps per pass (ceil(kf / kstep))
    int nb, passes;                        // Mel bins per pass (multiple of 16), number of passes over the bins
    int nk;                                // operand kinds per term: 4 (hi/lo x sum/diff) or 2
    // ---- tensor memory map (columns)
    int acc_cols, acc_stages, unit_cols, a_slots, a_col0;
    // ---- shared memory map (bytes from the dynamic smem base)
    int b_resident, b_slots;
    uint32_t unit_b_bytes;
    int stg_comb, stg_slots, chunk_units, stg_pitch, stg_slot_words;
    unsigned long long hop_inv40;          // ceil(2^40 / hop): exact division of sample indices < 2^24
    uint32_t off_b, off_stg, off_tab, off_dct, off_bar, smem_bytes;
    int dct_pitch;                         // floats per Mel bin in the DCT table (n_mfcc rounded up to 16)
    // ---- numerics
    float in_scale, out_scale, out_log10_offset;
    int output_power;                      // melt_output: 0 log10 clamp, 1 power, 2 ln(S + eps)
    float ln_eps;                          // MELT_OUTPUT_LN_EPS: eps
    // ---- batch
    const float *x;
    float *out, *tap;
    const long long *offsets;       // ragged: device sample offsets (n_clips + 1), else NULL
    const long long *frame_offsets; // ragged: device frame offsets written by the scan kernel
    const int *tile_prefix;         // ragged: device exclusive prefix of tiles per clip (n_clips + 1)
    int n_clips;
    long long len;                  // dense: samples per clip
    long long frames_per_clip;      // dense: T
    int tiles_per_clip, n_tiles;    // dense
    int pad, drop_last, feature_major;
    // ---- plan-owned device data
    const uint8_t *b_img;  // [passes][units] slabs of unit_b_bytes
    const uint32_t *tab;   // [units * kstep] packed staging offsets (lo16: a0 + j sample, hi16: b0 - j sample)
    const float *dct;      // [n_mels][dct_pitch]
};

// ---------------------------------------------------------------------------------------------- v2 (CTA-pair kernel)
constexpr int V2_CONV_GROUPS = 3;     // converter groups of 4 warps (one warp per tensor-memory lane quarter); they take K-steps round-robin
// Warps of melt_fwd2_kernel (512 threads): loader, MMA issuer R, basis / tensor-memory owner, MMA issuer I; then MODE 2 (plain
// log-Mel): three converter groups that also drain the accumulators; MODE 0 (power / tap / MFCCT outputs): four epilogue
// warps + two converter groups.  (A third converter group next to the epilogue warps, 640 threads at <= 102 registers, made the
// ragged MFCCT batch SLOWER: 300 vs 225 us -- the schedulers are already oversubscribed.)
constexpr int v2_threads(int mode) { return mode == 5 ? 128 * (3 + V2_CONV_GROUPS) : (mode == 3 ? 128 * (2 + V2_CONV_GROUPS) : 128 * (1 + V2_CONV_GROUPS)); }
constexpr int V2_MAX_UNITS = 128;     // K-steps per tile the per-unit load table covers
constexpr int V2_MAX_STG = 12;        // staging ring slots (32-frame chunks)
constexpr int V2_TAB = 12;            // int16 entries per unit: [0,4) forward quads, [4,8) backward quads, [8] single

struct K2Params {
    // ---- analysis geometry (as KParams)
    int n_fft, hop, n_mels, n_mfcc, n_ch;
    int kstep, units, nb, nk, unit_cols;
    int a0, b0;                // fold geometry: pairs (a0 + j, b0 - j)
    int acc_cols, acc_stages, a_slots, a_col0;
    // ---- staging ring of 32-frame chunks: rows of `hop` samples at a padded pitch
    int rows_per_chunk, pitch_bytes, slot_bytes, stg_slots;
    int kslot_bytes;           // K-step staging (direct form): bytes of one slot = forward + mirrored block of 32 x (kstep + 4) samples
    int stg_phases;            // ceil(stg_slots / 4): staging barriers are indexed [lane quarter + 4 (tile mod stg_phases)]
    int vpad;                  // MELT_PAD_REFLECT on this kernel: frames start vpad = n_fft/2 samples before sample t * hop, the
                               // samples beyond the clip are mirrored by the loader's edge path (0: no padding)
    int input_ready;           // MELT_OPT_INPUT_READY: x / offsets may be read before the predecessor kernel has completed
    // ---- basis (this CTA's half: nb/2 rows per kind)
    uint32_t unit_b_bytes, kind_bytes;
    uint32_t off_b, off_stg, off_dct, off_bar, smem_bytes;
    uint32_t off_epi;          // MFCCT, frame-major: per epilogue warp 32 x n_mfcc floats to transpose the cepstra for coalesced stores (0 = none)
    int dct_pitch;
    float in_scale, out_scale, out_log10_offset;
    int output_power, feature_major;   // output_power: melt_output (0 log10 clamp, 1 power, 2 ln(S + eps))
    float ln_eps;              // MELT_OUTPUT_LN_EPS: eps
    int out_dtype;             // melt_dtype of `out` (16-bit forms: plain log-Mel only; `out` is then addressed in bytes)
    // ---- batch (dense)
    const float *x;
    float *out, *tap;
    int n_clips;
    long long len, frames_per_clip;
    int chunks_per_clip, n_tiles; // dense: 32-frame chunks per clip; tiles of 8 consecutive chunks of the batch (256 frames)
    // ---- batch (ragged: clips packed back to back; offsets != nullptr selects this form, frame-major output only)
    const long long *offsets;        // device sample offsets (n_clips + 1)
    const long long *frame_offsets;  // device frame offsets (n_clips + 1), written by the scan kernel
    const int *tile_prefix;          // device exclusive prefix of 256-frame tiles per clip (n_clips + 1)
    // ---- plan-owned device data
    const uint8_t *b_img;  // [2 ranks][passes][units] slabs of unit_b_bytes
    int passes;                // passes over the Mel bins (nb bins each); > 1 needs the streamed basis
    int direct;                // very long windows: K-step staging (the loader stages two runs of kstep + 4 samples per frame and K-step)
    int b_resident, b_slots;   // basis half resident in shared memory (b_slots = units), or streamed through a ring of b_slots K-step slabs
    const float *dct;      // [n_mels][dct_pitch]
    // ---- conventional front end (melt_plan_create_stft_mel; MODE 4 of the kernel): the nb "bins" are the DFT bins 0 .. N/2, and a
    //      second tensor-core product with the triangular Mel filterbank follows their power.  fb_mels = 0: not in use.
    int fb_mels, fb_nb, fb_units;      // Mel filters, padded to a multiple of 16 (N of the second MMA), K-steps of 16 bins (= nb / 16)
    uint32_t fb_kind_bytes, off_fb;    // bytes of one K-step slab of one operand kind in this CTA (fb_nb / 2 rows x 32 B); where the image sits
    const uint8_t *fb_img;             // [2 ranks][fb_units][hi, mid][fb_nb / 2 rows][16 bins] bf16, no-swizzle K-major slabs
    // ---- per-unit shared-memory byte offsets (relative to the first sample of the thread's frame)
    short tab[V2_MAX_UNITS][V2_TAB];
    // ---- implicit im2col by the tensor-map engine: 3-D map over the raw signal, dims (sample-in-row: pitch words,
    //      hop-row: stride = hop, clip: stride = len); one box = one 32-frame chunk.  tma_rows = hop-rows per clip whose
    //      whole pitch-wide extent lies inside the clip (chunks reaching beyond take the per-row bulk-copy path); 0 = off.
    int tma_rows;
#ifdef MELT_TRACE
    int trace_slot;            // development builds only: region of the event-trace buffer this launch records into
#endif
    alignas(64) unsigned char tmap[128];
};

}  // namespace melt

struct melt_plan {
    double fs, fmin, fmax;
    int n_fft, hop, window, n_mels, mel_scale, n_mfcc;
    int layout, precision, drop_last, pad, in_scale_log2, output, input_ready, out_dtype, eps_exp10;
    int fb_mels;                       // > 0: conventional STFT + Mel filterbank plan (n_mels = n_fft / 2 + 1 DFT bins, fb_mels filters)
    std::vector<double> fb;            // its filterbank F[m][k], fb_mels x n_mels, fp64
    uint8_t *d_fbimg;
    mutable std::atomic<bool> used;    // set by the first forward call: options are frozen from then on
    int device, sm_count;
    std::vector<double> centres, win;
    melt::KParams kp;  // geometry + plan-owned device pointers (batch fields filled per call)
    melt::K2Params k2; // the CTA-pair kernel's view of the same plan (valid when v2_ok)
    bool v2_ok;        // the geometry is covered by melt_fwd2_kernel
    int v2_sigma;      // alignment class of the mirrored sample run (0 or 1)
    uint8_t *d_bimg2;
    uint8_t *d_bimg;
    uint32_t *d_tab;
    float *d_dct;
    cudaMemPool_t pool;                // per-call device scratch (ragged tile index, realigned copies, host-buffer staging):
                                       // stream-ordered allocations, so forward calls neither synchronise nor touch the plan
    cudaStream_t copy_in, copy_out;    // melt_forward_host: upload / download streams (ordered against the caller's by events)
    std::string desc;
};

namespace melt {
int plan_build_device(melt_plan *p);  // (re)builds geometry + operand images for the current options
int launch_forward(const melt_plan *p, const KParams &kp, cudaStream_t stream);
int plan_build_v2(melt_plan *p);   // fills p->k2 / p->v2_ok (never fails the plan: v1 remains the general path)
bool v2_accepts(const melt_plan *p, const float *x, long long len);
int launch_forward2(const melt_plan *p, const K2Params &kp, cudaStream_t stream);
int launch_forward2_fb(const K2Params &kp, int grid, int sigma, cudaStream_t stream);   // MODE 4 instantiations (melt_forward2_fb.cu)
int launch_reflect_pad(const float *x, float *xp, int batch, long long len, int pad, long long plen, cudaStream_t stream);
int v2_encode_tmap(K2Params &kp);
int v2_encode_tmap_ragged(K2Params &kp);   // 2-D map over the packed buffer (any start sample, rows of `hop` samples)   // fills kp.tmap / kp.tma_rows for this call's (x, len, batch); never fails the call
int launch_ragged_scan(const melt_plan *p, const long long *offsets, int n_clips, long long *frame_offsets, int *tile_prefix, int tile_m, cudaStream_t stream);
}  // namespace melt
