/*
 * melt.h -- C ABI of the B200-native (sm_100a) MelT / MFCCT hot path (arxiv/paper_2606_01009).
 *
 * The library computes, for framed audio, the Direct Mel Projection of PAPER.md section III-A:
 *
 *   Eq. (1)-(2) PAPER.md:126-136  M analysis frequencies f_m at the HTK-Mel filterbank centres
 *   Eq. (3)     PAPER.md:140-145  R_tm = sum_n w[n] x_t[n] cos(2 pi f_m n / fs),  I_tm with sin
 *   Eq. (4)/(7) PAPER.md:147-171  S = R^2 + I^2
 *   Eq. (5)-(6) PAPER.md:155-173  window folded into fixed basis matrices; R, I as one dense GEMM
 *   Eq. (8)     PAPER.md:179-183  MelT = log(S + eps)   -- contract form: log10(max(S, 1e-10))
 *   Eq. (9)     PAPER.md:187-191  MFCCT = MelT . D^T, D the K x M orthonormal DCT-II
 *
 * Every step runs in hand-written CUDA kernels (tcgen05 tensor-core MMAs accumulating in tensor memory,
 * fused power / log / DCT epilogue).  Frames are never materialised: the overlapping frames are formed
 * on chip from the raw signal (implicit im2col).  There is no CPU fallback: on a device that is not
 * sm_100 every entry point that needs the GPU fails with MELT_ERR_UNSUPPORTED.
 *
 * Conventions
 *   - "device" pointers are CUDA device memory of the device that was current at melt_plan_create;
 *     "host" pointers are ordinary host memory.  The library never takes ownership of caller buffers.
 *   - All forward calls are asynchronous on `stream` (a cudaStream_t passed as void*; NULL = the
 *     legacy default stream).  Caller buffers must stay valid until the stream reaches the call.
 *   - No host synchronisation happens inside a forward call, and the plan is never modified by one (forward calls take a
 *     const plan; concurrent calls on one plan from several threads / streams are safe).  Dense batches whose clips start on
 *     16-byte boundaries -- the fast path -- use no memory beyond the caller's buffers.  Three paths need per-call device
 *     scratch: packed (ragged) batches (4 (n_clips + 1) bytes), dense batches that are not 16-byte aligned (one realigned copy of
 *     the batch) and melt_forward_host (device copies of x and out).  That scratch is taken from a plan-owned stream-ordered
 *     pool (cudaMallocFromPoolAsync on `stream`, returned with cudaFreeAsync on `stream` inside the same call): asynchronous,
 *     and after the first call of a given size it is served from memory the pool already holds (melt_plan_reserve pre-sizes it).
 *   - Errors are detected on the host before any launch and returned as melt_status; the message is
 *     available from melt_last_error() (thread-local).  Kernel-side faults are not reported asynchronously.
 *   - Inputs must be finite; in MELT_PREC_COMPENSATED mode |x| must stay below 8 * 2^(12 - s) where s is
 *     MELT_OPT_INPUT_SCALE_LOG2 (default 12, i.e. |x| < 8: audio normalised to [-1, 1] has 8x headroom).
 */
#ifndef MELT_H_
#define MELT_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct melt_plan melt_plan; /* opaque, library-owned */

typedef enum {
    MELT_OK = 0,
    MELT_ERR_INVALID_ARG = 1, /* bad scalar, NULL pointer where data is needed, option out of range */
    MELT_ERR_UNSUPPORTED = 2, /* valid request the sm_100a kernels do not cover, or non-sm_100 device */
    MELT_ERR_ALIGNMENT = 3,   /* x / out not 4-byte aligned */
    MELT_ERR_CUDA = 4,        /* a CUDA runtime call failed; melt_last_error() has the CUDA string */
    MELT_ERR_ALLOC = 5        /* host or device allocation failed (plan creation only) */
} melt_status;

typedef enum {
    MELT_WINDOW_HANN_PERIODIC = 0, /* 0.5 - 0.5 cos(2 pi n / N): BASELINE.json configs[0] */
    MELT_WINDOW_HANN_SYMMETRIC = 1, /* 0.5 - 0.5 cos(2 pi n / (N-1)): PAPER.md:138 */
    MELT_WINDOW_RECT = 2
} melt_window;

typedef enum {
    MELT_MEL_HTK = 0,   /* Eq. (1)-(2) */
    MELT_MEL_SLANEY = 1 /* not defined by the paper: melt_plan_create returns NULL (UNSUPPORTED) */
} melt_mel_scale;

typedef enum {
    MELT_OPT_LAYOUT = 0,           /* melt_layout; default FRAME_MAJOR */
    MELT_OPT_PRECISION = 1,        /* melt_precision; default COMPENSATED */
    MELT_OPT_DROP_LAST = 2,        /* 0/1: drop the last frame of every clip (configs[1], [2]); default 0 */
    MELT_OPT_PAD = 3,              /* melt_pad; default NONE */
    MELT_OPT_INPUT_SCALE_LOG2 = 4, /* s in [-24, 24]: samples are multiplied by 2^s before the fp16 split of the
                                      COMPENSATED mode (exact; undone in the epilogue); default 12 */
    MELT_OPT_OUTPUT = 5,           /* melt_output; default LOG */
    MELT_OPT_OUTPUT_DTYPE = 7,     /* melt_dtype of `out`; default F32.  F16 / BF16 halve the bytes the kernel stores (the Whisper-shaped
                                      batch is bound by HBM traffic); log-Mel output (n_mfcc == 0, MELT_OUTPUT_LOG, no tap) only */
    MELT_OPT_LOG_EPS_EXP10 = 8,    /* e in [-30, 0]: the epsilon of MELT_OUTPUT_LN_EPS is 10^e; default -10 */
    MELT_OPT_INPUT_READY = 6       /* 0/1, default 0.  Consecutive forwards on one stream overlap on the device (programmatic
                                      dependent launch: the next forward's blocks start on the SMs the previous kernel has
                                      already vacated).  With 0 a forward waits for the completion of whatever precedes it in
                                      `stream` before its first read of x (and of offsets) -- correct for any producer, only the
                                      kernel's set-up and its reads of the plan's own tables overlap.  1 is the caller's promise
                                      that x / offsets are NOT written by the operation that directly precedes the call in
                                      `stream` (they were complete earlier: copied by a memcpy, or produced before an earlier
                                      kernel): the kernel then reads them while its predecessor is still draining and waits
                                      only before its first store.  bench.py's device-resident timing sets 1 and says so. */
} melt_option;

typedef enum {
    MELT_LAYOUT_FRAME_MAJOR = 0,  /* out[b][t][c]  (configs[0], [3]) */
    MELT_LAYOUT_FEATURE_MAJOR = 1 /* out[b][c][t]  (configs[1], [2], [4]); dense batches only */
} melt_layout;

typedef enum {
    MELT_PREC_COMPENSATED = 0, /* fp16 hi/lo split of both operands, 3 tensor-core products per term, fp32
                                  accumulate: meets every north-star tolerance */
    MELT_PREC_TF32 = 1,        /* single kind::tf32 pass (operands rounded to nearest-away tf32) */
    MELT_PREC_BF16 = 2         /* single kind::f16 pass on bf16 operands */
} melt_precision;

typedef enum {
    MELT_PAD_NONE = 0,   /* T = floor((len - n_fft)/hop) + 1 frames per clip; tail samples ignored */
    MELT_PAD_REFLECT = 1 /* the clip is reflect-padded by n_fft/2 per side (edge sample not repeated);
                            T = floor(len/hop) + 1 for even n_fft; needs len > n_fft/2.  The padding is virtual: the few frames per
                            clip that reach beyond the clip are staged through an edge path that mirrors the indices, every other
                            frame takes the same bulk-copy path as an unpadded clip -- no padded copy of the signal is made */
} melt_pad;

typedef enum {
    MELT_OUTPUT_LOG = 0,    /* log10(max(S, 1e-10)), then the DCT when n_mfcc > 0: the contract form (BASELINE.json north_star) */
    MELT_OUTPUT_POWER = 1,  /* S itself (Eq. 4); only with n_mfcc == 0 */
    MELT_OUTPUT_LOG_WHISPER = 3, /* the contract log10 form followed by Whisper's dynamic-range normalisation (PAPER.md:424 configures MelT
                               "to Whisper's 80-bin log-Mel specification"; the normalisation itself is Whisper's): per clip,
                               L <- max(L, max_clip(L) - 8), then (L + 4) / 4.  Dense batches, n_mfcc == 0, fp32 output.  Two small
                               kernels behind the forward kernel (per-clip maximum, rescale in place): two more passes over `out` */
    MELT_OUTPUT_LN_EPS = 2  /* the paper's own form, Eq. (8): ln(S + eps), natural logarithm (PAPER.md:343 measures
                               in nats), eps = 10^MELT_OPT_LOG_EPS_EXP10 (the paper does not state it); then the DCT when n_mfcc > 0 */
} melt_output;

typedef enum {
    MELT_DTYPE_F32 = 0,
    MELT_DTYPE_F16 = 1,  /* IEEE half, round to nearest even: |error| <= 2^-11 |value| (3.9e-3 at |log10| in [8, 16)) */
    MELT_DTYPE_BF16 = 2  /* bfloat16, round to nearest even: |error| <= 2^-8 |value| */
} melt_dtype;

/*
 * melt_plan_create -- builds the analysis frequencies (Eq. 1-2), the window, the window-folded cos/sin basis
 * (Eq. 5) and, when n_mfcc > 0, the DCT matrix (Eq. 9) in double precision on the host, converts them once to
 * the tensor-core operand format and uploads them to the current CUDA device.  Synchronous.
 *   fs > 0 sampling rate (Hz); n_fft >= 2 frame length N; hop >= 1; window: melt_window;
 *   n_mels >= 1 number of analysis frequencies M; 0 <= fmin < fmax <= fs/2 (Hz); mel_scale: melt_mel_scale;
 *   0 <= n_mfcc <= min(n_mels, 64): 0 -> log-Mel output with C = n_mels channels, > 0 -> MFCCT with C = n_mfcc.
 * Returns NULL on error (melt_last_error() says why).  The plan owns its device buffers until melt_plan_destroy.
 */
melt_plan *melt_plan_create(double fs, int n_fft, int hop, int window, int n_mels,
                            double fmin, double fmax, int mel_scale, int n_mfcc);

/* Frees the plan and its device buffers.  NULL is ignored.  Do not destroy a plan with work in flight. */
void melt_plan_destroy(melt_plan *plan);

/*
 * melt_plan_set_option -- sets one melt_option.  Allowed until the first forward call on the plan; afterwards the
 * plan is immutable (so concurrent forwards on different streams are safe) and MELT_ERR_INVALID_ARG is returned.
 * Changing MELT_OPT_PRECISION rebuilds and re-uploads the operand images (synchronous).
 */
int melt_plan_set_option(melt_plan *plan, int key, int value);

/* Frames per clip for a clip of `len` samples under the plan's pad / drop_last options (0 if too short). */
long long melt_num_frames(const melt_plan *plan, long long len);

/* The same count from the framing parameters alone (no plan, no GPU): T = floor((len + 2 p - n_fft) / hop) + 1 - drop_last with
 * p = n_fft/2 for MELT_PAD_REFLECT (which also needs len > n_fft/2) and 0 otherwise; 0 when the clip is too short.  Host-only
 * integer arithmetic, for callers that size buffers or shard batches before a plan exists. */
long long melt_count_frames(long long len, int n_fft, int hop, int pad, int drop_last);

/* Pre-sizes the plan's scratch pool so that later forward calls needing up to `bytes` of per-call scratch (see "Conventions")
 * are served without growing it.  Synchronous; optional.  Returns a melt_status. */
int melt_plan_reserve(melt_plan *plan, unsigned long long bytes);

/* Output channels per frame: n_mfcc if n_mfcc > 0 else n_mels. */
int melt_num_channels(const melt_plan *plan);

/* Test hook: copies the n_mels analysis frequencies (Hz) to host memory f_hz[n_mels]. */
int melt_plan_get_centres(const melt_plan *plan, double *f_hz);

/*
 * melt_plan_create_stft_mel -- a plan for the CONVENTIONAL front end, the comparator of the paper (a
 * hand-fused version is what PAPER.md:545 calls future work): frames and window as in melt_plan_create, then
 *   X_t[k] = sum_n w[n] x_t[n] exp(-2 pi i k n / N), k = 0 .. N/2;  P_t[k] = |X_t[k]|^2;
 *   S_t[m] = sum_k F[m][k] P_t[k],  F[m][k] = max(0, min((f_k - e_m) / (e_{m+1} - e_m), (e_{m+2} - f_k) / (e_{m+2} - e_{m+1}))),
 *            f_k = k fs / N, e = the n_mels + 2 points uniform in HTK mel between fmin and fmax (peak 1, no normalisation; the
 *            filter centres are the analysis frequencies of melt_plan_create with the same arguments);
 *   out    = log10(max(S, 1e-10)).
 * One kernel: the DFT as a tensor-core product on the same folded, compensated operands as the MelT projection, the power written
 * back to tensor memory as the operand of a second tensor-core product with F, the log in the epilogue -- nothing between the
 * signal and the log-Mel rows touches HBM.  Covered: even n_fft with n_fft / 2 + 1 <= 224 bins (n_fft <= 446), hop % 4 == 0,
 * n_mels <= 128, dense batches (melt_forward, melt_forward_host), fp32 output, MELT_OPT_LAYOUT / _PAD / _DROP_LAST /
 * _INPUT_SCALE_LOG2 / _INPUT_READY; anything else returns NULL here or MELT_ERR_UNSUPPORTED at the call.  melt_num_channels = n_mels.
 * Ownership and errors as melt_plan_create.
 */
melt_plan *melt_plan_create_stft_mel(double fs, int n_fft, int hop, int window, int n_mels, double fmin, double fmax);

/*
 * melt_forward -- the whole hot path on a dense batch.
 *   x    device, fp32, [batch, len] contiguous, 4-byte aligned.  When every clip start is 16-byte aligned (x and len*4)
 *        the kernel frames x in place; otherwise one pass first copies the batch into pool scratch at an aligned clip
 *        stride (see "Conventions");
 *   out  device, batch * C * T elements of MELT_OPT_OUTPUT_DTYPE (fp32 unless set otherwise), T = melt_num_frames(plan, len),
 *        layout per MELT_OPT_LAYOUT; aligned to its element size.
 * batch == 0 or T == 0 is a successful no-op.  Returns a melt_status.
 */
int melt_forward(const melt_plan *plan, const float *x, int batch, long long len, void *out, void *stream);

/*
 * melt_forward_host -- melt_forward on HOST buffers: x_host [batch, len] in, out_host (batch * C * T floats, layout per
 * MELT_OPT_LAYOUT) out.  The batch is cut into groups of clips and pipelined: the host-to-device copy of group k + 1, the
 * kernel of group k and the device-to-host copy of group k - 1 run at the same time (two plan-owned copy streams, ordered
 * against `stream` by events), so the call costs about max(upload, download) instead of their sum.  Everything is ordered
 * after the work already in `stream`, and `stream` waits for the last download: synchronise `stream` before reading out_host
 * or reusing x_host.  The call itself returns without waiting.  Pinned (page-locked) host buffers are needed for the copies
 * to be asynchronous.  Device copies of x and out come from the plan's scratch pool (see "Conventions").
 */
int melt_forward_host(const melt_plan *plan, const float *x_host, int batch, long long len, void *out_host, void *stream);

/*
 * melt_forward_ragged -- the whole hot path on clips packed back to back (configs[3]).
 *   x                  device, fp32, packed samples;
 *   offsets            device, int64, n_clips + 1 ascending sample offsets into x (clip i = [offsets[i], offsets[i+1]));
 *   out                device, MELT_OPT_OUTPUT_DTYPE (fp32 by default), packed frame-major [sum_i T_i, C]; the caller sizes it from the clip lengths
 *                      (an upper bound is sum_i melt_num_frames(len_i));
 *   out_frame_offsets  device, int64, n_clips + 1: written by the library, frame offset of every clip in `out`
 *                      (out_frame_offsets[n_clips] = total frames).  Must not be NULL.
 * n_clips <= 2^20.  Frame-major layout only.  No host synchronisation: tiles are assigned on the device.
 */
int melt_forward_ragged(const melt_plan *plan, const float *x, const long long *offsets, int n_clips,
                        void *out, long long *out_frame_offsets, void *stream);

/*
 * melt_forward_ragged_noalloc -- melt_forward_ragged (Eq. (3)-(4), (8)-(9) on packed clips; same arguments, same
 * results) for callers that must not allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc.  The call allocates and frees nothing, on the host or the device (no cudaMalloc / cudaFree, no memory-pool call):
 * the only per-call scratch of the ragged path, the device-side chunk prefix of n_clips + 1 ints, lives in a file-scope device
 * array of the library (MELT_NOALLOC_MAX_CLIPS + 1 ints = 256 KB that every GPU which loads the library holds until exit).
 *   n_clips > MELT_NOALLOC_MAX_CLIPS is rejected with MELT_ERR_UNSUPPORTED (use melt_forward_ragged);
 *   all calls on a device share the array: calls in ONE stream are ordered; calls that overlap on the GPU (different streams,
 *   or this entry point on two plans at once) RACE on it -- serialise them or use melt_forward_ragged, whose scratch is per call;
 *   the array keeps the last call's contents; every call rewrites the entries it reads, so nothing has to be cleared;
 *   the first call on a device looks the array's address up once (cudaGetSymbolAddress; no allocation).
 * Everything else (arguments, layouts, options, errors) as melt_forward_ragged; Whisper-normalised output is dense-only.
 */
#define MELT_NOALLOC_MAX_CLIPS 65536
int melt_forward_ragged_noalloc(const melt_plan *plan, const float *x, const long long *offsets, int n_clips,
                                void *out, long long *out_frame_offsets, void *stream);

/*
 * melt_forward_tap -- as melt_forward / melt_forward_ragged (offsets == NULL selects the dense form, in which
 * n_clips is the batch and len the clip length; otherwise len is ignored), and additionally writes the log-Mel
 * matrix that feeds the DCT to `logmel` (device, fp32, same frame order and layout as `out`, n_mels channels).
 * Only meaningful for MFCCT plans (n_mfcc > 0); used for two-stage parity checks.  logmel may be NULL.
 */
int melt_forward_tap(const melt_plan *plan, const float *x, const long long *offsets, int n_clips, long long len,
                     float *out, float *logmel, long long *out_frame_offsets, void *stream);

/* Thread-local message of the last error returned on this thread ("" if none). */
const char *melt_last_error(void);

/* Library / kernel configuration as a short human-readable string for logs (static storage per plan). */
const char *melt_plan_describe(const melt_plan *plan);

#ifdef __cplusplus
}
#endif
#endif /* MELT_H_ */
