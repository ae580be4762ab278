/*
 * melt_oracle.c -- fp64 CPU oracle for the MelT / MFCCT hot path (arxiv/paper_2606_01009).
 *
 * TEST INFRASTRUCTURE ONLY.  This file is the plain, slow, obviously-correct statement of what the
 * hot path computes.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call it.  It shares no code, header, table or constant with
 * the CUDA path under paper_2606_01009_b200/csrc/, and the product never falls back to it.
 *
 * The method reaches exactly (up to rounding order) a result with a plain definition, so the oracle
 * IS that definition written out in double precision, with direct sums and no blocking, folding or
 * reordering:
 *
 *   Eq. (1)  PAPER.md:126-129   mu(f)  = 2595 log10(1 + f/700)
 *   Eq. (2)  PAPER.md:133-136   f_m    = 700 (10^(mu_m/2595) - 1),  m = 0..M-1
 *            PAPER.md:131       mu_m uniformly spaced on the Mel scale between fmin and fmax, at the
 *                               centre frequencies of the HTK triangular filterbank, i.e. the M
 *                               interior points of an (M+2)-point grid (BASELINE.json configs[0]:
 *                               "endpoints excluded"; reading R1)
 *   Eq. (3)  PAPER.md:140-145   R_tm = sum_n w[n] x_t[n] cos(2 pi f_m n / fs),  I_tm likewise with sin
 *   Eq. (4)  PAPER.md:147-151   S_tm = R_tm^2 + I_tm^2
 *   Eq. (8)  PAPER.md:179-183   MelT = log(S + eps); contract form (BASELINE.json north_star,
 *                               DESIGN.md reading R2): log10(max(S, 1e-10))
 *   Eq. (9)  PAPER.md:187-191   MFCCT = MelT . D^T,  D the K x M orthonormal DCT-II
 *
 * Parity pins (tests/test_oracle_pins.py): every function below is pinned by closed forms, naive-DFT
 * special cases, invariants, SciPy's DCT and a pure-Python brute force.  Parity unpinned: nothing.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC melt_oracle.c -o libmelt_oracle.so -lm   (oracle/build.py)
 * The only parallelism is an OpenMP "parallel for" over frames; every frame is computed
 * independently by the same serial triple loop.
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>

#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_PI 3.14159265358979323846264338327950288

/* window kinds (reading R3; PAPER.md:138 says "symmetric Hann", configs[0] "periodic Hann") */
enum { ORACLE_HANN_PERIODIC = 0, ORACLE_HANN_SYMMETRIC = 1, ORACLE_RECT = 2 };
/* padding kinds (reading R5) */
enum { ORACLE_PAD_NONE = 0, ORACLE_PAD_REFLECT = 1 };

int melt_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Eq. (1). */
double melt_oracle_hz_to_mel(double f) { return 2595.0 * log10(1.0 + f / 700.0); }

/* Eq. (2). */
double melt_oracle_mel_to_hz(double mu) { return 700.0 * (pow(10.0, mu / 2595.0) - 1.0); }

/* M centres uniformly spaced on the Mel scale between fmin and fmax, endpoints excluded:
 * mu_m = mu_lo + (m+1)(mu_hi - mu_lo)/(M+1), then Eq. (2). */
int melt_oracle_centres(double fmin, double fmax, int n_mels, double *f_hz)
{
    if (n_mels < 1 || !(fmin >= 0.0) || !(fmax > fmin)) return 1;
    double mu_lo = melt_oracle_hz_to_mel(fmin);
    double mu_hi = melt_oracle_hz_to_mel(fmax);
    for (int m = 0; m < n_mels; ++m) {
        double mu_m = mu_lo + (double)(m + 1) * (mu_hi - mu_lo) / (double)(n_mels + 1);
        f_hz[m] = melt_oracle_mel_to_hz(mu_m);
    }
    return 0;
}

/* PAPER.md:138 (Hann window w[n]).  periodic: 0.5 - 0.5 cos(2 pi n / N); symmetric: denominator N-1. */
int melt_oracle_window(int kind, int n_fft, double *w)
{
    if (n_fft < 1) return 1;
    for (int n = 0; n < n_fft; ++n) {
        if (kind == ORACLE_HANN_PERIODIC)
            w[n] = 0.5 - 0.5 * cos(2.0 * ORACLE_PI * (double)n / (double)n_fft);
        else if (kind == ORACLE_HANN_SYMMETRIC)
            w[n] = (n_fft == 1) ? 1.0 : 0.5 - 0.5 * cos(2.0 * ORACLE_PI * (double)n / (double)(n_fft - 1));
        else if (kind == ORACLE_RECT)
            w[n] = 1.0;
        else
            return 1;
    }
    return 0;
}

/* Eq. (5): W^(r)_{m,n} = w[n] cos(2 pi f_m n / fs), W^(i)_{m,n} = w[n] sin(.).
 * Row-major [M, N] each.  Debug output for the pins (window-in-basis == window-on-frame). */
int melt_oracle_basis(double fs, int n_fft, int window, int n_mels, double fmin, double fmax,
                      double *Wr, double *Wi)
{
    double *f = (double *)malloc(sizeof(double) * (size_t)n_mels);
    double *w = (double *)malloc(sizeof(double) * (size_t)n_fft);
    if (!f || !w) { free(f); free(w); return 2; }
    int rc = melt_oracle_centres(fmin, fmax, n_mels, f);
    if (!rc) rc = melt_oracle_window(window, n_fft, w);
    if (!rc) {
        for (int m = 0; m < n_mels; ++m)
            for (int n = 0; n < n_fft; ++n) {
                double arg = 2.0 * ORACLE_PI * f[m] * (double)n / fs;
                Wr[(size_t)m * n_fft + n] = w[n] * cos(arg);
                Wi[(size_t)m * n_fft + n] = w[n] * sin(arg);
            }
    }
    free(f); free(w);
    return rc;
}

/* Eq. (9): orthonormal DCT-II, D in R^{K x M}:
 * D[0,m] = sqrt(1/M),  D[k,m] = sqrt(2/M) cos(pi k (2m+1) / (2M)),  k = 1..K-1. */
int melt_oracle_dct(int n_mfcc, int n_mels, double *D)
{
    if (n_mfcc < 1 || n_mfcc > n_mels) return 1;
    for (int k = 0; k < n_mfcc; ++k)
        for (int m = 0; m < n_mels; ++m)
            D[(size_t)k * n_mels + m] = (k == 0)
                ? sqrt(1.0 / (double)n_mels)
                : sqrt(2.0 / (double)n_mels) * cos(ORACLE_PI * (double)k * (double)(2 * m + 1) / (double)(2 * n_mels));
    return 0;
}

/* Frame count.  No padding: T = floor((L - N)/H) + 1 (0 if L < N).  Reflect padding by p = N/2 per
 * side: the padded length is L + 2p.  drop_last removes the final frame (BASELINE.json configs[1]:
 * "3000 frames per clip (last frame dropped)"). */
long long melt_oracle_num_frames(long long len, int n_fft, int hop, int pad, int drop_last)
{
    long long padded = len + (pad == ORACLE_PAD_REFLECT ? 2LL * (n_fft / 2) : 0LL);
    if (pad == ORACLE_PAD_REFLECT && len < (long long)(n_fft / 2) + 1) return 0; /* reflection undefined */
    if (padded < n_fft) return 0;
    long long T = (padded - n_fft) / hop + 1;
    if (drop_last) T -= 1;
    return T < 0 ? 0 : T;
}

/* Sample i of the (virtually) padded clip.  Reflect: padded[i] = x[rho(i - p)], rho(j) = -j for j < 0,
 * 2(L-1) - j for j >= L (edge sample not repeated; reading R5). */
static double padded_sample(const float *x, long long len, int pad, int n_fft, long long i)
{
    if (pad == ORACLE_PAD_REFLECT) {
        long long j = i - (long long)(n_fft / 2);
        if (j < 0) j = -j;
        if (j >= len) j = 2 * (len - 1) - j;
        return (double)x[j];
    }
    return (double)x[i];
}

/*
 * One clip, the whole path.  x: len fp32 samples (widened exactly to double).  Outputs are row-major
 * frame-major: R, I, P, L are [T, M]; C is [T, K].  Any output pointer may be NULL.
 * Eq. (3) is evaluated as written: for every frame t and bin m, a direct sum over n of
 * (w[n] * x_t[n]) * cos(2 pi f_m n / fs)  -- window applied to the frame, cos/sin from
 * a table computed once with libm in double.
 */
int melt_oracle_forward(const float *x, long long len,
                        double fs, int n_fft, int hop, int window,
                        int n_mels, double fmin, double fmax, int n_mfcc,
                        int pad, int drop_last,
                        double *R, double *I, double *P, double *L, double *C)
{
    if (!(fs > 0.0) || n_fft < 1 || hop < 1 || n_mels < 1 || n_mfcc < 0 || n_mfcc > n_mels) return 1;
    if (!(fmin >= 0.0) || !(fmax > fmin) || fmax > fs / 2.0 * (1.0 + 1e-12)) return 1;
    long long T = melt_oracle_num_frames(len, n_fft, hop, pad, drop_last);
    if (T == 0) return 0;

    double *f = (double *)malloc(sizeof(double) * (size_t)n_mels);
    double *w = (double *)malloc(sizeof(double) * (size_t)n_fft);
    double *ct = (double *)malloc(sizeof(double) * (size_t)n_mels * (size_t)n_fft);
    double *st = (double *)malloc(sizeof(double) * (size_t)n_mels * (size_t)n_fft);
    double *D = n_mfcc ? (double *)malloc(sizeof(double) * (size_t)n_mfcc * (size_t)n_mels) : NULL;
    if (!f || !w || !ct || !st || (n_mfcc && !D)) { free(f); free(w); free(ct); free(st); free(D); return 2; }
    int rc = melt_oracle_centres(fmin, fmax, n_mels, f);
    if (!rc) rc = melt_oracle_window(window, n_fft, w);
    if (!rc && n_mfcc) rc = melt_oracle_dct(n_mfcc, n_mels, D);
    if (rc) { free(f); free(w); free(ct); free(st); free(D); return rc; }

    for (int m = 0; m < n_mels; ++m)
        for (int n = 0; n < n_fft; ++n) {
            double arg = 2.0 * ORACLE_PI * f[m] * (double)n / fs;      /* Eq. (3) argument */
            ct[(size_t)m * n_fft + n] = cos(arg);
            st[(size_t)m * n_fft + n] = sin(arg);
        }

#pragma omp parallel
    {
        double *xw = (double *)malloc(sizeof(double) * (size_t)n_fft);     /* windowed frame x~_t */
        double *Lrow = (double *)malloc(sizeof(double) * (size_t)n_mels);
#pragma omp for schedule(static)
        for (long long t = 0; t < T; ++t) {
            for (int n = 0; n < n_fft; ++n)                                /* x~_t[n] = w[n] x_t[n] */
                xw[n] = w[n] * padded_sample(x, len, pad, n_fft, t * (long long)hop + n);
            for (int m = 0; m < n_mels; ++m) {
                const double *cr = ct + (size_t)m * n_fft;
                const double *sr = st + (size_t)m * n_fft;
                double r = 0.0, i = 0.0;
                for (int n = 0; n < n_fft; ++n) {                          /* Eq. (3) */
                    r += xw[n] * cr[n];
                    i += xw[n] * sr[n];
                }
                double s = r * r + i * i;                                  /* Eq. (4) */
                double l = log10(s > 1e-10 ? s : 1e-10);                   /* Eq. (8), contract form */
                size_t o = (size_t)t * n_mels + m;
                if (R) R[o] = r;
                if (I) I[o] = i;
                if (P) P[o] = s;
                if (L) L[o] = l;
                Lrow[m] = l;
            }
            if (n_mfcc && C)
                for (int k = 0; k < n_mfcc; ++k) {                         /* Eq. (9) */
                    double c = 0.0;
                    for (int m = 0; m < n_mels; ++m) c += D[(size_t)k * n_mels + m] * Lrow[m];
                    C[(size_t)t * n_mfcc + k] = c;
                }
        }
        free(xw); free(Lrow);
    }
    free(f); free(w); free(ct); free(st); free(D);
    return 0;
}

/* Eq. (9) alone on a caller-supplied log-Mel matrix Lin [T, M] -> C [T, K]; used by the two-stage
 * MFCCT parity check (reading R9): cepstra vs the oracle DCT of the GPU's own log-Mel. */
int melt_oracle_dct_apply(const double *Lin, long long T, int n_mels, int n_mfcc, double *C)
{
    double *D = (double *)malloc(sizeof(double) * (size_t)n_mfcc * (size_t)n_mels);
    if (!D) return 2;
    int rc = melt_oracle_dct(n_mfcc, n_mels, D);
    if (!rc)
        for (long long t = 0; t < T; ++t)
            for (int k = 0; k < n_mfcc; ++k) {
                double c = 0.0;
                for (int m = 0; m < n_mels; ++m) c += D[(size_t)k * n_mels + m] * Lin[(size_t)t * n_mels + m];
                C[(size_t)t * n_mfcc + k] = c;
            }
    free(D);
    return rc;
}
