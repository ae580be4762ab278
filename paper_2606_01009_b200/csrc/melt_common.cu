// melt_common.cu -- error reporting and host-side operand conversions.
#include "melt_internal.h"

namespace melt {

static thread_local char g_err[512] = "";

void set_error(const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}
int fail(int status, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return status;
}
int cuda_fail(cudaError_t e, const char *what) {
    snprintf(g_err, sizeof(g_err), "CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
    return MELT_ERR_CUDA;
}

// Round a double to a binary float format with `mant` explicit mantissa bits, exponent range [emin, emax]
// (emin = minimum normal exponent), round-to-nearest-even, gradual underflow, overflow to infinity.
// Returns sign, biased exponent field and mantissa field.
static void round_to_format(double v, int mant, int emin, int emax, int bias, uint32_t &sign, uint32_t &efield, uint32_t &mfield) {
    sign = std::signbit(v) ? 1u : 0u;
    double a = std::fabs(v);
    if (std::isnan(a)) { efield = (uint32_t)(emax + bias + 1); mfield = 1u << (mant - 1); return; }
    if (std::isinf(a)) { efield = (uint32_t)(emax + bias + 1); mfield = 0; return; }
    if (a == 0.0) { efield = 0; mfield = 0; return; }
    int e;
    (void)std::frexp(a, &e);  // a = f * 2^e, f in [0.5, 1)  ->  a = (2f) * 2^(e-1)
    int ex = e - 1;
    if (ex < emin) ex = emin;  // subnormal: fixed quantum 2^(emin - mant)
    double q = std::ldexp(a, mant - ex);           // a in units of the quantum; exact
    double r = std::nearbyint(q);                  // default rounding mode: to nearest even
    if (r >= std::ldexp(1.0, mant + 1)) { r *= 0.5; ex += 1; }  // mantissa overflow (only from the normal range)
    if (ex > emax) { efield = (uint32_t)(emax + bias + 1); mfield = 0; return; }
    uint64_t ri = (uint64_t)r;
    if (ri < (1ull << mant)) { efield = 0; mfield = (uint32_t)ri; }  // subnormal (or zero after rounding)
    else { efield = (uint32_t)(ex + bias); mfield = (uint32_t)(ri - (1ull << mant)); }
}

uint16_t f64_to_f16_bits(double v) {
    uint32_t s, e, m;
    round_to_format(v, 10, -14, 15, 15, s, e, m);
    return (uint16_t)((s << 15) | (e << 10) | m);
}
uint16_t f64_to_bf16_bits(double v) {
    uint32_t s, e, m;
    round_to_format(v, 7, -126, 127, 127, s, e, m);
    return (uint16_t)((s << 15) | (e << 7) | m);
}
uint32_t f64_to_tf32_bits(double v) {
    uint32_t s, e, m;
    round_to_format(v, 10, -126, 127, 127, s, e, m);
    return (s << 31) | (e << 23) | (m << 13);
}
double f16_bits_to_f64(uint16_t h) {
    int s = h >> 15, e = (h >> 10) & 31, m = h & 1023;
    double v;
    if (e == 0) v = std::ldexp((double)m, -24);
    else if (e == 31) v = m ? NAN : INFINITY;
    else v = std::ldexp((double)(m + 1024), e - 25);
    return s ? -v : v;
}
double bf16_bits_to_f64(uint16_t h) {
    uint32_t u = (uint32_t)h << 16;
    float f;
    memcpy(&f, &u, 4);
    return (double)f;
}
double tf32_bits_to_f64(uint32_t u) {
    float f;
    memcpy(&f, &u, 4);
    return (double)f;
}

}  // namespace melt

extern "C" const char *melt_last_error(void) { return melt::g_err; }
