// melt_internal.h -- host-side internals shared by the translation units of libmelt_b200.so.
#pragma once
#include <cmath>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/melt.h"

namespace melt {

// ------------------------------------------------------------------------------------------ errors
void set_error(const char *fmt, ...);
int fail(int status, const char *fmt, ...);
int cuda_fail(cudaError_t e, const char *what);
#define MELT_CUDA(call)                                                 \
    do {                                                                \
        cudaError_t e__ = (call);                                       \
        if (e__ != cudaSuccess) return ::melt::cuda_fail(e__, #call);   \
    } while (0)

// ------------------------------------------------------------------------------------------ operand formats
enum OperandKind : int { OP_F16 = 0, OP_BF16 = 1, OP_TF32 = 2 };
static inline int operand_bytes(int kind) { return kind == OP_TF32 ? 4 : 2; }
static inline int operand_kstep(int kind) { return kind == OP_TF32 ? 8 : 16; }  // K elements per tcgen05.mma (32 bytes)

// Round-to-nearest-even conversions from double, done in one step (no double rounding through float).
uint16_t f64_to_f16_bits(double v);
uint16_t f64_to_bf16_bits(double v);
uint32_t f64_to_tf32_bits(double v);  // fp32 bit pattern with the low 13 mantissa bits zero
double f16_bits_to_f64(uint16_t h);
double bf16_bits_to_f64(uint16_t h);
double tf32_bits_to_f64(uint32_t u);

// Writes one K-step slab of a K-major B operand in the no-swizzle canonical layout the UMMA shared-memory
// descriptor describes: [n_rows/8][2 K-halves][8 rows][16 bytes].  vals(row, k) gives the value (already scaled).
// dst must hold n_rows * 32 bytes.  Returns bytes written.
template <class F>
static inline size_t pack_b_slab(int kind, int n_rows, F vals, uint8_t *dst) {
    const int esz = operand_bytes(kind), kstep = operand_kstep(kind), per16 = 16 / esz;
    for (int r = 0; r < n_rows; ++r)
        for (int k = 0; k < kstep; ++k) {
            size_t off = (size_t)(r / 8) * 256 + (size_t)(k / per16) * 128 + (size_t)(r % 8) * 16 + (size_t)(k % per16) * esz;
            double v = vals(r, k);
            if (kind == OP_F16) { uint16_t b = f64_to_f16_bits(v); memcpy(dst + off, &b, 2); }
            else if (kind == OP_BF16) { uint16_t b = f64_to_bf16_bits(v); memcpy(dst + off, &b, 2); }
            else { uint32_t b = f64_to_tf32_bits(v); memcpy(dst + off, &b, 4); }
        }
    return (size_t)n_rows * 32;
}

}  // namespace melt
