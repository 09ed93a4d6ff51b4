// nspt_ozaki.cuh -- number format of the INT8-sliced mode-wise product (nspt_ozaki.cu); the transforms (nspt_fft.cu) use
// oz_abs_hi to record the per-mode maxima the format is relative to.  See nspt_ozaki.cu for the derivation.
#pragma once
#include <cstdint>

#include "nspt_internal.cuh"

namespace nspt {

constexpr int OZ_S = 7;                              // slices per plane
constexpr int OZ_PLANES = 3;                         // re, im, re + im
constexpr int OZ_FRAC_BITS = 54;                     // v = rint(x 2^(54-e)), |v| <= 2^54

// Slice layouts in global memory (of a row-major spectrum X[mode][row][col]):
//   ROWS layout (right factor B~, read MN-major):  [mode][plane][slice][row k][pitch bytes of col j]
//   QUAD layout (left factor A~, read K-major):    [mode][plane][row i][k-chunk of 32][8 slots][32 bytes of col k]
//     slot s < 7 holds slice s (slot 7 is padding): a 128-byte shared-memory row carries four slices of one k-chunk, and
//     the k-step of a tcgen05.mma selects the slice by a 32-byte offset inside the swizzled row.  k is padded to a multiple
//     of 32 with explicit zeros.
enum OzLayout { OZ_QUAD = 0, OZ_ROWS = 1 };
inline int oz_pitch_rows(int N) { return (N + 127) / 128 * 128; }   // rows start on 128-byte boundaries: a 128-byte box row is one line
inline int oz_pitch_quad(int N) { return (N + 31) / 32 * 256; }     // 8 slots x 32 bytes per chunk of 32 columns
inline size_t oz_bytes_quad(int N, size_t modes) { return (modes * OZ_PLANES * (size_t)N * oz_pitch_quad(N) + 255) / 256 * 256; }
inline size_t oz_bytes_rows(int N, size_t modes) { return (modes * OZ_PLANES * OZ_S * (size_t)N * oz_pitch_rows(N) + 255) / 256 * 256; }

// exponent e with max < 2^e from the bit pattern of the mode's maximum (0 for an all-zero mode)
__host__ __device__ __forceinline__ int oz_exponent(unsigned long long bits) {
    const int field = (int)((bits >> 52) & 0x7ff);
    if (bits == 0ull) return 0;
    if (field == 0x7ff) return 1 << 20;   // Inf / NaN in the spectrum: the product kernel answers NaN
    return field - 1022;   // max = m 2^(field-1023) with m in [1,2)  ->  max < 2^(field-1022)
}
#ifdef __CUDACC__
__device__ __forceinline__ double oz_pow2(int k) {   // 2^k, k in [-1022, 1023]
    k = k < -1022 ? -1022 : (k > 1023 ? 1023 : k);
    return __longlong_as_double((long long)(k + 1023) << 52);
}
// v = rint(x * scale), |v| <= 2^54, without a 64-bit float-to-int conversion: v = H 2^32 + l with H = rint(x scale 2^-32)
// and l = rint(x scale - H 2^32) (|l| <= 2^31), both read off the mantissa of a sum with M = 2^52 + 2^51
__device__ __forceinline__ long long oz_fixed(double x, double scale) {
    constexpr double M = 6755399441055744.0;
    const double xs = x * scale;
    const double t1 = fma(xs, 2.3283064365386963e-10, M);           // 2^-32
    const double hf = t1 - M;
    const double l = fma(hf, -4294967296.0, xs);
    const double t2 = l + M;
    return (long long)((unsigned long long)__double_as_longlong(t2) - 0x4338000000000000ull +
                       ((unsigned long long)(unsigned int)__double2loint(t1) << 32));
}
// balanced base-256 digits of an integer |v| <= 2^55 - 2^47 as bytes: lo = digits 0..3, hi = digits 4..6
__device__ __forceinline__ void oz_digits_of(long long v, unsigned int& lo, unsigned int& hi) {
    const unsigned long long u = (unsigned long long)v + 0x0000808080808080ull;
    lo = (unsigned int)u ^ 0x80808080u;
    hi = (unsigned int)(u >> 32) ^ 0x00008080u;
}
// in[e] = bytes (b0, b1, b2, b3) of element e  ->  out[d] = byte d of elements 0..3
__device__ __forceinline__ void transpose4x4(const unsigned int (&in)[4], unsigned int* out) {
    const unsigned int t0 = __byte_perm(in[0], in[1], 0x5140), t1 = __byte_perm(in[2], in[3], 0x5140);
    const unsigned int t2 = __byte_perm(in[0], in[1], 0x7362), t3 = __byte_perm(in[2], in[3], 0x7362);
    out[0] = __byte_perm(t0, t1, 0x5410);
    out[1] = __byte_perm(t0, t1, 0x7632);
    out[2] = __byte_perm(t2, t3, 0x5410);
    out[3] = __byte_perm(t2, t3, 0x7632);
}

// max(|re|, |im|) of a complex number as the high word of the bit pattern (non-negative doubles are ordered like their
// bit patterns, and the high word holds the exponent, which is all the slicing needs)
__device__ __forceinline__ unsigned int oz_abs_hi(double2 v) {
    const unsigned int a = (unsigned int)__double2hiint(v.x) & 0x7fffffffu, b = (unsigned int)__double2hiint(v.y) & 0x7fffffffu;
    return a > b ? a : b;
}
// running form for the transform kernels: m = max(m, 2 |re|_hi, 2 |im|_hi) -- the sign bit is shifted out instead of masked and
// the three-way maximum is one instruction; oz_abs_hi_shifted values are halved again when they are flushed
__device__ __forceinline__ unsigned int oz_max_hi2(unsigned int m, double2 v) {
    const unsigned int a = (unsigned int)__double2hiint(v.x) << 1, b = (unsigned int)__double2hiint(v.y) << 1;
    return __vimax3_u32(m, a, b);
}
#endif

}  // namespace nspt
