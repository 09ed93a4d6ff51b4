// nspt_ozaki.cu -- Step 3 of FFT-CONV (eq. 2.8) on the tcgen05 INT8 tensor cores: the mode-wise complex FP64
// product C~(p) = A~(p) B~(p) emulated with exact integer arithmetic (Ozaki-style slicing).  The paper
// finds ZGEMM dominant; on sm_100a the FP64 path is the DMMA pipe (37 TFLOP/s), the only way past it is the
// 4.5 POP/s INT8 path of the 5th-generation tensor cores.
//
// Number format.  Every real plane X of a spectrum (re, im, re+im -- the three operands of the 3-multiplication complex
// product) is written as fixed point relative to a power of two 2^e >= max|X| of its mode,
//     X = 2^e * sum_{s=0}^{6} q_s 2^(-6-8s) + r,        |r| <= 2^(e-55),
// with balanced base-256 digits q_s in [-128,127] (q_0 in [-64,64]): seven int8 "slices".  The product of two planes is
//     X Y = 2^(eX+eY-12) * sum_d 2^(-8d) * [ sum_{s+t=d} Q_s R_t ],
// each [..] an INT8 x INT8 -> INT32 matrix product that the tensor core evaluates EXACTLY (|q q'| <= 2^14, K <= 2^11 terms,
// <= 7 pairs per d: < 2^28).  Pairs with s + t > 6 are dropped (their total is below 2^-51 of the leading term), 28 pairs
// remain.  Only two roundings are not exact: the digit extraction (relative 2^-55 of the mode's largest element) and the
// final FP64 recombination.
//
// Kernel.  CTA tile 64 rows x 128 columns of one mode, computed transposed (see OZ_BM below); K-chunks of 32 arrive by TMA
// (SWIZZLE_128B) in a four-stage ring, all seven slices of both operands at once (44 KB per stage).  One thread issues
// tcgen05.mma.kind::i8 (M=128, N=64, K=32): 28 per stage, into seven TMEM accumulators (d = 0..6, 64 columns each, 448 of
// the 512 columns); runs of MMAs with the same M-side slice fetch it once (collector reuse).  The three planes run one
// after the other through the same accumulators; eight epilogue warps drain them with tcgen05.ld, recombine the seven
// INT32 sums in FP64 (Horner in 2^-8) and keep the running real / imaginary parts of the 3M product in registers.
#include <cuda.h>

#include "nspt_internal.cuh"
#include "nspt_tma.cuh"

namespace nspt {
namespace {

constexpr int OZ_S = 7;                              // slices per plane
constexpr int OZ_PLANES = 3;                         // re, im, re + im
// Operand staging, measured on B200 with probes of the TMA unit and of tcgen05.mma.kind::i8: the TMA unit is row-rate bound
// (1.9 cycles per row of <= 128 bytes with all SMs loading), so every shared-memory row is 128 bytes; a 128 x 64 x 32 MMA
// takes 46-58 cycles depending on the operand layouts (32 would be the tensor rate, reached only from N = 128 up, which the
// seven accumulators leave no room for in TMEM).  The tensor core computes the TRANSPOSED tile D[j][i] = sum_k B~[k][j] A~[i][k]:
// its M side (128 TMEM lanes) runs over output columns j and reads B~ slices MN-major -- the row-major layout the transforms
// write -- and its N side (64 TMEM columns) runs over output rows i and reads A~ slices K-major from 128-byte rows that carry
// four slices of one 32-column k-chunk (QUAD layout below; the slice is selected by a 32-byte offset inside the swizzled
// row).  The epilogue then writes 512 contiguous bytes of a row of C~ per warp.  (The untransposed arrangement, 64-byte rows
// for B~ and per-thread row segments in the epilogue, measured 9 % slower.)
constexpr int OZ_BM = 128, OZ_BN = 64, OZ_KC = 32;   // CTA tile (j x i) and K per stage = K of one tcgen05.mma.kind::i8
constexpr int OZ_STAGES = 4;
constexpr int OZ_M_SLICE = OZ_KC * OZ_BM;            // B~ slice of a stage: [32 k][128 bytes of j] = 4096
constexpr int OZ_M_STAGE = OZ_S * OZ_M_SLICE;        // 28672
constexpr int OZ_N_HALF = OZ_BN * 128;               // A~ slices 4h..4h+3 of a stage: [64 i][4 slices x 32 bytes of k] = 8192
constexpr int OZ_N_STAGE = 2 * OZ_N_HALF;            // 16384
constexpr int OZ_STAGE = OZ_M_STAGE + OZ_N_STAGE;    // 45056
constexpr int OZ_SMEM = OZ_STAGES * OZ_STAGE + 1024 + 128;
constexpr int OZ_THREADS = 384;                      // warp 0 TMA, warp 1 MMA, warp 2 TMEM allocator, warps 4-11 epilogue
constexpr int OZ_TMEM_COLS = 512;
constexpr int OZ_FRAC_BITS = 54;                     // v = rint(x 2^(54-e)), |v| <= 2^54

static_assert(OZ_STAGE % 1024 == 0 && OZ_M_STAGE % 1024 == 0, "stage alignment");

// ---- slicing ------------------------------------------------------------------------------------------------
// max over a mode of max(|re|, |im|) as the bit pattern of a non-negative double (ordered like an unsigned integer)
__global__ void __launch_bounds__(256) oz_absmax_kernel(const double2* __restrict__ X, unsigned long long* __restrict__ maxbits,
                                                      size_t NN, int modes) {
    __shared__ double red[8];
    for (int mode = blockIdx.y; mode < modes; mode += gridDim.y) {   // the grid's y extent is capped at 65535
    const double2* x = X + (size_t)mode * NN;
    double m = 0.0;
    for (size_t e = (size_t)blockIdx.x * 256 + threadIdx.x; e < NN; e += (size_t)gridDim.x * 256) {
        const double2 v = x[e];
        m = fmax(m, fmax(fabs(v.x), fabs(v.y)));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int w = 1; w < 8; ++w) m = fmax(m, red[w]);
        atomicMax(maxbits + mode, (unsigned long long)__double_as_longlong(m));
    }
    }
}

// exponent e with max < 2^e from the bit pattern of the mode's maximum (0 for an all-zero mode)
__device__ __forceinline__ int oz_exponent(unsigned long long bits) {
    const int field = (int)((bits >> 52) & 0x7ff);
    if (bits == 0ull) return 0;
    if (field == 0x7ff) return 1 << 20;   // Inf / NaN in the spectrum: the product kernel answers NaN
    return field - 1022;   // max = m 2^(field-1023) with m in [1,2)  ->  max < 2^(field-1022)
}
__device__ __forceinline__ double oz_pow2(int k) {   // 2^k, k in [-1022, 1023]
    k = k < -1022 ? -1022 : (k > 1023 ? 1023 : k);
    return __longlong_as_double((long long)(k + 1023) << 52);
}
// the seven digits of v = rint(x * scale), |v| <= 2^54, packed in bytes 0..6 of the result: byte j holds the balanced digit
// of weight 256^j (two's-complement int8), byte 6 the leading digit in [-64, 64]
__device__ __forceinline__ unsigned long long oz_digits(double x, double scale) {
    const long long v = __double2ll_rn(x * scale);
    const unsigned long long u = (unsigned long long)v + 0x0000808080808080ull;   // + 128 at digits 0..5
    return u ^ 0x0000808080808080ull;                                              // digit - 128 as int8
}

// Slice layouts in global memory (both from row-major FP64 spectra X[mode][row][col]):
//   ROWS layout (right factor B~, read MN-major):  [mode][plane][slice][row k][pitch bytes of col j]
//   QUAD layout (left factor A~, read K-major):    [mode][plane][row i][k-chunk of 32][8 slots][32 bytes of col k]
//     slot s < 7 holds slice s (slot 7 is padding): a 128-byte shared-memory row carries four slices of one k-chunk, and
//     the k-step of a tcgen05.mma selects the slice by a 32-byte offset inside the swizzled row.  k is padded to a multiple
//     of 32 with explicit zeros.
// thread = 4 consecutive columns of a row
template <bool QUAD>
__global__ void __launch_bounds__(256) oz_slice_kernel(const double2* __restrict__ X, int8_t* __restrict__ out,
                                                      const unsigned long long* __restrict__ maxbits, int* __restrict__ exps,
                                                      int N, int pitch, int modes) {
    for (int mode = blockIdx.y; mode < modes; mode += gridDim.y) {   // the grid's y extent is capped at 65535
    const int qpr = QUAD ? (pitch >> 5) : ((N + 3) >> 2);   // 4-column groups per row (QUAD: 256 bytes of pitch per 32 columns, k padded)
    const int t = blockIdx.x * 256 + threadIdx.x;
    const int e = oz_exponent(maxbits[mode]);
    if (t == 0) exps[mode] = e;
    if (t >= N * qpr) continue;
    const int row = t / qpr, j0 = (t % qpr) * 4;
    const double sc = oz_pow2(OZ_FRAC_BITS - e), sc_sum = oz_pow2(OZ_FRAC_BITS - e - 1);
    const double2* x = X + ((size_t)mode * N + row) * N + j0;
    unsigned long long w[OZ_PLANES][4];
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        double2 v = make_double2(0.0, 0.0);
        if (j0 + c < N) v = x[c];
        w[0][c] = oz_digits(v.x, sc);
        w[1][c] = oz_digits(v.y, sc);
        w[2][c] = oz_digits(v.x + v.y, sc_sum);
    }
    const size_t plane_stride = QUAD ? (size_t)N * pitch : (size_t)OZ_S * N * pitch;
    int8_t* base = out + (size_t)mode * OZ_PLANES * plane_stride + (size_t)row * pitch +
                   (QUAD ? (size_t)(j0 >> 5) * 256 + (j0 & 31) : (size_t)j0);
#pragma unroll
    for (int q = 0; q < OZ_PLANES; ++q) {
#pragma unroll
        for (int s = 0; s < OZ_S; ++s) {
            const int byte = OZ_S - 1 - s;   // slice s has weight 2^(-6-8s): digit 6 - s
            unsigned int word = 0;
#pragma unroll
            for (int c = 0; c < 4; ++c) word |= (unsigned int)((w[q][c] >> (8 * byte)) & 0xffull) << (8 * c);
            // ROWS: pitch is a multiple of 64 and j0 of 4; pad columns N..pitch-1 receive zeros (never read: TMA clips at N)
            *reinterpret_cast<unsigned int*>(base + (size_t)q * plane_stride + (QUAD ? (size_t)s * 32 : (size_t)s * N * pitch)) = word;
        }
    }
    }
}

// ---- tcgen05 wrappers ---------------------------------------------------------------------------------------
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_alloc(uint32_t smem_dst, uint32_t cols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tc_dealloc(uint32_t taddr, uint32_t cols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}
// COLLECT: use of the A-operand (M side) collector buffer -- consecutive MMAs with the same M-side slice read it from shared
// memory once: 0 = no reuse, 1 = fill (first of a run), 2 = use (middle), 3 = last use.  Without it a 128 x 64 x 32 MMA
// reads 6 KB of shared memory in 32 cycles, more than the 128 bytes per cycle an SM delivers.
template <int COLLECT>
__device__ __forceinline__ void tc_mma_i8(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
#define NSPT_OZ_MMA(Q)                                                                             \
    asm volatile(                                                                                  \
        "{\n"                                                                                      \
        ".reg .pred p;\n"                                                                          \
        "setp.ne.b32 p, %4, 0;\n"                                                                  \
        "tcgen05.mma.cta_group::1.kind::i8" Q " [%0], %1, %2, %3, p;\n"                            \
        "}\n" ::"r"(d_tmem),                                                                       \
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)                                      \
        : "memory")
    if constexpr (COLLECT == 1)
        NSPT_OZ_MMA(".collector::a::fill");
    else if constexpr (COLLECT == 2)
        NSPT_OZ_MMA(".collector::a::use");
    else if constexpr (COLLECT == 3)
        NSPT_OZ_MMA(".collector::a::lastuse");
    else
        NSPT_OZ_MMA("");
#undef NSPT_OZ_MMA
}
// arrive on an mbarrier once every tcgen05.mma issued so far by this thread has completed
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tc_ld8(uint32_t taddr, int (&r)[8]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr)
                 : "memory");
}
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tma_load_5d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2, int c3,
                                            int c4) {
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];" ::"r"(
            dst),
        "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
        : "memory");
}

// shared-memory matrix descriptor (SWIZZLE_128B): start address, leading / stride byte offsets in 16-byte units
__device__ __forceinline__ uint64_t oz_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    const uint32_t lo = ((addr >> 4) & 0x3fffu) | (((lbo_bytes >> 4) & 0x3fffu) << 16);
    const uint32_t hi = ((sbo_bytes >> 4) & 0x3fffu) | (1u << 14) /* version 1 (sm_100) */ | (2u << 29) /* SWIZZLE_128B */;
    return ((uint64_t)hi << 32) | lo;
}
// instruction descriptor: D = S32, A = B = signed int8, A (M side) MN-major, B (N side) K-major, N = 64, M = 128
constexpr uint32_t OZ_IDESC = (2u << 4) | (1u << 7) | (1u << 10) | (1u << 15) | (0u << 16) | ((OZ_BN >> 3) << 17) | ((OZ_BM >> 4) << 24);

// exact int32 -> double (no I2F): 2^52 + 2^31 + x has x + 2^31 in its low mantissa word
__device__ __forceinline__ double oz_i2d(int x) {
    return __hiloint2double(0x43300000, (int)((unsigned)x ^ 0x80000000u)) - 4503601774854144.0;
}

// All pairs (t, s), s + t <= 6, of one stage: B~ slice t (M side) times A~ slice s (N side) into accumulator d = s + t.
// Runs of equal t are consecutive (collector reuse of the M-side operand).
//   M side, slice t: [32 rows of k][128 bytes of j], MN-major: 8-row k groups 1024 bytes apart
//   N side, slice s: rows of [64 i][128 bytes] in half s / 4, K-major: 8-row groups 1024 bytes apart, slice = +32 (s % 4) bytes
template <int T0, int S0>
__device__ __forceinline__ void oz_issue_pairs(uint32_t tmem, uint32_t sm, uint32_t sn, bool not_first_k) {
    constexpr int LAST = OZ_S - 1 - T0;
    constexpr int COLLECT = (LAST == 0) ? 0 : (S0 == 0 ? 1 : (S0 == LAST ? 3 : 2));
    const uint64_t dm = oz_desc(sm + T0 * OZ_M_SLICE, 4096, 1024);
    const uint64_t dn = oz_desc(sn + (S0 >> 2) * OZ_N_HALF + (S0 & 3) * 32, 16, 1024);
    tc_mma_i8<COLLECT>(tmem + (uint32_t)((S0 + T0) * OZ_BN), dm, dn, OZ_IDESC, (not_first_k || T0 != 0) ? 1u : 0u);
    if constexpr (S0 < LAST)
        oz_issue_pairs<T0, S0 + 1>(tmem, sm, sn, not_first_k);
    else if constexpr (T0 + 1 < OZ_S)
        oz_issue_pairs<T0 + 1, 0>(tmem, sm, sn, not_first_k);
}

struct OzParams {
    double2* C;
    const int* expA;
    const int* expB;
    size_t NN;
    int N;
    int tiles_i, tiles_j;
    int nkc;
};

__global__ void __launch_bounds__(OZ_THREADS, 1)
zgemm_modes_ozaki_kernel(const __grid_constant__ CUtensorMap mapM, const __grid_constant__ CUtensorMap mapN, const OzParams P) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar_full = base + OZ_STAGES * OZ_STAGE;          // OZ_STAGES barriers
    const uint32_t bar_empty = bar_full + 8 * OZ_STAGES;
    const uint32_t bar_acc_full = bar_empty + 8 * OZ_STAGES;
    const uint32_t bar_acc_empty = bar_acc_full + 8;
    const uint32_t tmem_slot = bar_acc_empty + 8;
    volatile uint32_t* tmem_slot_gen =
        reinterpret_cast<volatile uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tiles = P.tiles_i * P.tiles_j;
    const int mode = blockIdx.x / tiles, tile = blockIdx.x % tiles;
    const int i0 = (tile / P.tiles_j) * OZ_BN, j0 = (tile % P.tiles_j) * OZ_BM;
    const int nkc = P.nkc;

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < OZ_STAGES; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, 1);
        }
        mbar_init(bar_acc_full, 1);
        mbar_init(bar_acc_empty, 8);
        mbar_fence_init();
    }
    if (warp == 2) tc_alloc(tmem_slot, OZ_TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot_gen;
    pdl_wait();
    pdl_trigger();

    // the epilogue keeps a 128 x 64 complex FP64 tile in registers (128 per thread): take them from the warps that only issue
    if (warp < 4) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
        if (warp == 0) {
            // ------------------------------------------------------------ TMA producer
            if (lane == 0) {
                int it = 0;
                for (int plane = 0; plane < OZ_PLANES; ++plane) {
                    const int pidx = mode * OZ_PLANES + plane;
                    for (int kc = 0; kc < nkc; ++kc, ++it) {
                        const int slot = it % OZ_STAGES;
                        mbar_wait(bar_empty + 8 * slot, ((it / OZ_STAGES) & 1) ^ 1);
                        mbar_expect_tx(bar_full + 8 * slot, OZ_STAGE);
                        const uint32_t st = base + slot * OZ_STAGE;
                        tma_load_4d(st, &mapM, bar_full + 8 * slot, j0, kc * OZ_KC, 0, pidx);
                        tma_load_5d(st + OZ_M_STAGE, &mapN, bar_full + 8 * slot, 0, i0, 0, kc, pidx);
                    }
                }
            }
        } else if (warp == 1) {
            // ------------------------------------------------------------ MMA issuer (one thread)
            if (lane == 0) {
                int it = 0;
                for (int plane = 0; plane < OZ_PLANES; ++plane) {
                    if (plane > 0) mbar_wait(bar_acc_empty, (plane - 1) & 1);
                    tc_fence_after();
                    for (int kc = 0; kc < nkc; ++kc, ++it) {
                        const int slot = it % OZ_STAGES;
                        mbar_wait(bar_full + 8 * slot, (it / OZ_STAGES) & 1);
                        tc_fence_after();
                        const uint32_t sm = base + slot * OZ_STAGE;
                        oz_issue_pairs<0, 0>(tmem, sm, sm + OZ_M_STAGE, kc != 0);
                        tc_commit(bar_empty + 8 * slot);   // the stage may be refilled once these MMAs have read it
                    }
                    tc_commit(bar_acc_full);
                }
            }
        }
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");
        // ------------------------------------------------------------ epilogue: 8 warps, warp w reads TMEM lanes 32 (w % 4) ..
        // lane of the accumulator = output column j, column of the accumulator = output row i
        const int we = warp - 4, quarter = we & 3, half = we >> 2;
        const int col = j0 + 32 * quarter + lane;
        const int row0 = i0 + 32 * half;
        double re[32], im[32];
#pragma unroll
        for (int j = 0; j < 32; ++j) re[j] = im[j] = 0.0;
        for (int plane = 0; plane < OZ_PLANES; ++plane) {
            // 3M: Cr = P1 - P2, Ci = 4 P3 - P1 - P2 (the sum planes carry one more exponent bit each)
            const double cr = plane == 0 ? 1.0 : (plane == 1 ? -1.0 : 0.0);
            const double ci = plane == 2 ? 4.0 : -1.0;
            mbar_wait(bar_acc_full, plane & 1);
            tc_fence_after();
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) {
                int a[OZ_S][8];
#pragma unroll
                for (int d = 0; d < OZ_S; ++d)
                    tc_ld8(tmem + ((uint32_t)(32 * quarter) << 16) + (uint32_t)(d * OZ_BN + 32 * half + 8 * cc), a[d]);
                tc_wait_ld();
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    double h = oz_i2d(a[OZ_S - 1][j]);
#pragma unroll
                    for (int d = OZ_S - 2; d >= 0; --d) h = fma(h, 0.00390625, oz_i2d(a[d][j]));
                    re[8 * cc + j] = fma(cr, h, re[8 * cc + j]);
                    im[8 * cc + j] = fma(ci, h, im[8 * cc + j]);
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_acc_empty);
        }
        const int esum = P.expA[mode] + P.expB[mode];
        const double sc = esum >= (1 << 20) ? __longlong_as_double(0x7ff8000000000000ll) : oz_pow2(esum - 12);
        if (col < P.N) {
            double2* c = P.C + (size_t)mode * P.NN + col;
#pragma unroll
            for (int j = 0; j < 32; ++j)   // the 32 lanes of a warp write 512 contiguous bytes of row row0 + j
                if (row0 + j < P.N) c[(size_t)(row0 + j) * P.N] = make_double2(sc * re[j], sc * im[j]);
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 2) tc_dealloc(tmem, OZ_TMEM_COLS);
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

cudaError_t encode_u8(CUtensorMap* map, const int8_t* basep, int rank, const cuuint64_t* dims, const cuuint64_t* strides,
                      const cuuint32_t* box, CUtensorMapSwizzle swizzle) {
    static EncodeTiledFn enc = nullptr;
    if (!enc) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
        if (e != cudaSuccess) return e;
        if (qres != cudaDriverEntryPointSuccess || !fn) return cudaErrorNotSupported;
        enc = reinterpret_cast<EncodeTiledFn>(fn);
    }
    const cuuint32_t es[5] = {1, 1, 1, 1, 1};
    const CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_UINT8, (cuuint32_t)rank, const_cast<int8_t*>(basep), dims, strides, box, es,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, swizzle, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

struct OzWs {
    int8_t* sA;                    // QUAD layout
    int8_t* sB;                    // ROWS layout
    unsigned long long* maxbits;   // [2][modes]
    int* exps;                     // [2][modes]
};
int oz_pitch_rows(int N) { return (N + 127) / 128 * 128; }   // rows start on 128-byte boundaries: a 128-byte box row is one line
int oz_pitch_quad(int N) { return (N + 31) / 32 * 256; }     // 8 slots x 32 bytes per chunk of 32 columns
size_t oz_bytes_quad(int N, size_t modes) { return (modes * OZ_PLANES * (size_t)N * oz_pitch_quad(N) + 255) / 256 * 256; }
size_t oz_bytes_rows(int N, size_t modes) { return (modes * OZ_PLANES * OZ_S * (size_t)N * oz_pitch_rows(N) + 255) / 256 * 256; }
OzWs oz_carve(const FreqLayout& f, int batch, void* ws) {
    const size_t modes = (size_t)batch * f.L;
    OzWs w;
    w.sA = static_cast<int8_t*>(ws);
    w.sB = w.sA + oz_bytes_quad(f.N, modes);
    w.maxbits = reinterpret_cast<unsigned long long*>(w.sB + oz_bytes_rows(f.N, modes));
    w.exps = reinterpret_cast<int*>(w.maxbits + 2 * modes);
    return w;
}

}  // namespace

size_t ozaki_workspace_bytes(const FreqLayout& f, int batch) {
    const size_t modes = (size_t)batch * f.L;
    return oz_bytes_quad(f.N, modes) + oz_bytes_rows(f.N, modes) + 2 * modes * 16 + 256;
}

// FP64 spectra A~, B~ (all batch * L modes) -> int8 slices, exponents (in `ws`, ozaki_workspace_bytes)
cudaError_t launch_ozaki_slice(const FreqLayout& f, int batch, const double* A, const double* B, void* ws, cudaStream_t st) {
    const int modes = batch * f.L;
    const int N = f.N;
    const OzWs w = oz_carve(f, batch, ws);
    cudaError_t e;
    if ((e = cudaMemsetAsync(w.maxbits, 0, sizeof(unsigned long long) * 2 * modes, st)) != cudaSuccess) return e;
    const unsigned chunks = (unsigned)((f.NN + 256 * 8 - 1) / (256 * 8));
    const unsigned gy = (unsigned)(modes < 65535 ? modes : 65535);
    oz_absmax_kernel<<<dim3(chunks, gy), 256, 0, st>>>(reinterpret_cast<const double2*>(A), w.maxbits, f.NN, modes);
    oz_absmax_kernel<<<dim3(chunks, gy), 256, 0, st>>>(reinterpret_cast<const double2*>(B), w.maxbits + modes, f.NN, modes);
    const int pq = oz_pitch_quad(N), pr = oz_pitch_rows(N);
    oz_slice_kernel<true><<<dim3((unsigned)((N * (pq / 256 * 8) + 255) / 256), gy), 256, 0, st>>>(
        reinterpret_cast<const double2*>(A), w.sA, w.maxbits, w.exps, N, pq, modes);
    oz_slice_kernel<false><<<dim3((unsigned)((N * ((N + 3) / 4) + 255) / 256), gy), 256, 0, st>>>(
        reinterpret_cast<const double2*>(B), w.sB, w.maxbits + modes, w.exps + modes, N, pr, modes);
    return cudaGetLastError();
}

// C~(p) = A~(p) B~(p) for all batch * L modes from the slices in `ws`
cudaError_t launch_ozaki_gemm(const FreqLayout& f, int batch, const void* ws, double* C, cudaStream_t st) {
    const int modes = batch * f.L;
    const int N = f.N;
    const OzWs w = oz_carve(f, batch, const_cast<void*>(ws));
    cudaError_t e;
    static bool attr_done[NSPT_MAX_DEVICES] = {};
    const int dev = current_device();
    if (!attr_done[dev]) {
        e = cudaFuncSetAttribute(zgemm_modes_ozaki_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, OZ_SMEM);
        if (e != cudaSuccess) return e;
        attr_done[dev] = true;
    }
    const int pq = oz_pitch_quad(N), pr = oz_pitch_rows(N), nkc = (N + OZ_KC - 1) / OZ_KC;
    CUtensorMap mapM, mapN;
    {   // B~ slices, ROWS layout: (col j, row k, slice, mode * plane); box = [7 slices][32 k][128 bytes of j]
        const cuuint64_t dims[4] = {(cuuint64_t)N, (cuuint64_t)N, (cuuint64_t)OZ_S, (cuuint64_t)modes * OZ_PLANES};
        const cuuint64_t strides[3] = {(cuuint64_t)pr, (cuuint64_t)N * pr, (cuuint64_t)OZ_S * N * pr};
        const cuuint32_t box[4] = {(cuuint32_t)OZ_BM, (cuuint32_t)OZ_KC, (cuuint32_t)OZ_S, 1};
        if ((e = encode_u8(&mapM, w.sB, 4, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B)) != cudaSuccess) return e;
    }
    {   // A~ slices, QUAD layout: (128 bytes = 4 slots, row i, half, k-chunk, mode * plane); box = [2 halves][64 i][128 bytes]
        const cuuint64_t dims[5] = {128, (cuuint64_t)N, 2, (cuuint64_t)nkc, (cuuint64_t)modes * OZ_PLANES};
        const cuuint64_t strides[4] = {(cuuint64_t)pq, 128, 256, (cuuint64_t)N * pq};
        const cuuint32_t box[5] = {128, (cuuint32_t)OZ_BN, 2, 1, 1};
        if ((e = encode_u8(&mapN, w.sA, 5, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B)) != cudaSuccess) return e;
    }
    OzParams P;
    P.C = reinterpret_cast<double2*>(C);
    P.expA = w.exps;
    P.expB = w.exps + modes;
    P.NN = f.NN;
    P.N = N;
    P.tiles_i = (N + OZ_BN - 1) / OZ_BN;
    P.tiles_j = (N + OZ_BM - 1) / OZ_BM;
    P.nkc = nkc;
    const unsigned grid = (unsigned)(modes * P.tiles_i * P.tiles_j);
    return launch_pdl(zgemm_modes_ozaki_kernel, grid, OZ_THREADS, OZ_SMEM, st, mapM, mapN, P);
}

}  // namespace nspt
