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
// final FP64 recombination.  The exponents e come from the forward transform, which records max(|re|, |im|) of every mode
// while it writes the FP64 spectra (nspt_fft.cu); one slicing pass then cuts both spectra.
//
// Product kernel.  Persistent CTAs, tile = 64 rows x 128 columns of one mode, computed transposed (the M side of the MMA,
// 128 TMEM lanes, runs over output columns j and reads B~ slices MN-major; the N side runs over output rows i and reads
// A~ slices K-major); K-chunks of 32 arrive by TMA (SWIZZLE_128B) in a ring, all seven slices of both operands at once
// (44 KB per stage).  One lane of warp 1 issues tcgen05.mma.kind::i8 (M=128, N=64, K=32): 28 per stage, into seven TMEM
// accumulators (d = 0..6, 64 columns each, 448 of the 512 columns); runs of MMAs with the same M-side slice fetch it once
// (collector reuse).  The three planes run one after the other through the same accumulators; eight epilogue warps drain
// them with tcgen05.ld, recombine the seven INT32 sums in FP64 (Horner in 2^-8) and keep the running real / imaginary
// parts of the 3M product in registers; the scaling and stores of a tile overlap the next tile's MMAs.  With CG = 2 a CTA
// PAIR computes 256 columns x 64 rows (tcgen05.mma.cta_group::2, M = 256): each CTA stages its own 128 columns of the
// M side and half of the N-side rows.  Measured on B200 at N = 225, L = 128: a stage of 28 MMAs takes
// 1200 cycles with one CTA per tile (bound by shared-memory bandwidth: 84 KB read by the tensor core + 44 KB written by
// TMA per stage) and 980 with pairs (the tensor-core rate), the drain of the seven accumulators 2200-2900 cycles per
// plane; 166 us per product either way against 325 us on the FP64 tensor pipe.
#include <cuda.h>

#include "nspt_internal.cuh"
#include "nspt_ozaki.cuh"
#include "nspt_tma.cuh"

namespace nspt {
namespace {

// Operand staging, measured on B200 with probes of the TMA unit and of tcgen05.mma.kind::i8: the TMA unit is
// row-rate bound (1.9 cycles per row of <= 128 bytes with all SMs loading), so every shared-memory row is 128 bytes; a
// 128 x 64 x 32 MMA takes 35 cycles in a run that reuses the M-side operand from the collector and 48 without (32 is the
// tensor rate; N = 128 and 256 reach it, but seven accumulators of 128 columns do not fit the 512 columns of TMEM).  The tensor
// core computes the TRANSPOSED tile D[j][i] = sum_k B~[k][j] A~[i][k]: its M side (128 TMEM lanes) runs over output columns j
// and reads B~ slices MN-major -- the row-major layout the transforms write -- and its N side (64 TMEM columns) runs over
// output rows i and reads A~ slices K-major from 128-byte rows that carry four slices of one 32-column k-chunk (QUAD layout;
// the slice is selected by a 32-byte offset inside the swizzled row).  The epilogue then writes 512 contiguous bytes of a row of
// C~ per warp.  (The untransposed arrangement, 64-byte rows for B~ and per-thread row segments in the epilogue, measured 9 %
// slower.)
constexpr int OZ_BM = 128, OZ_BN = 64, OZ_KC = 32;   // tile of one CTA (j x i) and K per stage = K of one tcgen05.mma.kind::i8
constexpr int OZ_M_SLICE = OZ_KC * OZ_BM;            // B~ slice of a stage: [32 k][128 bytes of j] = 4096
constexpr int OZ_M_STAGE = OZ_S * OZ_M_SLICE;        // 28672
constexpr int OZ_THREADS = 384;                      // warp 0 TMA, warp 1 MMA, warp 2 TMEM allocator, warps 4-11 epilogue
constexpr int OZ_TMEM_COLS = 512;

// ---- slicing ------------------------------------------------------------------------------------------------
// Slicing pass: up to OZ_MAX_JOBS spectra in one launch (blockIdx.z), each into the QUAD and / or the ROWS layout (a spectrum
// that serves as left factor of one product and as right factor of another is read and converted once); the per-mode maxima
// come from the transform that wrote the spectrum (maxbits); digits without 64-bit conversions (oz_fixed), 4 x 4 byte
// transposes for the packing.  thread = 4 consecutive columns of a row of one mode; a warp writes 128 contiguous bytes per
// (plane, slice).
constexpr int OZ_MAX_JOBS = 12;
struct SliceJobDev {
    const double2* X;
    const unsigned long long* maxbits;
    size_t maxbits_stride;
    int8_t* quad;      // slot base or null
    int8_t* rows;      // slot base or null
    int* exps_q;
    int* exps_r;
    int mirror_L;      // 0, or L: mode b L + p takes the maximum of entry b L + (L - p) % L (X is a dagger spectrum)
};
struct SliceParams {
    SliceJobDev job[OZ_MAX_JOBS];
    int pitch_q, pitch_r;
    int N, modes;
};
// consecutive modes per CTA: the loads of the second are in flight while the first is cut.  Short CTAs win: 8 modes per CTA
// (2.5 waves, all CTAs of a wave in step) measured 119 us at config 3, 4: 112, 2: 106, 1: 111; a one-wave persistent kernel
// 123-136 us (its CTAs load, convert and store in lockstep).
constexpr int OZ_SLICE_MODES = 2;   // consecutive modes per thread: the loads of the next mode are in flight while one is cut
// the 21 slice words of four columns of one mode: re and im planes from the fixed-point integers V1, V2, the re + im plane from
// floor((V1 + V2) / 2) (same accuracy as rounding (re + im) / 2, without a third conversion); w[plane][d] = digit of weight
// 256^d of the four columns = slice 6 - d
__device__ __forceinline__ void oz_slice4(const double2 (&v)[4], double sc, unsigned int (&w)[OZ_PLANES][8]) {
    unsigned int lo[OZ_PLANES][4], hi[OZ_PLANES][4];
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const long long v1 = oz_fixed(v[c].x, sc), v2 = oz_fixed(v[c].y, sc);
        oz_digits_of(v1, lo[0][c], hi[0][c]);
        oz_digits_of(v2, lo[1][c], hi[1][c]);
        oz_digits_of((v1 + v2) >> 1, lo[2][c], hi[2][c]);
    }
#pragma unroll
    for (int q = 0; q < OZ_PLANES; ++q) {
        transpose4x4(lo[q], w[q]);
        transpose4x4(hi[q], w[q] + 4);
    }
}
__device__ __forceinline__ void oz_store_words(const unsigned int (&w)[OZ_PLANES][8], int8_t* base, size_t plane_stride, size_t slice_stride) {
#pragma unroll
    for (int q = 0; q < OZ_PLANES; ++q) {
        int8_t* p = base + (size_t)q * plane_stride + (size_t)(OZ_S - 1) * slice_stride;
#pragma unroll
        for (int d = 0; d < OZ_S; ++d) {
            *reinterpret_cast<unsigned int*>(p) = w[q][d];
            p -= slice_stride;
        }
    }
}
// The spectrum of a mode is one contiguous array of N^2 elements and the 256 threads of a CTA (row-aligned groups of four
// columns, row-major) cover one contiguous range of it: the CTA copies that range to shared memory with 16-byte cp.async
// (coalesced, no registers, two modes in flight) and every thread then picks up its four columns from there.
constexpr int OZ_SLICE_BUF = 1024 + 8;   // elements per stage (256 groups of 4, plus slack for the row ends)
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int PENDING>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(PENDING) : "memory"); }
// position of element p of the staged range: XOR of the low two bits with bits 3-4, so that the 16-byte reads of a quarter
// warp (stride four elements) cover all banks
__device__ __forceinline__ int oz_swz(int p) { return p ^ ((p >> 3) & 3); }

__global__ void __launch_bounds__(256) oz_slice_kernel(const __grid_constant__ SliceParams P) {
    __shared__ double2 stage[2][OZ_SLICE_BUF];
    __shared__ double ssc[OZ_SLICE_MODES];
    const SliceJobDev& J = P.job[blockIdx.z];
    const int N = P.N;
    const bool quad = J.quad != nullptr, rows = J.rows != nullptr;
    // 4-column groups per row: the QUAD layout writes its k padding (zeros up to a multiple of 32 columns) as well
    const int qpr = quad ? (P.pitch_q >> 5) : ((N + 3) >> 2);
    const int total = N * qpr;
    const int t0 = blockIdx.x * 256, t = t0 + threadIdx.x;
    if (t0 >= total) return;
    const int m_begin = blockIdx.y * OZ_SLICE_MODES;
    const int nm = P.modes - m_begin < OZ_SLICE_MODES ? P.modes - m_begin : OZ_SLICE_MODES;
    // contiguous element range of this CTA: from the first column of its first group to the end of its last group
    const int tl = (t0 + 255 < total ? t0 + 255 : total - 1);
    const int c0 = 4 * (t0 % qpr), c1 = 4 * (tl % qpr) + 4;
    const int e0 = (t0 / qpr) * N + (c0 < N ? c0 : N), e1 = (tl / qpr) * N + (c1 < N ? c1 : N);
    const int count = e1 - e0;   // <= OZ_SLICE_BUF
    pdl_wait();
    pdl_trigger();
    if (threadIdx.x < nm) {
        int m = m_begin + threadIdx.x;
        if (J.mirror_L) {
            const int p = m % J.mirror_L;
            m = m - p + (J.mirror_L - p) % J.mirror_L;
        }
        unsigned long long mb = J.maxbits[m];
#pragma unroll
        for (int b = 1; b < NSPT_MAX_BUCKETS; ++b) {   // the transforms keep NSPT_MAX_BUCKETS copies (less atomic contention)
            const unsigned long long o = J.maxbits[m + (size_t)b * J.maxbits_stride];
            mb = o > mb ? o : mb;
        }
        const int e = oz_exponent(mb);
        ssc[threadIdx.x] = oz_pow2(OZ_FRAC_BITS - e);
        if (blockIdx.x == 0) {
            if (quad) J.exps_q[m_begin + threadIdx.x] = e;
            if (rows) J.exps_r[m_begin + threadIdx.x] = e;
        }
    }
    auto fetch = [&](int i) {   // mode m_begin + i -> stage i & 1
        if (i < nm) {
            const double2* src = J.X + (size_t)(m_begin + i) * N * N + e0;
            const uint32_t dst = smem_u32(&stage[i & 1][0]);
            for (int p = threadIdx.x; p < count; p += 256) cp_async16(dst + 16u * (uint32_t)oz_swz(p), src + p);
        }
        cp_async_commit();
    };
    fetch(0);
    const bool active = t < total;
    const int row = active ? t / qpr : 0, j0 = active ? (t % qpr) * 4 : 0;
    const int nvalid = active ? N - j0 : 0;   // columns of this group inside the matrix (<= 0: k padding of the QUAD layout)
    const int p0 = row * N + j0 - e0;
    const size_t q_plane = (size_t)N * P.pitch_q, q_mode = (size_t)OZ_PLANES * q_plane;
    const size_t r_slice = (size_t)N * P.pitch_r, r_plane = (size_t)OZ_S * r_slice, r_mode = (size_t)OZ_PLANES * r_plane;
    int8_t* outq = quad ? J.quad + (size_t)m_begin * q_mode + (size_t)row * P.pitch_q + (size_t)(j0 >> 5) * 256 + (j0 & 31) : nullptr;
    int8_t* outr = (rows && j0 < P.pitch_r) ? J.rows + (size_t)m_begin * r_mode + (size_t)row * P.pitch_r + j0 : nullptr;
#pragma unroll 1
    for (int i = 0; i < nm; ++i) {
        fetch(i + 1);
        cp_async_wait<1>();
        __syncthreads();   // mode i has landed (and the scales, first time round)
        if (active) {
            double2 v[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) v[c] = c < nvalid ? stage[i & 1][oz_swz(p0 + c)] : make_double2(0.0, 0.0);
            unsigned int w[OZ_PLANES][8];
            oz_slice4(v, ssc[i], w);
            if (outq) oz_store_words(w, outq + (size_t)i * q_mode, q_plane, 32);
            if (outr) oz_store_words(w, outr + (size_t)i * r_mode, r_plane, r_slice);
        }
        __syncthreads();   // stage i & 1 may be refilled
    }
}

// Per-mode maxima of a spectrum that no transform kernel has written (the block polynomials of the series exponential):
// max(|re|, |im|) as the high word of the bit pattern, one atomicMax per CTA and mode.
__global__ void __launch_bounds__(256) oz_absmax_kernel(const double2* __restrict__ X, unsigned long long* __restrict__ maxbits,
                                                      size_t NN, int modes) {
    __shared__ unsigned int red[8];
    for (int mode = blockIdx.y; mode < modes; mode += gridDim.y) {   // the grid's y extent is capped at 65535
        const double2* x = X + (size_t)mode * NN;
        unsigned int m = 0u;
        for (size_t e = (size_t)blockIdx.x * 256 + threadIdx.x; e < NN; e += (size_t)gridDim.x * 256) {
            const unsigned int a = oz_abs_hi(__ldg(&x[e]));
            m = a > m ? a : m;
        }
        m = __reduce_max_sync(0xffffffffu, m);
        __syncthreads();
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
        __syncthreads();
        if (threadIdx.x == 0) {
#pragma unroll
            for (int w = 1; w < 8; ++w) m = red[w] > m ? red[w] : m;
            if (m) atomicMax(maxbits + mode, (unsigned long long)m << 32);
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
// arrive on an mbarrier once every tcgen05.mma issued so far by this thread has completed
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tc_ld4(uint32_t taddr, int (&r)[4]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
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
// exact int32 -> double (no I2F): 2^52 + 2^31 + x has x + 2^31 in its low mantissa word
__device__ __forceinline__ double oz_i2d(int x) {
    return __hiloint2double(0x43300000, (int)((unsigned)x ^ 0x80000000u)) - 4503601774854144.0;
}

// =====================================================================================================================
// The product kernel (see the head of the file).  Barrier protocol with CG = 2: TMA loads of both CTAs report to the
// leader's "full" barrier, MMA completion is multicast to both CTAs' "empty" / "accumulator full" barriers, and the epilogue
// warps of both CTAs report to the leader's "accumulator empty" barrier.
// =====================================================================================================================
template <int CG>
struct OzCfg {
    static constexpr int N_ROWS = OZ_BN / CG;               // rows of the N-side operand staged by one CTA
    static constexpr int N_HALF = N_ROWS * 128;              // slices 4h..4h+3 of a stage
    static constexpr int N_STAGE = 2 * N_HALF;
    static constexpr int STAGE = OZ_M_STAGE + N_STAGE;       // 45056 (CG = 1) / 36864 (CG = 2)
    static constexpr int STAGES = CG == 2 ? 5 : 4;
    static constexpr int SMEM = STAGES * STAGE + 1024 + 256;
    static constexpr uint32_t IDESC = (2u << 4) | (1u << 7) | (1u << 10) | (1u << 15) | (0u << 16) | ((OZ_BN >> 3) << 17) |
                                      (((128 * CG) >> 4) << 24);
    static_assert(STAGE % 1024 == 0, "stage alignment");
};

__device__ __forceinline__ uint32_t cluster_rank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// shared::cluster address of the same shared-memory location in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t mapa_rank(uint32_t addr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
// mbarrier wait with a watchdog: a protocol error traps instead of hanging the GPU
__device__ __forceinline__ void mbar_wait_wd(uint32_t bar, uint32_t parity) {
    uint32_t done = 0;
    for (unsigned long long spins = 0; !done; ++spins) {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(done)
            : "r"(bar), "r"(parity)
            : "memory");
        if (spins > (1ull << 22)) __trap();
    }
}
// COLLECT: use of the A-operand (M side) collector buffer -- consecutive MMAs with the same M-side slice read it from shared
// memory once: 0 = no reuse, 1 = fill (first of a run), 2 = use (middle), 3 = last use.  Without it a 128 x 64 x 32 MMA
// reads 6 KB of shared memory in 32 cycles, more than the 128 bytes per cycle an SM delivers.
template <int CG, int COLLECT>
__device__ __forceinline__ void tc_mma_i8_cg(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
#define NSPT_OZ_MMA2(G, Q)                                                                         \
    asm volatile(                                                                                  \
        "{\n"                                                                                      \
        ".reg .pred p;\n"                                                                          \
        "setp.ne.b32 p, %4, 0;\n"                                                                  \
        "tcgen05.mma.cta_group::" G ".kind::i8" Q " [%0], %1, %2, %3, p;\n"                        \
        "}\n" ::"r"(d_tmem),                                                                       \
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)                                      \
        : "memory")
    if constexpr (CG == 2) {
        if constexpr (COLLECT == 1) NSPT_OZ_MMA2("2", ".collector::a::fill");
        else if constexpr (COLLECT == 2) NSPT_OZ_MMA2("2", ".collector::a::use");
        else if constexpr (COLLECT == 3) NSPT_OZ_MMA2("2", ".collector::a::lastuse");
        else NSPT_OZ_MMA2("2", "");
    } else {
        if constexpr (COLLECT == 1) NSPT_OZ_MMA2("1", ".collector::a::fill");
        else if constexpr (COLLECT == 2) NSPT_OZ_MMA2("1", ".collector::a::use");
        else if constexpr (COLLECT == 3) NSPT_OZ_MMA2("1", ".collector::a::lastuse");
        else NSPT_OZ_MMA2("1", "");
    }
#undef NSPT_OZ_MMA2
}
// completion of all MMAs issued so far -> arrive on the barrier at the same offset in every CTA of the pair
template <int CG>
__device__ __forceinline__ void tc_commit_cg(uint32_t bar) {
    if constexpr (CG == 2) {
        asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(bar),
                     "h"((uint16_t)3)
                     : "memory");
    } else {
        tc_commit(bar);
    }
}
// TMA loads whose completion is reported to a barrier that may live in the peer CTA (the leader's)
// The slices are streamed once (each operand tile is read by the two to five CTAs that need it at about the same time) while
// the C~ the epilogues write is read back by the next kernel: the operand loads carry an L2 evict_first policy (1-2 % measured).
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void tma_load_4d_hint(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2, int c3,
                                                 uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%3, %4, %5, %6}], "
        "[%2], %7;" ::"r"(dst),
        "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "l"(policy)
        : "memory");
}
__device__ __forceinline__ void tma_load_5d_hint(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2, int c3,
                                                 int c4, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%3, %4, %5, %6, "
        "%7}], [%2], %8;" ::"r"(dst),
        "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "l"(policy)
        : "memory");
}
template <int CG>
__device__ __forceinline__ void tma_load_4d_cg(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2, int c3) {
    if constexpr (CG == 2) {
        asm volatile(
            "cp.async.bulk.tensor.4d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], "
            "[%2];" ::"r"(dst),
            "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
            : "memory");
    } else {
        tma_load_4d(dst, map, bar, c0, c1, c2, c3);
    }
}
template <int CG>
__device__ __forceinline__ void tma_load_5d_cg(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2, int c3,
                                               int c4) {
    if constexpr (CG == 2) {
        asm volatile(
            "cp.async.bulk.tensor.5d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, "
            "%7}], [%2];" ::"r"(dst),
            "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
            : "memory");
    } else {
        tma_load_5d(dst, map, bar, c0, c1, c2, c3, c4);
    }
}
template <int CG>
__device__ __forceinline__ void tc_alloc_cg(uint32_t smem_dst, uint32_t cols) {
    if constexpr (CG == 2) {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(cols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    } else {
        tc_alloc(smem_dst, cols);
    }
}
template <int CG>
__device__ __forceinline__ void tc_dealloc_cg(uint32_t taddr, uint32_t cols) {
    if constexpr (CG == 2)
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
    else
        tc_dealloc(taddr, cols);
}

// One lane of the MMA warp issues; everything the instruction consumes (descriptors, TMEM address) is computed by the WHOLE
// warp from warp-uniform values so that the compiler keeps it in uniform registers -- inside a lane-0-only branch it falls
// back to a R2UR "waterfall" loop of ~17 instructions per MMA, which costs more than the 32 cycles an MMA takes.
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "elect.sync _|p, 0xffffffff;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(pred));
    return pred != 0;
}
template <int CG, int T0, int S0, bool FIRSTK>
__device__ __forceinline__ void oz_issue_pairs(uint32_t tmem, uint64_t dm0, uint64_t dn0, bool elected) {
    constexpr int LAST = OZ_S - 1 - T0;
    constexpr int COLLECT = (LAST == 0) ? 0 : (S0 == 0 ? 1 : (S0 == LAST ? 3 : 2));
    // descriptors differ from the stage's first ones by a constant in the 14-bit start-address field (no carry: < 256 KB)
    const uint64_t dm = dm0 + (uint64_t)((T0 * OZ_M_SLICE) >> 4);
    const uint64_t dn = dn0 + (uint64_t)(((S0 >> 2) * OzCfg<CG>::N_HALF + (S0 & 3) * 32) >> 4);
    const uint32_t d = tmem + (uint32_t)((S0 + T0) * OZ_BN);
    if (elected) tc_mma_i8_cg<CG, COLLECT>(d, dm, dn, OzCfg<CG>::IDESC, (!FIRSTK || T0 != 0) ? 1u : 0u);
    if constexpr (S0 < LAST)
        oz_issue_pairs<CG, T0, S0 + 1, FIRSTK>(tmem, dm0, dn0, elected);
    else if constexpr (T0 + 1 < OZ_S)
        oz_issue_pairs<CG, T0 + 1, 0, FIRSTK>(tmem, dm0, dn0, elected);
}

// exact conversion of the weighted sum of the seven accumulators of one output element:
//   h = sum_d a_d 2^(-8 d) = hi 2^-24 + lo 2^-48,  hi = a0 2^24 + a1 2^16 + a2 2^8 + a3,  lo = a4 2^16 + a5 2^8 + a6
// (|a_d| < 2^26, so |hi| < 2^51 and |lo| < 2^43: both convert exactly with the 2^52 + 2^51 trick); returns h * 2^24
// h = sum_d a_d 2^(-8 d) from the seven INT32 accumulators of one output element: every a_d converts exactly through the
// 2^52 + 2^31 bit trick (one LOP3 and one DADD, no I2F), then Horner in 2^-8 -- 7 LOP3, 7 DADD, 6 DFMA.  (The all-integer
// alternative, two 64-bit multiply-add chains, compiles to about 40 instructions per element on sm_100a: ptxas expands every
// mad.wide.s32 with a 64-bit addend into IMAD.HI + IMAD + IADD3 + IADD3.X.)  Returns h * 2^24 for the common scale below.
__device__ __forceinline__ double oz_combine(int a0, int a1, int a2, int a3, int a4, int a5, int a6) {
    double h = oz_i2d(a6);
    h = fma(h, 0.00390625, oz_i2d(a5));
    h = fma(h, 0.00390625, oz_i2d(a4));
    h = fma(h, 0.00390625, oz_i2d(a3));
    h = fma(h, 0.00390625, oz_i2d(a2));
    h = fma(h, 0.00390625, oz_i2d(a1));
    h = fma(h, 0.00390625, oz_i2d(a0));
    return h;
}

// One product of a launch: left factor = QUAD slot, right factor = ROWS slot (as (mode, plane) offsets of the tensor maps),
// the FP64 spectra they were cut from (tail of K), their exponent tables, and the epilogue of nspt_zgemm.cu's GemmOut:
//     C(p)            (+)= alpha * M(p) + diag * 1,        D((L - p) mod L) (+)= beta * M(p)^H.
struct OzGroupDev {
    const double2* At;
    const double2* Bt;
    const int* expA;
    const int* expB;
    double2* C;
    double2* D;
    double alpha_re, alpha_im, beta_re, beta_im, diag;
    int pbaseA, pbaseB;        // first (mode, plane) index of the slot in the N-side / M-side tensor map
    int accumulate, accumulate_d;
};
constexpr int OZ_MAX_GROUPS = 12;
struct OzParams {
    OzGroupDev g[OZ_MAX_GROUPS];
    unsigned long long* clear;   // per-mode maxima the slicing pass has consumed: zeroed here for the next transform (or null)
    int clear_count;
    size_t NN;
    int N, L;
    int modes;                 // modes per group (batch * L)
    int tiles_i, tiles_j;      // tiles per mode: rows in steps of 64, columns in steps of 128 * CG
    int total_tiles;           // groups * modes * tiles_i * tiles_j
    int nkc;                   // K-chunks of 32 that run on the tensor core
    int tail;                  // k >= 32 nkc (0 .. OZ_TAIL_MAX of them) are added in FP64 by the epilogue
};
// Every odd-L TEK size has N = 1 mod 8, and N = 225, 289 are 1 mod 32: a full K-chunk of 28 MMAs per plane would serve ONE
// column of A~.  When N mod 32 <= OZ_TAIL_MAX those columns are left out of the integer products and the epilogue adds
// their rank-1 updates from the FP64 spectra (7 instead of 8 chunks at N = 225: 12 % fewer MMAs).
constexpr int OZ_TAIL_MAX = 2;

template <int CG>
__global__ void __launch_bounds__(OZ_THREADS, 1)
zgemm_modes_i8_kernel(const __grid_constant__ CUtensorMap mapM, const __grid_constant__ CUtensorMap mapN,
                      const __grid_constant__ OzParams P) {
    using K = OzCfg<CG>;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar_full = base + K::STAGES * K::STAGE;
    const uint32_t bar_empty = bar_full + 8 * K::STAGES;
    const uint32_t bar_acc_full = bar_empty + 8 * K::STAGES;
    const uint32_t bar_acc_empty = bar_acc_full + 8;
    const uint32_t tmem_slot = bar_acc_empty + 8;
    volatile uint32_t* tmem_slot_gen = reinterpret_cast<volatile uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = CG == 2 ? cluster_rank() : 0u;
    const int cluster_id = blockIdx.x / CG, nclusters = gridDim.x / CG;
    const int nkc = P.nkc;
    const int tiles_per_mode = P.tiles_i * P.tiles_j;

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < K::STAGES; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, 1);
        }
        mbar_init(bar_acc_full, 1);
        mbar_init(bar_acc_empty, 8 * CG);
        mbar_fence_init();
    }
    if (warp == 2) tc_alloc_cg<CG>(tmem_slot, OZ_TMEM_COLS);
    tc_fence_before();
    if constexpr (CG == 2) cluster_sync_all(); else __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot_gen;
    pdl_wait();
    pdl_trigger();
    if (P.clear && blockIdx.x == 0)   // a memset between two kernels would cost a launch and the programmatic overlap of the next one
        for (int i = threadIdx.x; i < P.clear_count; i += OZ_THREADS) P.clear[i] = 0ull;
    // barriers of the leader CTA, as shared::cluster addresses (identity for CG = 1)
    const uint32_t lead_full = CG == 2 ? mapa_rank(bar_full, 0) : bar_full;
    const uint32_t lead_acc_empty = CG == 2 ? mapa_rank(bar_acc_empty, 0) : bar_acc_empty;

    if (warp < 4) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
        if (warp == 0) {
            // ------------------------------------------------------------ TMA producer (one thread per CTA)
            if (lane == 0) {
                int it = 0;
                const uint64_t policy = l2_policy_evict_first();
                for (int tile = cluster_id; tile < P.total_tiles; tile += nclusters) {
                    const int gm = tile / tiles_per_mode, rem = tile % tiles_per_mode;   // gm = group * modes + mode
                    const int grp = gm / P.modes, mode = gm % P.modes;
                    const int i0 = (rem / P.tiles_j) * OZ_BN + (int)rank * K::N_ROWS;
                    const int j0 = (rem % P.tiles_j) * (OZ_BM * CG) + (int)rank * OZ_BM;
                    const int pa = P.g[grp].pbaseA + mode * OZ_PLANES, pb = P.g[grp].pbaseB + mode * OZ_PLANES;
                    for (int plane = 0; plane < OZ_PLANES; ++plane) {
                        for (int kc = 0; kc < nkc; ++kc, ++it) {
                            const int slot = it % K::STAGES;
                            mbar_wait_wd(bar_empty + 8 * slot, ((it / K::STAGES) & 1) ^ 1);
                            if (rank == 0) mbar_expect_tx(bar_full + 8 * slot, K::STAGE * CG);
                            const uint32_t st = base + slot * K::STAGE;
                            if constexpr (CG == 1) {
                                tma_load_4d_hint(st, &mapM, bar_full + 8 * slot, j0, kc * OZ_KC, 0, pb + plane, policy);
                                tma_load_5d_hint(st + OZ_M_STAGE, &mapN, bar_full + 8 * slot, 0, i0, 0, kc, pa + plane, policy);
                            } else {
                                tma_load_4d_cg<CG>(st, &mapM, lead_full + 8 * slot, j0, kc * OZ_KC, 0, pb + plane);
                                tma_load_5d_cg<CG>(st + OZ_M_STAGE, &mapN, lead_full + 8 * slot, 0, i0, 0, kc, pa + plane);
                            }
                        }
                    }
                }
            }
        } else if (warp == 1) {
            // ------------------------------------------------------------ MMA issuer (warp 1 of the leader CTA, one lane issues)
            if (rank == 0) {
                const bool elected = elect_one();
                int it = 0, acc_it = 0;
                for (int tile = cluster_id; tile < P.total_tiles; tile += nclusters) {
                    for (int plane = 0; plane < OZ_PLANES; ++plane, ++acc_it) {
                        if (acc_it > 0) mbar_wait_wd(bar_acc_empty, (acc_it - 1) & 1);
                        tc_fence_after();
                        for (int kc = 0; kc < nkc; ++kc, ++it) {
                            const int slot = it % K::STAGES;
                            mbar_wait_wd(bar_full + 8 * slot, (it / K::STAGES) & 1);
                            tc_fence_after();
                            const uint32_t sm = base + slot * K::STAGE;
                            const uint64_t dm0 = oz_desc(sm, 4096, 1024), dn0 = oz_desc(sm + OZ_M_STAGE, 16, 1024);
                            if (kc == 0)
                                oz_issue_pairs<CG, 0, 0, true>(tmem, dm0, dn0, elected);
                            else
                                oz_issue_pairs<CG, 0, 0, false>(tmem, dm0, dn0, elected);
                            if (elected) tc_commit_cg<CG>(bar_empty + 8 * slot);   // the stage may be refilled once these MMAs have read it
                            __syncwarp();
                        }
                        if (elected) tc_commit_cg<CG>(bar_acc_full);
                        __syncwarp();
                    }
                }
            }
        }
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");
        // ------------------------------------------------------------ epilogue: 8 warps; warp w reads TMEM lanes 32 (w % 4) ..
        // lane of the accumulator = output column j, column of the accumulator = output row i
        const int we = warp - 4, quarter = we & 3, half = we >> 2;
        int acc_it = 0;
        uint64_t keep_policy;
        asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(keep_policy));
        // What a tile needs from global memory before its first drain -- the exponents of its mode and, for the tail of K
        // (k >= 32 nkc, added in FP64), lane l's element A~[row0 + l][k] and its own column of B~[k][.] -- is fetched BEFORE the
        // stores of the tile before it: behind 131 KB of stores per SM these loads waited 2800 cycles on the critical path.
        int esum_next = 0;
        double2 at_next[OZ_TAIL_MAX], bt_next[OZ_TAIL_MAX];
        auto prefetch = [&](int tile) {
            if (tile >= P.total_tiles) return;
            const int gm = tile / tiles_per_mode, rem = tile % tiles_per_mode;
            const int mode = gm % P.modes;
            const OzGroupDev& G = P.g[gm / P.modes];
            const int row0 = (rem / P.tiles_j) * OZ_BN + 32 * half;
            const int col = (rem % P.tiles_j) * (OZ_BM * CG) + (int)rank * OZ_BM + 32 * quarter + lane;
            esum_next = __ldg(G.expA + mode) + __ldg(G.expB + mode);
#pragma unroll
            for (int t = 0; t < OZ_TAIL_MAX; ++t) {
                at_next[t] = bt_next[t] = make_double2(0.0, 0.0);
                if (t < P.tail) {
                    const int k = OZ_KC * nkc + t;
                    if (row0 + lane < P.N) at_next[t] = __ldg(G.At + (size_t)mode * P.NN + (size_t)(row0 + lane) * P.N + k);
                    if (col < P.N) bt_next[t] = __ldg(G.Bt + (size_t)mode * P.NN + (size_t)k * P.N + col);
                }
            }
        };
        prefetch(cluster_id);
        for (int tile = cluster_id; tile < P.total_tiles; tile += nclusters) {
            const int gm = tile / tiles_per_mode, rem = tile % tiles_per_mode;
            const int mode = gm % P.modes;
            const OzGroupDev& G = P.g[gm / P.modes];
            const int row0 = (rem / P.tiles_j) * OZ_BN + 32 * half;
            const int col = (rem % P.tiles_j) * (OZ_BM * CG) + (int)rank * OZ_BM + 32 * quarter + lane;
            double re[32], im[32];
            const int esum = esum_next;
            const double sc = esum >= (1 << 20) ? __longlong_as_double(0x7ff8000000000000ll) : oz_pow2(esum - 12);
            // the running sums start from the tail product in units of the common scale (a power of two)
#pragma unroll
            for (int j = 0; j < 32; ++j) re[j] = im[j] = 0.0;
            if (P.tail) {
                const double isc = oz_pow2(12 - esum);
#pragma unroll
                for (int t = 0; t < OZ_TAIL_MAX; ++t) {
                    if (t < P.tail) {
                        const double2 at = at_next[t];
                        const double2 bt = make_double2(bt_next[t].x * isc, bt_next[t].y * isc);
#pragma unroll
                        for (int j = 0; j < 32; ++j) {
                            const double ax = __shfl_sync(0xffffffffu, at.x, j), ay = __shfl_sync(0xffffffffu, at.y, j);
                            re[j] = fma(ax, bt.x, fma(-ay, bt.y, re[j]));
                            im[j] = fma(ax, bt.y, fma(ay, bt.x, im[j]));
                        }
                    }
                }
            }
#pragma unroll
            for (int plane = 0; plane < OZ_PLANES; ++plane, ++acc_it) {
                mbar_wait_wd(bar_acc_full, acc_it & 1);
                tc_fence_after();
                // eight chunks of four columns; the loads of the next chunk are in flight while one is combined
                const uint32_t tbase = tmem + ((uint32_t)(32 * quarter) << 16) + (uint32_t)(32 * half);
                int a[2][OZ_S][4];
#pragma unroll
                for (int d = 0; d < OZ_S; ++d) tc_ld4(tbase + (uint32_t)(d * OZ_BN), a[0][d]);
#pragma unroll
                for (int cc = 0; cc < 8; ++cc) {
                    tc_wait_ld();
                    if (cc + 1 < 8) {
#pragma unroll
                        for (int d = 0; d < OZ_S; ++d) tc_ld4(tbase + (uint32_t)(d * OZ_BN + 4 * (cc + 1)), a[(cc + 1) & 1][d]);
                    }
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const int (&b)[OZ_S][4] = a[cc & 1];
                        const double h = oz_combine(b[0][j], b[1][j], b[2][j], b[3][j], b[4][j], b[5][j], b[6][j]);
                        // 3M: Cr = P1 - P2, Ci = 4 P3 - P1 - P2 (the sum planes carry one more exponent bit each)
                        if (plane == 0) {
                            re[4 * cc + j] += h;
                            im[4 * cc + j] -= h;
                        } else if (plane == 1) {
                            re[4 * cc + j] -= h;
                            im[4 * cc + j] -= h;
                        } else {
                            im[4 * cc + j] = fma(4.0, h, im[4 * cc + j]);
                        }
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) {
                    if (CG == 2) mbar_arrive_cluster(lead_acc_empty); else mbar_arrive(bar_acc_empty);
                }
            }
            prefetch(tile + nclusters);
            // scaling, epilogue and stores overlap the MMAs of the next tile
            if (col < P.N) {
                if (G.C) {
                    double2* c = G.C + (size_t)mode * P.NN + col;
                    const bool plain = G.alpha_re == 1.0 && G.alpha_im == 0.0 && G.diag == 0.0 && !G.accumulate;
                    if (plain) {
#pragma unroll
                        for (int j = 0; j < 32; ++j)   // the 32 lanes of a warp write 512 contiguous bytes of row row0 + j
                            if (row0 + j < P.N) {
                                double2* dst = &c[(size_t)(row0 + j) * P.N];
                                asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(dst), "d"(sc * re[j]), "d"(sc * im[j]), "l"(keep_policy) : "memory");
                            }
                    } else {
                        const double ar = sc * G.alpha_re, ai = sc * G.alpha_im;
#pragma unroll
                        for (int j = 0; j < 32; ++j) {
                            if (row0 + j < P.N) {
                                double2 o = make_double2(ar * re[j] - ai * im[j], ar * im[j] + ai * re[j]);
                                if (row0 + j == col) o.x += G.diag;
                                double2* dst = c + (size_t)(row0 + j) * P.N;
                                if (G.accumulate) {   // one contribution per element and launch: the sum keeps a fixed order
                                    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(&dst->x), "d"(o.x) : "memory");
                                    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(&dst->y), "d"(o.y) : "memory");
                                } else {
                                    *dst = o;
                                }
                            }
                        }
                    }
                }
                if (G.D) {
                    // spectrum of the daggered product series: D((L - p) mod L)[j][i] (+)= beta conj(M(p)[i][j])
                    const int pm = mode % P.L;
                    double2* d = G.D + (size_t)(mode - pm + (P.L - pm) % P.L) * P.NN + (size_t)col * P.N + row0;
                    const double br = sc * G.beta_re, bi = sc * G.beta_im;
#pragma unroll
                    for (int j = 0; j < 32; ++j) {
                        if (row0 + j < P.N) {
                            const double2 o = make_double2(br * re[j] + bi * im[j], bi * re[j] - br * im[j]);
                            if (G.accumulate_d) {
                                asm volatile("red.global.add.f64 [%0], %1;" ::"l"(&d[j].x), "d"(o.x) : "memory");
                                asm volatile("red.global.add.f64 [%0], %1;" ::"l"(&d[j].y), "d"(o.y) : "memory");
                            } else {
                                d[j] = o;
                            }
                        }
                    }
                }
            }
        }
    }
    __syncwarp();
    tc_fence_before();
    if constexpr (CG == 2) cluster_sync_all(); else __syncthreads();
    if (warp == 2) tc_dealloc_cg<CG>(tmem, OZ_TMEM_COLS);
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

size_t quad_slot_bytes(const FreqLayout& f, int modes) { return oz_bytes_quad(f.N, (size_t)modes); }
size_t rows_slot_bytes(const FreqLayout& f, int modes) { return oz_bytes_rows(f.N, (size_t)modes); }

// launch with programmatic stream serialization and (CG = 2) clusters of two CTAs
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl_cluster(void (*kernel)(KArgs...), unsigned grid, unsigned block, size_t smem, unsigned cluster,
                               cudaStream_t st, Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid, 1, 1);
    cfg.blockDim = dim3(block, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    attr[1].id = cudaLaunchAttributeClusterDimension;
    attr[1].val.clusterDim.x = cluster;
    attr[1].val.clusterDim.y = 1;
    attr[1].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = cluster > 1 ? 2 : 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// tensor maps over ALL slots of the store: a product addresses its operands by (mode, plane) offset
cudaError_t oz_maps(const FreqLayout& f, const OzStore& S, int n_rows, CUtensorMap* mapM, CUtensorMap* mapN) {
    const int N = f.N;
    const int pq = oz_pitch_quad(N), pr = oz_pitch_rows(N), nkc = (N + OZ_KC - 1) / OZ_KC;
    cudaError_t e;
    {   // right factors, ROWS layout: (col j, row k, slice, slot * mode * plane); box = [7 slices][32 k][128 bytes of j]
        const cuuint64_t dims[4] = {(cuuint64_t)N, (cuuint64_t)N, (cuuint64_t)OZ_S, (cuuint64_t)(S.nr > 0 ? S.nr : 1) * S.modes * OZ_PLANES};
        const cuuint64_t strides[3] = {(cuuint64_t)pr, (cuuint64_t)N * pr, (cuuint64_t)OZ_S * N * pr};
        const cuuint32_t box[4] = {(cuuint32_t)OZ_BM, (cuuint32_t)OZ_KC, (cuuint32_t)OZ_S, 1};
        if ((e = encode_u8(mapM, S.rows, 4, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B)) != cudaSuccess) return e;
    }
    {   // left factors, QUAD layout: (128 bytes = 4 slots, row i, half, k-chunk, slot * mode * plane); box = [2 halves][rows][128 bytes]
        const cuuint64_t dims[5] = {128, (cuuint64_t)N, 2, (cuuint64_t)nkc, (cuuint64_t)(S.nq > 0 ? S.nq : 1) * S.modes * OZ_PLANES};
        const cuuint64_t strides[4] = {(cuuint64_t)pq, 128, 256, (cuuint64_t)N * pq};
        const cuuint32_t box[5] = {128, (cuuint32_t)n_rows, 2, 1, 1};
        return encode_u8(mapN, S.quad, 5, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B);
    }
}

template <int CG>
cudaError_t launch_oz(const FreqLayout& f, const OzStore& S, const OzGemmGroup* groups, int ngroups, cudaStream_t st,
                      unsigned long long* clear, int clear_count) {
    using K = OzCfg<CG>;
    const int N = f.N;
    cudaError_t e;
    static bool attr_done[NSPT_MAX_DEVICES] = {};
    static int sms[NSPT_MAX_DEVICES] = {};
    const int dev = current_device();
    if (!attr_done[dev]) {
        e = cudaFuncSetAttribute(zgemm_modes_i8_kernel<CG>, cudaFuncAttributeMaxDynamicSharedMemorySize, K::SMEM);
        if (e != cudaSuccess) return e;
        sms[dev] = 148;
        cudaDeviceGetAttribute(&sms[dev], cudaDevAttrMultiProcessorCount, dev);
        attr_done[dev] = true;
    }
    CUtensorMap mapM, mapN;
    if ((e = oz_maps(f, S, K::N_ROWS, &mapM, &mapN)) != cudaSuccess) return e;
    OzParams P{};
    P.clear = clear;
    P.clear_count = clear_count;
    P.NN = f.NN;
    P.N = N;
    P.L = f.L;
    P.modes = S.modes;
    P.tiles_i = (N + OZ_BN - 1) / OZ_BN;
    P.tiles_j = (N + OZ_BM * CG - 1) / (OZ_BM * CG);
    P.total_tiles = ngroups * S.modes * P.tiles_i * P.tiles_j;
    P.nkc = (N + OZ_KC - 1) / OZ_KC;
    P.tail = 0;
    if (N >= 2 * OZ_KC && N % OZ_KC != 0 && N % OZ_KC <= OZ_TAIL_MAX) {
        P.nkc = N / OZ_KC;
        P.tail = N % OZ_KC;
    }
    for (int i = 0; i < ngroups; ++i) {
        const OzGemmGroup& g = groups[i];
        if (g.quad_slot < 0 || g.quad_slot >= S.nq || g.rows_slot < 0 || g.rows_slot >= S.nr || !g.A || !g.B || (!g.out.C && !g.out.D))
            return cudaErrorInvalidValue;
        OzGroupDev& d = P.g[i];
        d.At = reinterpret_cast<const double2*>(g.A);
        d.Bt = reinterpret_cast<const double2*>(g.B);
        d.expA = S.exps_q + (size_t)g.quad_slot * S.modes;
        d.expB = S.exps_r + (size_t)g.rows_slot * S.modes;
        d.C = reinterpret_cast<double2*>(g.out.C);
        d.D = reinterpret_cast<double2*>(g.out.D);
        d.alpha_re = g.out.alpha.re;
        d.alpha_im = g.out.alpha.im;
        d.beta_re = g.out.beta.re;
        d.beta_im = g.out.beta.im;
        d.diag = g.out.diag;
        d.pbaseA = g.quad_slot * S.modes * OZ_PLANES;
        d.pbaseB = g.rows_slot * S.modes * OZ_PLANES;
        d.accumulate = g.out.accumulate ? 1 : 0;
        d.accumulate_d = g.out.accumulate_d ? 1 : 0;
    }
    int clusters = sms[dev] / CG;
    if (clusters > P.total_tiles) clusters = P.total_tiles;
    return launch_pdl_cluster(zgemm_modes_i8_kernel<CG>, (unsigned)(clusters * CG), OZ_THREADS, K::SMEM, CG, st, mapM, mapN, P);
}

}  // namespace

size_t ozaki_store_bytes(const FreqLayout& f, int modes, int nq, int nr) {
    return (size_t)nq * quad_slot_bytes(f, modes) + (size_t)nr * rows_slot_bytes(f, modes) + (size_t)(nq + nr) * modes * sizeof(int) + 512;
}

OzStore ozaki_store(const FreqLayout& f, int modes, int nq, int nr, void* ws) {
    OzStore S;
    S.nq = nq;
    S.nr = nr;
    S.modes = modes;
    S.quad_slot_bytes = quad_slot_bytes(f, modes);
    S.rows_slot_bytes = rows_slot_bytes(f, modes);
    S.quad = static_cast<int8_t*>(ws);
    S.rows = S.quad + (size_t)nq * S.quad_slot_bytes;
    S.exps_q = reinterpret_cast<int*>(S.rows + (size_t)nr * S.rows_slot_bytes);
    S.exps_r = S.exps_q + (size_t)nq * modes;
    return S;
}

// FP64 spectra -> int8 slices, with the per-mode maxima the transforms recorded; up to OZ_MAX_JOBS spectra per launch
cudaError_t launch_ozaki_slice(const FreqLayout& f, const OzStore& S, const OzSliceJob* jobs, int njobs, cudaStream_t st) {
    const int N = f.N;
    for (int j0 = 0; j0 < njobs; j0 += OZ_MAX_JOBS) {
        const int nj = njobs - j0 < OZ_MAX_JOBS ? njobs - j0 : OZ_MAX_JOBS;
        SliceParams P{};
        P.pitch_q = oz_pitch_quad(N);
        P.pitch_r = oz_pitch_rows(N);
        P.N = N;
        P.modes = S.modes;
        bool any_quad = false;
        for (int j = 0; j < nj; ++j) {
            const OzSliceJob& s = jobs[j0 + j];
            if (!s.X || !s.maxbits || s.quad_slot >= S.nq || s.rows_slot >= S.nr || (s.quad_slot < 0 && s.rows_slot < 0))
                return cudaErrorInvalidValue;
            SliceJobDev& d = P.job[j];
            d.X = reinterpret_cast<const double2*>(s.X);
            d.maxbits = s.maxbits;
            d.maxbits_stride = s.maxbits_stride;
            d.quad = s.quad_slot >= 0 ? S.quad + (size_t)s.quad_slot * S.quad_slot_bytes : nullptr;
            d.rows = s.rows_slot >= 0 ? S.rows + (size_t)s.rows_slot * S.rows_slot_bytes : nullptr;
            d.exps_q = s.quad_slot >= 0 ? S.exps_q + (size_t)s.quad_slot * S.modes : nullptr;
            d.exps_r = s.rows_slot >= 0 ? S.exps_r + (size_t)s.rows_slot * S.modes : nullptr;
            d.mirror_L = s.mirror ? f.L : 0;
            any_quad = any_quad || s.quad_slot >= 0;
        }
        const int groups = N * (any_quad ? (P.pitch_q >> 5) : ((N + 3) >> 2));   // jobs without a QUAD target leave the rest of the grid at once
        const int my = (S.modes + OZ_SLICE_MODES - 1) / OZ_SLICE_MODES;
        if (my > 65535) return cudaErrorInvalidValue;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)((groups + 255) / 256), (unsigned)my, (unsigned)nj);
        cfg.blockDim = dim3(256, 1, 1);
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        cudaError_t e = cudaLaunchKernelEx(&cfg, oz_slice_kernel, P);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

cudaError_t launch_ozaki_absmax(const FreqLayout& f, int modes, const double* X, unsigned long long* maxbits, cudaStream_t st) {
    const unsigned chunks = (unsigned)((f.NN + 256 * 8 - 1) / (256 * 8));
    oz_absmax_kernel<<<dim3(chunks, (unsigned)(modes < 65535 ? modes : 65535)), 256, 0, st>>>(reinterpret_cast<const double2*>(X),
                                                                                             maxbits, f.NN, modes);
    return cudaGetLastError();
}

// Up to OZ_MAX_GROUPS independent products M(p) = A~(p) B~(p) of the same shape in one launch, operands from the slots of
// the store (and, for the last N mod 32 <= 2 values of k, from the FP64 spectra they were cut from), epilogues as in
// nspt_zgemm.cu; pairs = true runs every tile on a CTA pair (tcgen05.mma.cta_group::2); clear (optional): clear_count per-mode
// maxima that the slicing pass before this launch has consumed are zeroed for the next transform
cudaError_t launch_ozaki_gemm(const FreqLayout& f, const OzStore& S, const OzGemmGroup* groups, int ngroups, cudaStream_t st,
                              bool pairs, unsigned long long* clear, int clear_count) {
    if (ngroups < 1 || ngroups > OZ_MAX_GROUPS) return cudaErrorInvalidValue;
    return pairs ? launch_oz<2>(f, S, groups, ngroups, st, clear, clear_count) : launch_oz<1>(f, S, groups, ngroups, st, clear, clear_count);
}

}  // namespace nspt
