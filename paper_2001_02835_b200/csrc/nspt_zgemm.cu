// nspt_zgemm.cu -- Step 3 of FFT-CONV: the Fourier-mode-wise matrix product
//     C~(p) = A~(p) B~(p),   p = 0..L-1                          (eq. 2.8)
// one dense N x N x N complex FP64 product per mode, batched over modes.  The paper
// finds this step dominant on the GPU (cublasZgemm on streams).  Here it is one
// hand-written sm_100a kernel for all modes; no cuBLAS.
//
// Arithmetic.  tcgen05.mma has no FP64 kind, so the FP64 tensor path on sm_100a is the warp-level
// mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4); measured on B200 it sustains the full FP64 pipe rate
// (37.2 TFLOP/s at 1965 MHz) with 1/8 of the instructions of a DFMA kernel.  The complex product
// uses the 3-multiplication form on the interleaved (re, im) operands:
//     P1 = Ar Br,  P2 = Ai Bi,  P3 = (Ar+Ai)(Br+Bi);   Cr = P1 - P2,  Ci = P3 - P1 - P2
// (6 N^3 real flops instead of 8 N^3; normwise stable).  The sums Ar+Ai, Br+Bi are formed on the
// register fragments (6 DADD per 27 DMMA).
// This kernel runs the staple, the exponential and every product below N = 192; from there on
// nspt_series_mul and friends use the INT8 tensor-core path of nspt_ozaki.cu (same epilogues).
//
// Tiling.  Tiling A: CTA tile 48 x 48, four warps in 2 x 2, warp tile 24 x 24 = 3 x 3 DMMA blocks and
// three accumulator sets (108 registers); 128 threads and 159 registers per thread let three CTAs
// share an SM (12 warps, 3 per scheduler).  Tiling B: 32 x 32, warp tile 16 x 16, five CTAs per SM,
// chosen where the 8-row blocks of N do not fill the last 48-tile.  Operands arrive through TMA (cp.async.bulk.tensor, mbarrier
// complete_tx) in a ring of K-slices of 8; the refill of a slice is issued by the warps in turn, two
// iterations after the slice was consumed, so nobody waits on it.  Out-of-range rows / columns / k
// are zero-filled by TMA, so N need not be a multiple of anything; fully out-of-range 8-row /
// 8-column blocks of edge tiles are skipped (warp-uniform), and so is the odd half of the last slice.
//
// Shared-memory layout: every operand row is 8 complex128 = 128 bytes, written by TMA with
// SWIZZLE_128B (16-byte chunk index XOR row index mod 8).  A slice: [m 0..47][k 0..7]; B slice: six
// blocks [k 0..7][n 0..7], fetched by ONE box of a 4-D view of the operand (encode_operand_b4: two TMA
// instructions per slice; seven, one per block, cost 2.4 % of the kernel).  Lane (g = lane/4, t = lane%4) loads one complex element (re, im) per
// fragment with a 16-byte ld.shared; a slice is consumed as two k4 sub-steps whose k-slots are
// {0,2,4,6} and {1,3,5,7} (any k permutation is legal as long as A and B agree), which makes the
// eight lanes of every quarter-warp hit eight different 16-byte chunks: no bank conflicts.
#include <cuda.h>
#include "nspt_internal.cuh"
#include "nspt_tma.cuh"

namespace nspt {
namespace {

constexpr int BK = 8;
constexpr int B_BOX_BYTES = BK * 8 * 16;                       // 1024: [k][8 complex]

// Tiling of one kernel instance: a warp owns MB x NB DMMA blocks (8 MB rows x 8 NB columns), the CTA has
// WM x WN warps, MINB CTAs share an SM, the operand ring is NSTAGES K-slices deep.
template <int MB_, int NB_, int WM_, int WN_, int MINB_, int NSTAGES_, int LAG_ = 2>
struct Tile {
    static constexpr int LAG = LAG_;
    static constexpr int MB = MB_, NB = NB_, WM = WM_, WN = WN_, MINB = MINB_, STAGES = NSTAGES_;
    static constexpr int WARPS = WM * WN;
    static constexpr int THREADS = 32 * WARPS;
    static constexpr int BM = 8 * MB * WM, BN = 8 * NB * WN;
    static constexpr int A_STAGE_BYTES = BM * BK * 16;             // [m][8 complex]
    static constexpr int B_STAGE_BYTES = (BN / 8) * B_BOX_BYTES;   // BN/8 boxes [k][8 complex]
    static constexpr int STAGE_BYTES = A_STAGE_BYTES + B_STAGE_BYTES;
    static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 2 * STAGES * 8 + 1024;  // + barriers + alignment slack
    static_assert((WARPS & (WARPS - 1)) == 0, "warp count must be a power of two");
    static_assert(BM <= 256 && A_STAGE_BYTES % 1024 == 0, "A box");
};

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn g_encode = nullptr;

__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};"
        : "+d"(c0), "+d"(c1)
        : "d"(a), "d"(b));
}

// One product of a launch: modes [aoff, aoff + nmodes) of the A tensor map times modes [boff, ...) of the B map.
// *dst += v without reading it back (RED.E.ADD.F64)
__device__ __forceinline__ void red_add(double2& dst, double2 v) {
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(&dst.x), "d"(v.x) : "memory");
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(&dst.y), "d"(v.y) : "memory");
}

__device__ __forceinline__ uint64_t l2_keep_policy() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void st_keep(double2& dst, double2 v, uint64_t policy) {
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(&dst), "d"(v.x), "d"(v.y), "l"(policy) : "memory");
}

struct GemmGroupDev {
    double2* C;   // direct target:   C(p)            (+)= alpha * A(p) B(p) + diag   (may be null)
    double2* D;   // daggered target: D((L-p) mod L)  (+)= beta * (A(p) B(p))^H       (may be null)
    int aoff, boff;
    double alpha_re, alpha_im;
    double beta_re, beta_im;
    double diag;   // added to the diagonal of C after alpha
    int accumulate, accumulate_d;
};
constexpr int MAX_GROUPS = 12;

// Independent products of the same shape share one launch (the staple has up to twelve at a time): the grid is
// ngroups x nmodes x tiles, so a launch of g products has g times the waves and 1/g of the tail of a single one.
struct GemmParams {
    size_t NN;
    int N, L;
    int tiles_m, tiles_n;
    int nmodes;    // modes per group (batch * L)
    int ngroups;
    // Naive-CONV: the operands are the series themselves ("mode" = order index, n per batch element) and the
    // product of order k is ONE matrix product with the K dimension concatenated over l = 0..k, A^(l) against B^(k-l).
    int conv;      // 0 = mode-wise product, 1 = convolution over the order index
    int n;         // coefficients per series (conv only)
    GemmGroupDev g[MAX_GROUPS];
};

// Which slice of which matrices K-slice j of a CTA reads.
struct SliceMap {
    int conv, nk_seg, modeA, modeB;   // conv: modeA = first coefficient of A, modeB = coefficient k of B (l = 0)
    __device__ __forceinline__ void coords(int j, int& k0, int& ma, int& mb) const {
        if (!conv) {
            k0 = j * 8;
            ma = modeA;
            mb = modeB;
        } else {
            const int l = j / nk_seg;
            k0 = (j - l * nk_seg) * 8;
            ma = modeA + l;
            mb = modeB - l;
        }
    }
};

template <class TC>
__device__ __forceinline__ void issue_slice(const CUtensorMap* mapA, const CUtensorMap* mapB, uint32_t stage_addr,
                                            uint32_t full_bar, int k0, int m0, int n0, int modeA, int modeB) {
    mbar_expect_tx(full_bar, TC::STAGE_BYTES);
    tma_load_3d(stage_addr, mapA, full_bar, 2 * k0, m0, modeA);
    tma_load_4d(stage_addr + TC::A_STAGE_BYTES, mapB, full_bar, 0, k0, n0 / 8, modeB);
}
// The same slice with the B operand fetched as BN/8 boxes of a plain 3-D map (columns beyond N are zero-filled, nothing
// beyond the operand is touched): used when B is a caller's array (Naive-CONV), which has no pad behind its last row.
template <class TC>
__device__ __forceinline__ void issue_slice_b3(const CUtensorMap* mapA, const CUtensorMap* mapB, uint32_t stage_addr,
                                               uint32_t full_bar, int k0, int m0, int n0, int modeA, int modeB) {
    mbar_expect_tx(full_bar, TC::STAGE_BYTES);
    tma_load_3d(stage_addr, mapA, full_bar, 2 * k0, m0, modeA);
#pragma unroll
    for (int c = 0; c < TC::BN / 8; ++c)
        tma_load_3d(stage_addr + TC::A_STAGE_BYTES + c * B_BOX_BYTES, mapB, full_bar, 2 * (n0 + 8 * c), k0, modeB);
}
template <class TC>
__device__ __forceinline__ void issue_mapped(const CUtensorMap* mapA, const CUtensorMap* mapB, uint32_t stage_addr, uint32_t full_bar,
                                             const SliceMap& sm, int j, int m0, int n0) {
    int k0, ma, mb;
    sm.coords(j, k0, ma, mb);
    if (sm.conv)
        issue_slice_b3<TC>(mapA, mapB, stage_addr, full_bar, k0, m0, n0, ma, mb);
    else
        issue_slice<TC>(mapA, mapB, stage_addr, full_bar, k0, m0, n0, ma, mb);
}

template <class TC, bool FULL>
__device__ __forceinline__ void gemm_mainloop(const CUtensorMap& mapA, const CUtensorMap& mapB, const GemmParams& P,
                                              uint32_t base, const uint8_t* sgen, uint32_t bar_full, uint32_t bar_empty,
                                              int warp, int lane, int nk, int m0, int n0, const SliceMap smap, int nbm,
                                              int nbn,
                                              uint32_t offA0, uint32_t offA1, uint32_t offB0, uint32_t offB1,
                                              double (&p1)[TC::MB][TC::NB][2], double (&p2)[TC::MB][TC::NB][2],
                                              double (&p3)[TC::MB][TC::NB][2]) {
    constexpr int MB = TC::MB, NB = TC::NB, STAGES = TC::STAGES, STAGE_BYTES = TC::STAGE_BYTES;
    const int N = P.N;
    const bool active = FULL || ((nbm > 0) && (nbn > 0));
    int seg_it = 0;   // slice index inside the current K segment (one segment unless conv)
    for (int it = 0; it < nk; ++it) {
        // keep the four fragment offsets in registers (ptxas otherwise rematerialises them from the lane and
        // CTA indices inside every sub-step, ~20 dependent integer instructions in front of the loads)
        asm volatile("" : "+r"(offA0), "+r"(offA1), "+r"(offB0), "+r"(offB1));
        const int slot = it % STAGES;
        mbar_wait(bar_full + 8 * slot, (it / STAGES) & 1);
        if (active) {
            const uint8_t* st = sgen + slot * STAGE_BYTES;
            const int nsub = (seg_it * BK + 1 < N) ? 2 : 1;  // odd k-slots of the last slice may all be padding
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                if (s < nsub) {
                    double2 a[MB], b[NB];
                    double as[MB], bs[NB];
#pragma unroll
                    for (int bm = 0; bm < MB; ++bm) {
                        a[bm] = *reinterpret_cast<const double2*>(st + (s ? offA1 : offA0) + bm * 1024);
                        as[bm] = a[bm].x + a[bm].y;
                    }
#pragma unroll
                    for (int bn = 0; bn < NB; ++bn) {
                        b[bn] = *reinterpret_cast<const double2*>(st + (s ? offB1 : offB0) + bn * B_BOX_BYTES);
                        bs[bn] = b[bn].x + b[bn].y;
                    }
#pragma unroll
                    for (int bm = 0; bm < MB; ++bm) {
                        if (FULL || bm < nbm) {
#pragma unroll
                            for (int bn = 0; bn < NB; ++bn) {
                                if (FULL || bn < nbn) {
                                    dmma(p1[bm][bn][0], p1[bm][bn][1], a[bm].x, b[bn].x);
                                    dmma(p2[bm][bn][0], p2[bm][bn][1], a[bm].y, b[bn].y);
                                    dmma(p3[bm][bn][0], p3[bm][bn][1], as[bm], bs[bn]);
                                }
                            }
                        }
                    }
                }
            }
        }
        if (++seg_it == smap.nk_seg) seg_it = 0;
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8 * slot);
        if (it + 1 >= TC::LAG && warp == ((it + 1) & (TC::WARPS - 1))) {
            // refill of the slot released LAG iterations ago, by the warps in turn: by then even the slowest warp
            // has released it, so the wait below does not block (LAG = 1 or a refill by the last arriver costs 5 %)
            const int j = it + 1 - TC::LAG;
            if (j + STAGES < nk && lane == 0) {
                const int sl = j % STAGES;
                mbar_wait(bar_empty + 8 * sl, (j / STAGES) & 1);
                issue_mapped<TC>(&mapA, &mapB, base + sl * STAGE_BYTES, bar_full + 8 * sl, smap, j + STAGES, m0, n0);
            }
            __syncwarp();
        }
    }
}

// Epilogue of one warp: C = alpha AB (+ diag 1), C += alpha AB, and / or the conjugate-transposed (accumulating) store into
// the mirrored mode (the spectrum of the daggered product series, FFT[X^+](p') = (X~(p))^H with p' = (L - p) mod L).
template <class TC>
__device__ __forceinline__ void gemm_epilogue(const GemmParams& P, const GemmGroupDev& G, int mode, int m0, int n0, int mw, int nw,
                                              int nbm, int nbn, int g, int t, double (&p1)[TC::MB][TC::NB][2],
                                              double (&p2)[TC::MB][TC::NB][2], double (&p3)[TC::MB][TC::NB][2]) {
    constexpr int MB = TC::MB, NB = TC::NB;
    const int N = P.N;
    double2* Cm = G.C ? G.C + (size_t)mode * P.NN : nullptr;
    const int pm = mode % P.L;
    double2* Dm = G.D ? G.D + (size_t)(mode - pm + ((P.L - pm) % P.L)) * P.NN : nullptr;
    const double alpha_re = G.alpha_re, alpha_im = G.alpha_im, beta_re = G.beta_re, beta_im = G.beta_im;
    const int accumulate = G.accumulate, accumulate_d = G.accumulate_d;
    const double diag = G.diag;
    const uint64_t keep = l2_keep_policy();
#pragma unroll
    for (int bm = 0; bm < MB; ++bm) {
        const int m = m0 + mw + 8 * bm + g;
        if (bm < nbm && m < N) {
#pragma unroll
            for (int bn = 0; bn < NB; ++bn) {
                const int n = n0 + nw + 8 * bn + 2 * t;
                if (bn < nbn && n < N) {
                    const double cr0 = p1[bm][bn][0] - p2[bm][bn][0];
                    const double cr1 = p1[bm][bn][1] - p2[bm][bn][1];
                    const double ci0 = p3[bm][bn][0] - p1[bm][bn][0] - p2[bm][bn][0];
                    const double ci1 = p3[bm][bn][1] - p1[bm][bn][1] - p2[bm][bn][1];
                    const bool second = (n + 1 < N);
                    if (Cm) {
                        double2 o0 = make_double2(alpha_re * cr0 - alpha_im * ci0, alpha_re * ci0 + alpha_im * cr0);
                        double2 o1 = make_double2(alpha_re * cr1 - alpha_im * ci1, alpha_re * ci1 + alpha_im * cr1);
                        if (m == n) o0.x += diag;
                        if (m == n + 1) o1.x += diag;
                        double2* d = Cm + (size_t)m * N + n;
                        if (accumulate) {
                            // fire-and-forget reductions: every element receives exactly one contribution per launch
                            // (deterministic), and nothing waits for the old value to come back from L2 / HBM
                            red_add(d[0], o0);
                            if (second) red_add(d[1], o1);
                        } else {   // the transform that follows reads this spectrum at once: the lines stay in the L2 while they can
                            st_keep(d[0], o0, keep);
                            if (second) st_keep(d[1], o1, keep);
                        }
                    }
                    if (Dm) {
                        // beta * conj(c): the eight lanes g = 0..7 of a quarter-warp write 128 contiguous bytes
                        double2 o0 = make_double2(beta_re * cr0 + beta_im * ci0, beta_im * cr0 - beta_re * ci0);
                        double2 o1 = make_double2(beta_re * cr1 + beta_im * ci1, beta_im * cr1 - beta_re * ci1);
                        double2* d0 = Dm + (size_t)n * N + m;
                        double2* d1 = d0 + N;
                        if (accumulate_d) {
                            red_add(*d0, o0);
                            if (second) red_add(*d1, o1);
                        } else {
                            *d0 = o0;
                            if (second) *d1 = o1;
                        }
                    }
                }
            }
        }
    }
}

template <class TC>
__global__ void __launch_bounds__(TC::THREADS, TC::MINB)
zgemm_modes_dmma_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB,
                        const GemmParams P) {
    constexpr int MB = TC::MB, NB = TC::NB, STAGES = TC::STAGES, STAGE_BYTES = TC::STAGE_BYTES;
    constexpr int BM = TC::BM, BN = TC::BN;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint8_t* sgen = smem_raw + (base - smem_u32(smem_raw));  // same address, generic-shared pointer for loads
    const uint32_t bar_full = base + STAGES * STAGE_BYTES;
    const uint32_t bar_empty = bar_full + STAGES * 8;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tiles = P.tiles_m * P.tiles_n;
    const int grp = blockIdx.x / (tiles * P.nmodes);
    const int rest = blockIdx.x % (tiles * P.nmodes);
    int mode = rest / tiles;          // mode inside the group
    const int tile = rest % tiles;
    const int m0 = (tile / P.tiles_n) * BM, n0 = (tile % P.tiles_n) * BN;
    const int N = P.N;
    const GemmGroupDev& G = P.g[grp];
    SliceMap smap;
    smap.conv = P.conv;
    smap.nk_seg = (N + BK - 1) / BK;
    int nk = smap.nk_seg;
    if (P.conv) {
        // order k of batch element b; the heavy high orders come first in the grid, the light ones fill its tail
        const int b = mode / P.n, k = P.n - 1 - mode % P.n;
        mode = b * P.n + k;            // where the result goes
        nk = (k + 1) * smap.nk_seg;    // K runs over A^(0..k) against B^(k..0)
        smap.modeA = G.aoff + b * P.n;
        smap.modeB = G.boff + b * P.n + k;
    } else {
        smap.modeA = G.aoff + mode;
        smap.modeB = G.boff + mode;
    }

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, TC::WARPS);
        }
        mbar_fence_init();
    }
    pdl_wait();      // the set-up above overlaps the tail of the previous kernel of the stream
    pdl_trigger();
    if (threadIdx.x == 0) {
        const int pre = nk < STAGES ? nk : STAGES;
        for (int it = 0; it < pre; ++it)
            issue_mapped<TC>(&mapA, &mapB, base + it * STAGE_BYTES, bar_full + 8 * it, smap, it, m0, n0);
    }
    __syncthreads();

    const int g = lane >> 2, t = lane & 3;
    // Part of the CTA tile this warp owns.  Edge tiles give the warps unequal work (out-of-range 8-blocks are
    // skipped) and warp w always runs on scheduler w % 4 of its SM, each with its own DMMA pipe: rotating the
    // assignment with the CTA index spreads the light parts over the four schedulers.
    const int quad = (warp + blockIdx.x) & (TC::WARPS - 1);
    const int wm = quad / TC::WN, wn = quad % TC::WN;
    const int mw = 8 * MB * wm, nw = 8 * NB * wn;  // warp offsets inside the CTA tile
    // number of 8-row / 8-column blocks of this warp that intersect the matrix
    int nbm = (N - (m0 + mw) + 7) >> 3;
    nbm = nbm < 0 ? 0 : (nbm > MB ? MB : nbm);
    int nbn = (N - (n0 + nw) + 7) >> 3;
    nbn = nbn < 0 ? 0 : (nbn > NB ? NB : nbn);
    const bool active = (nbm > 0) && (nbn > 0);

    double p1[MB][NB][2], p2[MB][NB][2], p3[MB][NB][2];
#pragma unroll
    for (int i = 0; i < MB; ++i)
#pragma unroll
        for (int j = 0; j < NB; ++j) {
            p1[i][j][0] = p1[i][j][1] = 0.0;
            p2[i][j][0] = p2[i][j][1] = 0.0;
            p3[i][j][0] = p3[i][j][1] = 0.0;
        }

    // per-lane byte offsets of the fragment loads inside a stage (sub-step 0; sub-step 1 is derived)
    const uint32_t offA0 = (uint32_t)((mw + g) * 128 + (((2 * t) ^ g) << 4));           // + bm*1024
    const uint32_t offA1 = offA0 ^ 16u;                                                   // k-slot 2t+1
    const uint32_t offB0 =
        (uint32_t)(TC::A_STAGE_BYTES + (NB * wn) * B_BOX_BYTES + (2 * t) * 128 + ((g ^ (2 * t)) << 4));  // + bn*1024
    const uint32_t offB1 = (offB0 + 128u) ^ 16u;                                          // row 2t+1

    // Warps whose MB x NB blocks all intersect the matrix (all but those on the last tile row / column) run
    // an unpredicated copy of the loop: predicated mma.sync costs a WARPSYNC and issue bubbles per group.
    if (nbm == MB && nbn == NB)
        gemm_mainloop<TC, true>(mapA, mapB, P, base, sgen, bar_full, bar_empty, warp, lane, nk, m0, n0, smap, MB, NB,
                                offA0, offA1, offB0, offB1, p1, p2, p3);
    else
        gemm_mainloop<TC, false>(mapA, mapB, P, base, sgen, bar_full, bar_empty, warp, lane, nk, m0, n0, smap, nbm,
                                 nbn, offA0, offA1, offB0, offB1, p1, p2, p3);

    if (!active) return;
    gemm_epilogue<TC>(P, G, mode, m0, n0, mw, nw, nbm, nbn, g, t, p1, p2, p3);
}

// ---------------------------------------------------------------------------------------------------------------------
// Persistent, warp-specialised form of the same product (one CTA per SM).  Warp group 0 holds the producers: warp q feeds
// consumer group q -- four warps that own one CTA tile at a time, exactly the warp tile and inner loop of the kernel
// above -- through a ring of its own.  What changes: (1) a producer runs up to STAGES slices ahead across tile boundaries,
// so a consumer group never waits for the first slices of its next tile, and no warp spends registers or issue slots on
// refill bookkeeping; (2) consumer group q of SM b walks the tiles q * SMs + b, + GROUPS * SMs, ... : all groups of all SMs
// stay within a window of GROUPS * SMs consecutive tiles (the same L2 locality as block-order scheduling), every SM gets
// the same number of tiles up to one, and the surplus tiles of the last round land on group 0 of different SMs, where
// each has an SM's FP64 pipe to itself; (3) the register file is split with setmaxnreg (producers 32, consumers 160).
template <class TC, bool FULL>
__device__ __forceinline__ void ws_consume_tile(const GemmParams& P, const uint8_t* ring, uint32_t bar_full, uint32_t bar_empty,
                                                int lane, int nk, int nbm, int nbn, uint32_t offA0, uint32_t offA1,
                                                uint32_t offB0, uint32_t offB1, uint32_t& slot, uint32_t& phase,
                                                double (&p1)[TC::MB][TC::NB][2], double (&p2)[TC::MB][TC::NB][2],
                                                double (&p3)[TC::MB][TC::NB][2]) {
    constexpr int MB = TC::MB, NB = TC::NB, STAGES = TC::STAGES, STAGE_BYTES = TC::STAGE_BYTES;
    const int N = P.N;
    const bool active = FULL || ((nbm > 0) && (nbn > 0));
    for (int it = 0; it < nk; ++it) {
        asm volatile("" : "+r"(offA0), "+r"(offA1), "+r"(offB0), "+r"(offB1));
        mbar_wait(bar_full + 8 * slot, phase);
        if (active) {
            const uint8_t* st = ring + slot * STAGE_BYTES;
            const int nsub = (it * BK + 1 < N) ? 2 : 1;  // odd k-slots of the last slice may all be padding
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                if (s < nsub) {
                    double2 a[MB], b[NB];
                    double as[MB], bs[NB];
#pragma unroll
                    for (int bm = 0; bm < MB; ++bm) {
                        a[bm] = *reinterpret_cast<const double2*>(st + (s ? offA1 : offA0) + bm * 1024);
                        as[bm] = a[bm].x + a[bm].y;
                    }
#pragma unroll
                    for (int bn = 0; bn < NB; ++bn) {
                        b[bn] = *reinterpret_cast<const double2*>(st + (s ? offB1 : offB0) + bn * B_BOX_BYTES);
                        bs[bn] = b[bn].x + b[bn].y;
                    }
                    if constexpr (FULL) {
#pragma unroll
                        for (int bm = 0; bm < MB; ++bm)
#pragma unroll
                            for (int bn = 0; bn < NB; ++bn) {
                                dmma(p1[bm][bn][0], p1[bm][bn][1], a[bm].x, b[bn].x);
                                dmma(p2[bm][bn][0], p2[bm][bn][1], a[bm].y, b[bn].y);
                                dmma(p3[bm][bn][0], p3[bm][bn][1], as[bm], bs[bn]);
                            }
                    } else {
#pragma unroll
                        for (int bm = 0; bm < MB; ++bm)
                            if (bm < nbm) {
#pragma unroll
                                for (int bn = 0; bn < NB; ++bn)
                                    if (bn < nbn) {
                                        dmma(p1[bm][bn][0], p1[bm][bn][1], a[bm].x, b[bn].x);
                                        dmma(p2[bm][bn][0], p2[bm][bn][1], a[bm].y, b[bn].y);
                                        dmma(p3[bm][bn][0], p3[bm][bn][1], as[bm], bs[bn]);
                                    }
                            }
                    }
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8 * slot);
        if (++slot == STAGES) {
            slot = 0;
            phase ^= 1u;
        }
    }
}

template <class TC, int GROUPS, int PRODUCER_REGS, int CONSUMER_REGS>
__global__ void __launch_bounds__(128 * (GROUPS + 1), 1)
zgemm_modes_dmma_ws_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB,
                           const GemmParams P) {
    constexpr int MB = TC::MB, NB = TC::NB, STAGES = TC::STAGES, STAGE_BYTES = TC::STAGE_BYTES;
    constexpr int BM = TC::BM, BN = TC::BN;
    constexpr int RING_BYTES = STAGES * STAGE_BYTES;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint8_t* sgen = smem_raw + (base - smem_u32(smem_raw));
    const uint32_t bars = base + GROUPS * RING_BYTES;   // per group: STAGES full barriers, then STAGES empty barriers

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int wg = warp >> 2;
    const int tiles = P.tiles_m * P.tiles_n;
    const int per_product = tiles * P.nmodes;
    const int total = P.ngroups * per_product;
    const int stride = GROUPS * (int)gridDim.x;
    const int N = P.N;
    const int nk = (N + BK - 1) / BK;

    if (threadIdx.x == 0) {
        for (int q = 0; q < GROUPS; ++q)
            for (int s = 0; s < STAGES; ++s) {
                mbar_init(bars + (q * 2 * STAGES + s) * 8, 1);
                mbar_init(bars + (q * 2 * STAGES + STAGES + s) * 8, TC::WARPS);
            }
        mbar_fence_init();
    }
    pdl_wait();
    pdl_trigger();
    __syncthreads();

    if (wg == 0) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(PRODUCER_REGS));
        if (warp < GROUPS && lane == 0) {
            const uint32_t ring = base + warp * RING_BYTES;
            const uint32_t bar_full = bars + warp * 2 * STAGES * 8, bar_empty = bar_full + STAGES * 8;
            uint32_t slot = 0, phase = 0;
            for (int tl = warp * (int)gridDim.x + (int)blockIdx.x; tl < total; tl += stride) {
                const int grp = tl / per_product, rest = tl - grp * per_product;
                const int mode = rest / tiles, tile = rest - mode * tiles;
                const int m0 = (tile / P.tiles_n) * BM, n0 = (tile % P.tiles_n) * BN;
                const int modeA = P.g[grp].aoff + mode, modeB = P.g[grp].boff + mode;
                for (int it = 0; it < nk; ++it) {
                    mbar_wait(bar_empty + 8 * slot, phase ^ 1u);
                    issue_slice<TC>(&mapA, &mapB, ring + slot * STAGE_BYTES, bar_full + 8 * slot, it * BK, m0, n0, modeA, modeB);
                    if (++slot == STAGES) {
                        slot = 0;
                        phase ^= 1u;
                    }
                }
            }
        }
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(CONSUMER_REGS));
    const int q = wg - 1, w4 = warp & 3;
    const uint8_t* ring = sgen + q * RING_BYTES;
    const uint32_t bar_full = bars + q * 2 * STAGES * 8, bar_empty = bar_full + STAGES * 8;
    const int g = lane >> 2, t = lane & 3;
    uint32_t slot = 0, phase = 0;
    for (int tl = q * (int)gridDim.x + (int)blockIdx.x; tl < total; tl += stride) {
        const int grp = tl / per_product, rest = tl - grp * per_product;
        const int mode = rest / tiles, tile = rest - mode * tiles;
        const int m0 = (tile / P.tiles_n) * BM, n0 = (tile % P.tiles_n) * BN;
        // rotate the warp -> quarter-tile assignment with the tile: edge tiles give the warps unequal work
        const int quad = (w4 + tl) & (TC::WARPS - 1);
        const int wm = quad / TC::WN, wn = quad % TC::WN;
        const int mw = 8 * MB * wm, nw = 8 * NB * wn;
        int nbm = (N - (m0 + mw) + 7) >> 3;
        nbm = nbm < 0 ? 0 : (nbm > MB ? MB : nbm);
        int nbn = (N - (n0 + nw) + 7) >> 3;
        nbn = nbn < 0 ? 0 : (nbn > NB ? NB : nbn);
        double p1[MB][NB][2], p2[MB][NB][2], p3[MB][NB][2];
#pragma unroll
        for (int i = 0; i < MB; ++i)
#pragma unroll
            for (int j = 0; j < NB; ++j) {
                p1[i][j][0] = p1[i][j][1] = 0.0;
                p2[i][j][0] = p2[i][j][1] = 0.0;
                p3[i][j][0] = p3[i][j][1] = 0.0;
            }
        const uint32_t offA0 = (uint32_t)((mw + g) * 128 + (((2 * t) ^ g) << 4));
        const uint32_t offA1 = offA0 ^ 16u;
        const uint32_t offB0 =
            (uint32_t)(TC::A_STAGE_BYTES + (NB * wn) * B_BOX_BYTES + (2 * t) * 128 + ((g ^ (2 * t)) << 4));
        const uint32_t offB1 = (offB0 + 128u) ^ 16u;
        if (nbm == MB && nbn == NB)
            ws_consume_tile<TC, true>(P, ring, bar_full, bar_empty, lane, nk, nbm, nbn, offA0, offA1, offB0, offB1, slot, phase, p1,
                                      p2, p3);
        else
            ws_consume_tile<TC, false>(P, ring, bar_full, bar_empty, lane, nk, nbm, nbn, offA0, offA1, offB0, offB1, slot, phase, p1,
                                       p2, p3);
        if (nbm > 0 && nbn > 0) gemm_epilogue<TC>(P, P.g[grp], mode, m0, n0, mw, nw, nbm, nbn, g, t, p1, p2, p3);
    }
}

// Reference kernel (variant 0): one thread per output element, conventional 4-multiplication
// complex product with plain FMAs.  For debugging the tensor-core kernel; never the default.
__global__ void __launch_bounds__(256)
zgemm_modes_ref_kernel(const double2* __restrict__ A, const double2* __restrict__ B, const GemmGroupDev G, int N, size_t NN,
                       int L, int modes) {
    const int j = blockIdx.x * 16 + (threadIdx.x & 15);
    const int i = blockIdx.y * 16 + (threadIdx.x >> 4);
    if (i >= N || j >= N) return;
    for (int mode = blockIdx.z; mode < modes; mode += gridDim.z) {   // the grid's z extent is capped at 65535
    const double2* Am = A + (size_t)mode * NN;
    const double2* Bm = B + (size_t)mode * NN;
    double cr = 0.0, ci = 0.0;
    for (int k = 0; k < N; ++k) {
        const double2 a = Am[(size_t)i * N + k];
        const double2 b = Bm[(size_t)k * N + j];
        cr += a.x * b.x - a.y * b.y;
        ci += a.x * b.y + a.y * b.x;
    }
    if (G.C) {
        double2 out = make_double2(G.alpha_re * cr - G.alpha_im * ci, G.alpha_re * ci + G.alpha_im * cr);
        if (i == j) out.x += G.diag;
        double2* c = G.C + (size_t)mode * NN + (size_t)i * N + j;
        if (G.accumulate) {
            out.x += c->x;
            out.y += c->y;
        }
        *c = out;
    }
    if (G.D) {
        const int pm = mode % L;
        double2 out = make_double2(G.beta_re * cr + G.beta_im * ci, G.beta_im * cr - G.beta_re * ci);
        double2* d = G.D + (size_t)(mode - pm + ((L - pm) % L)) * NN + (size_t)j * N + i;
        if (G.accumulate_d) {
            out.x += d->x;
            out.y += d->y;
        }
        *d = out;
    }
    }
}

// 3-D view of a spectrum as doubles: (2N doubles per row, N rows, modes); boxes are 16 doubles wide
// (8 complex = 128 bytes, the swizzle span).
// B operand as (16 doubles of one 128-byte chunk, N rows, ceil(2N/16) chunks per row, modes): one box (16, 8, BN/8, 1)
// brings the BN/8 chunk columns of a K-slice with ONE instruction, laid out [chunk][k][8 complex] exactly like BN/8
// separate boxes.  The last chunk of a row runs into the next row (columns >= N of the tile hold garbage that only
// reaches output columns >= N, which are never stored); the caller's buffer must extend 128 bytes past the last row.
cudaError_t encode_operand_b4(CUtensorMap* map, const double* basep, const FreqLayout& f, int modes, int chunks_box) {
    const uint64_t dims[4] = {16, (uint64_t)f.N, (uint64_t)((2 * f.N + 15) / 16), (uint64_t)modes};
    const uint64_t strides[3] = {(uint64_t)f.N * 16, 128, (uint64_t)f.NN * 16};
    const uint32_t box[4] = {16, (uint32_t)BK, (uint32_t)chunks_box, 1};
    return tma_encode_f64(map, basep, 4, dims, strides, box, true);
}

cudaError_t encode_operand(CUtensorMap* map, const double* basep, const FreqLayout& f, int modes, int box_rows) {
    const uint64_t dims[3] = {(uint64_t)(2 * f.N), (uint64_t)f.N, (uint64_t)modes};
    const uint64_t strides[2] = {(uint64_t)f.N * 16, (uint64_t)f.NN * 16};
    const uint32_t box[3] = {16, (uint32_t)box_rows, 1};
    return tma_encode_f64(map, basep, 3, dims, strides, box, true);
}

}  // namespace

// A tensor map depends only on (pointer, shape, strides, box, swizzle); encoding one costs 1-2 us of host time and a product
// needs eight, which is most of the host cost of a small product.  Repeated calls on the same buffers (the normal case in an
// NSPT run) therefore reuse the last encodings: a small per-thread cache, most recently used first.
namespace {
struct MapKey {
    const void* base;
    int rank;
    int swizzle;
    uint64_t dims[4];
    uint64_t strides[3];
    uint32_t box[4];
    bool operator==(const MapKey& o) const {
        if (base != o.base || rank != o.rank || swizzle != o.swizzle) return false;
        for (int i = 0; i < 4; ++i)
            if (dims[i] != o.dims[i] || box[i] != o.box[i]) return false;
        for (int i = 0; i < 3; ++i)
            if (strides[i] != o.strides[i]) return false;
        return true;
    }
};
struct MapEntry {
    MapKey key;
    CUtensorMap map;
};
constexpr int MAP_CACHE = 48;
thread_local MapEntry t_maps[MAP_CACHE];
thread_local int t_nmaps = 0;
}  // namespace

cudaError_t tma_encode_f64(CUtensorMap* map, const void* base, int rank, const uint64_t* dims,
                           const uint64_t* strides_bytes, const uint32_t* box, bool swizzle128) {
    if (!g_encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
        if (e != cudaSuccess) return e;
        if (qres != cudaDriverEntryPointSuccess || !fn) return cudaErrorNotSupported;
        g_encode = reinterpret_cast<EncodeTiledFn>(fn);
    }
    MapKey key{};
    key.base = base;
    key.rank = rank;
    key.swizzle = swizzle128 ? 1 : 0;
    cuuint64_t d[4] = {1, 1, 1, 1}, st[3] = {16, 16, 16};
    cuuint32_t bx[4] = {1, 1, 1, 1}, es[4] = {1, 1, 1, 1};
    for (int i = 0; i < rank; ++i) {
        d[i] = dims[i];
        bx[i] = box[i];
    }
    for (int i = 0; i + 1 < rank; ++i) st[i] = strides_bytes[i];
    for (int i = 0; i < 4; ++i) {
        key.dims[i] = d[i];
        key.box[i] = bx[i];
    }
    for (int i = 0; i < 3; ++i) key.strides[i] = st[i];
    for (int i = 0; i < t_nmaps; ++i) {
        if (t_maps[i].key == key) {
            *map = t_maps[i].map;
            if (i > 0) {   // move to the front
                const MapEntry hit = t_maps[i];
                for (int j = i; j > 0; --j) t_maps[j] = t_maps[j - 1];
                t_maps[0] = hit;
            }
            return cudaSuccess;
        }
    }
    const CUresult r = g_encode(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, (cuuint32_t)rank, const_cast<void*>(base), d, st, bx, es,
                                CU_TENSOR_MAP_INTERLEAVE_NONE,
                                swizzle128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE,
                                CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
    if (t_nmaps < MAP_CACHE) ++t_nmaps;
    for (int j = t_nmaps - 1; j > 0; --j) t_maps[j] = t_maps[j - 1];
    t_maps[0].key = key;
    t_maps[0].map = *map;
    return cudaSuccess;
}

namespace {

template <class TC>
cudaError_t launch_dmma(const FreqLayout& f, const double* baseA, int modesA, const double* baseB, int modesB, GemmParams P,
                        cudaStream_t st) {
    static bool attr_done[NSPT_MAX_DEVICES] = {};   // the function attribute is per device
    cudaError_t e;
    const int dev = current_device();
    if (!attr_done[dev]) {
        e = cudaFuncSetAttribute(zgemm_modes_dmma_kernel<TC>, cudaFuncAttributeMaxDynamicSharedMemorySize, TC::SMEM_BYTES);
        if (e != cudaSuccess) return e;
        attr_done[dev] = true;
    }
    P.tiles_m = (f.N + TC::BM - 1) / TC::BM;
    P.tiles_n = (f.N + TC::BN - 1) / TC::BN;
    CUtensorMap mapA, mapB;
    if ((e = encode_operand(&mapA, baseA, f, modesA, TC::BM)) != cudaSuccess) return e;
    if (P.conv)   // a caller's array: plain 3-D map, one box per eight columns
        e = encode_operand(&mapB, baseB, f, modesB, BK);
    else
        e = encode_operand_b4(&mapB, baseB, f, modesB, TC::BN / 8);
    if (e != cudaSuccess) return e;
    const unsigned grid = (unsigned)(P.ngroups * P.nmodes * P.tiles_m * P.tiles_n);
    return launch_pdl(zgemm_modes_dmma_kernel<TC>, grid, TC::THREADS, TC::SMEM_BYTES, st, mapA, mapB, P);
}

template <class TC, int GROUPS, int PREGS, int CREGS>
cudaError_t launch_dmma_ws(const FreqLayout& f, const double* baseA, int modesA, const double* baseB, int modesB, GemmParams P,
                           cudaStream_t st) {
    constexpr int SMEM = GROUPS * TC::STAGES * TC::STAGE_BYTES + GROUPS * 2 * TC::STAGES * 8 + 1024;
    static bool attr_done[NSPT_MAX_DEVICES] = {};
    static int sms[NSPT_MAX_DEVICES] = {};
    cudaError_t e;
    const int dev = current_device();
    auto kern = zgemm_modes_dmma_ws_kernel<TC, GROUPS, PREGS, CREGS>;
    if (!attr_done[dev]) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
        if (e != cudaSuccess) return e;
        cudaDeviceGetAttribute(&sms[dev], cudaDevAttrMultiProcessorCount, dev);
        if (sms[dev] <= 0) sms[dev] = 148;
        attr_done[dev] = true;
    }
    P.tiles_m = (f.N + TC::BM - 1) / TC::BM;
    P.tiles_n = (f.N + TC::BN - 1) / TC::BN;
    CUtensorMap mapA, mapB;
    if ((e = encode_operand(&mapA, baseA, f, modesA, TC::BM)) != cudaSuccess) return e;
    if ((e = encode_operand_b4(&mapB, baseB, f, modesB, TC::BN / 8)) != cudaSuccess) return e;
    return launch_pdl(kern, (unsigned)sms[dev], 128 * (GROUPS + 1), SMEM, st, mapA, mapB, P);
}

GemmGroupDev to_dev(const GemmOut& out) {
    GemmGroupDev g{};
    g.C = reinterpret_cast<double2*>(out.C);
    g.D = reinterpret_cast<double2*>(out.D);
    g.alpha_re = out.alpha.re;
    g.alpha_im = out.alpha.im;
    g.beta_re = out.beta.re;
    g.beta_im = out.beta.im;
    g.diag = out.diag;
    g.accumulate = out.accumulate ? 1 : 0;
    g.accumulate_d = out.accumulate_d ? 1 : 0;
    return g;
}

}  // namespace

cudaError_t launch_zgemm_groups(const FreqLayout& f, int batch, const GemmGroup* groups, int ngroups, int variant,
                                cudaStream_t st) {
    const int modes = batch * f.L;
    if (ngroups < 1 || ngroups > MAX_GROUPS) return cudaErrorInvalidValue;
    for (int i = 0; i < ngroups; ++i)
        if (!groups[i].A || !groups[i].B || (!groups[i].out.C && !groups[i].out.D)) return cudaErrorInvalidValue;
    if (variant == 0) {
        for (int i = 0; i < ngroups; ++i) {
            dim3 grid((f.N + 15) / 16, (f.N + 15) / 16, modes < 65535 ? modes : 65535);
            zgemm_modes_ref_kernel<<<grid, 256, 0, st>>>(reinterpret_cast<const double2*>(groups[i].A),
                                                         reinterpret_cast<const double2*>(groups[i].B), to_dev(groups[i].out),
                                                         f.N, f.NN, f.L, modes);
            cudaError_t e = cudaGetLastError();
            if (e != cudaSuccess) return e;
        }
        return cudaSuccess;
    }
    if (variant != 1 && variant != 3) return cudaErrorInvalidValue;
    // one tensor map per operand side spans every group's spectrum: the groups address it by mode offset, so
    // their operands must sit a whole number of N x N matrices apart (spectra of one workspace always do)
    const double* baseA = groups[0].A;
    const double* baseB = groups[0].B;
    for (int i = 1; i < ngroups; ++i) {
        if (groups[i].A < baseA) baseA = groups[i].A;
        if (groups[i].B < baseB) baseB = groups[i].B;
    }
    GemmParams P{};
    P.NN = f.NN;
    P.N = f.N;
    P.L = f.L;
    P.nmodes = modes;
    P.ngroups = ngroups;
    const size_t mat = f.NN * 2;  // doubles per mode
    long long maxA = 0, maxB = 0;
    for (int i = 0; i < ngroups; ++i) {
        const size_t da = (size_t)(groups[i].A - baseA), db = (size_t)(groups[i].B - baseB);
        if (da % mat || db % mat) return cudaErrorInvalidValue;
        P.g[i] = to_dev(groups[i].out);
        P.g[i].aoff = (int)(da / mat);
        P.g[i].boff = (int)(db / mat);
        if ((long long)(da / mat) > maxA) maxA = (long long)(da / mat);
        if ((long long)(db / mat) > maxB) maxB = (long long)(db / mat);
    }
    // Two tilings.  A: 48 x 48 CTA tile, 4 warps of 24 x 24, 3 CTAs per SM -- the better inner loop (6 fragment loads
    // and 6 DADDs per 27 DMMAs); measured alternatives at N = 225, L = 128 (331 us): 64 x 48 / 8 warps of 16 x 24 / 2
    // CTAs 341 us, 48 x 64 / 8 warps of 24 x 16 354 us, 32 x 48 / 4 warps / 4 CTAs 338 us, 6-deep ring 331 us, 2 CTAs
    // with an 8-deep ring 359 us.  B: 32 x 32 CTA tile, 4 warps of 16 x 16, 5 CTAs per SM -- finer granularity.
    // Which one wins is decided by how the nb = ceil(N / 8) eight-blocks of a dimension fill the last tile: A when
    // they fill it (nb mod 6 = 0) or nearly (5, from nb = 29 up), B otherwise.  Measured per product at L = 64, A vs B in us:
    // N = 121: 67 / 48, 169: 119 / 111, 200: 172 / 156, 256: 306 / 268, 289: 449 / 430, 400: 988 / 979 (B wins);
    // N = 144: 72 / 74, 192: 122 / 126, 225: 213 / 226, 240: 220 / 244 (A wins); N = 184 (nb = 23): 126 / 121, hence nb >= 29 for the 'nearly' case.
    const int nb = (f.N + 7) / 8;
    if (variant == 3) return launch_dmma_ws<Tile<3, 3, 2, 2, 3, 5>, 3, 32, 160>(f, baseA, (int)maxA + modes, baseB, (int)maxB + modes, P, st);
    if (nb % 6 == 0 || (nb % 6 == 5 && nb >= 29))
        return launch_dmma<Tile<3, 3, 2, 2, 3, 5>>(f, baseA, (int)maxA + modes, baseB, (int)maxB + modes, P, st);
    return launch_dmma<Tile<2, 2, 2, 2, 5, 5>>(f, baseA, (int)maxA + modes, baseB, (int)maxB + modes, P, st);
}

// Naive-CONV (eq. 2.5 evaluated directly): C^(k) = sum_{l<=k} A^(l) B^(k-l) as ONE launch of the tensor-pipe
// kernel, each order a matrix product whose K dimension is concatenated over l.  No transforms, no workspace; N^3 n(n+1)/2
// multiplications instead of N^3 L, so it wins only for very low orders or launch-bound sizes.  C must not alias A or B.
cudaError_t launch_naive_conv(const FreqLayout& f, int batch, const nspt_c128* A, const nspt_c128* B, nspt_c128* C,
                              cudaStream_t st) {
    GemmParams P{};
    P.NN = f.NN;
    P.N = f.N;
    P.L = f.n;
    P.nmodes = batch * f.n;
    P.ngroups = 1;
    P.conv = 1;
    P.n = f.n;
    P.g[0].C = reinterpret_cast<double2*>(C);
    P.g[0].alpha_re = 1.0;
    const double* a = reinterpret_cast<const double*>(A);
    const double* b = reinterpret_cast<const double*>(B);
    const int nb = (f.N + 7) / 8;
    if (nb % 6 == 0 || (nb % 6 == 5 && nb >= 29))
        return launch_dmma<Tile<3, 3, 2, 2, 3, 5>>(f, a, P.nmodes, b, P.nmodes, P, st);
    return launch_dmma<Tile<2, 2, 2, 2, 5, 5>>(f, a, P.nmodes, b, P.nmodes, P, st);
}

cudaError_t launch_zgemm_modes(const FreqLayout& f, int batch, const double* A, const double* B, const GemmOut& out,
                               int variant, cudaStream_t st) {
    GemmGroup g;
    g.A = A;
    g.B = B;
    g.out = out;
    return launch_zgemm_groups(f, batch, &g, 1, variant, st);
}

}  // namespace nspt
