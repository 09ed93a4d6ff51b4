// nspt_zgemm.cu -- Step 3 of FFT-CONV: the Fourier-mode-wise matrix product
//     C~(p) = A~(p) B~(p),   p = 0..L-1                          (eq. 2.8)
// one dense N x N x N complex FP64 product per mode, batched over modes.  The paper
// finds this step dominant on the GPU (cublasZgemm on streams).  Here it is one
// hand-written sm_100a kernel for all modes; no cuBLAS.
//
// Arithmetic.  tcgen05.mma has no FP64 kind, so the FP64 tensor path on sm_100a is the warp-level
// mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4); measured on B200 it sustains the full FP64 pipe rate
// (37.2 TFLOP/s at 1965 MHz) with 1/8 of the instructions of a DFMA kernel.  The complex product
// uses the 3-multiplication form on planar operands:
//     P1 = Ar Br,  P2 = Ai Bi,  P3 = (Ar+Ai)(Br+Bi);   Cr = P1 - P2,  Ci = P3 - P1 - P2
// (6 N^3 real flops instead of 8 N^3; normwise stable).  The sums Ar+Ai, Br+Bi are formed on the
// register fragments (2 DADD per 9 DMMA).
//
// Tiling.  CTA tile 48 x 48, four consumer warps in 2 x 2, warp tile 24 x 24 = 3 x 3 DMMA blocks and
// three accumulator sets; one extra producer warp feeds a ring of K-slices of 8 through TMA
// (cp.async.bulk.tensor, mbarrier complete_tx).  Out-of-range rows / columns / k are zero-filled by
// TMA, so N need not be a multiple of anything; fully out-of-range 8-row / 8-column blocks of edge
// tiles are skipped (warp-uniform), and so is the odd half of the last K-slice.
//
// Shared-memory layouts are chosen so every fragment load is bank-conflict free:
//   A slice  [plane][m 0..47][k 0..7]            (64-byte rows, no swizzle).  Lane (g = lane/4, t = lane%4)
//            reads the pair A[m][2t], A[m][2t+1] with one 16-byte load; the slice is consumed as two
//            k4 sub-steps whose k-slots are {0,2,4,6} and {1,3,5,7} (any k permutation is legal as long
//            as A and B agree).
//   B slice  [chunk 0..2][plane][k 0..7][n 0..15] (128-byte rows, TMA SWIZZLE_128B).  Lane (g, t) reads
//            B[2t+s][n] with 8-byte loads; rows {0,2,4,6} (or {1,3,5,7}) XOR-swizzle onto disjoint banks.
#include <cuda.h>
#include "nspt_internal.cuh"

namespace nspt {
namespace {

constexpr int BM = 48, BN = 48, BK = 8;
constexpr int STAGES = 6;
constexpr int A_STAGE_BYTES = 2 * BM * BK * 8;                 // 6144
constexpr int B_CHUNK_BYTES = 2 * BK * 16 * 8;                 // 2048: [plane][k][16]
constexpr int B_STAGE_BYTES = (BN / 16) * B_CHUNK_BYTES;       // 6144
constexpr int STAGE_BYTES = A_STAGE_BYTES + B_STAGE_BYTES;     // 12288
constexpr int GEMM_THREADS = 160;                              // 4 consumer warps + 1 producer warp
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 2 * STAGES * 8 + 1024;  // + barriers + alignment slack

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn g_encode = nullptr;

// ---------------------------------------------------------------- PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(dst),
        "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}
__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};"
        : "+d"(c0), "+d"(c1)
        : "d"(a), "d"(b));
}

struct GemmParams {
    double* C;
    size_t ps;
    int N, ld;
    int tiles_m, tiles_n;
    double alpha_re, alpha_im;
    int accumulate;
};

__global__ void __launch_bounds__(GEMM_THREADS, 2)
zgemm_modes_dmma_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB,
                        const GemmParams P) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint8_t* sgen = smem_raw + (base - smem_u32(smem_raw));  // same address, generic-shared pointer for loads
    const uint32_t bar_full = base + STAGES * STAGE_BYTES;
    const uint32_t bar_empty = bar_full + STAGES * 8;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tiles = P.tiles_m * P.tiles_n;
    const int mode = blockIdx.x / tiles;
    const int tile = blockIdx.x % tiles;
    const int m0 = (tile / P.tiles_n) * BM, n0 = (tile % P.tiles_n) * BN;
    const int N = P.N;
    const int nk = (N + BK - 1) / BK;

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, 4);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == 4) {
        // ------------------------------------------------------------ producer
        if (lane == 0) {
            for (int it = 0; it < nk; ++it) {
                const int slot = it % STAGES;
                if (it >= STAGES) mbar_wait(bar_empty + 8 * slot, ((it / STAGES) - 1) & 1);
                const uint32_t full = bar_full + 8 * slot;
                mbar_expect_tx(full, STAGE_BYTES);
                const uint32_t sa = base + slot * STAGE_BYTES;
                const uint32_t sb = sa + A_STAGE_BYTES;
                const int k0 = it * BK;
                tma_load_3d(sa, &mapA, full, k0, m0, 2 * mode);
#pragma unroll
                for (int c = 0; c < BN / 16; ++c)
                    tma_load_3d(sb + c * B_CHUNK_BYTES, &mapB, full, n0 + 16 * c, k0, 2 * mode);
            }
        }
        return;
    }

    // ---------------------------------------------------------------- consumers
    const int g = lane >> 2, t = lane & 3;
    const int wm = warp >> 1, wn = warp & 1;
    const int mw = 24 * wm, nw = 24 * wn;  // warp offsets inside the CTA tile
    // number of 8-row / 8-column blocks of this warp that intersect the matrix
    int nbm = (N - (m0 + mw) + 7) >> 3;
    nbm = nbm < 0 ? 0 : (nbm > 3 ? 3 : nbm);
    int nbn = (N - (n0 + nw) + 7) >> 3;
    nbn = nbn < 0 ? 0 : (nbn > 3 ? 3 : nbn);
    const bool active = (nbm > 0) && (nbn > 0);

    double p1[3][3][2], p2[3][3][2], p3[3][3][2];
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            p1[i][j][0] = p1[i][j][1] = 0.0;
            p2[i][j][0] = p2[i][j][1] = 0.0;
            p3[i][j][0] = p3[i][j][1] = 0.0;
        }

    // per-lane constant byte offsets of the fragment loads inside a stage
    uint32_t offA[3];
#pragma unroll
    for (int bm = 0; bm < 3; ++bm) offA[bm] = (uint32_t)(((mw + 8 * bm + g) * BK + 2 * t) * 8);
    uint32_t offB[2][3];
#pragma unroll
    for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int bn = 0; bn < 3; ++bn) {
            const int k = 2 * t + s;
            const int n = nw + 8 * bn + g;
            const int chunk = n >> 4, n16 = n & 15;
            offB[s][bn] = (uint32_t)(A_STAGE_BYTES + chunk * B_CHUNK_BYTES + k * 128 + ((((n16 >> 1) ^ k) & 7) << 4) +
                                     (n16 & 1) * 8);
        }

    for (int it = 0; it < nk; ++it) {
        const int slot = it % STAGES;
        mbar_wait(bar_full + 8 * slot, (it / STAGES) & 1);
        if (active) {
            const uint8_t* st = sgen + slot * STAGE_BYTES;
            double2 ar[3], ai[3];
#pragma unroll
            for (int bm = 0; bm < 3; ++bm) {
                ar[bm] = *reinterpret_cast<const double2*>(st + offA[bm]);
                ai[bm] = *reinterpret_cast<const double2*>(st + offA[bm] + BM * BK * 8);
            }
            const int nsub = (it * BK + 1 < N) ? 2 : 1;  // odd k-slots of the last slice may all be padding
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                if (s < nsub) {
                    double br[3], bi[3], bs[3];
#pragma unroll
                    for (int bn = 0; bn < 3; ++bn) {
                        br[bn] = *reinterpret_cast<const double*>(st + offB[s][bn]);
                        bi[bn] = *reinterpret_cast<const double*>(st + offB[s][bn] + BK * 16 * 8);
                        bs[bn] = br[bn] + bi[bn];
                    }
#pragma unroll
                    for (int bm = 0; bm < 3; ++bm) {
                        if (bm < nbm) {
                            const double a_r = s ? ar[bm].y : ar[bm].x;
                            const double a_i = s ? ai[bm].y : ai[bm].x;
                            const double a_s = a_r + a_i;
#pragma unroll
                            for (int bn = 0; bn < 3; ++bn) {
                                if (bn < nbn) {
                                    dmma(p1[bm][bn][0], p1[bm][bn][1], a_r, br[bn]);
                                    dmma(p2[bm][bn][0], p2[bm][bn][1], a_i, bi[bn]);
                                    dmma(p3[bm][bn][0], p3[bm][bn][1], a_s, bs[bn]);
                                }
                            }
                        }
                    }
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8 * slot);
    }

    if (!active) return;
    // ---------------------------------------------------------------- epilogue
    double* Cr = P.C + (size_t)(2 * mode) * P.ps;
    double* Ci = Cr + P.ps;
#pragma unroll
    for (int bm = 0; bm < 3; ++bm) {
        const int m = m0 + mw + 8 * bm + g;
        if (bm < nbm && m < N) {
#pragma unroll
            for (int bn = 0; bn < 3; ++bn) {
                const int n = n0 + nw + 8 * bn + 2 * t;
                if (bn < nbn && n < N) {
                    double cr0 = p1[bm][bn][0] - p2[bm][bn][0];
                    double cr1 = p1[bm][bn][1] - p2[bm][bn][1];
                    double ci0 = p3[bm][bn][0] - p1[bm][bn][0] - p2[bm][bn][0];
                    double ci1 = p3[bm][bn][1] - p1[bm][bn][1] - p2[bm][bn][1];
                    double or0 = P.alpha_re * cr0 - P.alpha_im * ci0;
                    double oi0 = P.alpha_re * ci0 + P.alpha_im * cr0;
                    double or1 = P.alpha_re * cr1 - P.alpha_im * ci1;
                    double oi1 = P.alpha_re * ci1 + P.alpha_im * cr1;
                    double2* dr = reinterpret_cast<double2*>(Cr + (size_t)m * P.ld + n);
                    double2* di = reinterpret_cast<double2*>(Ci + (size_t)m * P.ld + n);
                    if (P.accumulate) {
                        const double2 oldr = *dr, oldi = *di;
                        or0 += oldr.x;
                        or1 += oldr.y;
                        oi0 += oldi.x;
                        oi1 += oldi.y;
                    }
                    *dr = make_double2(or0, or1);  // n+1 may be the first padding column (n+1 < ld): harmless
                    *di = make_double2(oi0, oi1);
                }
            }
        }
    }
}

// Reference kernel (variant 0): one thread per output element, conventional 4-multiplication
// complex product with plain FMAs.  For debugging the tensor-core kernel; never the default.
__global__ void __launch_bounds__(256)
zgemm_modes_ref_kernel(const double* __restrict__ A, const double* __restrict__ B, double* __restrict__ C, int N, int ld,
                       size_t ps, double alpha_re, double alpha_im, int accumulate) {
    const int mode = blockIdx.z;
    const int j = blockIdx.x * 16 + (threadIdx.x & 15);
    const int i = blockIdx.y * 16 + (threadIdx.x >> 4);
    if (i >= N || j >= N) return;
    const double* Ar = A + (size_t)(2 * mode) * ps;
    const double* Ai = Ar + ps;
    const double* Br = B + (size_t)(2 * mode) * ps;
    const double* Bi = Br + ps;
    double cr = 0.0, ci = 0.0;
    for (int k = 0; k < N; ++k) {
        const double ar = Ar[(size_t)i * ld + k], ai = Ai[(size_t)i * ld + k];
        const double br = Br[(size_t)k * ld + j], bi = Bi[(size_t)k * ld + j];
        cr += ar * br - ai * bi;
        ci += ar * bi + ai * br;
    }
    double outr = alpha_re * cr - alpha_im * ci;
    double outi = alpha_re * ci + alpha_im * cr;
    double* Cr = C + (size_t)(2 * mode) * ps;
    double* Ci = Cr + ps;
    if (accumulate) {
        outr += Cr[(size_t)i * ld + j];
        outi += Ci[(size_t)i * ld + j];
    }
    Cr[(size_t)i * ld + j] = outr;
    Ci[(size_t)i * ld + j] = outi;
}

CUresult encode_3d(CUtensorMap* map, const double* basep, const FreqLayout& f, int planes, int box0, int box1,
                   CUtensorMapSwizzle swz) {
    cuuint64_t dims[3] = {(cuuint64_t)f.N, (cuuint64_t)f.N, (cuuint64_t)planes};
    cuuint64_t strides[2] = {(cuuint64_t)f.ld * 8, (cuuint64_t)f.ps * 8};
    cuuint32_t box[3] = {(cuuint32_t)box0, (cuuint32_t)box1, 2};
    cuuint32_t estr[3] = {1, 1, 1};
    return g_encode(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<double*>(basep), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, swz, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
}

}  // namespace

cudaError_t zgemm_init() {
    if (g_encode) return cudaSuccess;
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess) return e;
    if (qres != cudaDriverEntryPointSuccess || !fn) return cudaErrorNotSupported;
    g_encode = reinterpret_cast<EncodeTiledFn>(fn);
    e = cudaFuncSetAttribute(zgemm_modes_dmma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    return e;
}

cudaError_t launch_zgemm_modes(const FreqLayout& f, int batch, const double* A, const double* B, double* C, Cplx alpha,
                               bool accumulate, int variant, cudaStream_t st) {
    const int modes = batch * f.L;
    if (variant == 0) {
        dim3 grid((f.N + 15) / 16, (f.N + 15) / 16, modes);
        zgemm_modes_ref_kernel<<<grid, 256, 0, st>>>(A, B, C, f.N, f.ld, f.ps, alpha.re, alpha.im, accumulate ? 1 : 0);
        return cudaGetLastError();
    }
    cudaError_t e = zgemm_init();
    if (e != cudaSuccess) return e;
    CUtensorMap mapA, mapB;
    if (encode_3d(&mapA, A, f, 2 * modes, BK, BM, CU_TENSOR_MAP_SWIZZLE_NONE) != CUDA_SUCCESS) return cudaErrorInvalidValue;
    if (encode_3d(&mapB, B, f, 2 * modes, 16, BK, CU_TENSOR_MAP_SWIZZLE_128B) != CUDA_SUCCESS) return cudaErrorInvalidValue;
    GemmParams P;
    P.C = C;
    P.ps = f.ps;
    P.N = f.N;
    P.ld = f.ld;
    P.tiles_m = (f.N + BM - 1) / BM;
    P.tiles_n = (f.N + BN - 1) / BN;
    P.alpha_re = alpha.re;
    P.alpha_im = alpha.im;
    P.accumulate = accumulate ? 1 : 0;
    const unsigned grid = (unsigned)(modes * P.tiles_m * P.tiles_n);
    zgemm_modes_dmma_kernel<<<grid, GEMM_THREADS, SMEM_BYTES, st>>>(mapA, mapB, P);
    return cudaGetLastError();
}

}  // namespace nspt
