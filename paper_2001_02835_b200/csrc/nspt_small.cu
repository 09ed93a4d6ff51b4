// nspt_small.cu -- FFT-CONV in ONE launch for small matrices (Steps 1-4 of Section 2 fused).
//
// Below N of a few dozen a product is bound by the three launches of the general path (forward, mode-wise product, inverse:
// 12-14 us at N = 16, of which the arithmetic is a fraction of a microsecond).  Here one CTA computes one output series
// C_ij = sum_k A_ik * B_kj entirely in shared memory:
//   1. the N series of row i of A and the N series of column j of B are loaded (zero-padded to L, order scale applied),
//   2. every warp transforms whole series by itself: radix-2 decimation in frequency, in place, natural order in,
//      bit-reversed order out -- no block barriers, and the permutation never has to be undone because
//   3. the mode-wise product sum_k A~_ik(p) B~_kj(p) is taken in the same (bit-reversed) order, and
//   4. the inverse is a decimation-in-time transform, bit-reversed in, natural out; 1/L, truncation and unscale on the way out.
// Every CTA redoes the transforms of the row and the column it needs (N-fold redundant flops, all of them in shared memory; the
// inputs are read from L2), which is what removes the spectra, the workspace and two launches.  Eligible while both operand
// blocks fit in shared memory (2 N (L + 1) + 256 complex128); the caller's output must not alias an input, because CTAs read A and
// B while others write C.
#include "nspt_internal.cuh"
#include "nspt_tma.cuh"

namespace nspt {
namespace {

constexpr int SMALL_THREADS = 256;
constexpr size_t SMALL_SMEM_MAX = 200 * 1024;

__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

struct SmallParams {
    const double2* A;
    const double2* B;
    double2* C;
    const double2* tw_fwd;    // w^m, m < L (eq. 2.7)
    const double2* tw_inv;    // w^-m       (eq. 2.9)
    const double* scale_in;   // s^k, or null when the order scale is off
    const double* scale_out;  // s^-k / L
    size_t NN;
    int N, n, L;
};

__global__ void __launch_bounds__(SMALL_THREADS) fftconv_small_kernel(const SmallParams P) {
    extern __shared__ double2 sm_small[];
    const int N = P.N, n = P.n, L = P.L;
    const int LP = L + 1;                      // series are L + 1 elements apart: consecutive series start in different banks
    double2* SA = sm_small;                    // [k][LP]: series of A_ik
    double2* SB = sm_small + (size_t)N * LP;   // [k][LP]: series of B_kj
    const int i = blockIdx.y, j = blockIdx.x, b = blockIdx.z;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const double2* A = P.A + (size_t)b * n * P.NN + (size_t)i * N;   // A^(o)_ik at A[o NN + k]
    const double2* B = P.B + (size_t)b * n * P.NN + j;               // B^(o)_kj at B[o NN + k N]
    pdl_wait();
    pdl_trigger();
    // Step 1 (eq. 2.6): the n coefficients of every series (order scale applied), four loads per operand in flight per thread,
    // and the zero padding up to L
    const int total = N * n;
    for (int e0 = tid; e0 < total; e0 += 4 * SMALL_THREADS) {
        double2 va[4], vb[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int e = e0 + u * SMALL_THREADS;
            if (e < total) {
                const int k = e % N, o = e / N;   // consecutive threads read consecutive k of one order of A
                va[u] = __ldg(&A[(size_t)o * P.NN + k]);
                vb[u] = __ldg(&B[(size_t)o * P.NN + (size_t)k * N]);
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int e = e0 + u * SMALL_THREADS;
            if (e < total) {
                const int k = e % N, o = e / N;
                const double s = P.scale_in ? __ldg(&P.scale_in[o]) : 1.0;
                SA[(size_t)k * LP + o] = make_double2(va[u].x * s, va[u].y * s);
                SB[(size_t)k * LP + o] = make_double2(vb[u].x * s, vb[u].y * s);
            }
        }
    }
    const int npad = L - n;
    for (int e = tid; e < 2 * N * npad; e += SMALL_THREADS) sm_small[(size_t)(e / npad) * LP + n + e % npad] = make_double2(0.0, 0.0);
    __syncthreads();
    // Step 2 (eq. 2.7): 2N transforms, whole series per warp, decimation in frequency
    for (int sidx = warp; sidx < 2 * N; sidx += SMALL_THREADS / 32) {
        double2* x = sm_small + (size_t)sidx * LP;
        for (int m = L >> 1, tstep = 1; m >= 1; m >>= 1, tstep <<= 1) {
            for (int q = lane; q < (L >> 1); q += 32) {
                const int jj = q & (m - 1), blk = q - jj;   // butterfly jj of the block starting at 2 blk
                const int p0 = 2 * blk + jj;
                const double2 u = x[p0], v = x[p0 + m];
                x[p0] = make_double2(u.x + v.x, u.y + v.y);
                x[p0 + m] = cmul(make_double2(u.x - v.x, u.y - v.y), __ldg(&P.tw_fwd[jj * tstep]));
            }
            __syncwarp();
        }
    }
    __syncthreads();
    // Step 3 (eq. 2.8) for the one element (i, j): C~(p) = sum_k A~_ik(p) B~_kj(p), p in bit-reversed order on both sides.
    // For L < 256 the sum over k is split over 256 / L thread groups whose partial sums are added through shared memory.
    double2* part = sm_small + (size_t)2 * N * LP;   // [group][L] partial sums, then the spectrum of C_ij in part[0 .. L)
    if (L >= SMALL_THREADS) {
        for (int p = tid; p < L; p += SMALL_THREADS) {
            double2 acc = make_double2(0.0, 0.0);
            for (int k = 0; k < N; ++k) {
                const double2 a = SA[(size_t)k * LP + p], bb = SB[(size_t)k * LP + p];
                acc.x = fma(a.x, bb.x, fma(-a.y, bb.y, acc.x));
                acc.y = fma(a.x, bb.y, fma(a.y, bb.x, acc.y));
            }
            part[p] = acc;
        }
        __syncthreads();
    } else {
        const int G = SMALL_THREADS / L, grp = tid / L, p = tid - grp * L;
        double2 acc = make_double2(0.0, 0.0);
        for (int k = grp; k < N; k += G) {
            const double2 a = SA[(size_t)k * LP + p], bb = SB[(size_t)k * LP + p];
            acc.x = fma(a.x, bb.x, fma(-a.y, bb.y, acc.x));
            acc.y = fma(a.x, bb.y, fma(a.y, bb.x, acc.y));
        }
        part[tid] = acc;
        __syncthreads();
        if (tid < L) {
            for (int q = 1; q < G; ++q) {   // fixed order: the result does not depend on scheduling
                acc.x += part[q * L + tid].x;
                acc.y += part[q * L + tid].y;
            }
        }
        __syncthreads();
        if (tid < L) part[tid] = acc;
        __syncthreads();
    }
    double2* SC = part;
    // Step 4 (eq. 2.9): inverse, decimation in time (bit-reversed in, natural out); one warp and warp barriers up to L = 64
    if (L <= 64) {
        if (warp == 0) {
            for (int m = 1, tstep = L >> 1; m < L; m <<= 1, tstep >>= 1) {
                if (lane < (L >> 1)) {
                    const int jj = lane & (m - 1), p0 = 2 * (lane - jj) + jj;
                    const double2 u = SC[p0], v = cmul(SC[p0 + m], __ldg(&P.tw_inv[jj * tstep]));
                    SC[p0] = make_double2(u.x + v.x, u.y + v.y);
                    SC[p0 + m] = make_double2(u.x - v.x, u.y - v.y);
                }
                __syncwarp();
            }
        }
        __syncthreads();
    } else {
        for (int m = 1, tstep = L >> 1; m < L; m <<= 1, tstep >>= 1) {
            for (int q = tid; q < (L >> 1); q += SMALL_THREADS) {
                const int jj = q & (m - 1), p0 = 2 * (q - jj) + jj;
                const double2 u = SC[p0], v = cmul(SC[p0 + m], __ldg(&P.tw_inv[jj * tstep]));
                SC[p0] = make_double2(u.x + v.x, u.y + v.y);
                SC[p0 + m] = make_double2(u.x - v.x, u.y - v.y);
            }
            __syncthreads();
        }
    }
    // truncation, 1/L and unscale
    double2* C = P.C + (size_t)b * n * P.NN + (size_t)i * N + j;
    for (int o = tid; o < n; o += SMALL_THREADS) {
        const double s = __ldg(&P.scale_out[o]);
        C[(size_t)o * P.NN] = make_double2(SC[o].x * s, SC[o].y * s);
    }
}

// both operand blocks and the partial sums / result spectrum
size_t small_smem_bytes(const FreqLayout& f) {
    return ((size_t)2 * f.N * (f.L + 1) + (size_t)(f.L > SMALL_THREADS ? f.L : SMALL_THREADS)) * sizeof(double2);
}

}  // namespace

bool fused_small_eligible(const FreqLayout& f, int batch) {
    if (f.L < 2 || f.L > 4 * SMALL_THREADS) return false;
    if (small_smem_bytes(f) > SMALL_SMEM_MAX) return false;
    return f.N <= 65535 && batch <= 65535;
}

cudaError_t launch_fused_small(const FreqLayout& f, const PlanTables& t, int batch, const nspt_c128* A, const nspt_c128* B,
                               nspt_c128* C, cudaStream_t st) {
    if (!fused_small_eligible(f, batch)) return cudaErrorInvalidValue;
    const size_t smem = small_smem_bytes(f);
    static bool attr_done[NSPT_MAX_DEVICES] = {};
    const int dev = current_device();
    if (!attr_done[dev]) {
        cudaError_t e = cudaFuncSetAttribute(fftconv_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMALL_SMEM_MAX);
        if (e != cudaSuccess) return e;
        attr_done[dev] = true;
    }
    SmallParams P{};
    P.A = reinterpret_cast<const double2*>(A);
    P.B = reinterpret_cast<const double2*>(B);
    P.C = reinterpret_cast<double2*>(C);
    P.tw_fwd = t.tw_fwd;
    P.tw_inv = t.tw_inv;
    P.scale_in = t.scale_in;
    P.scale_out = t.scale_out;
    P.NN = f.NN;
    P.N = f.N;
    P.n = f.n;
    P.L = f.L;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)f.N, (unsigned)f.N, (unsigned)batch);
    cfg.blockDim = dim3(SMALL_THREADS, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, fftconv_small_kernel, P);
}

}  // namespace nspt
