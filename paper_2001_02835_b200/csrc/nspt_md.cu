// nspt_md.cu -- the force projection that follows the staple in the NSPT update (eq. 2.3):
//     F^(k) = i c [ S^(k) - S^(k)+ - Tr(S^(k) - S^(k)+)/N ],   k = 0..Ntrunc,
// per order a traceless-Hermitian projection of the staple coefficient.  HBM-bound (each element of S is read
// twice, once transposed through shared memory, and F is written once): 48 N^2 bytes per order.
// With S^(k)_ij = a_ij + i b_ij and t = sum_i b_ii:
//     F_ij = -c (b_ij + b_ji) + i c (a_ij - a_ji)  +  delta_ij 2 c t / N.
#include "nspt_internal.cuh"

namespace nspt {
namespace {

__global__ void __launch_bounds__(256) force_kernel(const double2* __restrict__ S, double2* __restrict__ F, int N, size_t NN,
                                                   double c) {
    __shared__ double2 tile[32][33];
    __shared__ double red[8];
    const int k = blockIdx.z;
    const double2* s = S + (size_t)k * NN;
    double2* f = F + (size_t)k * NN;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;  // 32 x 8
    const int i0 = blockIdx.y * 32, j0 = blockIdx.x * 32;
    const bool diag_tile = (i0 == j0);
    // t = sum_i Im S_ii, needed by the diagonal tiles only (N values, L2-resident)
    double t = 0.0;
    if (diag_tile) {
        for (int i = threadIdx.x; i < N; i += 256) t += s[(size_t)i * N + i].y;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        if (tx == 0) red[ty] = t;
    }
    // transposed tile: tile[r][tx] = S[j0 + r][i0 + tx]
#pragma unroll
    for (int r = ty; r < 32; r += 8) {
        const int j = j0 + r, i = i0 + tx;
        tile[r][tx] = (j < N && i < N) ? s[(size_t)j * N + i] : make_double2(0.0, 0.0);
    }
    __syncthreads();
    if (diag_tile) {
        t = 0.0;
#pragma unroll
        for (int w = 0; w < 8; ++w) t += red[w];
    }
    const double shift = 2.0 * c * t / (double)N;
#pragma unroll
    for (int r = ty; r < 32; r += 8) {
        const int i = i0 + r, j = j0 + tx;
        if (i < N && j < N) {
            const double2 a = s[(size_t)i * N + j];  // S_ij
            const double2 b = tile[tx][r];           // S_ji
            double2 o = make_double2(-c * (a.y + b.y), c * (a.x - b.x));
            if (i == j) o.x += shift;
            f[(size_t)i * N + j] = o;
        }
    }
}

// Block polynomials of the Paterson-Stockmeyer form of exp(X) in frequency space (nspt_api.cu, series_exp_device):
//     B_j(p) = c[j][0] 1 + sum_{i=1}^{s-1} c[j][i] P_i(p),   j = 0..r-1,
// P_i = spectrum of the power X^{*i} (spectra `stride` doubles apart, P_1 first), B_j written `stride` apart.  One pass:
// every element of the s-1 powers is read once and the r results are written once.
struct PolyCoef {
    double c[12][12];
};
struct PolyCoefC {
    double c[12][12];
    double ci[12][12];   // imaginary parts: exp(lambda X) with a complex lambda (the link update has lambda = i eps)
};

__global__ void __launch_bounds__(256) freq_block_polys_kernel(const double2* __restrict__ pw, double2* __restrict__ out,
                                                              size_t stride_c, size_t total, int N, size_t NN, int s, int r,
                                                              const PolyCoef K) {
    const size_t e = (size_t)blockIdx.x * 256 + threadIdx.x;   // element of one (batched) spectrum
    if (e >= total) return;
    const size_t el = e % NN;
    const bool on_diag = (el / N == el % N);
    double2 acc[12];
#pragma unroll
    for (int j = 0; j < 12; ++j) acc[j] = make_double2((on_diag && j < r) ? K.c[j][0] : 0.0, 0.0);
    // all loads of a group of four powers are issued before the first is used (with a plain loop over i every load waited for the
    // arithmetic of the one before)
    for (int i0 = 1; i0 < s; i0 += 4) {
        double2 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = (i0 + u < s) ? __ldcs(&pw[(size_t)(i0 + u - 1) * stride_c + e]) : make_double2(0.0, 0.0);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (i0 + u < s) {
#pragma unroll
                for (int j = 0; j < 12; ++j) {
                    if (j < r) {
                        const double w = K.c[j][i0 + u];
                        acc[j].x += w * v[u].x;
                        acc[j].y += w * v[u].y;
                    }
                }
            }
        }
    }
#pragma unroll
    for (int j = 0; j < 12; ++j)
        if (j < r) out[(size_t)j * stride_c + e] = acc[j];
}

// the same with complex coefficients
__global__ void __launch_bounds__(256) freq_block_polys_cplx_kernel(const double2* __restrict__ pw, double2* __restrict__ out,
                                                                   size_t stride_c, size_t total, int N, size_t NN, int s, int r,
                                                                   const __grid_constant__ PolyCoefC K) {
    const size_t e = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (e >= total) return;
    const size_t el = e % NN;
    const bool on_diag = (el / N == el % N);
    double2 acc[12];
#pragma unroll
    for (int j = 0; j < 12; ++j) acc[j] = make_double2((on_diag && j < r) ? K.c[j][0] : 0.0, (on_diag && j < r) ? K.ci[j][0] : 0.0);
    for (int i0 = 1; i0 < s; i0 += 4) {
        double2 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = (i0 + u < s) ? __ldcs(&pw[(size_t)(i0 + u - 1) * stride_c + e]) : make_double2(0.0, 0.0);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (i0 + u < s) {
#pragma unroll
                for (int j = 0; j < 12; ++j) {
                    if (j < r) {
                        const double w = K.c[j][i0 + u], wi = K.ci[j][i0 + u];
                        acc[j].x += w * v[u].x - wi * v[u].y;
                        acc[j].y += w * v[u].y + wi * v[u].x;
                    }
                }
            }
        }
    }
#pragma unroll
    for (int j = 0; j < 12; ++j)
        if (j < r) out[(size_t)j * stride_c + e] = acc[j];
}

}  // namespace

cudaError_t launch_freq_block_polys(const FreqLayout& f, int batch, const double* powers, double* polys, int s, int r,
                                    const double* coef /* r x s, row-major */, cudaStream_t st, const double* coef_im) {
    if (s < 1 || s > 12 || r < 1 || r > 12) return cudaErrorInvalidValue;
    const size_t total = (size_t)batch * f.L * f.NN;
    const unsigned grid = (unsigned)((total + 255) / 256);
    if (coef_im) {
        PolyCoefC K{};
        for (int j = 0; j < r; ++j)
            for (int i = 0; i < s; ++i) {
                K.c[j][i] = coef[j * s + i];
                K.ci[j][i] = coef_im[j * s + i];
            }
        freq_block_polys_cplx_kernel<<<grid, 256, 0, st>>>(reinterpret_cast<const double2*>(powers), reinterpret_cast<double2*>(polys),
                                                           total, total, f.N, f.NN, s, r, K);
    } else {
        PolyCoef K{};
        for (int j = 0; j < r; ++j)
            for (int i = 0; i < s; ++i) K.c[j][i] = coef[j * s + i];
        freq_block_polys_kernel<<<grid, 256, 0, st>>>(reinterpret_cast<const double2*>(powers), reinterpret_cast<double2*>(polys),
                                                      total, total, f.N, f.NN, s, r, K);
    }
    return cudaGetLastError();
}

cudaError_t launch_force(const nspt_c128* S, nspt_c128* F, double c, int N, int n, cudaStream_t st) {
    dim3 grid((N + 31) / 32, (N + 31) / 32, (unsigned)n);
    force_kernel<<<grid, 256, 0, st>>>(reinterpret_cast<const double2*>(S), reinterpret_cast<double2*>(F), N, (size_t)N * N, c);
    return cudaGetLastError();
}

}  // namespace nspt
