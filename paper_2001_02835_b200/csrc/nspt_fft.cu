// nspt_fft.cu -- transforms along the perturbative-order axis (Steps 1-2 and 4-5 of FFT-CONV,
// PAPER.md:70-77 eqs. 2.6-2.7 and PAPER.md:96-100 eq. 2.9), batched over the N^2 matrix elements
// (PAPER.md:106).  Hand-written for sm_100a; no cuFFT.
//
// Layout.  A series is [k][i][j] interleaved complex128, so for a fixed order k the N^2 elements
// are contiguous: threads run along the element index (coalesced 16-byte loads) and the transform
// runs along the strided k axis in registers + shared memory.  The paper's index permutations
// (MKL_ZOMATCOPY / cublasZgeam in Table 2) therefore cost nothing here: they are the
// addressing of these kernels.
//
// Algorithm.  L = R*S (R, S <= 16 powers of two).  A CTA owns T consecutive matrix elements and
// S threads cooperate on each element:
//   phase 1: thread s transforms the stride-S subsequence x[S r + s], r < R, in registers
//            (R-point DFT), multiplies by the twiddles w_L^(s p1) and parks Y_s[p1] in shared memory;
//   phase 2: thread q reads Y_s[p1], s < S, for p1 = q + S a and finishes with S-point DFTs:
//            X[p1 + R p2] = sum_s Y_s[p1] w_S^(s p2).
// Pruning.  Forward: orders >= L/2 are the zero padding of Step 1 (eq. 2.6) and are never loaded
// nor stored anywhere; the leaf butterflies of phase 1 degenerate to copies.  Inverse: Step 5
// discards orders >= L/2, so the last butterfly stage of phase 2 computes only the kept half.
// Re-truncation (needed between chained products in the staple) fuses inverse, truncation and
// forward: the orders a thread holds after the pruned inverse are exactly its phase-1 inputs of
// the forward transform, so no extra exchange is needed.
#include "nspt_internal.cuh"

namespace nspt {
namespace {

// cos / sin of 2 pi m / 16, m = 0..15
__host__ __device__ constexpr double c16(int m) {
    switch (m & 15) {
        case 0: return 1.0;
        case 1: return 0.92387953251128673848;
        case 2: return 0.70710678118654752440;
        case 3: return 0.38268343236508977173;
        case 4: return 0.0;
        case 5: return -0.38268343236508977173;
        case 6: return -0.70710678118654752440;
        case 7: return -0.92387953251128673848;
        case 8: return -1.0;
        case 9: return -0.92387953251128673848;
        case 10: return -0.70710678118654752440;
        case 11: return -0.38268343236508977173;
        case 12: return 0.0;
        case 13: return 0.38268343236508977173;
        case 14: return 0.70710678118654752440;
        default: return 0.92387953251128673848;
    }
}
__host__ __device__ constexpr double s16(int m) { return c16((m + 12) & 15); }  // sin x = cos(x - pi/2)

__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 cmul(double2 a, double2 w) {
    return make_double2(a.x * w.x - a.y * w.y, a.x * w.y + a.y * w.x);
}

// v * w_R^(SIGN*Q), compile-time twiddle
template <int R, int Q, int SIGN>
__device__ __forceinline__ double2 twmul(double2 v) {
    static_assert(R <= 16, "codelets are limited to 16 points");
    constexpr int m = (Q * (16 / R)) & 15;
    if constexpr (m == 0) {
        return v;
    } else if constexpr (m == 4) {
        return SIGN > 0 ? make_double2(-v.y, v.x) : make_double2(v.y, -v.x);
    } else if constexpr (m == 8) {
        return make_double2(-v.x, -v.y);
    } else if constexpr (m == 12) {
        return SIGN > 0 ? make_double2(v.y, -v.x) : make_double2(-v.y, v.x);
    } else {
        constexpr double c = c16(m);
        constexpr double s = SIGN * s16(m);
        return make_double2(v.x * c - v.y * s, v.x * s + v.y * c);
    }
}

// Radix-2 decimation-in-time DFT in registers: X[p] = sum_r x[r] w_R^(SIGN r p).
// ZERO_UPPER: x[R/2..R-1] are zero (never read).  HALF_OUT: only X[0..R/2-1] is produced.
template <int R, int SIGN, bool ZERO_UPPER, bool HALF_OUT>
struct Dft {
    template <int Q>
    static __device__ __forceinline__ void combine(const double2 (&E)[R / 2], const double2 (&O)[R / 2],
                                                   double2 (&X)[R]) {
        if constexpr (Q < R / 2) {
            const double2 t = twmul<R, Q, SIGN>(O[Q]);
            X[Q] = cadd(E[Q], t);
            if constexpr (!HALF_OUT) X[Q + R / 2] = csub(E[Q], t);
            combine<Q + 1>(E, O, X);
        }
    }
    static __device__ __forceinline__ void run(const double2 (&x)[R], double2 (&X)[R]) {
        double2 e[R / 2], o[R / 2], E[R / 2], O[R / 2];
#pragma unroll
        for (int q = 0; q < R / 2; ++q) {
            e[q] = x[2 * q];
            o[q] = x[2 * q + 1];
        }
        Dft<R / 2, SIGN, ZERO_UPPER, false>::run(e, E);
        Dft<R / 2, SIGN, ZERO_UPPER, false>::run(o, O);
        combine<0>(E, O, X);
    }
};
template <int SIGN, bool ZERO_UPPER, bool HALF_OUT>
struct Dft<2, SIGN, ZERO_UPPER, HALF_OUT> {
    static __device__ __forceinline__ void run(const double2 (&x)[2], double2 (&X)[2]) {
        if constexpr (ZERO_UPPER) {
            X[0] = x[0];
            if constexpr (!HALF_OUT) X[1] = x[0];
        } else {
            X[0] = cadd(x[0], x[1]);
            if constexpr (!HALF_OUT) X[1] = csub(x[0], x[1]);
        }
    }
};
template <int SIGN, bool ZERO_UPPER, bool HALF_OUT>
struct Dft<1, SIGN, ZERO_UPPER, HALF_OUT> {
    static __device__ __forceinline__ void run(const double2 (&x)[1], double2 (&X)[1]) { X[0] = x[0]; }
};

struct XformParams {
    const double2* src_series[2];  // forward input (interleaved)
    const double* src_freq;        // inverse / retruncate input (planar)
    double* dst_freq[2];           // forward / retruncate output (planar)
    double2* dst_series;           // inverse output
    size_t NN;
    size_t ps;
    int N, ld, n;
    const double2* tw_fwd;
    const double2* tw_inv;
    const double* scale_in;
    const double* scale_out;
    double inv_L;
    int use_scale;
};

// ---- forward phases: registers x[r] = coefficient of order S*r + s (r < R/2 non-zero) -> planes
template <int R, int S, int T>
__device__ __forceinline__ void forward_from_regs(double2 (&x)[R], int s, int c, bool valid, double* out_re,
                                                  size_t ps, const double2* __restrict__ tw, double2* sm) {
    constexpr bool ZU = (R >= 2);
    double2 Y[R];
    Dft<R, +1, ZU, false>::run(x, Y);
    if constexpr (S == 1) {
        if (valid) {
#pragma unroll
            for (int p1 = 0; p1 < R; ++p1) {
                out_re[(size_t)(2 * p1) * ps] = Y[p1].x;
                out_re[(size_t)(2 * p1 + 1) * ps] = Y[p1].y;
            }
        }
    } else {
#pragma unroll
        for (int p1 = 0; p1 < R; ++p1) {
            const double2 w = __ldg(&tw[s * p1]);  // w_L^(s p1), s p1 < L
            sm[(p1 * S + s) * T + c] = (p1 == 0) ? Y[p1] : cmul(Y[p1], w);
        }
        __syncthreads();
#pragma unroll
        for (int a = 0; a < R / S; ++a) {
            const int p1 = s + S * a;
            double2 y[S], X[S];
#pragma unroll
            for (int sp = 0; sp < S; ++sp) y[sp] = sm[(p1 * S + sp) * T + c];
            Dft<S, +1, false, false>::run(y, X);
            if (valid) {
#pragma unroll
                for (int p2 = 0; p2 < S; ++p2) {
                    const int p = p1 + R * p2;
                    out_re[(size_t)(2 * p) * ps] = X[p2].x;
                    out_re[(size_t)(2 * p + 1) * ps] = X[p2].y;
                }
            }
        }
    }
}

// ---- inverse phases: planes -> registers.  On return, for S > 1, xk[a][k2] holds the UNSCALED
// sum for order k = (s + S a) + R k2 (k2 < S/2); for S == 1, xk[0][k1] holds order k1 (k1 < R).
template <int R, int S, int T>
struct InvRegs {
    static constexpr int A = (S == 1) ? 1 : R / S;
    static constexpr int K2 = (S == 1) ? R : (S / 2);
    double2 v[A][K2];
};

template <int R, int S, int T>
__device__ __forceinline__ void inverse_to_regs(const double* in_re, size_t ps, int s, int c, bool valid,
                                                const double2* __restrict__ tw, double2* sm,
                                                InvRegs<R, S, T>& out) {
    double2 x[R], Y[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int p = S * r + s;
        x[r] = valid ? make_double2(__ldg(&in_re[(size_t)(2 * p) * ps]), __ldg(&in_re[(size_t)(2 * p + 1) * ps]))
                     : make_double2(0.0, 0.0);
    }
    Dft<R, -1, false, false>::run(x, Y);
    if constexpr (S == 1) {
#pragma unroll
        for (int k1 = 0; k1 < R; ++k1) out.v[0][k1] = Y[k1];
    } else {
#pragma unroll
        for (int k1 = 0; k1 < R; ++k1) {
            const double2 w = __ldg(&tw[s * k1]);
            sm[(k1 * S + s) * T + c] = (k1 == 0) ? Y[k1] : cmul(Y[k1], w);
        }
        __syncthreads();
#pragma unroll
        for (int a = 0; a < R / S; ++a) {
            const int k1 = s + S * a;
            double2 y[S], X[S];
#pragma unroll
            for (int sp = 0; sp < S; ++sp) y[sp] = sm[(k1 * S + sp) * T + c];
            Dft<S, -1, false, true>::run(y, X);
#pragma unroll
            for (int k2 = 0; k2 < S / 2; ++k2) out.v[a][k2] = X[k2];
        }
    }
}

template <int R, int S, int T>
__global__ void __launch_bounds__(T* S) fft_forward_kernel(const XformParams P) {
    extern __shared__ double2 sm[];
    const int c = threadIdx.x % T, s = threadIdx.x / T;
    const size_t e = (size_t)blockIdx.x * T + c;
    const bool valid = e < P.NN;
    const int b = blockIdx.y, z = blockIdx.z;
    constexpr int L = R * S;
    const double2* in = (z ? P.src_series[1] : P.src_series[0]) + (size_t)b * P.n * P.NN + e;
    double2 x[R];
    constexpr int RH = (R >= 2) ? R / 2 : 1;
#pragma unroll
    for (int r = 0; r < RH; ++r) {
        const int k = S * r + s;
        double2 v = make_double2(0.0, 0.0);
        if (valid && k < P.n) {
            v = __ldg(&in[(size_t)k * P.NN]);
            if (P.use_scale) {
                const double sc = __ldg(&P.scale_in[k]);
                v.x *= sc;
                v.y *= sc;
            }
        }
        x[r] = v;
    }
#pragma unroll
    for (int r = RH; r < R; ++r) x[r] = make_double2(0.0, 0.0);
    const size_t off = valid ? (e / P.N) * P.ld + (e % P.N) : 0;
    double* out_re = (z ? P.dst_freq[1] : P.dst_freq[0]) + (size_t)b * L * 2 * P.ps + off;
    forward_from_regs<R, S, T>(x, s, c, valid, out_re, P.ps, P.tw_fwd, sm);
}

template <int R, int S, int T>
__global__ void __launch_bounds__(T* S) fft_inverse_kernel(const XformParams P) {
    extern __shared__ double2 sm[];
    const int c = threadIdx.x % T, s = threadIdx.x / T;
    const size_t e = (size_t)blockIdx.x * T + c;
    const bool valid = e < P.NN;
    const int b = blockIdx.y;
    constexpr int L = R * S;
    const size_t off = valid ? (e / P.N) * P.ld + (e % P.N) : 0;
    const double* in_re = P.src_freq + (size_t)b * L * 2 * P.ps + off;
    InvRegs<R, S, T> q;
    inverse_to_regs<R, S, T>(in_re, P.ps, s, c, valid, P.tw_inv, sm, q);
    if (!valid) return;
    double2* out = P.dst_series + (size_t)b * P.n * P.NN + e;
#pragma unroll
    for (int a = 0; a < InvRegs<R, S, T>::A; ++a)
#pragma unroll
        for (int k2 = 0; k2 < InvRegs<R, S, T>::K2; ++k2) {
            const int k = (S == 1) ? k2 : (s + S * a) + R * k2;
            if (k < P.n) {
                const double sc = __ldg(&P.scale_out[k]);  // s^-k / L
                out[(size_t)k * P.NN] = make_double2(q.v[a][k2].x * sc, q.v[a][k2].y * sc);
            }
        }
}

template <int R, int S, int T>
__global__ void __launch_bounds__(T* S) fft_retruncate_kernel(const XformParams P) {
    extern __shared__ double2 sm[];
    const int c = threadIdx.x % T, s = threadIdx.x / T;
    const size_t e = (size_t)blockIdx.x * T + c;
    const bool valid = e < P.NN;
    const int b = blockIdx.y;
    constexpr int L = R * S;
    const size_t off = valid ? (e / P.N) * P.ld + (e % P.N) : 0;
    const double* in_re = P.src_freq + (size_t)b * L * 2 * P.ps + off;
    InvRegs<R, S, T> q;
    inverse_to_regs<R, S, T>(in_re, P.ps, s, c, valid, P.tw_inv, sm, q);
    // orders this thread holds are k = s + S r with r = a + (R/S) k2 (S > 1) or r = k1 (S == 1)
    double2 x[R];
    constexpr int RH = (R >= 2) ? R / 2 : 1;
#pragma unroll
    for (int r = 0; r < R; ++r) x[r] = make_double2(0.0, 0.0);
    if constexpr (S == 1) {
#pragma unroll
        for (int r = 0; r < RH; ++r)
            if (r < P.n) x[r] = make_double2(q.v[0][r].x * P.inv_L, q.v[0][r].y * P.inv_L);
    } else {
#pragma unroll
        for (int a = 0; a < R / S; ++a)
#pragma unroll
            for (int k2 = 0; k2 < S / 2; ++k2) {
                const int r = a + (R / S) * k2;
                const int k = s + S * r;
                if (k < P.n) x[r] = make_double2(q.v[a][k2].x * P.inv_L, q.v[a][k2].y * P.inv_L);
            }
        __syncthreads();  // shared memory is reused by the forward phases
    }
    double* out_re = P.dst_freq[0] + (size_t)b * L * 2 * P.ps + off;
    forward_from_regs<R, S, T>(x, s, c, valid, out_re, P.ps, P.tw_fwd, sm);
}

// Spectrum of the daggered series (g is real): FFT[X^+](p) = (X~((L-p) mod L))^H.
// dst(b,p,c)[i*ld+j] = (c ? -1 : +1) * src(b,(L-p)%L,c)[j*ld+i]; 32x32 tiles through shared memory.
__global__ void __launch_bounds__(256) freq_dagger_kernel(const double* __restrict__ src, double* __restrict__ dst,
                                                         int N, int ld, size_t ps, int L) {
    __shared__ double tile[32][33];
    const int plane = blockIdx.z;  // (b*L + p)*2 + c
    const int c = plane & 1;
    const int bp = plane >> 1;
    const int b = bp / L, p = bp % L;
    const int ps_src = (L - p) % L;
    const double* s = src + ((size_t)(b * L + ps_src) * 2 + c) * ps;
    double* d = dst + (size_t)plane * ps;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;  // 32 x 8
    const int i0 = blockIdx.y * 32, j0 = blockIdx.x * 32;
    // read src rows j0.., cols i0..  (src[j][i])
#pragma unroll
    for (int r = ty; r < 32; r += 8) {
        const int j = j0 + r, i = i0 + tx;
        tile[r][tx] = (j < N && i < N) ? s[(size_t)j * ld + i] : 0.0;
    }
    __syncthreads();
    const double sgn = c ? -1.0 : 1.0;
#pragma unroll
    for (int r = ty; r < 32; r += 8) {
        const int i = i0 + r, j = j0 + tx;
        if (i < N && j < N) d[(size_t)i * ld + j] = sgn * tile[tx][r];
    }
}

template <int R, int S, int T>
struct Launcher {
    static constexpr int L = R * S;
    static constexpr size_t smem = (S == 1) ? 0 : (size_t)L * T * sizeof(double2);
    template <typename K>
    static cudaError_t prep(K kernel) {
        if (smem > 48 * 1024)
            return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        return cudaSuccess;
    }
    static cudaError_t forward(const XformParams& P, int batch, int nops, cudaStream_t st) {
        cudaError_t e = prep(fft_forward_kernel<R, S, T>);
        if (e != cudaSuccess) return e;
        dim3 grid((unsigned)((P.NN + T - 1) / T), batch, nops);
        fft_forward_kernel<R, S, T><<<grid, T * S, smem, st>>>(P);
        return cudaGetLastError();
    }
    static cudaError_t inverse(const XformParams& P, int batch, cudaStream_t st) {
        cudaError_t e = prep(fft_inverse_kernel<R, S, T>);
        if (e != cudaSuccess) return e;
        dim3 grid((unsigned)((P.NN + T - 1) / T), batch, 1);
        fft_inverse_kernel<R, S, T><<<grid, T * S, smem, st>>>(P);
        return cudaGetLastError();
    }
    static cudaError_t retruncate(const XformParams& P, int batch, cudaStream_t st) {
        cudaError_t e = prep(fft_retruncate_kernel<R, S, T>);
        if (e != cudaSuccess) return e;
        dim3 grid((unsigned)((P.NN + T - 1) / T), batch, 1);
        fft_retruncate_kernel<R, S, T><<<grid, T * S, smem, st>>>(P);
        return cudaGetLastError();
    }
};

enum Which { W_FWD, W_INV, W_RET };

template <int R, int S, int T>
cudaError_t run_cfg(Which w, const XformParams& P, int batch, int nops, cudaStream_t st) {
    switch (w) {
        case W_FWD: return Launcher<R, S, T>::forward(P, batch, nops, st);
        case W_INV: return Launcher<R, S, T>::inverse(P, batch, st);
        default: return Launcher<R, S, T>::retruncate(P, batch, st);
    }
}

cudaError_t dispatch(int L, Which w, const XformParams& P, int batch, int nops, cudaStream_t st) {
    switch (L) {
        case 1: return run_cfg<1, 1, 128>(w, P, batch, nops, st);
        case 2: return run_cfg<2, 1, 128>(w, P, batch, nops, st);
        case 4: return run_cfg<4, 1, 128>(w, P, batch, nops, st);
        case 8: return run_cfg<8, 1, 128>(w, P, batch, nops, st);
        case 16: return run_cfg<4, 4, 32>(w, P, batch, nops, st);
        case 32: return run_cfg<8, 4, 32>(w, P, batch, nops, st);
        case 64: return run_cfg<8, 8, 32>(w, P, batch, nops, st);
        case 128: return run_cfg<16, 8, 32>(w, P, batch, nops, st);
        case 256: return run_cfg<16, 16, 16>(w, P, batch, nops, st);
        default: return cudaErrorInvalidValue;
    }
}

XformParams base_params(const FreqLayout& f, const PlanTables& t) {
    XformParams P{};
    P.NN = f.NN;
    P.ps = f.ps;
    P.N = f.N;
    P.ld = f.ld;
    P.n = f.n;
    P.tw_fwd = t.tw_fwd;
    P.tw_inv = t.tw_inv;
    P.scale_in = t.scale_in;
    P.scale_out = t.scale_out;
    P.inv_L = t.inv_L;
    P.use_scale = 0;
    return P;
}

}  // namespace

bool fft_length_supported(int L) { return L >= 1 && L <= 256 && (L & (L - 1)) == 0; }

cudaError_t launch_fft_forward(const FreqLayout& f, const PlanTables& t, int batch, const nspt_c128* src0,
                               double* dst0, const nspt_c128* src1, double* dst1, cudaStream_t st) {
    XformParams P = base_params(f, t);
    P.src_series[0] = reinterpret_cast<const double2*>(src0);
    P.src_series[1] = reinterpret_cast<const double2*>(src1);
    P.dst_freq[0] = dst0;
    P.dst_freq[1] = dst1;
    P.use_scale = (t.scale_in != nullptr) ? 1 : 0;
    return dispatch(f.L, W_FWD, P, batch, src1 ? 2 : 1, st);
}

cudaError_t launch_fft_inverse(const FreqLayout& f, const PlanTables& t, int batch, const double* src,
                               nspt_c128* dst, cudaStream_t st) {
    XformParams P = base_params(f, t);
    P.src_freq = src;
    P.dst_series = reinterpret_cast<double2*>(dst);
    return dispatch(f.L, W_INV, P, batch, 1, st);
}

cudaError_t launch_fft_retruncate(const FreqLayout& f, const PlanTables& t, int batch, const double* src,
                                  double* dst, cudaStream_t st) {
    XformParams P = base_params(f, t);
    P.src_freq = src;
    P.dst_freq[0] = dst;
    return dispatch(f.L, W_RET, P, batch, 1, st);
}

cudaError_t launch_freq_dagger(const FreqLayout& f, int batch, const double* src, double* dst, cudaStream_t st) {
    dim3 grid((f.N + 31) / 32, (f.N + 31) / 32, (unsigned)(batch * f.L * 2));
    freq_dagger_kernel<<<grid, 256, 0, st>>>(src, dst, f.N, f.ld, f.ps, f.L);
    return cudaGetLastError();
}

}  // namespace nspt
