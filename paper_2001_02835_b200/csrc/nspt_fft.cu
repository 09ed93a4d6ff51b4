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
//
// Data movement.  The kernels are HBM-bound (about 1.5 flop per byte), so what matters is keeping
// loads in flight while a tile is being transformed.  For L >= 16 the kernels are persistent: each
// CTA walks over tiles of T elements, and the [order][T] input tile of the tile after next is
// fetched by one TMA box load (cp.async.bulk.tensor, mbarrier complete_tx) into a ring of
// shared-memory stages (three deep in the forward pass, two in the others) while the current tile is
// in registers.  Rows beyond Ntrunc and elements beyond N^2 are zero-filled by TMA, which is exactly
// the zero padding of Step 1.  Output tiles are formed in place in the exchange buffer and leave by
// one TMA box store each (double-buffered in the forward pass).  L <= 8 needs one thread per element
// and no shared memory; those kernels use plain loads and stores.
//
// INT8 product (nspt_ozaki.cu).  The kernels that write spectra (forward, re-truncation) can also
// record max(|re|, |im|) of every mode they write -- a running maximum of the high words per thread,
// one redux.sync and one atomicMax per mode and CTA at the end -- which is the scale of the fixed-point
// slices of that mode.
#include <cstdlib>
#include <map>
#include <mutex>

#include "nspt_internal.cuh"
#include "nspt_ozaki.cuh"
#include "nspt_tma.cuh"

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
    const double2* src_freq;       // inverse / retruncate input (spectrum)
    double2* dst_freq[2];          // forward / retruncate output (spectrum)
    double2* dst_series;           // inverse output
    size_t NN;
    int N, n;
    int batch;
    unsigned tiles_x;              // tiles per (operand, batch) = ceil(NN / T)
    unsigned total_tiles;
    const double2* tw_fwd;
    const double2* tw_inv;
    const double* scale_in;
    const double* scale_out;
    double inv_L;
    int use_scale;
    int skip_order0;               // forward only: treat the coefficient of g^0 as zero (series exponential)
    // forward / re-truncation, optional (INT8 product): maxbits[z][b * L + p] receives, by atomicMax, the high word (shifted
    // to the high half of a 64-bit pattern) of max(|re|, |im|) over mode p of the spectrum written for operand z
    unsigned long long* maxbits[2];
    size_t maxbits_stride;         // distance (entries) between the NSPT_MAX_BUCKETS copies of the maxima
};

// ---- forward phases: registers x[r] = coefficient of order S*r + s (r < R/2 non-zero) -> spectrum.
// For S > 1 the exchange buffer `sm` must be free on entry; on return every thread has passed the
// __syncthreads that follows the phase-1 writes, but phase-2 reads of `sm` may still be in flight.
template <int R, int S, int T>
__device__ __forceinline__ void forward_from_regs(double2 (&x)[R], int s, int c, bool valid, double2* out,
                                                  size_t NN, const double2* __restrict__ tw, double2* sm) {
    constexpr bool ZU = (R >= 2);
    double2 Y[R];
    Dft<R, +1, ZU, false>::run(x, Y);
    if constexpr (S == 1) {
        if (valid) {
#pragma unroll
            for (int p1 = 0; p1 < R; ++p1) out[(size_t)p1 * NN] = Y[p1];
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
                for (int p2 = 0; p2 < S; ++p2) out[(size_t)(p1 + R * p2) * NN] = X[p2];
            }
        }
    }
}

// ---- inverse phases: registers x[r] = mode S*r + s -> registers.  On return, for S > 1, v[a][k2]
// holds the UNSCALED sum for order k = (s + S a) + R k2 (k2 < S/2); for S == 1, v[0][k1] holds
// order k1 (k1 < R).  Same shared-memory contract as forward_from_regs.
template <int R, int S, int T>
struct InvRegs {
    static constexpr int A = (S == 1) ? 1 : R / S;
    static constexpr int K2 = (S == 1) ? R : (S / 2);
    double2 v[A][K2];
};

// The twiddles w^(+-s k1), k1 < R, of a thread do not change from tile to tile: the persistent kernels load them
// once into registers (twr) instead of once per tile from the global table (18 % of the inverse pass's warp samples
// were waiting for those loads).  TWREG selects the register copy.
template <int R, int S, int T, bool TWREG = false>
__device__ __forceinline__ void inverse_from_regs(double2 (&x)[R], int s, int c, const double2* __restrict__ tw,
                                                  double2* sm, InvRegs<R, S, T>& out, const double2* twr = nullptr) {
    double2 Y[R];
    Dft<R, -1, false, false>::run(x, Y);
    if constexpr (S == 1) {
#pragma unroll
        for (int k1 = 0; k1 < R; ++k1) out.v[0][k1] = Y[k1];
    } else {
#pragma unroll
        for (int k1 = 0; k1 < R; ++k1) {
            double2 w;
            if constexpr (TWREG)
                w = twr[k1];
            else
                w = __ldg(&tw[s * k1]);
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

// orders held after the pruned inverse -> phase-1 inputs of the forward transform (times 1/L,
// orders > Ntrunc dropped)
template <int R, int S, int T>
__device__ __forceinline__ void retruncate_regs(const InvRegs<R, S, T>& q, int s, int n, double inv_L, double2 (&x)[R]) {
    constexpr int RH = (R >= 2) ? R / 2 : 1;
#pragma unroll
    for (int r = 0; r < R; ++r) x[r] = make_double2(0.0, 0.0);
    if constexpr (S == 1) {
#pragma unroll
        for (int r = 0; r < RH; ++r)
            if (r < n) x[r] = make_double2(q.v[0][r].x * inv_L, q.v[0][r].y * inv_L);
    } else {
#pragma unroll
        for (int a = 0; a < R / S; ++a)
#pragma unroll
            for (int k2 = 0; k2 < S / 2; ++k2) {
                const int r = a + (R / S) * k2;
                const int k = s + S * r;
                if (k < n) x[r] = make_double2(q.v[a][k2].x * inv_L, q.v[a][k2].y * inv_L);
            }
    }
}

template <int R, int S, int T>
__device__ __forceinline__ void store_series(const InvRegs<R, S, T>& q, int s, int n, const double* __restrict__ scale_out,
                                             double2* out, size_t NN) {
#pragma unroll
    for (int a = 0; a < InvRegs<R, S, T>::A; ++a)
#pragma unroll
        for (int k2 = 0; k2 < InvRegs<R, S, T>::K2; ++k2) {
            const int k = (S == 1) ? k2 : (s + S * a) + R * k2;
            if (k < n) {
                const double sc = __ldg(&scale_out[k]);  // s^-k / L
                out[(size_t)k * NN] = make_double2(q.v[a][k2].x * sc, q.v[a][k2].y * sc);
            }
        }
}

// =================================================================================================
// L <= 8: one thread per element, plain loads (S == 1)
// =================================================================================================
template <int R, int T>
__global__ void __launch_bounds__(T) fft_forward_small_kernel(const XformParams P) {
    const int c = threadIdx.x;
    const size_t e = (size_t)blockIdx.x * T + c;
    const bool valid = e < P.NN;
    const int b = blockIdx.y, z = blockIdx.z;
    const double2* in = (z ? P.src_series[1] : P.src_series[0]) + (size_t)b * P.n * P.NN + e;
    double2 x[R];
    constexpr int RH = (R >= 2) ? R / 2 : 1;
#pragma unroll
    for (int r = 0; r < R; ++r) x[r] = make_double2(0.0, 0.0);
#pragma unroll
    for (int r = 0; r < RH; ++r) {
        if (valid && r < P.n && !(P.skip_order0 && r == 0)) {
            double2 v = __ldg(&in[(size_t)r * P.NN]);
            if (P.use_scale) {
                const double sc = __ldg(&P.scale_in[r]);
                v.x *= sc;
                v.y *= sc;
            }
            x[r] = v;
        }
    }
    double2* out = (z ? P.dst_freq[1] : P.dst_freq[0]) + (size_t)b * R * P.NN + e;
    forward_from_regs<R, 1, T>(x, 0, c, valid, out, P.NN, P.tw_fwd, nullptr);
}

template <int R, int T, bool RETRUNC>
__global__ void __launch_bounds__(T) fft_inverse_small_kernel(const XformParams P) {
    const int c = threadIdx.x;
    const size_t e = (size_t)blockIdx.x * T + c;
    if (e >= P.NN) return;
    const int b = blockIdx.y;
    const double2* in = P.src_freq + (size_t)b * R * P.NN + e;
    double2 x[R];
#pragma unroll
    for (int r = 0; r < R; ++r) x[r] = __ldg(&in[(size_t)r * P.NN]);
    InvRegs<R, 1, T> q;
    inverse_from_regs<R, 1, T>(x, 0, c, P.tw_inv, nullptr, q);
    if constexpr (RETRUNC) {
        double2 xf[R];
        retruncate_regs<R, 1, T>(q, 0, P.n, P.inv_L, xf);
        forward_from_regs<R, 1, T>(xf, 0, c, true, P.dst_freq[0] + (size_t)b * R * P.NN + e, P.NN, P.tw_fwd, nullptr);
    } else {
        store_series<R, 1, T>(q, 0, P.n, P.scale_out, P.dst_series + (size_t)b * P.n * P.NN + e, P.NN);
    }
}

// =================================================================================================
// L >= 16: persistent CTAs, TMA-staged input tiles
// =================================================================================================
template <int R, int S, int T>
struct Cfg {
    static constexpr int L = R * S;
    static constexpr int THREADS = T * S;
    static constexpr int FULL_TILE_BYTES = L * T * 16;        // [mode][T] tile, also the exchange buffer
    static constexpr int HALF_TILE_BYTES = (L / 2) * T * 16;  // [order < L/2][T] tile
    // forward: ring of input tiles (orders) + two exchange buffers that double as TMA-store sources
    static constexpr int FWD_STAGES = 3, FWD_OUTS = 2;
    static constexpr int FWD_SMEM = FWD_STAGES * HALF_TILE_BYTES + FWD_OUTS * FULL_TILE_BYTES + 64 + 128;
    // inverse: ring of input tiles (modes) + exchange buffer + one output tile (orders)
    static constexpr int INV_STAGES = 2;
    static constexpr int INV_SMEM = INV_STAGES * FULL_TILE_BYTES + FULL_TILE_BYTES + HALF_TILE_BYTES + 64 + 128;
    // re-truncation: ring of input tiles (modes) + one exchange buffer that is also the store source
    static constexpr int RET_STAGES = 2;
    static constexpr int RET_SMEM = RET_STAGES * FULL_TILE_BYTES + FULL_TILE_BYTES + 64 + 128;
};

__device__ __forceinline__ void tile_coords(unsigned tile, const XformParams& P, unsigned& tx, unsigned& b, unsigned& z) {
    tx = tile % P.tiles_x;
    const unsigned zb = tile / P.tiles_x;
    b = zb % (unsigned)P.batch;
    z = zb / (unsigned)P.batch;
}

// Forward phases on shared memory.  Phase 1: thread s parks Y_s[p1] w_L^(s p1) at slot [s][p1]; phase 2: thread q
// owns p1 = q + S a, reads slots [sp][p1] (all sp) and overwrites THE SAME slots with X[p1 + R p2] at [p2][p1],
// which is the natural mode order p = p1 + R p2: the exchange buffer becomes the [mode][T] output tile in place.
template <int R, int S, int T, bool TWREG = false>
__device__ __forceinline__ void forward_phase1_smem(const double2 (&x)[R], int s, int c, const double2* __restrict__ tw,
                                                    double2* exch, const double2* twr = nullptr) {
    double2 Y[R];
    Dft<R, +1, true, false>::run(x, Y);
#pragma unroll
    for (int p1 = 0; p1 < R; ++p1) {
        // w_L^(s p1), s p1 < L: from the thread's register copy in the persistent kernels, else from the global table
        double2 w;
        if constexpr (TWREG)
            w = twr[p1];
        else
            w = __ldg(&tw[s * p1]);
        exch[(s * R + p1) * T + c] = (p1 == 0) ? Y[p1] : cmul(Y[p1], w);
    }
}
template <int R, int S, int T, bool TRACK = false>
__device__ __forceinline__ void forward_phase2_smem(int s, int c, double2* exch, unsigned int* mx = nullptr) {
#pragma unroll
    for (int a = 0; a < R / S; ++a) {
        const int p1 = s + S * a;
        double2 y[S], X[S];
#pragma unroll
        for (int sp = 0; sp < S; ++sp) y[sp] = exch[(sp * R + p1) * T + c];
        Dft<S, +1, false, false>::run(y, X);
#pragma unroll
        for (int p2 = 0; p2 < S; ++p2) {
            exch[(p2 * R + p1) * T + c] = X[p2];
            if constexpr (TRACK)   // running maximum of mode p1 + R p2 over the elements this thread has transformed
                mx[a * S + p2] = oz_max_hi2(mx[a * S + p2], X[p2]);
        }
    }
}
// Flush the per-thread running maxima of the modes: reduce over the T lanes that share s (a warp, or an aligned part of one),
// one atomicMax per mode, and reset.  mx[a * S + p2] belongs to mode (s + S a) + R p2.
template <int R, int S, int T>
__device__ __forceinline__ void flush_mode_max(unsigned int (&mx)[R], int s, int c, unsigned long long* dst) {
    static_assert(T <= 32 && (32 % T) == 0, "T lanes form a part of a warp");
    const unsigned mask = (T == 32) ? 0xffffffffu : (((1u << T) - 1u) << (T * ((threadIdx.x & 31) / T)));
    // what the table holds already (high words, read from L2; a stale value is a lower one): an atomic is issued only where this
    // CTA raises the maximum -- the k-th CTA to arrive does so with probability ~1/k, so a mode sees a handful of atomics
    // instead of one per CTA
    // (measured: L = 128 forward pass 60 -> 57 us; at L <= 32 a CTA lives for two or three tiles and the extra L2 round trip
    // costs more than it saves, 17 -> 19 us at L = 16, so short transforms issue their atomics unconditionally)
    constexpr bool PEEK = R * S >= 128;
    unsigned int cur[R];
#pragma unroll
    for (int a = 0; a < R / S; ++a)
#pragma unroll
        for (int p2 = 0; p2 < S; ++p2)
            cur[a * S + p2] = (PEEK && c == 0) ? __ldcg(reinterpret_cast<const unsigned int*>(dst + ((s + S * a) + R * p2)) + 1) : 0u;
#pragma unroll
    for (int a = 0; a < R / S; ++a)
#pragma unroll
        for (int p2 = 0; p2 < S; ++p2) {
            const unsigned int v = __reduce_max_sync(mask, mx[a * S + p2]) >> 1;   // the running values carry 2 |x|_hi (oz_max_hi2)
            if (c == 0 && v > cur[a * S + p2]) atomicMax(dst + ((s + S * a) + R * p2), (unsigned long long)v << 32);
            mx[a * S + p2] = 0u;
        }
}

template <int R, int S, int T>
__global__ void __launch_bounds__(T* S, 1) fft_forward_tma_kernel(const __grid_constant__ CUtensorMap in0,
                                                              const __grid_constant__ CUtensorMap in1,
                                                              const __grid_constant__ CUtensorMap out0,
                                                              const __grid_constant__ CUtensorMap out1,
                                                              const XformParams P) {
    using C = Cfg<R, S, T>;
    constexpr int NS = C::FWD_STAGES;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 127u) & ~127u;
    uint8_t* sgen = smem_raw + (base - smem_u32(smem_raw));
    const uint32_t out_addr = base + NS * C::HALF_TILE_BYTES;
    const uint32_t bar = out_addr + C::FWD_OUTS * C::FULL_TILE_BYTES;  // NS 8-byte mbarriers

    const int c = threadIdx.x % T, s = threadIdx.x / T;

    auto issue = [&](unsigned tile, int stage) {
        unsigned tx, b, z;
        tile_coords(tile, P, tx, b, z);
        mbar_expect_tx(bar + 8 * stage, C::HALF_TILE_BYTES);
        tma_load_3d(base + stage * C::HALF_TILE_BYTES, z ? &in1 : &in0, bar + 8 * stage, (int)(2 * tx * T), 0, (int)b);
    };

    if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < NS; ++i) mbar_init(bar + 8 * i, 1);
        mbar_fence_init();
    }
    pdl_wait();      // everything above overlaps the tail of the previous kernel of the stream
    pdl_trigger();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < NS; ++i)
            if (blockIdx.x + i * gridDim.x < P.total_tiles) issue(blockIdx.x + i * gridDim.x, i);
    }
    __syncthreads();

    double2 twr[R];   // this thread's forward twiddles w_L^(s p1), loaded once
#pragma unroll
    for (int p1 = 0; p1 < R; ++p1) twr[p1] = __ldg(&P.tw_fwd[s * p1]);
    unsigned int mx[R];   // running maxima of this thread's modes (INT8 product only)
#pragma unroll
    for (int i = 0; i < R; ++i) mx[i] = 0u;
    const bool track = P.maxbits[0] != nullptr;
    const size_t bucket = (size_t)(blockIdx.x % NSPT_MAX_BUCKETS) * P.maxbits_stride;
    unsigned cur_zb = 0xffffffffu;
    unsigned it = 0;
    for (unsigned tile = blockIdx.x; tile < P.total_tiles; tile += gridDim.x, ++it) {
        const int stage = it % NS;
        unsigned tx, b, z;
        tile_coords(tile, P, tx, b, z);
        if (track) {
            const unsigned zb = z * (unsigned)P.batch + b;
            if (zb != cur_zb) {
                if (cur_zb != 0xffffffffu)
                    flush_mode_max<R, S, T>(mx, s, c, P.maxbits[cur_zb / (unsigned)P.batch] + bucket + (size_t)(cur_zb % (unsigned)P.batch) * C::L);
                cur_zb = zb;
            }
        }
        mbar_wait(bar + 8 * stage, (it / NS) & 1);
        const double2* in = reinterpret_cast<const double2*>(sgen + stage * C::HALF_TILE_BYTES);
        double2 x[R];
#pragma unroll
        for (int r = 0; r < R / 2; ++r) {
            const int k = S * r + s;
            double2 v = in[k * T + c];  // rows >= n and elements >= N^2 were zero-filled by TMA (Step 1's padding)
            if (P.use_scale && k < P.n) {
                const double sc = __ldg(&P.scale_in[k]);
                v.x *= sc;
                v.y *= sc;
            }
            if (P.skip_order0 && k == 0) v = make_double2(0.0, 0.0);
            x[r] = v;
        }
#pragma unroll
        for (int r = R / 2; r < R; ++r) x[r] = make_double2(0.0, 0.0);
        const int ob = it & 1;
        double2* exch = reinterpret_cast<double2*>(sgen + NS * C::HALF_TILE_BYTES + ob * C::FULL_TILE_BYTES);
        if (threadIdx.x == 0) tma_store_wait_read<1>();  // the store issued two tiles ago has left buffer `ob`
        __syncthreads();  // input stage consumed by everyone; exchange buffer `ob` is free
        if (threadIdx.x == 0) {
            const unsigned next = tile + NS * gridDim.x;
            if (next < P.total_tiles) issue(next, stage);
        }
        forward_phase1_smem<R, S, T, true>(x, s, c, P.tw_fwd, exch, twr);
        __syncthreads();
        if (track)
            forward_phase2_smem<R, S, T, true>(s, c, exch, mx);
        else
            forward_phase2_smem<R, S, T>(s, c, exch);
        fence_proxy_async_smem();
        __syncthreads();
        if (threadIdx.x == 0) {
            // INT8 path: the slicing pass reads the spectrum at once -- the lines written stay in the L2 as long as they can
            if (track)
                tma_store_3d_hint(z ? &out1 : &out0, out_addr + ob * C::FULL_TILE_BYTES, (int)(2 * tx * T), 0, (int)b, l2_keep_policy());
            else
                tma_store_3d(z ? &out1 : &out0, out_addr + ob * C::FULL_TILE_BYTES, (int)(2 * tx * T), 0, (int)b);
            tma_store_commit();
        }
    }
    if (track && cur_zb != 0xffffffffu)
        flush_mode_max<R, S, T>(mx, s, c, P.maxbits[cur_zb / (unsigned)P.batch] + bucket + (size_t)(cur_zb % (unsigned)P.batch) * C::L);
    if (threadIdx.x == 0) tma_store_wait_read<0>();
}

// Inverse (+ 1/L, truncation, unscale) and, with RETRUNC, the fused inverse -> truncate -> forward pass.
template <int R, int S, int T, bool RETRUNC>
__global__ void __launch_bounds__(T* S) fft_inverse_tma_kernel(const __grid_constant__ CUtensorMap in_map,
                                                              const __grid_constant__ CUtensorMap out_map,
                                                              const XformParams P) {
    using C = Cfg<R, S, T>;
    constexpr int NS = RETRUNC ? C::RET_STAGES : C::INV_STAGES;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 127u) & ~127u;
    uint8_t* sgen = smem_raw + (base - smem_u32(smem_raw));
    const uint32_t exch_addr = base + NS * C::FULL_TILE_BYTES;
    double2* exch = reinterpret_cast<double2*>(sgen + NS * C::FULL_TILE_BYTES);
    const uint32_t outb_addr = exch_addr + C::FULL_TILE_BYTES;  // [order][T] output tile (plain inverse only)
    double2* outb = reinterpret_cast<double2*>(sgen + (NS + 1) * C::FULL_TILE_BYTES);
    const uint32_t bar = RETRUNC ? outb_addr : outb_addr + C::HALF_TILE_BYTES;

    const int c = threadIdx.x % T, s = threadIdx.x / T;

    auto issue = [&](unsigned tile, int stage) {
        unsigned tx, b, z;
        tile_coords(tile, P, tx, b, z);
        mbar_expect_tx(bar + 8 * stage, C::FULL_TILE_BYTES);
        tma_load_3d(base + stage * C::FULL_TILE_BYTES, &in_map, bar + 8 * stage, (int)(2 * tx * T), 0, (int)b);
    };

    if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < NS; ++i) mbar_init(bar + 8 * i, 1);
        mbar_fence_init();
    }
    pdl_wait();      // everything above overlaps the tail of the previous kernel of the stream
    pdl_trigger();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < NS; ++i)
            if (blockIdx.x + i * gridDim.x < P.total_tiles) issue(blockIdx.x + i * gridDim.x, i);
    }
    __syncthreads();

    double2 twr[R];   // this thread's inverse twiddles w_L^-(s k1), loaded once
#pragma unroll
    for (int k1 = 0; k1 < R; ++k1) twr[k1] = __ldg(&P.tw_inv[s * k1]);
    // the output scales s^-k / L of the orders this thread stores (plain inverse), loaded once as well
    double sco[InvRegs<R, S, T>::A][InvRegs<R, S, T>::K2];
    if constexpr (!RETRUNC) {
#pragma unroll
        for (int a = 0; a < InvRegs<R, S, T>::A; ++a)
#pragma unroll
            for (int k2 = 0; k2 < InvRegs<R, S, T>::K2; ++k2) {
                const int k = (s + S * a) + R * k2;
                sco[a][k2] = (k < P.n) ? __ldg(&P.scale_out[k]) : 0.0;
            }
    }
    unsigned int mx[RETRUNC ? R : 1];   // re-truncation for the INT8 path: running maxima of the modes written (see the forward kernel)
    const bool track = RETRUNC && P.maxbits[0] != nullptr;
    const size_t bucket = (size_t)(blockIdx.x % NSPT_MAX_BUCKETS) * P.maxbits_stride;
    unsigned cur_b = 0xffffffffu;
    if constexpr (RETRUNC) {
#pragma unroll
        for (int i = 0; i < R; ++i) mx[i] = 0u;
    }
    // re-truncation: the forward twiddles too where the register budget allows (R <= 8)
    constexpr bool FWD_TWREG = RETRUNC && (R <= 8);
    double2 twf[FWD_TWREG ? R : 1];
    if constexpr (FWD_TWREG) {
#pragma unroll
        for (int p1 = 0; p1 < R; ++p1) twf[p1] = __ldg(&P.tw_fwd[s * p1]);
    }
    unsigned it = 0;
    for (unsigned tile = blockIdx.x; tile < P.total_tiles; tile += gridDim.x, ++it) {
        const int stage = it % NS;
        unsigned tx, b, z;
        tile_coords(tile, P, tx, b, z);
        mbar_wait(bar + 8 * stage, (it / NS) & 1);
        const double2* in = reinterpret_cast<const double2*>(sgen + stage * C::FULL_TILE_BYTES);
        double2 x[R];
#pragma unroll
        for (int r = 0; r < R; ++r) x[r] = in[(S * r + s) * T + c];
        if (threadIdx.x == 0) tma_store_wait_read<0>();  // the previous tile's store has left `exch` / `outb`
        __syncthreads();  // input stage consumed; exchange buffer free
        if (threadIdx.x == 0) {
            const unsigned next = tile + NS * gridDim.x;
            if (next < P.total_tiles) issue(next, stage);
        }
        InvRegs<R, S, T> q;
        inverse_from_regs<R, S, T, true>(x, s, c, P.tw_inv, exch, q, twr);
        if constexpr (RETRUNC) {
            if (track && b != cur_b) {   // the spectra of a launch are its batch elements
                if (cur_b != 0xffffffffu) flush_mode_max<R, S, T>(mx, s, c, P.maxbits[0] + bucket + (size_t)cur_b * C::L);
                cur_b = b;
            }
            double2 xf[R];
            retruncate_regs<R, S, T>(q, s, P.n, P.inv_L, xf);
            __syncthreads();  // phase-2 reads of the inverse are done
            forward_phase1_smem<R, S, T, FWD_TWREG>(xf, s, c, P.tw_fwd, exch, twf);
            __syncthreads();
            if (track)
                forward_phase2_smem<R, S, T, true>(s, c, exch, mx);
            else
                forward_phase2_smem<R, S, T>(s, c, exch);
            fence_proxy_async_smem();
            __syncthreads();
            if (threadIdx.x == 0) {
                if (track)
                    tma_store_3d_hint(&out_map, exch_addr, (int)(2 * tx * T), 0, (int)b, l2_keep_policy());
                else
                    tma_store_3d(&out_map, exch_addr, (int)(2 * tx * T), 0, (int)b);
                tma_store_commit();
            }
        } else {
            // rows k >= n of the tile are never written: the series tensor has n rows, TMA clips the rest (Step 5)
#pragma unroll
            for (int a = 0; a < InvRegs<R, S, T>::A; ++a)
#pragma unroll
                for (int k2 = 0; k2 < InvRegs<R, S, T>::K2; ++k2) {
                    const int k = (s + S * a) + R * k2;
                    if (k < P.n) {
                        const double sc = sco[a][k2];  // s^-k / L
                        outb[k * T + c] = make_double2(q.v[a][k2].x * sc, q.v[a][k2].y * sc);
                    }
                }
            fence_proxy_async_smem();
            __syncthreads();
            if (threadIdx.x == 0) {
                tma_store_3d(&out_map, outb_addr, (int)(2 * tx * T), 0, (int)b);
                tma_store_commit();
            }
        }
    }
    if constexpr (RETRUNC) {
        if (track && cur_b != 0xffffffffu) flush_mode_max<R, S, T>(mx, s, c, P.maxbits[0] + bucket + (size_t)cur_b * C::L);
    }
    if (threadIdx.x == 0) tma_store_wait_read<0>();
}

// Spectrum of the daggered series (g is real): FFT[X^+](p) = (X~((L-p) mod L))^H.
// dst(b,p)[i][j] = conj(src(b,(L-p)%L)[j][i]); 32x32 tiles through shared memory.
__global__ void __launch_bounds__(256) freq_dagger_kernel(const double2* __restrict__ src, double2* __restrict__ dst,
                                                         int N, size_t NN, int L, int modes) {
    __shared__ double2 tile[32][33];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;  // 32 x 8
    const int i0 = blockIdx.y * 32, j0 = blockIdx.x * 32;
    for (int bp = blockIdx.z; bp < modes; bp += gridDim.z) {  // b*L + p (the grid's z extent is capped at 65535)
        const int b = bp / L, p = bp % L;
        const double2* s = src + (size_t)(b * L + (L - p) % L) * NN;
        double2* d = dst + (size_t)bp * NN;
        __syncthreads();
#pragma unroll
        for (int r = ty; r < 32; r += 8) {
            const int j = j0 + r, i = i0 + tx;
            tile[r][tx] = (j < N && i < N) ? s[(size_t)j * N + i] : make_double2(0.0, 0.0);
        }
        __syncthreads();
#pragma unroll
        for (int r = ty; r < 32; r += 8) {
            const int i = i0 + r, j = j0 + tx;
            if (i < N && j < N) {
                const double2 v = tile[tx][r];
                d[(size_t)i * N + j] = make_double2(v.x, -v.y);
            }
        }
    }
}

// dst(p) = alpha * src(p) + 1 for every mode p: alpha X + (identity series), whose spectrum is the unit matrix
// at every mode.  First Horner step of the series exponential.
__global__ void __launch_bounds__(256) freq_scale_identity_kernel(const double2* __restrict__ src, double2* __restrict__ dst,
                                                                 int N, size_t NN, double alpha, double alpha_im, int modes) {
    const size_t e = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (e >= NN) return;
    for (int m = blockIdx.y; m < modes; m += gridDim.y) {   // the grid's y extent is capped at 65535
        const size_t o = (size_t)m * NN + e;
        const double2 u = src[o];
        double2 v = make_double2(alpha * u.x - alpha_im * u.y, alpha * u.y + alpha_im * u.x);
        if (e / N == e % N) v.x += 1.0;
        dst[o] = v;
    }
}

// ------------------------------------------------------------------------------------ host side
enum Which { W_FWD, W_INV, W_RET };

int num_sms() {
    static int sms[NSPT_MAX_DEVICES] = {};
    const int dev = current_device();
    if (!sms[dev]) {
        cudaDeviceGetAttribute(&sms[dev], cudaDevAttrMultiProcessorCount, dev);
        if (sms[dev] <= 0) sms[dev] = 148;
    }
    return sms[dev];
}

// Resident CTAs per SM of a kernel, looked up once per kernel (the attribute and occupancy calls cost more host
// time than a small transform takes on the device).
template <typename K>
cudaError_t persistent_grid(K kernel, int threads, int smem, unsigned total_tiles, unsigned* grid) {
    static std::map<std::pair<int, const void*>, int> cache;   // (device, kernel): function attributes are per device
    static std::mutex mu;
    std::lock_guard<std::mutex> lk(mu);
    const std::pair<int, const void*> key(current_device(), reinterpret_cast<const void*>(kernel));
    auto it = cache.find(key);
    int occ;
    if (it == cache.end()) {
        cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        occ = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, threads, smem);
        if (e != cudaSuccess) return e;
        if (occ < 1) occ = 1;
        cache[key] = occ;
    } else {
        occ = it->second;
    }
    const unsigned cap = (unsigned)(occ * num_sms());
    *grid = total_tiles < cap ? total_tiles : cap;
    return cudaSuccess;
}

template <int R, int T>
cudaError_t run_small(Which w, XformParams P, int nops, cudaStream_t st) {
    dim3 grid((unsigned)((P.NN + T - 1) / T), P.batch, nops);
    switch (w) {
        case W_FWD: fft_forward_small_kernel<R, T><<<grid, T, 0, st>>>(P); break;
        case W_INV: fft_inverse_small_kernel<R, T, false><<<grid, T, 0, st>>>(P); break;
        default: fft_inverse_small_kernel<R, T, true><<<grid, T, 0, st>>>(P); break;
    }
    return cudaGetLastError();
}

template <int R, int S, int T>
cudaError_t run_tma(Which w, XformParams P, int nops, cudaStream_t st) {
    using C = Cfg<R, S, T>;
    P.tiles_x = (unsigned)((P.NN + T - 1) / T);
    P.total_tiles = P.tiles_x * (unsigned)P.batch * (unsigned)nops;
    cudaError_t e;
    unsigned grid = 0;
    // series viewed as doubles: (2 N^2 per order, n orders, batch); spectrum: (2 N^2 per mode, L modes, batch)
    const uint64_t sdims[3] = {(uint64_t)(2 * P.NN), (uint64_t)P.n, (uint64_t)P.batch};
    const uint64_t sstrides[2] = {(uint64_t)P.NN * 16, (uint64_t)P.n * P.NN * 16};
    const uint32_t sbox[3] = {2 * T, (uint32_t)(C::L / 2), 1};
    const uint64_t fdims[3] = {(uint64_t)(2 * P.NN), (uint64_t)C::L, (uint64_t)P.batch};
    const uint64_t fstrides[2] = {(uint64_t)P.NN * 16, (uint64_t)C::L * P.NN * 16};
    const uint32_t fbox[3] = {2 * T, (uint32_t)C::L, 1};
    if (w == W_FWD) {
        CUtensorMap in[2], out[2];
        for (int z = 0; z < 2; ++z) {
            const void* src = P.src_series[z] ? (const void*)P.src_series[z] : (const void*)P.src_series[0];
            const void* dst = P.dst_freq[z] ? (const void*)P.dst_freq[z] : (const void*)P.dst_freq[0];
            if ((e = tma_encode_f64(&in[z], src, 3, sdims, sstrides, sbox, false)) != cudaSuccess) return e;
            if ((e = tma_encode_f64(&out[z], dst, 3, fdims, fstrides, fbox, false)) != cudaSuccess) return e;
        }
        auto kern = fft_forward_tma_kernel<R, S, T>;
        if ((e = persistent_grid(kern, C::THREADS, C::FWD_SMEM, P.total_tiles, &grid)) != cudaSuccess) return e;
        return launch_pdl(kern, grid, C::THREADS, C::FWD_SMEM, st, in[0], in[1], out[0], out[1], P);
    } else {
        CUtensorMap in, out;
        if ((e = tma_encode_f64(&in, P.src_freq, 3, fdims, fstrides, fbox, false)) != cudaSuccess) return e;
        if (w == W_INV) {
            if ((e = tma_encode_f64(&out, P.dst_series, 3, sdims, sstrides, sbox, false)) != cudaSuccess) return e;
            auto kern = fft_inverse_tma_kernel<R, S, T, false>;
            if ((e = persistent_grid(kern, C::THREADS, C::INV_SMEM, P.total_tiles, &grid)) != cudaSuccess) return e;
            return launch_pdl(kern, grid, C::THREADS, C::INV_SMEM, st, in, out, P);
        } else {
            if ((e = tma_encode_f64(&out, P.dst_freq[0], 3, fdims, fstrides, fbox, false)) != cudaSuccess) return e;
            auto kern = fft_inverse_tma_kernel<R, S, T, true>;
            if ((e = persistent_grid(kern, C::THREADS, C::RET_SMEM, P.total_tiles, &grid)) != cudaSuccess) return e;
            return launch_pdl(kern, grid, C::THREADS, C::RET_SMEM, st, in, out, P);
        }
    }
    return cudaGetLastError();
}

cudaError_t dispatch(int L, Which w, const XformParams& P, int nops, cudaStream_t st) {
    switch (L) {
        case 1: return run_small<1, 128>(w, P, nops, st);
        case 2: return run_small<2, 128>(w, P, nops, st);
        case 4: return run_small<4, 128>(w, P, nops, st);
        case 8: return run_small<8, 128>(w, P, nops, st);
        case 16: return run_tma<4, 4, 32>(w, P, nops, st);
        case 32: return run_tma<8, 4, 32>(w, P, nops, st);
        // The forward pass (1 byte read : 2 written) gains from wider rows per TMA box -- measured at N = 225: L = 64
        // 32.8 -> 32.0 us, L = 128 63.9 -> 60.2 us, L = 256 140 -> 129 us -- while the inverse and re-truncation passes lose
        // with them (L = 128: 34.2 -> 37.2 us, L = 256: 58.5 -> 68.9 us) and keep the narrower tiles.
        case 64: return w == W_FWD ? run_tma<8, 8, 32>(w, P, nops, st) : run_tma<8, 8, 16>(w, P, nops, st);
        case 128: return w == W_FWD ? run_tma<16, 8, 32>(w, P, nops, st) : run_tma<16, 8, 16>(w, P, nops, st);
        case 256: return w == W_FWD ? run_tma<16, 16, 16>(w, P, nops, st) : run_tma<16, 16, 8>(w, P, nops, st);
        default: return cudaErrorInvalidValue;
    }
}

XformParams base_params(const FreqLayout& f, const PlanTables& t, int batch) {
    XformParams P{};
    P.NN = f.NN;
    P.N = f.N;
    P.n = f.n;
    P.batch = batch;
    P.tw_fwd = t.tw_fwd;
    P.tw_inv = t.tw_inv;
    P.scale_in = t.scale_in;
    P.scale_out = t.scale_out;
    P.inv_L = t.inv_L;
    P.use_scale = 0;
    P.skip_order0 = 0;
    return P;
}

}  // namespace

bool fft_length_supported(int L) { return L >= 1 && L <= 256 && (L & (L - 1)) == 0; }

cudaError_t launch_fft_forward(const FreqLayout& f, const PlanTables& t, int batch, const nspt_c128* src0,
                               double* dst0, const nspt_c128* src1, double* dst1, cudaStream_t st, bool skip_order0,
                               unsigned long long* maxbits0, unsigned long long* maxbits1, size_t maxbits_stride) {
    XformParams P = base_params(f, t, batch);
    P.skip_order0 = skip_order0 ? 1 : 0;
    P.maxbits[0] = maxbits0;
    P.maxbits[1] = maxbits1 ? maxbits1 : maxbits0;
    P.maxbits_stride = maxbits_stride;
    P.src_series[0] = reinterpret_cast<const double2*>(src0);
    P.src_series[1] = reinterpret_cast<const double2*>(src1);
    P.dst_freq[0] = reinterpret_cast<double2*>(dst0);
    P.dst_freq[1] = reinterpret_cast<double2*>(dst1);
    P.use_scale = (t.scale_in != nullptr) ? 1 : 0;
    return dispatch(f.L, W_FWD, P, src1 ? 2 : 1, st);
}

cudaError_t launch_fft_inverse(const FreqLayout& f, const PlanTables& t, int batch, const double* src,
                               nspt_c128* dst, cudaStream_t st) {
    XformParams P = base_params(f, t, batch);
    P.src_freq = reinterpret_cast<const double2*>(src);
    P.dst_series = reinterpret_cast<double2*>(dst);
    return dispatch(f.L, W_INV, P, 1, st);
}

cudaError_t launch_fft_retruncate(const FreqLayout& f, const PlanTables& t, int batch, const double* src,
                                  double* dst, cudaStream_t st, unsigned long long* maxbits, size_t maxbits_stride) {
    XformParams P = base_params(f, t, batch);
    P.maxbits[0] = P.maxbits[1] = maxbits;
    P.maxbits_stride = maxbits_stride;
    P.src_freq = reinterpret_cast<const double2*>(src);
    P.dst_freq[0] = reinterpret_cast<double2*>(dst);
    return dispatch(f.L, W_RET, P, 1, st);
}

cudaError_t launch_freq_dagger(const FreqLayout& f, int batch, const double* src, double* dst, cudaStream_t st) {
    const int modes = batch * f.L;
    dim3 grid((f.N + 31) / 32, (f.N + 31) / 32, (unsigned)(modes < 65535 ? modes : 65535));
    freq_dagger_kernel<<<grid, 256, 0, st>>>(reinterpret_cast<const double2*>(src), reinterpret_cast<double2*>(dst), f.N,
                                             f.NN, f.L, modes);
    return cudaGetLastError();
}

cudaError_t launch_freq_scale_identity(const FreqLayout& f, int batch, const double* src, double* dst, double alpha,
                                       cudaStream_t st, double alpha_im) {
    const int modes = batch * f.L;
    dim3 grid((unsigned)((f.NN + 255) / 256), (unsigned)(modes < 65535 ? modes : 65535));
    freq_scale_identity_kernel<<<grid, 256, 0, st>>>(reinterpret_cast<const double2*>(src), reinterpret_cast<double2*>(dst),
                                                     f.N, f.NN, alpha, alpha_im, modes);
    return cudaGetLastError();
}

}  // namespace nspt
