// nspt_internal.cuh -- shared declarations of libnspt (CUDA path only; the oracle shares nothing with this).
#pragma once
#include <cuda_runtime.h>
#include <cstddef>
#include <cstdint>
#include "../../include/nspt.h"
#include "../../include/nspt_debug.h"

namespace nspt {

// ---------------------------------------------------------------------------------------------
// Frequency-domain workspace layout (internal; eq. 2.7 defines the content).
// One "spectrum" holds the Fourier coefficients X~(p), p = 0..L-1, of `batch` series in the same
// shape as a series, with the mode index in place of the order index:
//     X~[((b*L + p)*N + i)*N + j]   interleaved complex128, row-major N x N per mode.
// The transforms write / read 16-byte complex elements with the threads running along (i,j); the
// mode-wise matrix product loads 128-byte rows of 8 complex through TMA (row pitch N*16 bytes is
// always a multiple of 16, so no padding is needed for any N).
// ---------------------------------------------------------------------------------------------
struct FreqLayout {
    int N;        // matrix dimension
    int n;        // Ntrunc + 1 coefficients
    int L;        // transform length: power of two >= 2*Ntrunc + 1
    size_t NN;    // N*N
    size_t spectrum_doubles(int batch) const { return (size_t)batch * L * NN * 2; }
};

inline int transform_length(int Ntrunc) {
    int need = 2 * Ntrunc + 1, L = 1;
    while (L < need) L <<= 1;
    return L;
}

inline FreqLayout make_layout(int N, int Ntrunc) {
    FreqLayout f;
    f.N = N;
    f.n = Ntrunc + 1;
    f.L = transform_length(Ntrunc);
    f.NN = (size_t)N * N;
    return f;
}

// Per-L tables living in device memory (built on the host in long double).
struct PlanTables {
    const double2* tw_fwd;   // w^m  = exp(+2 pi i m / L), m < L      (eq. 2.7)
    const double2* tw_inv;   // w^-m                                   (eq. 2.9)
    const double* scale_in;  // s^k, k < n          (order scale, 1 when off)
    const double* scale_out; // s^-k / L, k < n     (unscale and the 1/L of eq. 2.9)
    double inv_L;
};

// Launcher-side caches (function attributes, occupancy, SM counts) are per device.
constexpr int NSPT_MAX_DEVICES = 64;
inline int current_device() {
    int d = 0;
    if (cudaGetDevice(&d) != cudaSuccess) {
        cudaGetLastError();
        d = 0;
    }
    return (d < 0 || d >= NSPT_MAX_DEVICES) ? 0 : d;
}

enum Stage { ST_FWD = 0, ST_GEMM = 1, ST_INV = 2, ST_RETRUNC = 3, ST_OTHER = 4, ST_POLY = 5, ST_SLICE = 6, ST_COUNT = 7 };

// Complex scalar for epilogues.
struct Cplx { double re, im; };

// ---- transforms (nspt_fft.cu) ---------------------------------------------------------------
// Forward: up to two operands per launch (src1 may be null). series -> spectrum.
cudaError_t launch_fft_forward(const FreqLayout& f, const PlanTables& t, int batch,
                               const nspt_c128* src0, double* dst0,
                               const nspt_c128* src1, double* dst1, cudaStream_t st,
                               bool skip_order0 = false, unsigned long long* maxbits0 = nullptr,
                               unsigned long long* maxbits1 = nullptr, size_t maxbits_stride = 0);
// Inverse + 1/L + truncation (+ unscale): spectrum -> series.
cudaError_t launch_fft_inverse(const FreqLayout& f, const PlanTables& t, int batch,
                               const double* src, nspt_c128* dst, cudaStream_t st);
// Re-truncation in place in frequency space: inverse, zero orders > Ntrunc, forward.
// maxbits (optional, INT8 path): [batch][L] entries that receive, by atomicMax, the per-mode maxima of the spectra written
// (L >= 16 only; the caller clears them).
cudaError_t launch_fft_retruncate(const FreqLayout& f, const PlanTables& t, int batch,
                                  const double* src, double* dst, cudaStream_t st, unsigned long long* maxbits = nullptr,
                                  size_t maxbits_stride = 0);
// The per-mode maxima are kept in NSPT_MAX_BUCKETS copies `maxbits_stride` entries apart: CTA c of a transform kernel updates
// copy c % NSPT_MAX_BUCKETS (148+ atomicMax on ONE address per mode serialise in L2: 6 us on a 30-60 us transform), the
// slicing pass takes the maximum over the copies.
constexpr int NSPT_MAX_BUCKETS = 8;
// Spectrum of the daggered series: Xd~(p) = (X~((L - p) mod L))^H.
cudaError_t launch_freq_dagger(const FreqLayout& f, int batch, const double* src, double* dst,
                               cudaStream_t st);
// dst(p) = (alpha + i alpha_im) * src(p) + 1 (unit matrix) for every mode: spectrum of alpha X + identity series.
cudaError_t launch_freq_scale_identity(const FreqLayout& f, int batch, const double* src, double* dst, double alpha,
                                       cudaStream_t st, double alpha_im = 0.0);
bool fft_length_supported(int L);

// ---- force projection (nspt_md.cu) -------------------------------------------------------------
// F^(k) = i c [ S^(k) - S^(k)+ - Tr(S^(k) - S^(k)+)/N ] for k < n (eq. 2.3).  F must not alias S.
cudaError_t launch_force(const nspt_c128* S, nspt_c128* F, double c, int N, int n, cudaStream_t st);
// Block polynomials B_j = coef[j][0] 1 + sum_{i=1}^{s-1} coef[j][i] P_i (j < r) of spectra packed back to back:
// powers = P_1, P_2, ... (s-1 of them), polys = B_0 .. B_{r-1}; s, r <= 12.  Used by the series exponential.
// coef_im (optional, r x s): imaginary parts of the coefficients (exp(lambda X) with a complex lambda).
cudaError_t launch_freq_block_polys(const FreqLayout& f, int batch, const double* powers, double* polys, int s, int r,
                                    const double* coef, cudaStream_t st, const double* coef_im = nullptr);

// ---- mode-wise matrix product (nspt_zgemm.cu) -----------------------------------------------
// For all batch*L modes p, with M(p) = A~(p) B~(p):
//     C(p)             (+)= alpha * M(p) + diag*1   if C is not null  (accumulate selects +=)
//     D((L-p) mod L)   (+)= beta  * M(p)^H      if D is not null  (accumulate_d selects +=)
// The second form adds the spectrum of the DAGGERED product series, FFT[X^+](p') = (X~((L-p') mod L))^H.
struct GemmOut {
    double* C = nullptr;
    Cplx alpha{1.0, 0.0};
    bool accumulate = false;
    double* D = nullptr;
    Cplx beta{1.0, 0.0};
    bool accumulate_d = false;
    double diag = 0.0;   // added to the diagonal of C(p) after alpha (the identity series in frequency space)
};
cudaError_t launch_zgemm_modes(const FreqLayout& f, int batch, const double* A, const double* B,
                               const GemmOut& out, int variant, cudaStream_t st);
// Up to 12 independent products of the same shape in ONE launch (their outputs must not overlap).  The operands
// of all groups must lie a whole number of N x N matrices apart (spectra of one workspace do).
struct GemmGroup {
    const double* A = nullptr;
    const double* B = nullptr;
    GemmOut out;
};
cudaError_t launch_zgemm_groups(const FreqLayout& f, int batch, const GemmGroup* groups, int ngroups, int variant,
                                cudaStream_t st);

// Naive-CONV: eq. 2.5 evaluated directly on the series (no transforms, no workspace), one launch.  C must not alias A, B.
cudaError_t launch_naive_conv(const FreqLayout& f, int batch, const nspt_c128* A, const nspt_c128* B, nspt_c128* C,
                              cudaStream_t st);

// FFT-CONV fused into one launch for small matrices (nspt_small.cu): one CTA per output series, everything in shared memory,
// no workspace.  C must not alias A, B.
bool fused_small_eligible(const FreqLayout& f, int batch);
cudaError_t launch_fused_small(const FreqLayout& f, const PlanTables& t, int batch, const nspt_c128* A, const nspt_c128* B,
                               nspt_c128* C, cudaStream_t st);

// ---- mode-wise matrix product on the INT8 tensor cores (nspt_ozaki.cu) -----------------------------------------
// FP64 spectra, whose per-mode maxima the transforms have recorded (maxbits), are cut into int8 slices (launch_ozaki_slice),
// multiplied exactly by tcgen05.mma.kind::i8 and recombined in FP64 (launch_ozaki_gemm, same epilogues as launch_zgemm_groups).
// A left factor must be sliced in the QUAD layout, a right factor in the ROWS layout; the store holds nq + nr such slots of
// `modes` = batch * L modes each.
struct OzStore {
    int8_t* quad = nullptr;
    int8_t* rows = nullptr;
    int* exps_q = nullptr;     // [nq][modes]: exponent of every mode of a QUAD slot (written by the slicing pass)
    int* exps_r = nullptr;     // [nr][modes]
    size_t quad_slot_bytes = 0, rows_slot_bytes = 0;
    int nq = 0, nr = 0, modes = 0;
};
size_t ozaki_store_bytes(const FreqLayout& f, int modes, int nq, int nr);
OzStore ozaki_store(const FreqLayout& f, int modes, int nq, int nr, void* ws);
struct OzSliceJob {
    const double* X = nullptr;                      // FP64 spectrum, modes x N x N
    const unsigned long long* maxbits = nullptr;    // [NSPT_MAX_BUCKETS][stride] maxima of the modes of X, entry of mode m at [m] ...
    size_t maxbits_stride = 0;
    bool mirror = false;                            // ... or of the series X is the dagger spectrum of: mode p takes entry (L - p) % L
    int quad_slot = -1, rows_slot = -1;             // -1: not needed in that layout
};
cudaError_t launch_ozaki_slice(const FreqLayout& f, const OzStore& S, const OzSliceJob* jobs, int njobs, cudaStream_t st);
// maxbits[mode] = max(maxbits[mode], max over the mode of X) for spectra no transform kernel has written (caller clears)
cudaError_t launch_ozaki_absmax(const FreqLayout& f, int modes, const double* X, unsigned long long* maxbits, cudaStream_t st);
struct OzGemmGroup {
    int quad_slot = -1;        // left factor
    int rows_slot = -1;        // right factor
    const double* A = nullptr; // the FP64 spectra the two slots were cut from
    const double* B = nullptr;
    GemmOut out;
};
cudaError_t launch_ozaki_gemm(const FreqLayout& f, const OzStore& S, const OzGemmGroup* groups, int ngroups, cudaStream_t st,
                              bool pairs = false, unsigned long long* clear = nullptr, int clear_count = 0);

}  // namespace nspt
