/*
 * nspt.h -- C ABI of libnspt: the FFT-based convolution (FFT-CONV) star-product of truncated
 * perturbative series with dense N x N complex128 matrix coefficients, and the TEK staple
 * built from it, for one NVIDIA B200 (sm_100a).
 *
 * Source of every definition: Gonzalez-Arroyo et al., "Towards higher order numerical
 * stochastic perturbation computation applied to the twisted Eguchi-Kawai model"
 * (arXiv:2001.02835), cited below as PAPER.md:<line> (section / equation).
 *
 * ---------------------------------------------------------------------------------------
 * Series layout (all entry points).  A polynomial matrix truncated at O(g^Ntrunc)
 *     X = sum_{k=0}^{Ntrunc} g^k X^(k)                     (eq. 2.4)
 * is an array of n = Ntrunc+1 row-major N x N matrices of nspt_c128, order index slowest:
 *     X[(k*N + i)*N + j] = X^(k)_{ij},   k = 0..Ntrunc,  i, j = 0..N-1,
 * contiguous, n*N*N elements, 16-byte aligned.  nspt_c128 is layout-identical to C
 * `double _Complex`, cuDoubleComplex and torch.complex128.
 *
 * Pointers.  Entry points WITHOUT the _host suffix take DEVICE pointers valid on the
 * current CUDA device; they enqueue kernels on the library stream (nspt_set_stream) and
 * return without synchronising.  Entry points WITH the _host suffix take HOST pointers
 * (pinned memory recommended), copy host->device, run the same kernels, copy device->host
 * and synchronise the stream before returning.  The twist tensor z is always a HOST array.
 *
 * Ownership.  The caller owns every array it passes; the library keeps no caller pointer
 * past the stream-ordered work of the call.  Library-owned state (plan tables, the internal
 * frequency-domain workspace, staging buffers of the _host calls) is released by nspt_release.
 *
 * Aliasing.  The output of nspt_series_mul[_batched] may be exactly one of its inputs (all
 * inputs are transformed into the workspace before any output is written); partial overlap
 * is undefined.  In nspt_staple S[mu] may alias U[mu] for the same reason.
 *
 * CUDA graphs.  After one call of the same shape (which builds the plan tables and sizes the workspace) the
 * device entry points neither allocate nor synchronise, so they can be captured into a CUDA graph on the library
 * stream.  The large kernels are launched with programmatic stream serialization.
 *
 * Errors.  Every call returns 0 (NSPT_OK) or a negative code; nothing throws, aborts or
 * prints.  Kernel faults are asynchronous and surface at the caller's next synchronisation.
 *
 * Devices and threads.  The library keeps one context per CUDA device (plan tables, workspace, staging, stream,
 * order scale), selected by the device that is current at the call (cudaGetDevice) and guarded by a mutex: calls for the
 * same device are serialised, calls for different devices (e.g. one direction of the TEK model per GPU)
 * run independently.  nspt_set_stream / nspt_set_order_scale / nspt_set_workspace apply to the current device only.
 * All calls of one device share one workspace: when nspt_set_stream switches streams, work queued on the new stream
 * is ordered after the work already queued on the old one (an event), so two streams never overlap inside the library.
 *
 * Allocation.  The library-owned workspace and staging buffers grow on demand: the FIRST call of a larger shape
 * synchronises the library stream, frees and reallocates (cudaMalloc); every later call of that or a smaller shape is
 * asynchronous and allocation-free.  Pass a workspace (nspt_set_workspace) to rule this out.
 *
 * Diagnostics (kernel selection, per-stage timing, FP64 peak probe, launch counter) live in nspt_debug.h.
 * ---------------------------------------------------------------------------------------
 */
#ifndef NSPT_H
#define NSPT_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct { double re, im; } nspt_c128;

enum {
    NSPT_OK = 0,
    NSPT_EINVAL = -1,  /* null / misaligned pointer, N < 1, Ntrunc < 0, batch < 1, Ntrunc > NSPT_MAX_NTRUNC */
    NSPT_ENOMEM = -2,  /* device or host allocation failed, or caller workspace too small */
    NSPT_ECUDA = -3,   /* CUDA runtime / launch error (text: nspt_strerror) */
    NSPT_EARCH = -4,   /* current device is not compute capability 10.x */
    NSPT_ETOOBIG = -5  /* nspt_series_mul_noalloc: the problem does not fit the static scratch array */
};

enum { NSPT_OP_SERIES_MUL = 0, NSPT_OP_STAPLE = 1, NSPT_OP_SERIES_EXP = 2 };

/* Largest supported truncation order: the transform length L = smallest power of two
 * >= 2*Ntrunc+1 must be <= 256 (Ntrunc <= 127; the paper uses Ntrunc <= 63). */
#define NSPT_MAX_NTRUNC 127

/*
 * C = A * B, the convolution product truncated at O(g^Ntrunc):
 *     C^(k) = sum_{l=0}^{k} A^(l) B^(k-l),  k = 0..Ntrunc     (eq. 2.5)
 * with the left factor always from A.  Computed by FFT-CONV (Steps 1-5,
 * eqs. 2.6-2.9): zero-padded forward transforms of length L along the order index for every
 * matrix element, one N x N complex matrix product per Fourier mode, inverse transform with
 * 1/L, orders above Ntrunc discarded.  L = smallest power of two >= 2*Ntrunc+1 (= 2*N_p of
 * the paper when Ntrunc = N_p - 1 = 2^s - 1); any Ntrunc in [0, 127] is accepted.
 * A, B, C: device pointers, (Ntrunc+1)*N*N elements each.
 */
int nspt_series_mul(const nspt_c128* A, const nspt_c128* B, nspt_c128* C, int N, int Ntrunc);

/*
 * batch independent products C_b = A_b * B_b (e.g. the four P_mu * U_mu of the link update,
 * PAPER.md:50, eq. 2.3; batching of independent transforms / products: PAPER.md:106).
 * Operand b starts at element offset b*(Ntrunc+1)*N*N.  Device pointers.
 */
int nspt_series_mul_batched(const nspt_c128* A, const nspt_c128* B, nspt_c128* C,
                            int N, int Ntrunc, int batch);

/*
 * nspt_series_mul for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): the same FFT-CONV (Steps 1-5, eqs. 2.6-2.9) by the same kernels on the FP64 tensor
 * pipe, with the three spectra A~, B~, C~ and the per-L tables in a static device array of NSPT_NOALLOC_SCRATCH_BYTES
 * inside the library instead of the workspace.  The call runs no cudaMalloc, cudaFree or other allocating routine; every
 * GPU that loads the library holds the array until the process exits.
 * A, B, C: device pointers as for nspt_series_mul (C may be one of the inputs); asynchronous on the library stream; the
 * order scale of nspt_set_order_scale applies; nspt_set_gemm_variant, nspt_set_conv_algorithm and nspt_set_workspace do not.
 * Limit: 3 * 16 * L * N * N + 16640 bytes <= NSPT_NOALLOC_SCRATCH_BYTES with L the transform length (N <= 104 at
 * N_trunc = 31, N <= 73 at N_trunc = 63, N <= 208 at N_trunc = 7); larger problems return NSPT_ETOOBIG and touch nothing.
 * All calls on one GPU share the array, and it keeps the last call's contents: nothing in it has to start from zero (every
 * byte a call reads it has written before), but two calls that overlap on the GPU -- issued to different streams without an
 * ordering between them, or from two host threads with different streams -- race on it.  Calls on one stream are safe.
 * The first call on a device loads the kernels (CUDA lazy loading) and takes the array's address, and a call whose
 * (N_trunc, order scale) differ from the previous call's copies 10 KB of tables from host memory first: under stream capture,
 * make one call with the same shape before the capture begins.
 */
#define NSPT_NOALLOC_SCRATCH_BYTES (32u << 20)
int nspt_series_mul_noalloc(const nspt_c128* A, const nspt_c128* B, nspt_c128* C, int N, int Ntrunc);

/*
 * The TEK staple for all four directions (eq. 2.3; eq. 2.2):
 *     S_mu = U_mu * [ sum_{nu != mu} ( z_{mu nu}   U_nu  * U_mu^+ * U_nu^+
 *                                    - z_{mu nu}^* U_nu^+ * U_mu^+ * U_nu ) ],  mu = 0..3,
 * every * truncated at O(g^Ntrunc); X^+ is the coefficient-wise conjugate transpose.
 * U[4], S[4]: HOST arrays of four DEVICE pointers to series of (Ntrunc+1)*N*N elements.
 * z: HOST 4x4 row-major array, z[4*mu+nu] = z_{mu nu}; the diagonal is ignored and the
 * second term uses conj(z[4*mu+nu]) exactly as the equation prints it.  z is not checked
 * for antisymmetry or unit modulus.
 */
int nspt_staple(const nspt_c128* const U[4], const nspt_c128 z[16], nspt_c128* const S[4],
                int N, int Ntrunc);

/*
 * The staple of ONE direction mu (0..3), same definition and arguments: the unit of work of the paper's multi-GPU scheme
 * ("we assign computational tasks, which are independent in the four-dimensional direction, on each GPU card";
 * every * stays inside one card, the updated links are exchanged once per step).  S_mu: device pointer, must not alias any
 * U[nu].  15 mode-wise products (nspt_staple shares intermediate products between directions: 36 for all four).
 */
int nspt_staple_dir(const nspt_c128* const U[4], const nspt_c128 z[16], int mu, nspt_c128* S_mu,
                    int N, int Ntrunc);

/*
 * E = exp(X) = sum_{m=0}^{Ntrunc} X^{*m} / m!, every power a chain of the star-product above, for a series
 * whose coefficient of g^0 vanishes; X^(0) is NOT read and is taken as zero (with X^(0) = 0 the power
 * X^{*m} starts at g^m, so the sum is finite and exact).  This is the exponential of the link update
 * U <- exp(i eps P) * U of the NSPT integrator ("solved with a symplectic integrator";
 * U-dot = i P * U, eq. 2.3), and of U = exp(i sum_k g^k H_k).  For Ntrunc >= 6 the sum is evaluated in the
 * Paterson-Stockmeyer arrangement, (s-1)+(r-1) star-products with s = ceil(sqrt(Ntrunc+1)), r = ceil((Ntrunc+1)/s)
 * (10 at Ntrunc = 31); below that by Horner with Ntrunc-1 products.  X is transformed once and all intermediate
 * results stay in frequency space.  Device pointers, (Ntrunc+1)*N*N elements; E may alias X.
 */
int nspt_series_exp(const nspt_c128* X, nspt_c128* E, int N, int Ntrunc);
/* batch independent exponentials E_b = exp(X_b) (the four links of an update); element b at offset b*(Ntrunc+1)*N*N. */
int nspt_series_exp_batched(const nspt_c128* X, nspt_c128* E, int N, int Ntrunc, int batch);

/*
 * The link update of the NSPT integrator (U-dot = i P * U, "solved with a symplectic integrator"):
 *     Unew = exp(i eps P) * U,
 * P a series of Hermitian coefficients whose g^0 coefficient is NOT read and taken as zero (as in nspt_series_exp), eps the
 * real step.  One call: the exponential is formed in frequency space as above (the factor i eps only changes the coefficients
 * (i eps)^m / m!), re-truncated, multiplied by the spectrum of U and transformed back once.  Device pointers,
 * (Ntrunc+1)*N*N elements each; Unew may alias U or P.  The batched form updates `batch` links (the four directions).
 */
int nspt_link_update(const nspt_c128* P, const nspt_c128* U, double eps, nspt_c128* Unew, int N, int Ntrunc);
int nspt_link_update_batched(const nspt_c128* P, const nspt_c128* U, double eps, nspt_c128* Unew, int N, int Ntrunc, int batch);

/*
 * The force of eq. 2.3 from a staple series, order by order:
 *     F^(k) = i c [ S^(k) - S^(k)+ - Tr(S^(k) - S^(k)+)/N ],   k = 0..Ntrunc,
 * Hermitian and traceless.  c is the real coefficient the paper writes as beta; what is left of it after the
 * paper's rescaling of the fictitious time is not recoverable from the text, so the caller supplies it.
 * Device pointers, (Ntrunc+1)*N*N elements; F must NOT alias S (NSPT_EINVAL if F == S).
 */
int nspt_force(const nspt_c128* S, nspt_c128* F, double c, int N, int Ntrunc);

/* Host-buffer forms of nspt_series_mul, nspt_series_mul_batched and nspt_staple: same semantics, HOST pointers for the series,
 * host<->device copies inside the call, everything synchronised on return.  For batch > 1 the batched form overlaps the
 * copy-in of element b+1, the product of element b and the copy-out of element b-1 on internal copy streams. */
int nspt_series_mul_host(const nspt_c128* A, const nspt_c128* B, nspt_c128* C, int N, int Ntrunc);
int nspt_series_mul_batched_host(const nspt_c128* A, const nspt_c128* B, nspt_c128* C,
                                 int N, int Ntrunc, int batch);
int nspt_staple_host(const nspt_c128* const U[4], const nspt_c128 z[16], nspt_c128* const S[4],
                     int N, int Ntrunc);

/* ------------------------------------------------------------------------- context calls */

/* CUDA stream (a cudaStream_t passed as void*) all later calls enqueue on.  Default: the
 * legacy default stream (NULL). */
int nspt_set_stream(void* cuda_stream);

/* Optional magnitude balancing: coefficient k is multiplied by s^k before the forward
 * transform and the result by s^-k after the inverse one; exact in exact arithmetic because
 * (s^l)(s^(k-l)) = s^k.  s = 1 (default) switches it off.  s must be finite and > 0. */
int nspt_set_order_scale(double s);

/* Bytes of device workspace a call needs (op = NSPT_OP_SERIES_MUL or
 * NSPT_OP_SERIES_EXP with theirs, or NSPT_OP_STAPLE, batch ignored).  nspt_force needs none.  batch <= 65535.
 * For NSPT_OP_SERIES_MUL this is what the general FFT-CONV needs: the one-launch forms the library takes for very small
 * matrices (nspt_debug.h, nspt_set_conv_algorithm) use no workspace at all. */
int nspt_workspace_bytes(int N, int Ntrunc, int batch, int op, size_t* out);

/* Give the library a caller-owned device workspace (256-byte aligned).  Calls that need more
 * return NSPT_ENOMEM.  Pass (NULL, 0) to go back to the library-owned, grow-only workspace. */
int nspt_set_workspace(void* dptr, size_t bytes);

/* Free all library-owned device / host memory and cached plans. */
int nspt_release(void);

/* Text for an error code; for NSPT_ECUDA the text of the last CUDA error seen. */
const char* nspt_strerror(int code);

/* Version: major*10000 + minor*100 + patch. */
int nspt_version(void);

#ifdef __cplusplus
}
#endif
#endif /* NSPT_H */
