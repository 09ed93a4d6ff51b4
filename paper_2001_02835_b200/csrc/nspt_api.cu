// nspt_api.cu -- the C ABI of libnspt (include/nspt.h): context, plans, workspace, and the
// composition of the kernels into nspt_series_mul / _batched (FFT-CONV Steps 1-5,
// PAPER.md:68-102) and nspt_staple (eq. 2.3).
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>

#include "nspt_internal.cuh"

namespace nspt {
namespace {

struct Plan {
    int L, n;
    double s;
    double2* tw_fwd = nullptr;
    double2* tw_inv = nullptr;
    double* scale_in = nullptr;   // null when s == 1
    double* scale_out = nullptr;  // s^-k / L
};

struct ProfEvent {
    cudaEvent_t a, b;
    int stage;
};

struct Context {
    std::mutex mu;
    cudaStream_t stream = nullptr;
    cudaEvent_t order_event = nullptr;   // orders a newly set stream after the work of the previous one
    bool used = false;                   // a kernel has been enqueued since the library was loaded / released
    double order_scale = 1.0;
    int gemm_variant = -1;               // nspt_debug.h: -1 = automatic
    int conv_algorithm = 0;              // 0 = automatic, 1 = FFT-CONV, 2 = Naive-CONV, 3 = FFT-CONV in one launch (nspt_debug.h)
    bool arch_checked = false;
    // workspace
    void* user_ws = nullptr;
    size_t user_ws_bytes = 0;
    void* own_ws = nullptr;
    size_t own_ws_bytes = 0;
    // staging for the _host calls; copy streams and events of the pipelined batched call
    void* stage_dev = nullptr;
    size_t stage_dev_bytes = 0;
    cudaStream_t h2d = nullptr, d2h = nullptr;
    std::vector<cudaEvent_t> copy_events;
    std::vector<Plan> plans;
    // per-mode maxima of the INT8 product path that are known to be zero (left so by the last product kernel)
    const void* clean_maxbits = nullptr;
    size_t clean_maxbits_count = 0;
    // profiling
    bool profiling = false;
    std::vector<ProfEvent> prof_used;
    std::vector<ProfEvent> prof_free;
    double prof_ms[ST_COUNT] = {};
    long long prof_n[ST_COUNT] = {};
    long long launches = 0;
    char cuda_msg[256] = "no CUDA error recorded";
};

// One context per CUDA device, selected by the device current at the call (cudaGetDevice): plans, workspace, staging,
// stream and profiling state never cross devices, so one process can drive several GPUs (one direction of the TEK model per
// GPU) from one or several host threads.
constexpr int MAX_DEVICES = 64;
Context g_contexts[MAX_DEVICES];
thread_local Context* g_current = &g_contexts[0];
#define g (*g_current)

struct ContextLock {
    bool ok = false;
    Context* c = nullptr;
    ContextLock() {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess) {   // no device at all: argument checks still work (context 0)
            cudaGetLastError();
            dev = 0;
        }
        if (dev < 0 || dev >= MAX_DEVICES) return;
        c = &g_contexts[dev];
        c->mu.lock();
        g_current = c;
        ok = true;
    }
    ~ContextLock() {
        if (ok) c->mu.unlock();
    }
};
#define NSPT_LOCK()     \
    ContextLock lk__;   \
    if (!lk__.ok) return NSPT_ECUDA

int cuda_fail(cudaError_t e) {
    snprintf(g.cuda_msg, sizeof(g.cuda_msg), "CUDA error: %s", cudaGetErrorString(e));
    if (e == cudaErrorMemoryAllocation) return NSPT_ENOMEM;
    return NSPT_ECUDA;
}

#define NSPT_CUDA(x)                                 \
    do {                                             \
        cudaError_t e__ = (x);                       \
        if (e__ != cudaSuccess) return cuda_fail(e__); \
    } while (0)

int check_arch() {
    if (g.arch_checked) return NSPT_OK;
    int dev = 0;
    NSPT_CUDA(cudaGetDevice(&dev));
    int major = 0;
    NSPT_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) return NSPT_EARCH;
    g.arch_checked = true;
    return NSPT_OK;
}

int check_dims(int N, int Ntrunc, int batch) {
    if (N < 1 || Ntrunc < 0 || batch < 1) return NSPT_EINVAL;
    if (Ntrunc > NSPT_MAX_NTRUNC || batch > 65535) return NSPT_EINVAL;
    if ((long long)N * N > (1ll << 40)) return NSPT_EINVAL;
    return NSPT_OK;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

// ---- plans ---------------------------------------------------------------------------------
int get_plan(int L, int n, double s, PlanTables* out) {
    for (const Plan& p : g.plans) {
        if (p.L == L && p.n == n && p.s == s) {
            *out = PlanTables{p.tw_fwd, p.tw_inv, p.scale_in, p.scale_out, 1.0 / L};
            return NSPT_OK;
        }
    }
    Plan p;
    p.L = L;
    p.n = n;
    p.s = s;
    std::vector<double2> f(L), b(L);
    const long double two_pi = 6.283185307179586476925286766559005768L;
    for (int m = 0; m < L; ++m) {
        // exact values on the axes and diagonals, long double elsewhere
        long double ang = two_pi * (long double)m / (long double)L;
        double c = (double)cosl(ang), sn = (double)sinl(ang);
        if ((4 * m) % L == 0) {  // multiples of pi/2
            const int q = (4 * m) / L;
            c = (q == 0) ? 1.0 : (q == 2 ? -1.0 : 0.0);
            sn = (q == 1) ? 1.0 : (q == 3 ? -1.0 : 0.0);
        }
        f[m] = make_double2(c, sn);   // w^m,  w = exp(+2 pi i / L)   (eq. 2.7)
        b[m] = make_double2(c, -sn);  // w^-m                          (eq. 2.9)
    }
    std::vector<double> so(n), si(n);
    for (int k = 0; k < n; ++k) {
        si[k] = (double)powl((long double)s, (long double)k);
        so[k] = (double)(powl((long double)s, -(long double)k) / (long double)L);
    }
    NSPT_CUDA(cudaMalloc(&p.tw_fwd, sizeof(double2) * L));
    NSPT_CUDA(cudaMalloc(&p.tw_inv, sizeof(double2) * L));
    NSPT_CUDA(cudaMalloc(&p.scale_out, sizeof(double) * n));
    NSPT_CUDA(cudaMemcpy(p.tw_fwd, f.data(), sizeof(double2) * L, cudaMemcpyHostToDevice));
    NSPT_CUDA(cudaMemcpy(p.tw_inv, b.data(), sizeof(double2) * L, cudaMemcpyHostToDevice));
    NSPT_CUDA(cudaMemcpy(p.scale_out, so.data(), sizeof(double) * n, cudaMemcpyHostToDevice));
    if (s != 1.0) {
        NSPT_CUDA(cudaMalloc(&p.scale_in, sizeof(double) * n));
        NSPT_CUDA(cudaMemcpy(p.scale_in, si.data(), sizeof(double) * n, cudaMemcpyHostToDevice));
    }
    g.plans.push_back(p);
    *out = PlanTables{p.tw_fwd, p.tw_inv, p.scale_in, p.scale_out, 1.0 / L};
    return NSPT_OK;
}

// ---- workspace -----------------------------------------------------------------------------
size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Spectra are packed back to back (a whole number of N x N matrices apart) so that one tensor map can address
// several of them by mode offset; 16-byte alignment is all the TMA maps need.
size_t spectrum_bytes(const FreqLayout& f, int batch) { return f.spectrum_doubles(batch) * 8; }

// Paterson-Stockmeyer split of exp(X) = sum_{m <= n} X^m / m!: powers X^1..X^s and r = ceil((n+1)/s) block polynomials
// (series_exp_device).  Below n = 6 the plain Horner form is used (s = 0).
void exp_split(int Ntrunc, int* s, int* r) {
    *s = 0;
    *r = 0;
    if (Ntrunc < 6) return;
    int q = 1;
    while (q * q < Ntrunc + 1) ++q;
    *s = q;                                  // <= 12 for Ntrunc <= 127
    *r = (Ntrunc + 1 + q - 1) / q;           // <= 12
}

// The B-operand tensor map of the mode-wise product reads up to 112 bytes past the last row of the last spectrum (its
// last 128-byte chunk of a row runs into what follows, nspt_zgemm.cu), so every workspace ends with a 256-byte pad.
constexpr size_t WS_PAD = 256;

// Mode-wise product of nspt_series_mul[_batched] on the INT8 tensor cores (nspt_ozaki.cu) or on the FP64 tensor pipe
// (nspt_zgemm.cu).  Automatic choice, measured on one B200: the INT8 path pays a slicing pass of O(N^2 L) bytes
// for a product kernel that is about twice as fast, so it wins from N = 192 up -- from N = 160 for the staple and the
// exponential (`chained`), whose slicing is shared between products and whose grouped launches have no partial last wave
// (N = 169: staple 3.17 -> 2.94 ms, four exponentials 3.90 -> 3.49 ms; a single product 108 -> 125 us); between 129 and 159 the
// second 128-column tile is nearly empty and the FP64 pipe wins everywhere; at L = 16 (N_trunc <= 7) the threshold is 192 for all
// operations (N = 225: product 64 -> 56 us, staple 1.66 -> 1.25 ms; N = 169: staple 0.85 -> 0.85 ms, four exponentials 0.43 -> 0.46 ms).
// It is limited to L <= 128 (N_trunc <= 63), where
// its error stays two orders of magnitude below the 1e-11 tolerance on series shaped like the paper's (at N_trunc = 127 the
// margin shrinks to a factor of five to eight: that range stays on the FP64 pipe unless the variant is forced).
bool use_int8(const FreqLayout& f, bool chained = false) {
    if (f.L < 16) return false;   // the slicing pass takes its maxima from the TMA transform kernels
    if (g.gemm_variant == 2 || g.gemm_variant == 4) return true;
    if (g.gemm_variant != -1) return false;
    return f.N >= ((chained && f.L >= 32) ? 160 : 192) && f.L <= 128;
}

// INT8 staple (staple_device): slice slots per layout and per-mode maxima tables (see the slot maps there)
constexpr int STAPLE_NQ = 25, STAPLE_NR = 19, STAPLE_MAXBITS = 22;

// per-mode maxima (one 64-bit pattern per mode) recorded by the transforms for the INT8 path
size_t maxbits_bytes(int modes) { return align_up((size_t)NSPT_MAX_BUCKETS * modes * sizeof(unsigned long long), 256); }   // all copies

size_t ws_bytes_for(const FreqLayout& f, int batch, int op) {
    if (op == NSPT_OP_SERIES_MUL && use_int8(f))
        return 3 * spectrum_bytes(f, batch) + WS_PAD + maxbits_bytes(2 * batch * f.L) + ozaki_store_bytes(f, batch * f.L, 1, 1);
    if (op == NSPT_OP_STAPLE) {
        size_t b = 30 * spectrum_bytes(f, 1) + WS_PAD;
        if (use_int8(f, true)) b += maxbits_bytes(STAPLE_MAXBITS * f.L) + ozaki_store_bytes(f, f.L, STAPLE_NQ, STAPLE_NR);
        return b;
    }
    if (op == NSPT_OP_SERIES_EXP) {
        int s, r;
        exp_split(f.n - 1, &s, &r);
        size_t b = (size_t)(s ? s + r : 3) * spectrum_bytes(f, batch) + WS_PAD;
        if (s && use_int8(f, true)) b += maxbits_bytes((s + r + 1) * batch * f.L) + ozaki_store_bytes(f, batch * f.L, s + r, s);
        return b;
    }
    return 3 * spectrum_bytes(f, batch) + WS_PAD;
}

int get_workspace(size_t bytes, char** out, bool keeps_maxima = false) {
    if (!keeps_maxima) g.clean_maxbits = nullptr;   // every caller but the INT8 product overwrites the region of its maxima
    if (g.user_ws) {
        if (g.user_ws_bytes < bytes) return NSPT_ENOMEM;
        *out = static_cast<char*>(g.user_ws);
        return NSPT_OK;
    }
    if (g.own_ws_bytes < bytes) {
        g.clean_maxbits = nullptr;
        if (g.own_ws) {
            NSPT_CUDA(cudaStreamSynchronize(g.stream));
            NSPT_CUDA(cudaFree(g.own_ws));
            g.own_ws = nullptr;
            g.own_ws_bytes = 0;
        }
        NSPT_CUDA(cudaMalloc(&g.own_ws, bytes));
        g.own_ws_bytes = bytes;
    }
    *out = static_cast<char*>(g.own_ws);
    return NSPT_OK;
}

int get_staging(size_t bytes, char** out) {
    if (g.stage_dev_bytes < bytes) {
        if (g.stage_dev) {
            NSPT_CUDA(cudaStreamSynchronize(g.stream));
            NSPT_CUDA(cudaFree(g.stage_dev));
            g.stage_dev = nullptr;
            g.stage_dev_bytes = 0;
        }
        NSPT_CUDA(cudaMalloc(&g.stage_dev, bytes));
        g.stage_dev_bytes = bytes;
    }
    *out = static_cast<char*>(g.stage_dev);
    return NSPT_OK;
}

// ---- profiling -----------------------------------------------------------------------------
int prof_flush() {
    if (g.prof_used.empty()) return NSPT_OK;
    NSPT_CUDA(cudaStreamSynchronize(g.stream));
    for (ProfEvent& e : g.prof_used) {
        float ms = 0.f;
        NSPT_CUDA(cudaEventElapsedTime(&ms, e.a, e.b));
        g.prof_ms[e.stage] += ms;
        g.prof_n[e.stage] += 1;
        g.prof_free.push_back(e);
    }
    g.prof_used.clear();
    return NSPT_OK;
}

struct StageTimer {
    bool on = false;
    ProfEvent ev{};
    int begin(int stage) {
        g.launches += 1;
        g.used = true;
        if (!g.profiling) return NSPT_OK;
        if (g.prof_used.size() >= 4096) {
            int rc = prof_flush();
            if (rc) return rc;
        }
        if (!g.prof_free.empty()) {
            ev = g.prof_free.back();
            g.prof_free.pop_back();
        } else {
            NSPT_CUDA(cudaEventCreate(&ev.a));
            NSPT_CUDA(cudaEventCreate(&ev.b));
        }
        ev.stage = stage;
        on = true;
        NSPT_CUDA(cudaEventRecord(ev.a, g.stream));
        return NSPT_OK;
    }
    int end() {
        if (!on) return NSPT_OK;
        NSPT_CUDA(cudaEventRecord(ev.b, g.stream));
        g.prof_used.push_back(ev);
        on = false;
        return NSPT_OK;
    }
};

#define NSPT_TRY(x)            \
    do {                       \
        int rc__ = (x);        \
        if (rc__) return rc__; \
    } while (0)

// Each helper = one kernel launch, bracketed for the profiler.
int k_forward(const FreqLayout& f, const PlanTables& t, int batch, const nspt_c128* s0, double* d0,
              const nspt_c128* s1, double* d1) {
    StageTimer tm;
    NSPT_TRY(tm.begin(ST_FWD));
    NSPT_CUDA(launch_fft_forward(f, t, batch, s0, d0, s1, d1, g.stream));
    return tm.end();
}
int k_inverse(const FreqLayout& f, const PlanTables& t, int batch, const double* src, nspt_c128* dst) {
    StageTimer tm;
    NSPT_TRY(tm.begin(ST_INV));
    NSPT_CUDA(launch_fft_inverse(f, t, batch, src, dst, g.stream));
    return tm.end();
}
int k_retrunc(const FreqLayout& f, const PlanTables& t, int batch, const double* src, double* dst,
              unsigned long long* maxbits = nullptr, size_t maxbits_stride = 0) {
    StageTimer tm;
    NSPT_TRY(tm.begin(ST_RETRUNC));
    NSPT_CUDA(launch_fft_retruncate(f, t, batch, src, dst, g.stream, maxbits, maxbits_stride));
    return tm.end();
}
// maxbits_stride: distance between the copies of the maxima of the calling operation (all its jobs share it)
int k_slice(const FreqLayout& f, const OzStore& store, OzSliceJob* jobs, int njobs, size_t maxbits_stride) {
    for (int i = 0; i < njobs; ++i) jobs[i].maxbits_stride = maxbits_stride;
    StageTimer tm;
    NSPT_TRY(tm.begin(ST_SLICE));
    NSPT_CUDA(launch_ozaki_slice(f, store, jobs, njobs, g.stream));
    return tm.end();
}
int k_gemm_i8(const FreqLayout& f, const OzStore& store, const OzGemmGroup* groups, int ngroups) {
    StageTimer tm;
    NSPT_TRY(tm.begin(ST_GEMM));
    NSPT_CUDA(launch_ozaki_gemm(f, store, groups, ngroups, g.stream, g.gemm_variant == 4));
    return tm.end();
}
int k_dagger(const FreqLayout& f, int batch, const double* src, double* dst) {
    StageTimer tm;
    NSPT_TRY(tm.begin(ST_OTHER));
    NSPT_CUDA(launch_freq_dagger(f, batch, src, dst, g.stream));
    return tm.end();
}
// kernel of nspt_zgemm.cu behind the staple, the exponential and the FP64 products: 0 = debug, 1 = block-scheduled, 3 = persistent
int dmma_variant() { return (g.gemm_variant == 0 || g.gemm_variant == 3) ? g.gemm_variant : 1; }

int k_gemm(const FreqLayout& f, int batch, const double* A, const double* B, const GemmOut& out) {
    StageTimer tm;
    NSPT_TRY(tm.begin(ST_GEMM));
    NSPT_CUDA(launch_zgemm_modes(f, batch, A, B, out, dmma_variant(), g.stream));
    return tm.end();
}
int k_gemm_groups(const FreqLayout& f, const GemmGroup* groups, int ngroups, int batch = 1) {
    StageTimer tm;
    NSPT_TRY(tm.begin(ST_GEMM));
    NSPT_CUDA(launch_zgemm_groups(f, batch, groups, ngroups, dmma_variant(), g.stream));
    return tm.end();
}
int k_gemm(const FreqLayout& f, int batch, const double* A, const double* B, double* C) {
    GemmOut out;
    out.C = C;
    return k_gemm(f, batch, A, B, out);
}

// ---- the products --------------------------------------------------------------------------
// Naive-CONV or FFT-CONV (PAPER.md:66 vs :68-102).  The direct evaluation needs N^3 n(n+1)/2 matrix multiplications against
// N^3 L plus three transform passes, but it is a single launch without workspace traffic: it wins where the product is
// launch- or transform-bound (see DESIGN.md 5.5 for the measured crossover).  It reads A and B while it writes C, so an
// output that aliases an input always takes FFT-CONV.
// Automatic choice of the one-launch FFT-CONV: its N^2 CTAs each redo the transforms of 2N series, so its time grows like
// N^3 L, against three launches (12.5 us through the binding) of the general path.  Measured per product (one B200, us, general /
// one-launch): N = 8, N_trunc = 63: 12.7 / 9.8; N = 12, 31: 12.7 / 9.9; N = 16, 15: 12.6 / 9.2; N = 20, 7: 12.9 / 10.7;
// N = 16, 31: 12.5 / 12.2; N = 12, 63: 12.5 / 13.1; N = 20, 15: 12.5 / 13.5; N = 24, 31: 13.5 / 29.3.
constexpr double FUSED_SMALL_MAX_N3L = 150000.0;

bool use_naive_conv(const FreqLayout& f, const nspt_c128* A, const nspt_c128* B, const nspt_c128* C) {
    if (C == A || C == B || g.gemm_variant == 0 || g.gemm_variant == 2 || g.gemm_variant == 4) return false;
    if (g.conv_algorithm == 1) return false;
    if (g.conv_algorithm == 2) return true;
    // measured crossover (one B200, time per product through the binding): the direct form is one launch
    // (7.5 us) against three (13 us) and wins while its n(n+1)/2 products stay a fraction of a wave
    if (f.n == 1) return true;                 // a single matrix product: nothing to transform
    if (f.N <= 16) return f.n <= 8;
    if (f.N <= 32) return f.n <= 4;
    if (f.N <= 64) return f.n <= 2;
    return false;
}

// FFT-CONV in one launch (nspt_small.cu) where the general path is bound by its three launches.  Like Naive-CONV it reads
// A and B while it writes C, so an aliased output takes the general path.
bool use_fused_small(const FreqLayout& f, int batch, const nspt_c128* A, const nspt_c128* B, const nspt_c128* C) {
    if (C == A || C == B || (g.gemm_variant != -1 && g.gemm_variant != 1)) return false;
    if (!fused_small_eligible(f, batch)) return false;
    if (g.conv_algorithm == 3) return true;
    if (g.conv_algorithm != 0) return false;
    return (double)f.N * f.N * f.N * f.L <= FUSED_SMALL_MAX_N3L;
}

int series_mul_device(const nspt_c128* A, const nspt_c128* B, nspt_c128* C, int N, int Ntrunc, int batch) {
    NSPT_TRY(check_dims(N, Ntrunc, batch));
    if (!A || !B || !C || !aligned16(A) || !aligned16(B) || !aligned16(C)) return NSPT_EINVAL;
    NSPT_TRY(check_arch());
    const FreqLayout f = make_layout(N, Ntrunc);
    if (!fft_length_supported(f.L)) return NSPT_EINVAL;
    if (use_naive_conv(f, A, B, C)) {
        // eq. 2.5 directly: one launch, no transforms, no workspace
        StageTimer tm;
        NSPT_TRY(tm.begin(ST_GEMM));
        NSPT_CUDA(launch_naive_conv(f, batch, A, B, C, g.stream));
        return tm.end();
    }
    PlanTables t;
    NSPT_TRY(get_plan(f.L, f.n, g.order_scale, &t));
    if (use_fused_small(f, batch, A, B, C)) {
        // Steps 1-4 in one launch, one CTA per output series (nspt_small.cu)
        StageTimer tm;
        NSPT_TRY(tm.begin(ST_GEMM));
        NSPT_CUDA(launch_fused_small(f, t, batch, A, B, C, g.stream));
        return tm.end();
    }
    char* ws = nullptr;
    NSPT_TRY(get_workspace(ws_bytes_for(f, batch, NSPT_OP_SERIES_MUL), &ws, use_int8(f)));
    const size_t sb = spectrum_bytes(f, batch);
    double* At = reinterpret_cast<double*>(ws);
    double* Bt = reinterpret_cast<double*>(ws + sb);
    double* Ct = reinterpret_cast<double*>(ws + 2 * sb);
    if (use_int8(f)) {
        const int modes = batch * f.L;
        unsigned long long* mbA = reinterpret_cast<unsigned long long*>(ws + 3 * sb + WS_PAD);
        unsigned long long* mbB = mbA + modes;
        const size_t mbs = (size_t)2 * modes, mbn = (size_t)NSPT_MAX_BUCKETS * mbs;   // stride between the copies, all entries
        const OzStore store = ozaki_store(f, modes, 1, 1, ws + 3 * sb + WS_PAD + maxbits_bytes(2 * modes));
        {
            // Steps 1-2 (eqs. 2.6-2.7); the transform also records max(|re|, |im|) of every mode of both spectra
            // (the maxima start from zero: the product kernel of the previous call has cleared them, else a memset does)
            if (g.clean_maxbits != mbA || g.clean_maxbits_count != mbn)
                NSPT_CUDA(cudaMemsetAsync(mbA, 0, sizeof(unsigned long long) * mbn, g.stream));
            g.clean_maxbits = nullptr;
            StageTimer tm;
            NSPT_TRY(tm.begin(ST_FWD));
            NSPT_CUDA(launch_fft_forward(f, t, batch, A, At, B, Bt, g.stream, false, mbA, mbB, mbs));
            NSPT_TRY(tm.end());
        }
        {
            // both spectra cut into seven int8 slices per plane, fixed point relative to the largest element of each mode:
            // A~ as a left factor (QUAD layout), B~ as a right factor (ROWS layout)
            OzSliceJob jobs[2];
            jobs[0].X = At;
            jobs[0].maxbits = mbA;
            jobs[0].maxbits_stride = mbs;
            jobs[0].quad_slot = 0;
            jobs[1].X = Bt;
            jobs[1].maxbits = mbB;
            jobs[1].maxbits_stride = mbs;
            jobs[1].rows_slot = 0;
            StageTimer tm;
            NSPT_TRY(tm.begin(ST_SLICE));
            NSPT_CUDA(launch_ozaki_slice(f, store, jobs, 2, g.stream));
            NSPT_TRY(tm.end());
        }
        // Step 3 (eq. 2.8): exact integer products on the INT8 tensor cores, recombined in FP64
        OzGemmGroup grp;
        grp.quad_slot = 0;
        grp.rows_slot = 0;
        grp.A = At;
        grp.B = Bt;
        grp.out.C = Ct;
        StageTimer tm;
        NSPT_TRY(tm.begin(ST_GEMM));
        NSPT_CUDA(launch_ozaki_gemm(f, store, &grp, 1, g.stream, g.gemm_variant == 4, mbA, (int)mbn));
        NSPT_TRY(tm.end());
        g.clean_maxbits = mbA;
        g.clean_maxbits_count = mbn;
    } else {
        // Steps 1-2 (eqs. 2.6-2.7): zero-padded forward transforms of A and B, one launch
        NSPT_TRY(k_forward(f, t, batch, A, At, B, Bt));
        // Step 3 (eq. 2.8): mode-wise matrix products on the FP64 tensor pipe
        NSPT_TRY(k_gemm(f, batch, At, Bt, Ct));
    }
    // Steps 4-5 (eq. 2.9): inverse transform, 1/L, truncation
    NSPT_TRY(k_inverse(f, t, batch, Ct, C));
    return NSPT_OK;
}

// exp(X) = sum_{m <= n} X^{*m}/m!, n = Ntrunc, in frequency space (reading c17).  X~ is transformed once, every
// product is followed by a re-truncation pass (a length-L cyclic transform protects one product only), and the last
// product goes straight to the inverse transform.
//   n >= 6: Paterson-Stockmeyer.  With s = ceil(sqrt(n+1)), r = ceil((n+1)/s):
//       exp(X) = sum_{j<r} (X^s)^j B_j(X),   B_j(X) = sum_{i<s} X^i / (s j + i)!   (terms beyond m = n dropped),
//     the powers X^2..X^s by doubling (X^2; X^3, X^4; X^5..X^8; ...: each wave ONE grouped launch and one batched
//     re-truncation), all B_j by one elementwise pass over the powers, then Horner in X^s: r-1 products whose
//     epilogue accumulates acc * X^s onto B_j.  s - 1 + r - 1 products instead of n - 1 (10 instead of 30 at n = 31).
//   n < 6: plain Horner, T_n = 1 + X/n, T_m = 1 + (X * T_{m+1})/m, exp(X) = T_1; the GEMM epilogue scales by 1/m and
//     adds the identity series (the unit matrix at every mode).
// With a prefactor lambda and a second series U the same machinery gives E = exp(lambda X) * U without leaving frequency
// space (the link update U <- exp(i eps P) * U): lambda only changes the coefficients lambda^m / m! of the block
// polynomials (or the Horner factors), and the product with U~ follows the last Horner step after one re-truncation pass.
int series_exp_device(const nspt_c128* X, nspt_c128* E, int N, int Ntrunc, int batch, Cplx lambda = Cplx{1.0, 0.0},
                      const nspt_c128* Umul = nullptr) {
    NSPT_TRY(check_dims(N, Ntrunc, batch));
    if (!X || !E || !aligned16(X) || !aligned16(E) || (Umul && !aligned16(Umul))) return NSPT_EINVAL;
    NSPT_TRY(check_arch());
    const FreqLayout f = make_layout(N, Ntrunc);
    if (!fft_length_supported(f.L)) return NSPT_EINVAL;
    PlanTables t;
    NSPT_TRY(get_plan(f.L, f.n, g.order_scale, &t));
    char* ws = nullptr;
    NSPT_TRY(get_workspace(ws_bytes_for(f, batch, NSPT_OP_SERIES_EXP), &ws));
    const size_t sb = spectrum_bytes(f, batch);
    double* Xt = reinterpret_cast<double*>(ws);
    double* Tt = reinterpret_cast<double*>(ws + sb);
    double* Pt = reinterpret_cast<double*>(ws + 2 * sb);
    int ps, pr;
    exp_split(Ntrunc, &ps, &pr);
    const bool i8 = ps && use_int8(f, true);
    const int modes = batch * f.L;
    // INT8 path (use_int8): per-mode maxima of spectrum i (0-based: X^1..X^s, then B_0..B_{r-1}) and the slice store, QUAD slot
    // = spectrum index (left factors: powers and Horner sums), ROWS slot = power index (right factors: X^1..X^s)
    unsigned long long* mb = nullptr;
    OzStore store;
    if (i8) {
        char* extra = ws + (size_t)(ps + pr) * sb + WS_PAD;
        mb = reinterpret_cast<unsigned long long*>(extra);
        store = ozaki_store(f, modes, ps + pr, ps, extra + maxbits_bytes((ps + pr + 1) * modes));
        NSPT_CUDA(cudaMemsetAsync(mb, 0, sizeof(unsigned long long) * NSPT_MAX_BUCKETS * (size_t)(ps + pr + 1) * modes, g.stream));
    }
    const size_t mbs = (size_t)(ps + pr + 1) * modes;   // distance between the copies of the maxima (one extra table: U~)
    const bool unit_lambda = lambda.re == 1.0 && lambda.im == 0.0;
    {   // X~ with the coefficient of g^0 taken as zero
        StageTimer tm;
        NSPT_TRY(tm.begin(ST_FWD));
        NSPT_CUDA(launch_fft_forward(f, t, batch, X, Xt, nullptr, nullptr, g.stream, true, mb, nullptr, mbs));
        NSPT_TRY(tm.end());
    }
    if (ps) {
        auto pw = [&](int i) { return reinterpret_cast<double*>(ws + (size_t)(i - 1) * sb); };     // spectrum of X^i, i = 1..s
        auto bj = [&](int j) { return reinterpret_cast<double*>(ws + (size_t)(ps + j) * sb); };    // B_j, later the Horner sums
        // which powers serve as left factors (QUAD layout: the doubling bases X^1, X^2, X^4, ...) and as right factors (ROWS
        // layout: X^1 .. X^cnt of the later waves, and X^s for the Horner steps); the others are only read by the block polynomials
        bool left[13] = {}, right[13] = {};
        for (int h = 1; h < ps;) {
            const int cnt = (ps - h) < h ? (ps - h) : h;
            left[h] = true;
            for (int i = 1; i <= cnt; ++i) right[i] = true;
            h += cnt;
        }
        right[ps] = true;
        auto slice_powers = [&](int first, int cnt) -> int {   // X^first .. X^(first+cnt-1) into the layouts they are needed in
            OzSliceJob jobs[12];
            int nj = 0;
            for (int i = 0; i < cnt; ++i) {
                const int pwr = first + i;
                if (!left[pwr] && !right[pwr]) continue;
                jobs[nj].X = pw(pwr);
                jobs[nj].maxbits = mb + (size_t)(pwr - 1) * modes;
                jobs[nj].quad_slot = left[pwr] ? pwr - 1 : -1;
                jobs[nj].rows_slot = right[pwr] ? pwr - 1 : -1;
                ++nj;
            }
            return nj ? k_slice(f, store, jobs, nj, mbs) : NSPT_OK;
        };
        if (i8) NSPT_TRY(slice_powers(1, 1));
        // powers by doubling: with X^1..X^h known, X^(h+i) = X^h * X^i for i = 1..min(h, s-h)
        for (int h = 1; h < ps;) {
            const int cnt = (ps - h) < h ? (ps - h) : h;
            if (i8) {
                OzGemmGroup gr[12];
                for (int i = 1; i <= cnt; ++i) {
                    gr[i - 1].quad_slot = h - 1;
                    gr[i - 1].rows_slot = i - 1;
                    gr[i - 1].A = pw(h);
                    gr[i - 1].B = pw(i);
                    gr[i - 1].out.C = pw(h + i);
                }
                NSPT_TRY(k_gemm_i8(f, store, gr, cnt));
                NSPT_TRY(k_retrunc(f, t, cnt * batch, pw(h + 1), pw(h + 1), mb + (size_t)h * modes, mbs));
                NSPT_TRY(slice_powers(h + 1, cnt));
            } else {
                GemmGroup gr[12];
                for (int i = 1; i <= cnt; ++i) {
                    gr[i - 1].A = pw(h);
                    gr[i - 1].B = pw(i);
                    gr[i - 1].out.C = pw(h + i);
                }
                NSPT_TRY(k_gemm_groups(f, gr, cnt, batch));
                NSPT_TRY(k_retrunc(f, t, cnt * batch, pw(h + 1), pw(h + 1)));   // the new powers are contiguous
            }
            h += cnt;
        }
        {   // all block polynomials in one pass over X^1..X^(s-1)
            double coef[144], coef_im[144];
            for (int j = 0; j < pr; ++j)
                for (int i = 0; i < ps; ++i) {
                    const int m = ps * j + i;
                    // lambda^m / m!, in long double
                    long double cr = 1.0L, ci = 0.0L;
                    for (int q = 1; q <= m; ++q) {
                        const long double nr = (cr * lambda.re - ci * lambda.im) / q, ni = (cr * lambda.im + ci * lambda.re) / q;
                        cr = nr;
                        ci = ni;
                    }
                    coef[j * ps + i] = (m <= Ntrunc) ? (double)cr : 0.0;
                    coef_im[j * ps + i] = (m <= Ntrunc) ? (double)ci : 0.0;
                }
            StageTimer tm;
            NSPT_TRY(tm.begin(ST_POLY));
            NSPT_CUDA(launch_freq_block_polys(f, batch, pw(1), bj(0), ps, pr, coef, g.stream, unit_lambda ? nullptr : coef_im));
            NSPT_TRY(tm.end());
        }
        // Horner in X^s: acc = B_{r-1}; acc = acc * X^s + B_j for j = r-2 .. 0 (the product is accumulated onto B_j)
        for (int j = pr - 2; j >= 0; --j) {
            GemmOut o;
            o.C = bj(j);
            o.accumulate = true;
            if (i8) {
                // the left factor: B_{r-1} (no transform has seen it: one max pass) or the re-truncated sum of the previous step
                unsigned long long* mbl = mb + (size_t)(ps + j + 1) * modes;
                if (j == pr - 2) {
                    StageTimer tm;
                    NSPT_TRY(tm.begin(ST_SLICE));
                    NSPT_CUDA(launch_ozaki_absmax(f, modes, bj(j + 1), mbl, g.stream));
                    NSPT_TRY(tm.end());
                }
                OzSliceJob job;
                job.X = bj(j + 1);
                job.maxbits = mbl;
                job.quad_slot = ps + j + 1;
                NSPT_TRY(k_slice(f, store, &job, 1, mbs));
                OzGemmGroup gr;
                gr.quad_slot = ps + j + 1;
                gr.rows_slot = ps - 1;
                gr.A = bj(j + 1);
                gr.B = pw(ps);
                gr.out = o;
                NSPT_TRY(k_gemm_i8(f, store, &gr, 1));
                if (j > 0) NSPT_TRY(k_retrunc(f, t, batch, bj(j), bj(j), mb + (size_t)(ps + j) * modes, mbs));
            } else {
                NSPT_TRY(k_gemm(f, batch, bj(j + 1), pw(ps), o));
                if (j > 0) NSPT_TRY(k_retrunc(f, t, batch, bj(j), bj(j)));
            }
        }
        if (!Umul) return k_inverse(f, t, batch, bj(0), E);
        // exp(lambda X) * U: re-truncate the exponential, transform U into the (free) place of X~, multiply into the place of X^2
        double* Ut = pw(1);
        double* Vt = pw(2);
        if (i8) {
            unsigned long long* mbE = mb + (size_t)ps * modes;          // B_0's table: not used so far
            unsigned long long* mbUm = mb + (size_t)(ps + pr) * modes;  // the extra table
            NSPT_TRY(k_retrunc(f, t, batch, bj(0), bj(0), mbE, mbs));
            {
                StageTimer tm;
                NSPT_TRY(tm.begin(ST_FWD));
                NSPT_CUDA(launch_fft_forward(f, t, batch, Umul, Ut, nullptr, nullptr, g.stream, false, mbUm, nullptr, mbs));
                NSPT_TRY(tm.end());
            }
            OzSliceJob jobs[2];
            jobs[0].X = bj(0);
            jobs[0].maxbits = mbE;
            jobs[0].quad_slot = ps;
            jobs[1].X = Ut;
            jobs[1].maxbits = mbUm;
            jobs[1].rows_slot = 0;
            NSPT_TRY(k_slice(f, store, jobs, 2, mbs));
            OzGemmGroup gr;
            gr.quad_slot = ps;
            gr.rows_slot = 0;
            gr.A = bj(0);
            gr.B = Ut;
            gr.out.C = Vt;
            NSPT_TRY(k_gemm_i8(f, store, &gr, 1));
        } else {
            NSPT_TRY(k_retrunc(f, t, batch, bj(0), bj(0)));
            NSPT_TRY(k_forward(f, t, batch, Umul, Ut, nullptr, nullptr));
            NSPT_TRY(k_gemm(f, batch, bj(0), Ut, Vt));
        }
        return k_inverse(f, t, batch, Vt, E);
    }
    const int n = Ntrunc > 0 ? Ntrunc : 1;
    {   // T_n = 1 + lambda X / n
        StageTimer tm;
        NSPT_TRY(tm.begin(ST_OTHER));
        NSPT_CUDA(launch_freq_scale_identity(f, batch, Xt, Tt, lambda.re / n, g.stream, lambda.im / n));
        NSPT_TRY(tm.end());
    }
    double* cur = Tt;
    double* other = Pt;
    for (int m = n - 1; m >= 1; --m) {
        GemmOut o;
        o.C = other;
        o.alpha = Cplx{lambda.re / m, lambda.im / m};
        o.diag = 1.0;
        NSPT_TRY(k_gemm(f, batch, Xt, cur, o));
        if (m > 1 || Umul) NSPT_TRY(k_retrunc(f, t, batch, other, other));
        double* tmp = cur;
        cur = other;
        other = tmp;
    }
    if (!Umul) return k_inverse(f, t, batch, cur, E);
    if (n == 1) NSPT_TRY(k_retrunc(f, t, batch, cur, cur));   // no product has run: 1 + lambda X is already truncated, but keep one code path
    NSPT_TRY(k_forward(f, t, batch, Umul, Xt, nullptr, nullptr));   // X~ is no longer needed
    NSPT_TRY(k_gemm(f, batch, cur, Xt, other));
    return k_inverse(f, t, batch, other, E);
}

int force_device(const nspt_c128* S, nspt_c128* F, double c, int N, int Ntrunc) {
    NSPT_TRY(check_dims(N, Ntrunc, 1));
    if (!S || !F || S == F || !aligned16(S) || !aligned16(F) || !std::isfinite(c)) return NSPT_EINVAL;
    NSPT_TRY(check_arch());
    StageTimer tm;
    NSPT_TRY(tm.begin(ST_OTHER));
    NSPT_CUDA(launch_force(S, F, c, N, Ntrunc + 1, g.stream));
    return tm.end();
}

int staple_device(const nspt_c128* const U[4], const nspt_c128 z[16], nspt_c128* const S[4], int N, int Ntrunc) {
    NSPT_TRY(check_dims(N, Ntrunc, 1));
    if (!U || !z || !S) return NSPT_EINVAL;
    for (int mu = 0; mu < 4; ++mu)
        if (!U[mu] || !S[mu] || !aligned16(U[mu]) || !aligned16(S[mu])) return NSPT_EINVAL;
    NSPT_TRY(check_arch());
    const FreqLayout f = make_layout(N, Ntrunc);
    if (!fft_length_supported(f.L)) return NSPT_EINVAL;
    PlanTables t;
    NSPT_TRY(get_plan(f.L, f.n, g.order_scale, &t));
    char* ws = nullptr;
    NSPT_TRY(get_workspace(ws_bytes_for(f, 1, NSPT_OP_STAPLE), &ws));
    const size_t sb = spectrum_bytes(f, 1);
    auto spec = [&](int i) { return reinterpret_cast<double*>(ws + (size_t)i * sb); };
    double* Ut[4] = {spec(0), spec(1), spec(2), spec(3)};      // U~_mu
    double* Ud[4] = {spec(4), spec(5), spec(6), spec(7)};      // spectrum of U_mu^+
    double* St[4] = {spec(8), spec(9), spec(10), spec(11)};    // S~_mu, accumulated in frequency space
    // per unordered pair p = (mu < nu): W_p = U_mu * U_nu^+, Y_p = U_mu^+ * U_nu, T_p = U_nu * W_p
    double* W[6];
    double* Y[6];
    double* T[6];
    int pmu[6], pnu[6], np = 0;
    for (int mu = 0; mu < 4; ++mu)
        for (int nu = mu + 1; nu < 4; ++nu) {
            pmu[np] = mu;
            pnu[np] = nu;
            W[np] = spec(12 + np);
            Y[np] = spec(18 + np);
            T[np] = spec(24 + np);
            ++np;
        }
    // Eq. 2.3 with U_mu distributed over the sum (the truncated series form a ring, so this is exact):
    //     S_mu = sum_{nu != mu} ( z_{mu nu} P_{mu nu} - z_{mu nu}^* R_{mu nu} ),
    //     P_{mu nu} = U_mu U_nu U_mu^+ U_nu^+,     R_{mu nu} = U_mu U_nu^+ U_mu^+ U_nu       (all products are *).
    // For each unordered pair mu < nu, with W = U_mu U_nu^+ and Y = U_mu^+ U_nu:
    //     R_{mu nu} = W Y,   R_{nu mu} = (Y W)^+,   P_{nu mu} = (U_nu W) U_mu^+,   P_{mu nu} = P_{nu mu}^+ .
    // Six mode-wise products per pair, 36 in all (the literal form needs 52).  The daggers of PRODUCTS are
    // taken by the GEMM epilogue (conjugate-transposed accumulate into the mirrored mode), the sums over
    // nu are accumulated in frequency space, and each S_mu is inverse-transformed once.
    // Products that do not depend on one another share a launch (8 launches for the 36 products): a single
    // product at L = 64 is 3.6 waves of CTAs and loses a tenth of its time to the last, partly filled wave.
    // All four links are transformed before any output is written (S may alias U).
    // The same launch plan runs on the FP64 tensor pipe or, from N = 192 (use_int8), on the INT8 tensor cores: there every
    // spectrum is also cut into int8 slices -- in the QUAD layout where it is a left factor, in the ROWS layout where it is a
    // right factor (one pass per wave of spectra, both layouts from one read) -- with the per-mode maxima the transforms record.
    const bool i8 = use_int8(f, true);
    const int L = f.L;
    unsigned long long* mb = reinterpret_cast<unsigned long long*>(ws + 30 * sb + WS_PAD);   // [U 0..3][W 0..5][Y 0..5][T 0..5] x L
    unsigned long long *mbU = mb, *mbW = mb + 4 * L, *mbY = mb + 10 * L, *mbT = mb + 16 * L;
    const size_t mbs = (size_t)STAPLE_MAXBITS * L;   // distance between the copies of the maxima
    OzStore store;
    // slots.  QUAD (left factors): U~_mu -> mu, Ud_mu (mu < 3) -> 4 + mu, W_p -> 7 + p, Y_p -> 13 + p, T_p -> 19 + p;
    //         ROWS (right factors): U~_mu (mu > 0) -> mu - 1, Ud_mu -> 3 + mu, W_p -> 7 + p, Y_p -> 13 + p
    auto qU = [](int mu) { return mu; };
    auto qUd = [](int mu) { return 4 + mu; };
    auto rU = [](int mu) { return mu - 1; };
    auto rUd = [](int mu) { return 3 + mu; };
    if (i8) {
        store = ozaki_store(f, L, STAPLE_NQ, STAPLE_NR, ws + 30 * sb + WS_PAD + maxbits_bytes(STAPLE_MAXBITS * L));
        NSPT_CUDA(cudaMemsetAsync(mb, 0, sizeof(unsigned long long) * NSPT_MAX_BUCKETS * STAPLE_MAXBITS * L, g.stream));
    }
    auto gemm_groups = [&](const GemmGroup* gr, const int (*slots)[2], int n) -> int {
        if (!i8) return k_gemm_groups(f, gr, n);
        OzGemmGroup og[12];
        for (int i = 0; i < n; ++i) {
            og[i].quad_slot = slots[i][0];
            og[i].rows_slot = slots[i][1];
            og[i].A = gr[i].A;
            og[i].B = gr[i].B;
            og[i].out = gr[i].out;
        }
        return k_gemm_i8(f, store, og, n);
    };
    {
        StageTimer tm;
        NSPT_TRY(tm.begin(ST_FWD));
        NSPT_CUDA(launch_fft_forward(f, t, 1, U[0], Ut[0], U[1], Ut[1], g.stream, false, i8 ? mbU : nullptr, i8 ? mbU + L : nullptr, mbs));
        NSPT_TRY(tm.end());
        NSPT_TRY(tm.begin(ST_FWD));
        NSPT_CUDA(launch_fft_forward(f, t, 1, U[2], Ut[2], U[3], Ut[3], g.stream, false, i8 ? mbU + 2 * L : nullptr,
                                     i8 ? mbU + 3 * L : nullptr, mbs));
        NSPT_TRY(tm.end());
    }
    NSPT_TRY(k_dagger(f, 4, Ut[0], Ud[0]));
    if (i8) {
        OzSliceJob jobs[8];
        for (int mu = 0; mu < 4; ++mu) {
            jobs[mu].X = Ut[mu];
            jobs[mu].maxbits = mbU + mu * L;
            jobs[mu].quad_slot = qU(mu);
            jobs[mu].rows_slot = mu > 0 ? rU(mu) : -1;
            jobs[4 + mu].X = Ud[mu];
            jobs[4 + mu].maxbits = mbU + mu * L;   // |Ud(p)| = |U~((L - p) mod L)|
            jobs[4 + mu].mirror = true;
            jobs[4 + mu].quad_slot = mu < 3 ? qUd(mu) : -1;
            jobs[4 + mu].rows_slot = rUd(mu);
        }
        NSPT_TRY(k_slice(f, store, jobs, 8, mbs));
    }
    {   // W_p and Y_p for the six pairs: twelve products, one launch; then one re-truncation pass over all twelve
        GemmGroup gr[12];
        int sl[12][2];
        for (int p = 0; p < 6; ++p) {
            gr[p].A = Ut[pmu[p]];
            gr[p].B = Ud[pnu[p]];
            gr[p].out.C = W[p];
            sl[p][0] = qU(pmu[p]);
            sl[p][1] = rUd(pnu[p]);
            gr[6 + p].A = Ud[pmu[p]];
            gr[6 + p].B = Ut[pnu[p]];
            gr[6 + p].out.C = Y[p];
            sl[6 + p][0] = qUd(pmu[p]);
            sl[6 + p][1] = rU(pnu[p]);
        }
        NSPT_TRY(gemm_groups(gr, sl, 12));
        NSPT_TRY(k_retrunc(f, t, 12, W[0], W[0], i8 ? mbW : nullptr, mbs));   // W[0..5], Y[0..5] are contiguous (and so are mbW, mbY)
        if (i8) {
            OzSliceJob jobs[12];
            for (int p = 0; p < 6; ++p) {
                jobs[p].X = W[p];
                jobs[p].maxbits = mbW + p * L;
                jobs[p].quad_slot = 7 + p;
                jobs[p].rows_slot = 7 + p;
                jobs[6 + p].X = Y[p];
                jobs[6 + p].maxbits = mbY + p * L;
                jobs[6 + p].quad_slot = 13 + p;
                jobs[6 + p].rows_slot = 13 + p;
            }
            NSPT_TRY(k_slice(f, store, jobs, 12, mbs));
        }
    }
    {   // T_p = U_nu W_p: six products, one launch, one re-truncation pass
        GemmGroup gr[6];
        int sl[6][2];
        for (int p = 0; p < 6; ++p) {
            gr[p].A = Ut[pnu[p]];
            gr[p].B = W[p];
            gr[p].out.C = T[p];
            sl[p][0] = qU(pnu[p]);
            sl[p][1] = 7 + p;
        }
        NSPT_TRY(gemm_groups(gr, sl, 6));
        NSPT_TRY(k_retrunc(f, t, 6, T[0], T[0], i8 ? mbT : nullptr, mbs));
        if (i8) {
            OzSliceJob jobs[6];
            for (int p = 0; p < 6; ++p) {
                jobs[p].X = T[p];
                jobs[p].maxbits = mbT + p * L;
                jobs[p].quad_slot = 19 + p;
            }
            NSPT_TRY(k_slice(f, store, jobs, 6, mbs));
        }
    }
    // Accumulation into S~: three rounds, each a perfect matching of the four directions, so that the products of
    // one launch write different S~_mu.  Round r: pairs (0, r+1) and the complementary pair.
    bool touched[4] = {false, false, false, false};
    const int match[3][2] = {{0, 5}, {1, 4}, {2, 3}};   // pair indices: (0,1)+(2,3), (0,2)+(1,3), (0,3)+(1,2)
    for (int r = 0; r < 3; ++r) {
        GemmGroup ga[4], gb[2];
        int sa[4][2], sbk[2][2];
        for (int q = 0; q < 2; ++q) {
            const int p = match[r][q], mu = pmu[p], nu = pnu[p];
            const Cplx zmn{z[4 * mu + nu].re, z[4 * mu + nu].im};
            const Cplx znm{z[4 * nu + mu].re, z[4 * nu + mu].im};
            // S_mu -= z_{mu nu}^* R_{mu nu},  R_{mu nu} = W Y
            ga[2 * q].A = W[p];
            ga[2 * q].B = Y[p];
            ga[2 * q].out.C = St[mu];
            ga[2 * q].out.alpha = Cplx{-zmn.re, zmn.im};
            ga[2 * q].out.accumulate = touched[mu];
            sa[2 * q][0] = 7 + p;
            sa[2 * q][1] = 13 + p;
            // S_nu -= z_{nu mu}^* R_{nu mu},  R_{nu mu} = (Y W)^+
            ga[2 * q + 1].A = Y[p];
            ga[2 * q + 1].B = W[p];
            ga[2 * q + 1].out.D = St[nu];
            ga[2 * q + 1].out.beta = Cplx{-znm.re, znm.im};
            ga[2 * q + 1].out.accumulate_d = touched[nu];
            sa[2 * q + 1][0] = 13 + p;
            sa[2 * q + 1][1] = 7 + p;
            // S_nu += z_{nu mu} P_{nu mu},  S_mu += z_{mu nu} P_{nu mu}^+,  P_{nu mu} = T U_mu^+
            gb[q].A = T[p];
            gb[q].B = Ud[mu];
            gb[q].out.C = St[nu];
            gb[q].out.alpha = znm;
            gb[q].out.accumulate = true;
            gb[q].out.D = St[mu];
            gb[q].out.beta = zmn;
            gb[q].out.accumulate_d = true;
            sbk[q][0] = 19 + p;
            sbk[q][1] = rUd(mu);
        }
        NSPT_TRY(gemm_groups(ga, sa, 4));
        for (int q = 0; q < 2; ++q) touched[pmu[match[r][q]]] = touched[pnu[match[r][q]]] = true;
        NSPT_TRY(gemm_groups(gb, sbk, 2));
    }
    for (int mu = 0; mu < 4; ++mu) NSPT_TRY(k_inverse(f, t, 1, St[mu], S[mu]));
    return NSPT_OK;
}

// The staple of ONE direction: the unit of work a GPU owns in the paper's four-GPU scheme ("we assign
// computational tasks, which are independent in the four-dimensional direction, on each GPU card").  With W = U_mu U_nu^+,
// Y = U_mu^+ U_nu, T = U_nu W (all *):
//     S_mu = sum_{nu != mu} ( -z_{mu nu}^* W Y + z_{mu nu} (T U_mu^+)^+ ),
// five mode-wise products per nu, 15 in all (the four-direction call shares W, Y, T between the two directions of a pair:
// 36 for four directions).  Every contribution to S~_mu is its own launch, so the sum has a fixed order.
int staple_dir_device(const nspt_c128* const U[4], const nspt_c128 z[16], int mu, nspt_c128* Smu, int N, int Ntrunc) {
    NSPT_TRY(check_dims(N, Ntrunc, 1));
    if (!U || !z || !Smu || mu < 0 || mu > 3 || !aligned16(Smu)) return NSPT_EINVAL;
    for (int d = 0; d < 4; ++d)
        if (!U[d] || !aligned16(U[d])) return NSPT_EINVAL;
    NSPT_TRY(check_arch());
    const FreqLayout f = make_layout(N, Ntrunc);
    if (!fft_length_supported(f.L)) return NSPT_EINVAL;
    PlanTables t;
    NSPT_TRY(get_plan(f.L, f.n, g.order_scale, &t));
    char* ws = nullptr;
    NSPT_TRY(get_workspace(ws_bytes_for(f, 1, NSPT_OP_STAPLE), &ws));
    const size_t sb = spectrum_bytes(f, 1);
    auto spec = [&](int i) { return reinterpret_cast<double*>(ws + (size_t)i * sb); };
    double* Ut[4] = {spec(0), spec(1), spec(2), spec(3)};
    double* Ud[4] = {spec(4), spec(5), spec(6), spec(7)};
    double* St = spec(8);
    double *W[3], *Y[3], *T[3];
    int nus[3], k = 0;
    for (int nu = 0; nu < 4; ++nu)
        if (nu != mu) {
            nus[k] = nu;
            W[k] = spec(9 + k);
            Y[k] = spec(12 + k);
            T[k] = spec(15 + k);
            ++k;
        }
    // FP64 tensor pipe or, from N = 192 (use_int8), INT8 tensor cores -- see staple_device.  Slots of the slice store:
    //   QUAD (left factors):  U~_d -> d, Ud_mu -> 4, W_q -> 5 + q, T_q -> 8 + q;   ROWS (right factors): Ud_d -> d, U~_d -> 4 + d,
    //   W_q -> 8 + q, Y_q -> 11 + q
    const bool i8 = use_int8(f, true);
    const int L = f.L;
    unsigned long long* mb = reinterpret_cast<unsigned long long*>(ws + 30 * sb + WS_PAD);   // [U 0..3][W 0..2][Y 0..2][T 0..2] x L
    unsigned long long *mbU = mb, *mbW = mb + 4 * L, *mbY = mb + 7 * L, *mbT = mb + 10 * L;
    const size_t mbs = (size_t)STAPLE_MAXBITS * L;   // distance between the copies of the maxima
    OzStore store;
    if (i8) {
        store = ozaki_store(f, L, STAPLE_NQ, STAPLE_NR, ws + 30 * sb + WS_PAD + maxbits_bytes(STAPLE_MAXBITS * L));
        NSPT_CUDA(cudaMemsetAsync(mb, 0, sizeof(unsigned long long) * NSPT_MAX_BUCKETS * STAPLE_MAXBITS * L, g.stream));
    }
    auto gemm_groups = [&](const GemmGroup* gr, const int (*slots)[2], int n) -> int {
        if (!i8) return n == 1 ? k_gemm(f, 1, gr[0].A, gr[0].B, gr[0].out) : k_gemm_groups(f, gr, n);
        OzGemmGroup og[12];
        for (int i = 0; i < n; ++i) {
            og[i].quad_slot = slots[i][0];
            og[i].rows_slot = slots[i][1];
            og[i].A = gr[i].A;
            og[i].B = gr[i].B;
            og[i].out = gr[i].out;
        }
        return k_gemm_i8(f, store, og, n);
    };
    {
        StageTimer tm;
        NSPT_TRY(tm.begin(ST_FWD));
        NSPT_CUDA(launch_fft_forward(f, t, 1, U[0], Ut[0], U[1], Ut[1], g.stream, false, i8 ? mbU : nullptr, i8 ? mbU + L : nullptr, mbs));
        NSPT_TRY(tm.end());
        NSPT_TRY(tm.begin(ST_FWD));
        NSPT_CUDA(launch_fft_forward(f, t, 1, U[2], Ut[2], U[3], Ut[3], g.stream, false, i8 ? mbU + 2 * L : nullptr,
                                     i8 ? mbU + 3 * L : nullptr, mbs));
        NSPT_TRY(tm.end());
    }
    NSPT_TRY(k_dagger(f, 4, Ut[0], Ud[0]));
    if (i8) {
        OzSliceJob jobs[8];
        for (int d = 0; d < 4; ++d) {
            jobs[d].X = Ut[d];
            jobs[d].maxbits = mbU + d * L;
            jobs[d].quad_slot = d;
            jobs[d].rows_slot = d != mu ? 4 + d : -1;
            jobs[4 + d].X = Ud[d];
            jobs[4 + d].maxbits = mbU + d * L;   // |Ud(p)| = |U~((L - p) mod L)|
            jobs[4 + d].mirror = true;
            jobs[4 + d].quad_slot = d == mu ? 4 : -1;
            jobs[4 + d].rows_slot = d;
        }
        NSPT_TRY(k_slice(f, store, jobs, 8, mbs));
    }
    {
        GemmGroup gr[6];
        int sl[6][2];
        for (int q = 0; q < 3; ++q) {
            gr[q].A = Ut[mu];
            gr[q].B = Ud[nus[q]];
            gr[q].out.C = W[q];
            sl[q][0] = mu;
            sl[q][1] = nus[q];
            gr[3 + q].A = Ud[mu];
            gr[3 + q].B = Ut[nus[q]];
            gr[3 + q].out.C = Y[q];
            sl[3 + q][0] = 4;
            sl[3 + q][1] = 4 + nus[q];
        }
        NSPT_TRY(gemm_groups(gr, sl, 6));
        NSPT_TRY(k_retrunc(f, t, 6, W[0], W[0], i8 ? mbW : nullptr, mbs));   // W[0..2], Y[0..2] are contiguous (and so are mbW, mbY)
        if (i8) {
            OzSliceJob jobs[6];
            for (int q = 0; q < 3; ++q) {
                jobs[q].X = W[q];
                jobs[q].maxbits = mbW + q * L;
                jobs[q].quad_slot = 5 + q;
                jobs[q].rows_slot = 8 + q;
                jobs[3 + q].X = Y[q];
                jobs[3 + q].maxbits = mbY + q * L;
                jobs[3 + q].rows_slot = 11 + q;
            }
            NSPT_TRY(k_slice(f, store, jobs, 6, mbs));
        }
    }
    {
        GemmGroup gr[3];
        int sl[3][2];
        for (int q = 0; q < 3; ++q) {
            gr[q].A = Ut[nus[q]];
            gr[q].B = W[q];
            gr[q].out.C = T[q];
            sl[q][0] = nus[q];
            sl[q][1] = 8 + q;
        }
        NSPT_TRY(gemm_groups(gr, sl, 3));
        NSPT_TRY(k_retrunc(f, t, 3, T[0], T[0], i8 ? mbT : nullptr, mbs));
        if (i8) {
            OzSliceJob jobs[3];
            for (int q = 0; q < 3; ++q) {
                jobs[q].X = T[q];
                jobs[q].maxbits = mbT + q * L;
                jobs[q].quad_slot = 8 + q;
            }
            NSPT_TRY(k_slice(f, store, jobs, 3, mbs));
        }
    }
    for (int q = 0; q < 3; ++q) {
        const Cplx zmn{z[4 * mu + nus[q]].re, z[4 * mu + nus[q]].im};
        GemmGroup r;   // S_mu -= z_{mu nu}^* W Y
        r.A = W[q];
        r.B = Y[q];
        r.out.C = St;
        r.out.alpha = Cplx{-zmn.re, zmn.im};
        r.out.accumulate = q > 0;
        const int sr[1][2] = {{5 + q, 11 + q}};
        NSPT_TRY(gemm_groups(&r, sr, 1));
        GemmGroup p;   // S_mu += z_{mu nu} (T U_mu^+)^+ : conjugate-transposed accumulate into the mirrored mode
        p.A = T[q];
        p.B = Ud[mu];
        p.out.D = St;
        p.out.beta = zmn;
        p.out.accumulate_d = true;
        const int sp[1][2] = {{8 + q, mu}};
        NSPT_TRY(gemm_groups(&p, sp, 1));
    }
    return k_inverse(f, t, 1, St, Smu);
}

// ---- nspt_series_mul_noalloc: FFT-CONV with its frequency-domain scratch in a file-scope device array ----------------------
// For callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc): the three spectra and
// the per-L tables live in ONE static array of NSPT_NOALLOC_SCRATCH_BYTES that every GPU loading the library holds until exit.
// Layout: [0, NOALLOC_TABLE_BYTES) tables (w^m, w^-m, s^k, s^-k / L), then A~, B~, C~ back to back and the 256-byte pad.
// In host code `noalloc_scratch` is only a handle: the device address comes from cudaGetSymbolAddress, once per device with
// that device current (noalloc_base), and that address is what the kernels of the other files receive.
constexpr size_t NOALLOC_TABLE_BYTES = 16384;
constexpr int NOALLOC_MAX_L = 256;   // = transform length at NSPT_MAX_NTRUNC
static __device__ __align__(256) unsigned char noalloc_scratch[NSPT_NOALLOC_SCRATCH_BYTES];

struct NoallocState {
    unsigned char* base = nullptr;   // device address of noalloc_scratch on this device
    int L = 0, n = 0;                // tables currently in the array
    double s = 0.0;
};
NoallocState noalloc_state[MAX_DEVICES];
// host copies of the tables (static: nothing is allocated per call); protected by the context lock of the calling device,
// and cudaMemcpyAsync from pageable memory has staged its source before it returns
struct NoallocHostTables {
    double2 f[NOALLOC_MAX_L], b[NOALLOC_MAX_L];
    double si[NSPT_MAX_NTRUNC + 1], so[NSPT_MAX_NTRUNC + 1];
};
NoallocHostTables noalloc_host[MAX_DEVICES];

int noalloc_base(int dev, NoallocState** out) {
    NoallocState& st = noalloc_state[dev];
    if (!st.base) {
        void* ptr = nullptr;
        NSPT_CUDA(cudaGetSymbolAddress(&ptr, noalloc_scratch));
        if (!ptr) return NSPT_ECUDA;
        st.base = static_cast<unsigned char*>(ptr);
    }
    *out = &st;
    return NSPT_OK;
}

// the tables of get_plan (same formulas, eqs. 2.7 / 2.9), written into the static array when (L, n, s) changed
int noalloc_tables(int dev, NoallocState& st, int L, int n, double s, PlanTables* out) {
    double2* d_f = reinterpret_cast<double2*>(st.base);
    double2* d_b = d_f + NOALLOC_MAX_L;
    double* d_si = reinterpret_cast<double*>(d_b + NOALLOC_MAX_L);
    double* d_so = d_si + (NSPT_MAX_NTRUNC + 1);
    static_assert(2 * NOALLOC_MAX_L * sizeof(double2) + 2 * (NSPT_MAX_NTRUNC + 1) * sizeof(double) <= NOALLOC_TABLE_BYTES, "table region");
    if (st.L != L || st.n != n || st.s != s) {
        NoallocHostTables& h = noalloc_host[dev];
        const long double two_pi = 6.283185307179586476925286766559005768L;
        for (int m = 0; m < L; ++m) {
            const long double ang = two_pi * (long double)m / (long double)L;
            double c = (double)cosl(ang), sn = (double)sinl(ang);
            if ((4 * m) % L == 0) {   // multiples of pi/2: exact
                const int q = (4 * m) / L;
                c = (q == 0) ? 1.0 : (q == 2 ? -1.0 : 0.0);
                sn = (q == 1) ? 1.0 : (q == 3 ? -1.0 : 0.0);
            }
            h.f[m] = make_double2(c, sn);
            h.b[m] = make_double2(c, -sn);
        }
        for (int k = 0; k < n; ++k) {
            h.si[k] = (double)powl((long double)s, (long double)k);
            h.so[k] = (double)(powl((long double)s, -(long double)k) / (long double)L);
        }
        st.L = 0;   // not valid until all four copies are enqueued
        NSPT_CUDA(cudaMemcpyAsync(d_f, h.f, sizeof(double2) * L, cudaMemcpyHostToDevice, g.stream));
        NSPT_CUDA(cudaMemcpyAsync(d_b, h.b, sizeof(double2) * L, cudaMemcpyHostToDevice, g.stream));
        NSPT_CUDA(cudaMemcpyAsync(d_si, h.si, sizeof(double) * n, cudaMemcpyHostToDevice, g.stream));
        NSPT_CUDA(cudaMemcpyAsync(d_so, h.so, sizeof(double) * n, cudaMemcpyHostToDevice, g.stream));
        st.L = L;
        st.n = n;
        st.s = s;
    }
    *out = PlanTables{d_f, d_b, s != 1.0 ? d_si : nullptr, d_so, 1.0 / L};
    return NSPT_OK;
}

int series_mul_noalloc_device(const nspt_c128* A, const nspt_c128* B, nspt_c128* C, int N, int Ntrunc) {
    NSPT_TRY(check_dims(N, Ntrunc, 1));
    if (!A || !B || !C || !aligned16(A) || !aligned16(B) || !aligned16(C)) return NSPT_EINVAL;
    const FreqLayout f = make_layout(N, Ntrunc);
    if (!fft_length_supported(f.L) || f.L > NOALLOC_MAX_L) return NSPT_EINVAL;
    const size_t sb = spectrum_bytes(f, 1);
    if (sb > NSPT_NOALLOC_SCRATCH_BYTES || NOALLOC_TABLE_BYTES + 3 * sb + WS_PAD > NSPT_NOALLOC_SCRATCH_BYTES) return NSPT_ETOOBIG;
    NSPT_TRY(check_arch());
    int dev = 0;
    NSPT_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEVICES) return NSPT_EINVAL;
    NoallocState* st = nullptr;
    NSPT_TRY(noalloc_base(dev, &st));
    PlanTables t;
    NSPT_TRY(noalloc_tables(dev, *st, f.L, f.n, g.order_scale, &t));
    unsigned char* ws = st->base + NOALLOC_TABLE_BYTES;
    double* At = reinterpret_cast<double*>(ws);
    double* Bt = reinterpret_cast<double*>(ws + sb);
    double* Ct = reinterpret_cast<double*>(ws + 2 * sb);
    // Every scratch byte a kernel reads has been written by this call: the forward pass writes both spectra completely
    // (Steps 1-2), the product writes the third (Step 3); nothing has to start from zero.
    g.used = true;
    g.launches += 3;
    NSPT_CUDA(launch_fft_forward(f, t, 1, A, At, B, Bt, g.stream));
    GemmOut out;
    out.C = Ct;
    NSPT_CUDA(launch_zgemm_modes(f, 1, At, Bt, out, 1, g.stream));   // FP64 tensor pipe (the sizes that fit are below the INT8 range)
    NSPT_CUDA(launch_fft_inverse(f, t, 1, Ct, C, g.stream));         // Steps 4-5
    return NSPT_OK;
}

}  // namespace
}  // namespace nspt

using namespace nspt;

extern "C" {

int nspt_series_mul_noalloc(const nspt_c128* A, const nspt_c128* B, nspt_c128* C, int N, int Ntrunc) {
    NSPT_LOCK();
    return series_mul_noalloc_device(A, B, C, N, Ntrunc);
}

int nspt_series_mul(const nspt_c128* A, const nspt_c128* B, nspt_c128* C, int N, int Ntrunc) {
    NSPT_LOCK();
    return series_mul_device(A, B, C, N, Ntrunc, 1);
}

int nspt_series_mul_batched(const nspt_c128* A, const nspt_c128* B, nspt_c128* C, int N, int Ntrunc, int batch) {
    NSPT_LOCK();
    return series_mul_device(A, B, C, N, Ntrunc, batch);
}

int nspt_staple(const nspt_c128* const U[4], const nspt_c128 z[16], nspt_c128* const S[4], int N, int Ntrunc) {
    NSPT_LOCK();
    return staple_device(U, z, S, N, Ntrunc);
}

int nspt_staple_dir(const nspt_c128* const U[4], const nspt_c128 z[16], int mu, nspt_c128* S_mu, int N, int Ntrunc) {
    NSPT_LOCK();
    return staple_dir_device(U, z, mu, S_mu, N, Ntrunc);
}

int nspt_series_exp(const nspt_c128* X, nspt_c128* E, int N, int Ntrunc) {
    NSPT_LOCK();
    return series_exp_device(X, E, N, Ntrunc, 1);
}

int nspt_series_exp_batched(const nspt_c128* X, nspt_c128* E, int N, int Ntrunc, int batch) {
    NSPT_LOCK();
    return series_exp_device(X, E, N, Ntrunc, batch);
}

int nspt_link_update(const nspt_c128* P, const nspt_c128* U, double eps, nspt_c128* Unew, int N, int Ntrunc) {
    NSPT_LOCK();
    if (!U) return NSPT_EINVAL;
    return series_exp_device(P, Unew, N, Ntrunc, 1, Cplx{0.0, eps}, U);
}

int nspt_link_update_batched(const nspt_c128* P, const nspt_c128* U, double eps, nspt_c128* Unew, int N, int Ntrunc, int batch) {
    NSPT_LOCK();
    if (!U) return NSPT_EINVAL;
    return series_exp_device(P, Unew, N, Ntrunc, batch, Cplx{0.0, eps}, U);
}

int nspt_force(const nspt_c128* S, nspt_c128* F, double c, int N, int Ntrunc) {
    NSPT_LOCK();
    return force_device(S, F, c, N, Ntrunc);
}

int nspt_series_mul_batched_host(const nspt_c128* A, const nspt_c128* B, nspt_c128* C, int N, int Ntrunc, int batch) {
    NSPT_LOCK();
    NSPT_TRY(check_dims(N, Ntrunc, batch));
    if (!A || !B || !C) return NSPT_EINVAL;
    const size_t bytes = (size_t)batch * (Ntrunc + 1) * N * N * sizeof(nspt_c128);
    const size_t slot = align_up(bytes, 256);
    char* dev = nullptr;
    NSPT_TRY(get_staging(3 * slot, &dev));
    nspt_c128* dA = reinterpret_cast<nspt_c128*>(dev);
    nspt_c128* dB = reinterpret_cast<nspt_c128*>(dev + slot);
    nspt_c128* dC = reinterpret_cast<nspt_c128*>(dev + 2 * slot);
    if (batch == 1) {
        NSPT_CUDA(cudaMemcpyAsync(dA, A, bytes, cudaMemcpyHostToDevice, g.stream));
        NSPT_CUDA(cudaMemcpyAsync(dB, B, bytes, cudaMemcpyHostToDevice, g.stream));
        NSPT_TRY(series_mul_device(dA, dB, dC, N, Ntrunc, 1));
        NSPT_CUDA(cudaMemcpyAsync(C, dC, bytes, cudaMemcpyDeviceToHost, g.stream));
        NSPT_CUDA(cudaStreamSynchronize(g.stream));
        return NSPT_OK;
    }
    // batch > 1: the products are independent, so element b+1 is copied in (one copy stream) while element b is
    // multiplied (library stream) and element b-1 is copied out (second copy stream, PCIe is full duplex).
    if (!g.h2d) NSPT_CUDA(cudaStreamCreateWithFlags(&g.h2d, cudaStreamNonBlocking));
    if (!g.d2h) NSPT_CUDA(cudaStreamCreateWithFlags(&g.d2h, cudaStreamNonBlocking));
    while (g.copy_events.size() < (size_t)(2 * batch + 1)) {
        cudaEvent_t e;
        NSPT_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        g.copy_events.push_back(e);
    }
    const size_t one = bytes / batch;
    const size_t elems = one / sizeof(nspt_c128);
    // the copy-in stream must not overtake earlier work of the library stream that may still read the staging area
    NSPT_CUDA(cudaEventRecord(g.copy_events[2 * batch], g.stream));
    NSPT_CUDA(cudaStreamWaitEvent(g.h2d, g.copy_events[2 * batch], 0));
    for (int b = 0; b < batch; ++b) {
        NSPT_CUDA(cudaMemcpyAsync(dA + b * elems, A + b * elems, one, cudaMemcpyHostToDevice, g.h2d));
        NSPT_CUDA(cudaMemcpyAsync(dB + b * elems, B + b * elems, one, cudaMemcpyHostToDevice, g.h2d));
        NSPT_CUDA(cudaEventRecord(g.copy_events[2 * b], g.h2d));
        NSPT_CUDA(cudaStreamWaitEvent(g.stream, g.copy_events[2 * b], 0));
        NSPT_TRY(series_mul_device(dA + b * elems, dB + b * elems, dC + b * elems, N, Ntrunc, 1));
        NSPT_CUDA(cudaEventRecord(g.copy_events[2 * b + 1], g.stream));
        NSPT_CUDA(cudaStreamWaitEvent(g.d2h, g.copy_events[2 * b + 1], 0));
        NSPT_CUDA(cudaMemcpyAsync(C + b * elems, dC + b * elems, one, cudaMemcpyDeviceToHost, g.d2h));
    }
    NSPT_CUDA(cudaStreamSynchronize(g.d2h));
    NSPT_CUDA(cudaStreamSynchronize(g.stream));
    return NSPT_OK;
}

int nspt_series_mul_host(const nspt_c128* A, const nspt_c128* B, nspt_c128* C, int N, int Ntrunc) {
    return nspt_series_mul_batched_host(A, B, C, N, Ntrunc, 1);
}

int nspt_staple_host(const nspt_c128* const U[4], const nspt_c128 z[16], nspt_c128* const S[4], int N, int Ntrunc) {
    NSPT_LOCK();
    NSPT_TRY(check_dims(N, Ntrunc, 1));
    if (!U || !z || !S) return NSPT_EINVAL;
    for (int mu = 0; mu < 4; ++mu)
        if (!U[mu] || !S[mu]) return NSPT_EINVAL;
    const size_t bytes = (size_t)(Ntrunc + 1) * N * N * sizeof(nspt_c128);
    const size_t slot = align_up(bytes, 256);
    char* dev = nullptr;
    NSPT_TRY(get_staging(8 * slot, &dev));
    const nspt_c128* dU[4];
    nspt_c128* dS[4];
    for (int mu = 0; mu < 4; ++mu) {
        dU[mu] = reinterpret_cast<nspt_c128*>(dev + (size_t)mu * slot);
        dS[mu] = reinterpret_cast<nspt_c128*>(dev + (size_t)(4 + mu) * slot);
        NSPT_CUDA(cudaMemcpyAsync(const_cast<nspt_c128*>(dU[mu]), U[mu], bytes, cudaMemcpyHostToDevice, g.stream));
    }
    NSPT_TRY(staple_device(dU, z, dS, N, Ntrunc));
    for (int mu = 0; mu < 4; ++mu) NSPT_CUDA(cudaMemcpyAsync(S[mu], dS[mu], bytes, cudaMemcpyDeviceToHost, g.stream));
    NSPT_CUDA(cudaStreamSynchronize(g.stream));
    return NSPT_OK;
}

int nspt_set_stream(void* cuda_stream) {
    NSPT_LOCK();
    if (g.profiling) NSPT_TRY(prof_flush());
    cudaStream_t next = static_cast<cudaStream_t>(cuda_stream);
    if (next != g.stream && g.used) {
        // all calls share one workspace: work queued on the new stream must not overtake what the old one still runs.
        // (Skipped while either stream is capturing: a captured stream cannot wait on work outside its graph.)
        cudaStreamCaptureStatus a = cudaStreamCaptureStatusNone, b = cudaStreamCaptureStatusNone;
        cudaStreamIsCapturing(g.stream, &a);
        cudaStreamIsCapturing(next, &b);
        if (a == cudaStreamCaptureStatusNone && b == cudaStreamCaptureStatusNone) {
            if (!g.order_event) NSPT_CUDA(cudaEventCreateWithFlags(&g.order_event, cudaEventDisableTiming));
            NSPT_CUDA(cudaEventRecord(g.order_event, g.stream));
            NSPT_CUDA(cudaStreamWaitEvent(next, g.order_event, 0));
        } else {
            cudaGetLastError();
        }
    }
    g.stream = next;
    return NSPT_OK;
}

int nspt_set_order_scale(double s) {
    NSPT_LOCK();
    if (!(s > 0.0) || !std::isfinite(s)) return NSPT_EINVAL;
    g.order_scale = s;
    return NSPT_OK;
}

int nspt_workspace_bytes(int N, int Ntrunc, int batch, int op, size_t* out) {
    if (!out) return NSPT_EINVAL;
    NSPT_LOCK();
    if (op != NSPT_OP_SERIES_MUL && op != NSPT_OP_STAPLE && op != NSPT_OP_SERIES_EXP) return NSPT_EINVAL;
    if (op == NSPT_OP_STAPLE) batch = 1;
    NSPT_TRY(check_dims(N, Ntrunc, batch));
    const FreqLayout f = make_layout(N, Ntrunc);
    if (!fft_length_supported(f.L)) return NSPT_EINVAL;
    *out = ws_bytes_for(f, batch, op);
    return NSPT_OK;
}

int nspt_set_workspace(void* dptr, size_t bytes) {
    NSPT_LOCK();
    if (dptr && (reinterpret_cast<uintptr_t>(dptr) & 255)) return NSPT_EINVAL;
    if (!dptr && bytes) return NSPT_EINVAL;
    g.clean_maxbits = nullptr;
    g.user_ws = dptr;
    g.user_ws_bytes = dptr ? bytes : 0;
    return NSPT_OK;
}

int nspt_set_gemm_variant(int variant) {
    NSPT_LOCK();
    if (variant < -1 || variant > 4) return NSPT_EINVAL;
    g.gemm_variant = variant;
    return NSPT_OK;
}

int nspt_set_conv_algorithm(int algorithm) {
    NSPT_LOCK();
    if (algorithm < 0 || algorithm > 3) return NSPT_EINVAL;
    g.conv_algorithm = algorithm;
    return NSPT_OK;
}

int nspt_profile(int enable) {
    NSPT_LOCK();
    if (!enable && g.profiling) NSPT_TRY(prof_flush());
    g.profiling = enable != 0;
    return NSPT_OK;
}

int nspt_profile_read(int stage, double* ms, long long* launches) {
    NSPT_LOCK();
    if (stage < 0 || stage >= ST_COUNT || !ms || !launches) return NSPT_EINVAL;
    NSPT_TRY(prof_flush());
    *ms = g.prof_ms[stage];
    *launches = g.prof_n[stage];
    g.prof_ms[stage] = 0.0;
    g.prof_n[stage] = 0;
    return NSPT_OK;
}

long long nspt_launch_count(void) {
    ContextLock lk;
    return lk.ok ? g.launches : 0;
}

int nspt_release(void) {
    NSPT_LOCK();
    cudaStreamSynchronize(g.stream);
    for (Plan& p : g.plans) {
        cudaFree(p.tw_fwd);
        cudaFree(p.tw_inv);
        cudaFree(p.scale_in);
        cudaFree(p.scale_out);
    }
    g.plans.clear();
    if (g.own_ws) cudaFree(g.own_ws);
    g.own_ws = nullptr;
    g.own_ws_bytes = 0;
    g.clean_maxbits = nullptr;
    if (g.stage_dev) cudaFree(g.stage_dev);
    g.stage_dev = nullptr;
    g.stage_dev_bytes = 0;
    for (cudaEvent_t e : g.copy_events) cudaEventDestroy(e);
    g.copy_events.clear();
    if (g.h2d) cudaStreamDestroy(g.h2d);
    if (g.d2h) cudaStreamDestroy(g.d2h);
    g.h2d = g.d2h = nullptr;
    for (ProfEvent& e : g.prof_used) {
        cudaEventDestroy(e.a);
        cudaEventDestroy(e.b);
    }
    for (ProfEvent& e : g.prof_free) {
        cudaEventDestroy(e.a);
        cudaEventDestroy(e.b);
    }
    g.prof_used.clear();
    g.prof_free.clear();
    if (g.order_event) cudaEventDestroy(g.order_event);
    g.order_event = nullptr;
    g.used = false;
    return NSPT_OK;
}

const char* nspt_strerror(int code) {
    switch (code) {
        case NSPT_OK: return "ok";
        case NSPT_EINVAL: return "invalid argument (null or misaligned pointer, N < 1, Ntrunc outside [0,127], batch < 1)";
        case NSPT_ENOMEM: return "out of memory, or the caller's workspace is too small";
        case NSPT_ECUDA: return g.cuda_msg;
        case NSPT_EARCH: return "the current CUDA device is not compute capability 10.x (B200, sm_100a)";
        case NSPT_ETOOBIG:
            return "nspt_series_mul_noalloc: the problem needs more than the static scratch (3 * 16 * L * N * N + 16640 bytes "
                   "must not exceed NSPT_NOALLOC_SCRATCH_BYTES); use nspt_series_mul";
        default: return "unknown error code";
    }
}

int nspt_version(void) { return 400; }

}  // extern "C"
