/*
 * nspt_oracle.c -- CPU ORACLE for the truncated series star-product.  TEST INFRASTRUCTURE ONLY.
 *
 * This file is the plain definition of the operation the CUDA library computes, written out
 * from the paper and nothing else.  It is slow on purpose (O(N^3 * Ntrunc^2)), shares no code,
 * header, table or helper with paper_2001_02835_b200/csrc, and may be used only by tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
 *
 * Definition followed (eqs. 2.4-2.5, section 2):
 *     A = sum_{k=0}^{Ntrunc} g^k A^(k),  B likewise,  N x N complex coefficient matrices,
 *     C^(k) = sum_{l=0}^{k} A^(l) B^(k-l)  ==  (A * B)^(k),      k = 0..Ntrunc,
 * "the ordering of multiplication have to be kept": the left factor is always taken from A.
 * Each matrix product is the textbook (XY)_{ij} = sum_m X_{im} Y_{mj}.
 * (reading c1: the paper prints the upper index of B as "k-l" beside a summation
 *  index "ell"; it is read as B^(k-ell).)
 *
 * There is NO FFT in this file: FFT-CONV reaches exactly this result
 * (zero padding removes the wrap-around), so the oracle is the definition, not the algorithm.
 *
 * Storage (reading c5; the paper does not fix one): series X is an array of
 * (Ntrunc+1) row-major N x N matrices of interleaved (re, im) doubles,
 *     X[k][i][j] = X_{ij}^{(k)}  at double offset 2*((k*N + i)*N + j).
 *
 * Arithmetic: IEEE double, explicit real/imaginary products (no _Complex multiply, which
 * would call __muldc3), accumulation in index order l = 0..k (outer), m = 0..N-1 (inner).
 * The OpenMP loop is over output rows i only, so every C^(k)_{ij} is summed by one thread
 * in a fixed order: the result is deterministic and independent of the thread count.
 *
 * Pins (tests/test_oracle_pins.py, all run with -m "not gpu"): N=1 equals textbook
 * polynomial multiplication; a hand-worked non-commuting 2x2 example (tests/golden);
 * a pure-Python five-loop brute force; unit element; exact associativity on integers;
 * (1 - gX) * sum g^k X^k = 1 exactly; exp(gX)*exp(gY) = exp(g(X+Y)) for commuting X, Y;
 * evaluation at a numeric g0 against the untruncated product; U * U^dagger = 1 for
 * U = exp(i sum g^k H_k); numpy FFT-CONV (paper Steps 1-5) agrees to rounding.
 */
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* C = A * B truncated at order Ntrunc (eq. 2.5).  C must not alias A or B. Returns 0, or -1
 * on bad arguments / allocation failure. */
int oracle_series_mul(const double *A, const double *B, double *C, int N, int Ntrunc)
{
    if (!A || !B || !C || N < 1 || Ntrunc < 0) return -1;
    const size_t mat = (size_t)N * (size_t)N * 2;      /* doubles per coefficient matrix */
    int fail = 0;
    for (int k = 0; k <= Ntrunc; ++k) {
        double *Ck = C + (size_t)k * mat;
#pragma omp parallel
        {
            double *cr = (double *)malloc(sizeof(double) * (size_t)N);
            double *ci = (double *)malloc(sizeof(double) * (size_t)N);
            if (!cr || !ci) {
#pragma omp atomic write
                fail = 1;
            } else {
#pragma omp for schedule(static)
                for (int i = 0; i < N; ++i) {
                    for (int j = 0; j < N; ++j) { cr[j] = 0.0; ci[j] = 0.0; }
                    for (int l = 0; l <= k; ++l) {                 /* sum over l of A^(l) B^(k-l) */
                        const double *Al = A + (size_t)l * mat + (size_t)i * N * 2;
                        const double *Bkl = B + (size_t)(k - l) * mat;
                        for (int m = 0; m < N; ++m) {              /* (XY)_ij = sum_m X_im Y_mj */
                            const double ar = Al[2 * m], ai = Al[2 * m + 1];
                            const double *b = Bkl + (size_t)m * N * 2;
                            for (int j = 0; j < N; ++j) {
                                const double br = b[2 * j], bi = b[2 * j + 1];
                                cr[j] += ar * br - ai * bi;
                                ci[j] += ar * bi + ai * br;
                            }
                        }
                    }
                    double *c = Ck + (size_t)i * N * 2;
                    for (int j = 0; j < N; ++j) { c[2 * j] = cr[j]; c[2 * j + 1] = ci[j]; }
                }
            }
            free(cr); free(ci);
        }
        if (fail) return -1;
    }
    return 0;
}

/* Selected rows of C = A * B: for every order k and every r < nrows, row rows[r] of C^(k),
 * written to out[k][r][j].  Same arithmetic and order as oracle_series_mul; lets a test
 * check full-size outputs "one by one" without forming the whole product. */
int oracle_series_mul_rows(const double *A, const double *B, double *out, int N, int Ntrunc,
                           const int *rows, int nrows)
{
    if (!A || !B || !out || !rows || N < 1 || Ntrunc < 0 || nrows < 0) return -1;
    const size_t mat = (size_t)N * (size_t)N * 2;
    for (int r = 0; r < nrows; ++r) if (rows[r] < 0 || rows[r] >= N) return -1;
#pragma omp parallel for collapse(2) schedule(dynamic)
    for (int k = 0; k <= Ntrunc; ++k) {
        for (int r = 0; r < nrows; ++r) {
            const int i = rows[r];
            double *c = out + ((size_t)k * nrows + r) * (size_t)N * 2;
            for (int j = 0; j < 2 * N; ++j) c[j] = 0.0;
            for (int l = 0; l <= k; ++l) {
                const double *Al = A + (size_t)l * mat + (size_t)i * N * 2;
                const double *Bkl = B + (size_t)(k - l) * mat;
                for (int m = 0; m < N; ++m) {
                    const double ar = Al[2 * m], ai = Al[2 * m + 1];
                    const double *b = Bkl + (size_t)m * N * 2;
                    for (int j = 0; j < N; ++j) {
                        const double br = b[2 * j], bi = b[2 * j + 1];
                        c[2 * j] += ar * br - ai * bi;
                        c[2 * j + 1] += ar * bi + ai * br;
                    }
                }
            }
        }
    }
    return 0;
}

/* (A^dagger)^(k) = (A^(k))^dagger: coefficient-wise conjugate transpose; g is real
 * (g = 1/sqrt(beta); reading c9).  Out must not alias A. */
int oracle_dagger(const double *A, double *Out, int N, int Ntrunc)
{
    if (!A || !Out || N < 1 || Ntrunc < 0) return -1;
    const size_t mat = (size_t)N * (size_t)N * 2;
    for (int k = 0; k <= Ntrunc; ++k)
        for (int i = 0; i < N; ++i)
            for (int j = 0; j < N; ++j) {
                const double *a = A + (size_t)k * mat + ((size_t)j * N + i) * 2;
                double *o = Out + (size_t)k * mat + ((size_t)i * N + j) * 2;
                o[0] = a[0];
                o[1] = -a[1];
            }
    return 0;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
