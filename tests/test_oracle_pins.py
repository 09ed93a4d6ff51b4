"""Pins for the CPU oracle (oracle/): everything here runs without a GPU.

Each test checks the oracle against something fixed by the paper's definition (eq. 2.5,
PAPER.md:62-66; eq. 2.3) or by mathematics -- never against the oracle itself
and never against the CUDA path.  A dropped term, a wrong sign or index, a swapped or
transposed operand fails at least one of them.
"""
import itertools
import math

import numpy as np
import pytest

import oracle
from paper_2001_02835_b200 import workloads as wl


# ----------------------------------------------------------------------------- helpers

def read_golden(path):
    out = {}
    for line in path.read_text().splitlines():
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        name, vals = line.split(":")
        entries = [complex(*map(float, v.split(","))) for v in vals.split()]
        n = int(round(math.sqrt(len(entries))))
        out[name.strip()] = np.array(entries, dtype=np.complex128).reshape(n, n)
    return out


def brute_force_product(A, B):
    """Scalar five-loop evaluation of eq. 2.5 in pure Python complex arithmetic."""
    n, N, _ = A.shape
    C = np.zeros((n, N, N), dtype=np.complex128)
    for k in range(n):
        for i in range(N):
            for j in range(N):
                s = 0j
                for l in range(k + 1):
                    for m in range(N):
                        s += complex(A[l, i, m]) * complex(B[k - l, m, j])
                C[k, i, j] = s
    return C


def identity_series(N, Ntrunc):
    one = np.zeros((Ntrunc + 1, N, N), dtype=np.complex128)
    one[0] = np.eye(N)
    return one


def fro(X):
    return np.sqrt((np.abs(X.reshape(X.shape[0], -1)) ** 2).sum(axis=1))


# ----------------------------------------------------------------------------- the product

def test_golden_noncommuting_2x2(golden_dir):
    g = read_golden(golden_dir / "noncommuting_2x2.txt")
    A = np.stack([g["A0"], g["A1"], g["A2"]])
    B = np.stack([g["B0"], g["B1"], g["B2"]])
    C = oracle.series_mul(A, B)
    assert np.array_equal(C, np.stack([g["C0"], g["C1"], g["C2"]]))
    # operand order matters and the oracle keeps A on the left
    assert np.array_equal(oracle.series_mul(B, A)[0], g["BA0"])
    assert not np.array_equal(C[0], g["BA0"])


def test_golden_complex_2x2(golden_dir):
    g = read_golden(golden_dir / "complex_2x2.txt")
    C = oracle.series_mul(g["A0"][None], g["B0"][None])
    assert np.array_equal(C[0], g["C0"])
    assert np.array_equal(oracle.dagger(g["A0"][None])[0], g["A0dag"])


def test_n1_is_polynomial_multiplication():
    # N = 1: eq. 2.5 is the textbook Cauchy product; compare with numpy.convolve, truncated.
    rng = np.random.default_rng(11)
    for Ntrunc in (0, 1, 5, 12):
        a = rng.integers(-9, 10, Ntrunc + 1) + 1j * rng.integers(-9, 10, Ntrunc + 1)
        b = rng.integers(-9, 10, Ntrunc + 1) + 1j * rng.integers(-9, 10, Ntrunc + 1)
        C = oracle.series_mul(a.reshape(-1, 1, 1), b.reshape(-1, 1, 1)).ravel()
        assert np.array_equal(C, np.convolve(a, b)[: Ntrunc + 1])


def test_n1_binomial_closed_form():
    # (1+g)^a (1+g)^b = (1+g)^(a+b): coefficients are binomials, exact in double here.
    Ntrunc = 10
    for a, b in ((3, 4), (7, 9), (10, 10)):
        pa = np.array([math.comb(a, k) for k in range(Ntrunc + 1)], dtype=np.complex128)
        pb = np.array([math.comb(b, k) for k in range(Ntrunc + 1)], dtype=np.complex128)
        want = np.array([math.comb(a + b, k) for k in range(Ntrunc + 1)], dtype=np.complex128)
        got = oracle.series_mul(pa.reshape(-1, 1, 1), pb.reshape(-1, 1, 1)).ravel()
        assert np.array_equal(got, want)


@pytest.mark.parametrize("N,Ntrunc", [(1, 3), (2, 0), (3, 4), (4, 2)])
def test_brute_force_tiny(N, Ntrunc):
    rng = np.random.default_rng(100 + 10 * N + Ntrunc)
    A = wl.gaussian_series(N, Ntrunc, rng)
    B = wl.gaussian_series(N, Ntrunc, rng)
    ref = brute_force_product(A, B)
    got = oracle.series_mul(A, B)
    assert np.abs(got - ref).max() <= 1e-14 * np.abs(ref).max()
    Ai = wl.integer_series(N, Ntrunc, rng)
    Bi = wl.integer_series(N, Ntrunc, rng)
    assert np.array_equal(oracle.series_mul(Ai, Bi), brute_force_product(Ai, Bi))


def test_unit_element_is_bitwise():
    rng = np.random.default_rng(5)
    A = wl.gaussian_series(7, 6, rng)
    one = identity_series(7, 6)
    assert np.array_equal(oracle.series_mul(one, A), A)
    assert np.array_equal(oracle.series_mul(A, one), A)


def test_associativity_exact_on_integers():
    rng = np.random.default_rng(0)
    A, B, C = (wl.integer_series(9, 7, rng) for _ in range(3))
    left = oracle.series_mul(oracle.series_mul(A, B), C)
    right = oracle.series_mul(A, oracle.series_mul(B, C))
    assert np.array_equal(left, right)


def test_geometric_series_inverse_exact():
    # (1 - g X) * sum_k g^k X^k = 1 exactly under truncation, X a small integer matrix.
    X = np.array([[1, 2, 0], [0, -1, 1], [2, 0, 1]], dtype=np.complex128) + 1j * np.array(
        [[0, 1, 0], [1, 0, 0], [0, 0, -1]])
    Ntrunc = 7
    geo = np.stack([np.linalg.matrix_power(X, k) for k in range(Ntrunc + 1)])
    lin = np.zeros_like(geo)
    lin[0] = np.eye(3)
    lin[1] = -X
    assert np.array_equal(oracle.series_mul(lin, geo), identity_series(3, Ntrunc))
    assert np.array_equal(oracle.series_mul(geo, lin), identity_series(3, Ntrunc))


def test_commuting_exponentials():
    # exp(gX) * exp(gY) = exp(g(X+Y)) when [X, Y] = 0; coefficients X^k / k!.
    rng = np.random.default_rng(3)
    M = rng.standard_normal((5, 5)) + 1j * rng.standard_normal((5, 5))
    X, Y = 0.3 * M, 0.2 * (M @ M) - 0.1 * M          # polynomials in M commute
    Ntrunc = 12

    def expser(Z):
        return np.stack([np.linalg.matrix_power(Z, k) / math.factorial(k) for k in range(Ntrunc + 1)])

    got = oracle.series_mul(expser(X), expser(Y))
    want = expser(X + Y)
    scale = oracle.product_bound(expser(X), expser(Y))
    assert (fro(got - want) / scale).max() < 1e-14


def test_evaluation_at_numeric_g_against_untruncated_product():
    # Independent identity: A(g0) B(g0) = C_full(g0), C_full the product with enough orders
    # that nothing is truncated (degree 2 Ntrunc); and truncation only drops orders.
    rng = np.random.default_rng(8)
    N, Ntrunc = 6, 5
    A = wl.gaussian_series(N, Ntrunc, rng)
    B = wl.gaussian_series(N, Ntrunc, rng)
    pad = np.zeros((Ntrunc, N, N), dtype=np.complex128)
    Cfull = oracle.series_mul(np.concatenate([A, pad]), np.concatenate([B, pad]))
    assert np.array_equal(Cfull[: Ntrunc + 1], oracle.series_mul(A, B))

    def horner(S, g0):
        acc = np.zeros((N, N), dtype=np.complex128)
        for k in range(S.shape[0] - 1, -1, -1):
            acc = acc * g0 + S[k]
        return acc

    g0 = 0.37 - 0.21j
    lhs = horner(A, g0) @ horner(B, g0)
    rhs = horner(Cfull, g0)
    assert np.abs(lhs - rhs).max() < 1e-13 * np.abs(lhs).max()


def test_fft_conv_steps_1_to_5_agree_with_definition():
    # The paper's algorithm (eqs. 2.6-2.9) written with numpy.fft must give
    # the oracle's result to rounding: zero padding removes the wrap-around.
    rng = np.random.default_rng(21)
    N, Np = 5, 8                      # Ntrunc = Np - 1
    A = wl.gaussian_series(N, Np - 1, rng)
    B = wl.gaussian_series(N, Np - 1, rng)
    pad = np.zeros_like(A)
    Ap, Bp = np.concatenate([A, pad]), np.concatenate([B, pad])          # Step 1, eq. 2.6
    # Step 2, eq. 2.7 uses w = exp(+2 pi i / 2Np): that is numpy's *inverse* kernel times 2Np
    At = np.fft.ifft(Ap, axis=0) * (2 * Np)
    Bt = np.fft.ifft(Bp, axis=0) * (2 * Np)
    Ct = np.einsum("pim,pmj->pij", At, Bt)                                  # Step 3, eq. 2.8
    C = np.fft.fft(Ct, axis=0) / (2 * Np)                                   # Step 4, eq. 2.9
    C = C[:Np]                                                              # Step 5
    ref = oracle.series_mul(A, B)
    err = oracle.per_order_error(C, ref, oracle.product_bound(A, B))
    assert err.max() < 1e-14
    # and too short a transform (no padding) does wrap around: the padding is necessary
    Cbad = np.fft.fft(np.einsum("pim,pmj->pij", np.fft.ifft(A, axis=0) * Np,
                                np.fft.ifft(B, axis=0) * Np), axis=0) / Np
    assert oracle.per_order_error(Cbad, ref, oracle.product_bound(A, B)).max() > 1e-3


def test_rows_variant_matches_full_product():
    rng = np.random.default_rng(4)
    A = wl.gaussian_series(11, 5, rng)
    B = wl.gaussian_series(11, 5, rng)
    rows = [0, 3, 10]
    full = oracle.series_mul(A, B)
    part = oracle.series_mul_rows(A, B, rows)
    assert np.array_equal(part, full[:, rows, :])
    assert np.abs(part - brute_force_product(A, B)[:, rows, :]).max() < 1e-13


def test_matches_numpy_matmul_medium():
    # Library-routine pin at a size spanning many rows per thread: numpy's matmul per term.
    rng = np.random.default_rng(17)
    N, Ntrunc = 40, 9
    A = wl.gaussian_series(N, Ntrunc, rng)
    B = wl.gaussian_series(N, Ntrunc, rng)
    ref = np.stack([sum(A[l] @ B[k - l] for l in range(k + 1)) for k in range(Ntrunc + 1)])
    err = oracle.per_order_error(oracle.series_mul(A, B), ref, oracle.product_bound(A, B))
    assert err.max() < 1e-15


# ----------------------------------------------------------------------------- generator + unitarity

@pytest.mark.parametrize("N,Ntrunc", [(9, 7), (16, 15), (49, 31)])
def test_unitarity_of_generated_series(N, Ntrunc):
    # U = exp(i sum g^k H_k), H_k Hermitian  =>  U * U^+ = 1 order by order.  Checks the
    # oracle product, the dagger and the input generator together.
    U = wl.unitary_series(N, Ntrunc, np.random.default_rng([7, N, Ntrunc]))
    assert np.allclose(U[0], np.eye(N), atol=0)
    for prod in (oracle.series_mul(U, oracle.dagger(U)), oracle.series_mul(oracle.dagger(U), U)):
        resid = prod - identity_series(N, Ntrunc)
        assert (fro(resid) / oracle.product_bound(U, U)).max() < 1e-14
    # first order of exp(i g H_1 + ...) is i H_1: anti-Hermitian and traceless
    assert np.abs(U[1] + U[1].conj().T).max() < 1e-15
    assert abs(np.trace(U[1])) < 1e-13


def test_generator_is_seeded_and_structured():
    A1, B1 = wl.config1_gaussian()
    A2, B2 = wl.config1_gaussian()
    assert np.array_equal(A1, A2) and np.array_equal(B1, B2) and not np.array_equal(A1, B1)
    assert A1.shape == (8, 9, 9) and A1.dtype == np.complex128
    Ai, Bi = wl.config1_integer()
    assert np.array_equal(Ai, np.round(Ai)) and np.abs(Ai.real).max() <= 3 and np.abs(Ai.imag).max() <= 3
    H = wl.hermitian_traceless(30, np.random.default_rng(1))
    assert np.abs(H - H.conj().T).max() == 0 and abs(np.trace(H)) < 1e-14
    z = wl.twist_tensor(15, 4)
    assert np.allclose(z[0, 1], np.exp(2j * np.pi * 4 / 15)) and np.allclose(z[1, 0], np.conj(z[0, 1]))


# ----------------------------------------------------------------------------- the staple (eq. 2.3)

def clock_shift(L):
    w = np.exp(2j * np.pi / L)
    P = np.diag(w ** np.arange(L))
    Q = np.roll(np.eye(L), 1, axis=0)
    return P, Q


def twist_eaters(L, k):
    """Gamma_mu = P^a Q^b (x) P^c Q^d with Gamma_mu Gamma_nu = z_{nu mu} Gamma_nu Gamma_mu for
    z = twist_tensor(L, k).  Found by a search over exponent vectors; the relation is asserted
    numerically by the caller, so the search itself need not be trusted."""
    P, Q = clock_shift(L)
    z = wl.twist_tensor(L, k)

    def gamma(v):
        a, b, c, d = v
        return np.kron(np.linalg.matrix_power(P, a) @ np.linalg.matrix_power(Q, b),
                       np.linalg.matrix_power(P, c) @ np.linalg.matrix_power(Q, d))

    def ok(gm, gn, mu, nu):
        return np.abs(gm @ gn - z[nu, mu] * (gn @ gm)).max() < 1e-12

    gammas = [gamma(v) for v in itertools.product(range(L), repeat=4)]

    def extend(chosen):                      # depth-first search with backtracking
        mu = len(chosen)
        if mu == 4:
            return chosen
        for g in gammas:
            if all(ok(chosen[nu], g, nu, mu) for nu in range(mu)):
                found = extend(chosen + [g])
                if found is not None:
                    return found
        return None

    chosen = extend([gamma((1, 0, 0, 0))])
    assert chosen is not None, "no twist eater found"
    return chosen, z


def test_staple_vanishes_on_twist_eater_vacuum():
    # Classical vacuum of eq. 2.1 (refs [9,10]): z_{mu nu} U_mu U_nu U_mu^+ U_nu^+ = 1,
    # i.e. Gamma_mu Gamma_nu = z_{nu mu} Gamma_nu Gamma_mu.  Then both triple products in eq. 2.3
    # equal z^* z Gamma_mu^+ and cancel: S_mu = 0.  With z conjugated they do not.  Pins the
    # orientation of z and of both triple products.
    L, k, Ntrunc = 3, 1, 2
    G, z = twist_eaters(L, k)
    for mu in range(4):
        for nu in range(4):
            if mu != nu:
                assert np.abs(G[mu] @ G[nu] - z[nu, mu] * (G[nu] @ G[mu])).max() < 1e-12
    U = []
    for g in G:
        s = np.zeros((Ntrunc + 1, L * L, L * L), dtype=np.complex128)
        s[0] = g
        U.append(s)
    S = oracle.staple(U, z)
    assert max(np.abs(s).max() for s in S) < 1e-13
    Sbad = oracle.staple(U, np.conj(z))
    assert min(np.abs(s[0]).max() for s in Sbad) > 0.5


def test_staple_of_identity_links():
    # All U_mu = 1: every triple product is 1, so S_mu^(0) = sum_{nu != mu} (z - z^*) = 2i sum Im z_{mu nu}.
    N, Ntrunc = 4, 3
    z = wl.twist_tensor(5, 2)
    U = [identity_series(N, Ntrunc) for _ in range(4)]
    S = oracle.staple(U, z)
    for mu in range(4):
        c = sum(2j * z[mu, nu].imag for nu in range(4) if nu != mu)
        assert np.allclose(S[mu][0], c * np.eye(N), atol=1e-15)
        assert np.abs(S[mu][1:]).max() == 0


def test_staple_of_commuting_diagonal_links():
    # Diagonal unitary series commute, so U_nu U_mu^+ U_nu^+ = U_mu^+ and S_mu = (sum 2i Im z) * 1.
    rng = np.random.default_rng(9)
    N, Ntrunc = 5, 6
    U = []
    for _ in range(4):
        s = np.zeros((Ntrunc + 1, N, N), dtype=np.complex128)
        theta = rng.standard_normal((Ntrunc, N))
        # exp(i sum_k g^k theta_k) per diagonal entry, by polynomial exponentiation
        for j in range(N):
            x = np.zeros(Ntrunc + 1, dtype=np.complex128)
            x[1:] = 1j * theta[:, j]
            e = np.zeros(Ntrunc + 1, dtype=np.complex128)
            e[0] = 1
            term = e.copy()
            for m in range(1, Ntrunc + 1):
                term = np.convolve(term, x)[: Ntrunc + 1] / m
                e = e + term
            s[:, j, j] = e
        U.append(s)
    z = wl.twist_tensor(7, 3)
    S = oracle.staple(U, z)
    for mu in range(4):
        c = sum(2j * z[mu, nu].imag for nu in range(4) if nu != mu)
        want = c * identity_series(N, Ntrunc)
        assert np.abs(S[mu] - want).max() < 1e-13


def test_staple_against_dense_matrix_evaluation():
    # Evaluate the links at a numeric g0 as plain matrices, form eq. 2.2's staple with dense
    # algebra, and compare with the series staple summed at g0.  With only U^(0), U^(1)
    # non-zero and Ntrunc >= 4 nothing is truncated (degree of S is 4).
    rng = np.random.default_rng(12)
    N, Ntrunc = 3, 4
    U = []
    for _ in range(4):
        s = np.zeros((Ntrunc + 1, N, N), dtype=np.complex128)
        s[0] = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
        s[1] = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
        U.append(s)
    z = wl.twist_tensor(4, 1)
    S = oracle.staple(U, z)
    g0 = 0.6
    M = [u[0] + g0 * u[1] for u in U]
    for mu in range(4):
        X = np.zeros((N, N), dtype=np.complex128)
        for nu in range(4):
            if nu == mu:
                continue
            X += z[mu, nu] * M[nu] @ M[mu].conj().T @ M[nu].conj().T
            X -= np.conj(z[mu, nu]) * M[nu].conj().T @ M[mu].conj().T @ M[nu]
        want = M[mu] @ X
        got = sum(S[mu][k] * g0 ** k for k in range(Ntrunc + 1))
        assert np.abs(got - want).max() < 1e-12 * np.abs(want).max()


def test_error_metric_definition():
    rng = np.random.default_rng(2)
    A = wl.gaussian_series(3, 2, rng)
    B = wl.gaussian_series(3, 2, rng)
    a, b = fro(A), fro(B)
    want = np.array([a[0] * b[0], a[0] * b[1] + a[1] * b[0], a[0] * b[2] + a[1] * b[1] + a[2] * b[0]])
    assert np.allclose(oracle.product_bound(A, B), want, rtol=1e-15)
    C = oracle.series_mul(A, B)
    D = C.copy()
    D[1] += 1e-6
    err = oracle.per_order_error(D, C, want)
    assert err[0] == 0 and err[2] == 0 and np.isclose(err[1], 3e-6 / want[1])


# ----------------------------------------------------------------------------- series exponential and force
# (the steps on either side of the staple in one NSPT update)

def test_exp_of_log_series_is_one_plus_g():
    # N = 1: X = log(1+g) = sum_{k>=1} (-1)^(k+1) g^k / k  =>  exp(X) = 1 + g exactly
    n = 24
    X = np.zeros((n, 1, 1), dtype=np.complex128)
    for k in range(1, n):
        X[k, 0, 0] = (-1.0) ** (k + 1) / k
    E = oracle.series_exp(X)
    want = np.zeros(n)
    want[0] = want[1] = 1.0
    assert np.abs(E[:, 0, 0] - want).max() < 5e-15


def test_exp_of_g_times_scalar_is_taylor_series():
    n = 16
    X = np.zeros((n, 1, 1), dtype=np.complex128)
    X[1, 0, 0] = 0.75 - 0.5j
    E = oracle.series_exp(X)
    want = np.array([(0.75 - 0.5j) ** k / math.factorial(k) for k in range(n)])
    assert np.abs(E[:, 0, 0] - want).max() < 1e-15


def test_exp_of_commuting_diagonal_series_matches_scalar_recurrence():
    # for commuting coefficients E' = X' E holds, i.e. k e_k = sum_j j x_j e_{k-j}: an independent formula
    rng = np.random.default_rng(70)
    n, N = 10, 4
    x = rng.standard_normal((n, N)) + 1j * rng.standard_normal((n, N))
    x[0] = 0
    X = np.zeros((n, N, N), dtype=np.complex128)
    for k in range(n):
        X[k] = np.diag(x[k])
    E = oracle.series_exp(X)
    e = np.zeros((n, N), dtype=np.complex128)
    e[0] = 1
    for k in range(1, n):
        e[k] = sum(j * x[j] * e[k - j] for j in range(1, k + 1)) / k
    for k in range(n):
        assert np.abs(E[k] - np.diag(e[k])).max() < 1e-12 * max(1.0, np.abs(e[k]).max())


def test_exp_low_orders_noncommuting_by_hand():
    # X = g A + g^2 B, [A, B] != 0: orders 0..3 of exp(X) written out by hand
    A = np.array([[0, 1], [2, 0]], dtype=np.complex128)
    B = np.array([[1, 0], [3, -1j]], dtype=np.complex128)
    X = np.zeros((4, 2, 2), dtype=np.complex128)
    X[1], X[2] = A, B
    E = oracle.series_exp(X)
    assert np.allclose(E[0], np.eye(2), atol=0)
    assert np.allclose(E[1], A, atol=1e-15)
    assert np.allclose(E[2], B + A @ A / 2, atol=1e-15)
    assert np.allclose(E[3], (A @ B + B @ A) / 2 + A @ A @ A / 6, atol=1e-15)
    assert not np.allclose(A @ B, B @ A)


def test_exp_of_nilpotent_generator_terminates():
    M = np.array([[0, 3, 1], [0, 0, -2], [0, 0, 0]], dtype=np.complex128)
    X = np.zeros((6, 3, 3), dtype=np.complex128)
    X[1] = M
    E = oracle.series_exp(X)
    assert np.array_equal(E[0], np.eye(3)) and np.array_equal(E[1], M)
    assert np.allclose(E[2], M @ M / 2, atol=0) and np.abs(E[3:]).max() == 0


def test_exp_inverse_and_unitarity():
    rng = np.random.default_rng(71)
    n, N = 9, 5
    X = np.zeros((n, N, N), dtype=np.complex128)
    for k in range(1, n):
        X[k] = 1j * wl.hermitian_traceless(N, rng)       # anti-Hermitian => exp(X) unitary order by order
    E = oracle.series_exp(X)
    one = identity_series(N, n - 1)
    assert np.abs(oracle.series_mul(E, oracle.series_exp(-X)) - one).max() < 1e-13
    assert np.abs(oracle.series_mul(E, oracle.dagger(E)) - one).max() < 1e-13


def test_exp_evaluated_at_numeric_g_matches_matrix_exponential():
    from scipy.linalg import expm
    rng = np.random.default_rng(72)
    n, N, g0 = 14, 4, 0.05
    X = 0.5 * wl.gaussian_series(N, n - 1, rng)
    X[0] = 0
    E = oracle.series_exp(X)
    Xg = sum(g0 ** k * X[k] for k in range(n))
    Eg = sum(g0 ** k * E[k] for k in range(n))
    assert np.abs(Eg - expm(Xg)).max() < 1e-14        # truncation error ~ g0^14


def test_exp_agrees_with_the_input_generator():
    # workloads._input_series_exp is a different arrangement (Horner, stacked products); both must give exp(X)
    rng = np.random.default_rng(73)
    n, N = 8, 6
    X = np.zeros((n, N, N), dtype=np.complex128)
    for k in range(1, n):
        X[k] = 1j * wl.hermitian_traceless(N, rng)
    E = oracle.series_exp(X)
    assert oracle.per_order_error(wl._input_series_exp(X), E, oracle.exp_bound(X)).max() < 1e-14


def test_exp_rejects_zeroth_order():
    X = np.zeros((3, 2, 2), dtype=np.complex128)
    X[0, 0, 0] = 1.0
    with pytest.raises(ValueError):
        oracle.series_exp(X)


def test_force_by_hand_2x2():
    # S = [[1+2i, 3], [4i, 5-i]]: S - S^+ = [[4i, 3+4i], [-3+4i, -2i]], Tr = 2i, /N = i
    S = np.zeros((1, 2, 2), dtype=np.complex128)
    S[0] = [[1 + 2j, 3], [4j, 5 - 1j]]
    F = oracle.force(S, 2.0)
    want = 2j * np.array([[4j - 1j, 3 + 4j], [-3 + 4j, -2j - 1j]])
    assert np.allclose(F[0], want, atol=0)


def test_force_is_hermitian_traceless_and_kills_hermitian_input():
    rng = np.random.default_rng(74)
    n, N = 5, 7
    S = wl.gaussian_series(N, n - 1, rng)
    F = oracle.force(S, 1.7)
    for k in range(n):
        assert np.abs(F[k] - F[k].conj().T).max() < 1e-15
        assert abs(np.trace(F[k])) < 1e-14
    H = S + np.conj(np.transpose(S, (0, 2, 1)))
    assert np.abs(oracle.force(H, 3.0)).max() == 0
    iden = np.zeros((1, N, N), dtype=np.complex128)
    iden[0] = 1j * np.eye(N)                                # S - S^+ = 2i 1 is pure trace
    assert np.abs(oracle.force(iden, 1.0)).max() == 0


def test_force_matches_scalar_loops():
    rng = np.random.default_rng(75)
    n, N, c = 3, 4, -0.6
    S = wl.gaussian_series(N, n - 1, rng)
    F = oracle.force(S, c)
    for k in range(n):
        tr = sum(complex(S[k, i, i]) - complex(S[k, i, i]).conjugate() for i in range(N))
        for i in range(N):
            for j in range(N):
                d = complex(S[k, i, j]) - complex(S[k, j, i]).conjugate() - (tr / N if i == j else 0)
                assert abs(F[k, i, j] - 1j * c * d) < 1e-15


def test_staple_is_covariant_under_a_constant_gauge_rotation():
    # eq. 2.3 is built from products U ... U^+ only, so U_mu -> W U_mu W^+ with one constant unitary W maps
    # S_mu -> W S_mu W^+ order by order: a structural check of the staple (operand order, daggers) at once
    rng = np.random.default_rng(76)
    N, Ntrunc = 4, 3
    U = [wl.unitary_series(N, Ntrunc, rng) for _ in range(4)]
    z = wl.twist_tensor(2, 1)
    H = wl.hermitian_traceless(N, rng)
    evals, V = np.linalg.eigh(H)
    W = (V * np.exp(1j * evals)) @ V.conj().T
    assert np.abs(W @ W.conj().T - np.eye(N)).max() < 1e-14
    rot = lambda X: np.einsum("ab,kbc,dc->kad", W, X, W.conj())
    S = oracle.staple(U, z)
    Sr = oracle.staple([rot(u) for u in U], z)
    for mu in range(4):
        assert np.abs(Sr[mu] - rot(S[mu])).max() < 1e-12


def test_exp_of_a_sum_of_commuting_series_factorises():
    # X and Y polynomials in one matrix commute, so exp(X + Y) = exp(X) * exp(Y) order by order
    rng = np.random.default_rng(77)
    N, n = 5, 8
    M = 0.4 * (rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N)))
    P = [np.eye(N, dtype=np.complex128)]
    for _ in range(3):
        P.append(P[-1] @ M)
    X = np.zeros((n, N, N), dtype=np.complex128)
    Y = np.zeros((n, N, N), dtype=np.complex128)
    for k in range(1, n):
        X[k] = rng.standard_normal() * P[1] + rng.standard_normal() * P[2]
        Y[k] = rng.standard_normal() * P[0] + rng.standard_normal() * P[3]
    lhs = oracle.series_exp(X + Y)
    rhs = oracle.series_mul(oracle.series_exp(X), oracle.series_exp(Y))
    assert oracle.per_order_error(lhs, rhs, oracle.exp_bound(X + Y)).max() < 1e-13


# ----------------------------------------------------------------------------- tolerance denominators, by hand

def test_staple_bound_by_hand_two_orders():
    # reading c12 with 1 x 1 "matrices" so that Frobenius norms are absolute values: a = (1, 2, 1, 3) at order 0,
    # b = (2, 1, 1, 0) at order 1.  (u_nu * u_mu * u_nu)_0 = a_nu^2 a_mu, (..)_1 = 2 a_nu b_nu a_mu + a_nu^2 b_mu;
    # acc = 2 * sum over nu != mu; bound = u_mu * acc.
    #   mu = 0: acc = (2*14*1, 2*[(4+8)+(2+2)+(0+18)]) = (28, 68)  ->  bound = (28, 1*68 + 2*28) = (28, 124)
    #   mu = 3: acc = (2*6*3, 2*(12+12+6)) = (36, 60)              ->  bound = (108, 3*60 + 0*36) = (108, 180)
    U = [np.array([[[1.0]], [[-2.0j]]]), np.array([[[2.0j]], [[1.0]]]), np.array([[[-1.0]], [[1.0j]]]),
         np.array([[[3.0]], [[0.0]]])]
    b = oracle.staple_bound([u.astype(np.complex128) for u in U])
    assert np.array_equal(b[0], [28.0, 124.0])
    assert np.array_equal(b[3], [108.0, 180.0])


def test_exp_bound_by_hand_three_orders():
    # x = (0, 3, 4) -> exp(x) = 1 + 3 g + (4 + 9/2) g^2; the order-0 entry is sqrt(N) for the identity
    X = np.zeros((3, 2, 2), dtype=np.complex128)
    X[1, 0, 0] = 3.0
    X[2, 0, 1] = 4.0j
    e = oracle.exp_bound(X)
    assert np.allclose(e, [np.sqrt(2.0), 3.0, 8.5], rtol=0, atol=1e-15)
