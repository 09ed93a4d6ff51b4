"""Seeded synthetic inputs shaped like the paper's workloads.  numpy only.

This module serves BOTH the oracle tests and the CUDA path's tests / bench, and therefore
holds none of the method's hot-path arithmetic: it imports neither ``oracle`` nor the CUDA
binding.  The one series operation it needs -- the exponential that turns Hermitian
traceless generators into a unitary series -- is a private numpy helper used only to
*prepare inputs* (reading c15); a bug in it would change the inputs both sides
see, not their agreement, and tests/test_oracle_pins.py checks its output independently
(U * U^+ = 1 order by order, computed with the oracle).

The paper's real workload is NSPT field configurations of the TEK model (Table 3,
PAPER.md:132-138: N in {121,169,225,289}, N_trunc in {7,15,31,63}) produced by the authors'
own program; those ensembles are not available, so the series below take their shape:
dense N x N complex128 coefficients, unitary order by order, identity leading term.

Layout everywhere: complex128, C-contiguous, shape (Ntrunc+1, N, N), X[k,i,j] = X^(k)_ij.
"""
from __future__ import annotations

import numpy as np

__all__ = [
    "gaussian_series", "integer_series", "hermitian_traceless", "unitary_series",
    "twist_tensor", "config1_gaussian", "config1_integer", "config_product",
    "config_staple", "sweep_points",
]


def gaussian_series(N: int, Ntrunc: int, rng: np.random.Generator) -> np.ndarray:
    """iid complex Gaussian coefficients, re and im ~ N(0, 1/2)  (BASELINE.json configs[0])."""
    shape = (Ntrunc + 1, N, N)
    return (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)) / np.sqrt(2.0)


def integer_series(N: int, Ntrunc: int, rng: np.random.Generator, lo: int = -3, hi: int = 3) -> np.ndarray:
    """Small-integer real and imaginary parts in [lo, hi] (bit-exact checks, configs[0])."""
    shape = (Ntrunc + 1, N, N)
    re = rng.integers(lo, hi + 1, shape)
    im = rng.integers(lo, hi + 1, shape)
    return (re + 1j * im).astype(np.complex128)


def hermitian_traceless(N: int, rng: np.random.Generator) -> np.ndarray:
    """Random Hermitian traceless N x N matrix with E|H_ij|^2 = 1/N (configs[1])."""
    G = (rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))) / np.sqrt(2.0)
    H = (G + G.conj().T) / np.sqrt(2.0) / np.sqrt(N)
    H -= (np.trace(H) / N) * np.eye(N)
    return H


def _input_series_exp(X: np.ndarray) -> np.ndarray:
    """exp of a series X with X^(0) = 0, truncated at the order of X  (reading c15).

    exp(X) = sum_{m=0}^{n} X^m / m!  exactly (X^m starts at g^m), by Horner
    T <- 1 + (X T)/m for m = n..1, where at step m only orders <= n-m+1 of the partial
    result are needed.  Each order of X T is one stacked matrix product
    [X^(1) ... X^(k)] [T^(k-1); ...; T^(0)].  Input preparation only."""
    n = X.shape[0] - 1
    N = X.shape[1]
    eye = np.eye(N, dtype=np.complex128)
    T = np.zeros_like(X)
    T[0] = eye
    # Xrow[i, l, m] = X^(l)_{im}: lets [X^(1)..X^(k)] be sliced as an N x (k N) matrix
    Xrow = np.ascontiguousarray(X.transpose(1, 0, 2))
    for m in range(n, 0, -1):
        d = n - m + 1                      # orders of X*T needed at this step: 1..d
        new = np.zeros_like(T)
        new[0] = eye
        for k in range(1, d + 1):
            left = Xrow[:, 1:k + 1, :].reshape(N, k * N)
            right = T[k - 1::-1].reshape(k * N, N) if k > 1 else T[0]
            new[k] = (left @ right) / m
        T = new
    return T


def unitary_series(N: int, Ntrunc: int, rng: np.random.Generator) -> np.ndarray:
    """U = exp(i sum_{k>=1} g^k H_k), H_k Hermitian traceless (configs[1]); U^(0) = 1."""
    X = np.zeros((Ntrunc + 1, N, N), dtype=np.complex128)
    for k in range(1, Ntrunc + 1):
        X[k] = 1j * hermitian_traceless(N, rng)
    return _input_series_exp(X)


def twist_tensor(L: int, k: int) -> np.ndarray:
    """z_{mu nu} = exp(2 pi i k eps_{mu nu} / L), eps = +1 (mu<nu), -1 (mu>nu), 1 on the
    diagonal (ignored by the staple).  configs[3]: L = sqrt(N) = 15, k = 4."""
    z = np.ones((4, 4), dtype=np.complex128)
    for mu in range(4):
        for nu in range(4):
            if mu != nu:
                eps = 1.0 if mu < nu else -1.0
                z[mu, nu] = np.exp(2j * np.pi * k * eps / L)
    return z


# ------------------------------------------------------------------ BASELINE.json configs

def config1_gaussian():
    """configs[0]: N=9, N_trunc=7, iid complex Gaussian, seed 0; A drawn before B."""
    rng = np.random.default_rng(0)
    return gaussian_series(9, 7, rng), gaussian_series(9, 7, rng)


def config1_integer():
    """configs[0], integer variant: entries in [-3,3], fresh rng seed 0; A before B."""
    rng = np.random.default_rng(0)
    return integer_series(9, 7, rng), integer_series(9, 7, rng)


def config_product(N: int, Ntrunc: int, seed):
    """configs[1], [2], [4]: A and B unitary series; A drawn before B."""
    rng = np.random.default_rng(seed)
    A = unitary_series(N, Ntrunc, rng)
    B = unitary_series(N, Ntrunc, rng)
    return A, B


def config_staple(N: int = 225, Ntrunc: int = 31, seed=4, twist_k: int = 4):
    """configs[3]: four unitary link series U_1..U_4 (drawn in order) and the twist tensor
    with L = sqrt(N)."""
    L = int(round(np.sqrt(N)))
    if L * L != N:
        raise ValueError("the symmetric twist needs N = L^2")
    rng = np.random.default_rng(seed)
    U = [unitary_series(N, Ntrunc, rng) for _ in range(4)]
    return U, twist_tensor(L, twist_k)


def sweep_points():
    """configs[4]: (N, N_trunc) points of the scaling sweep; seed for a point is [5, N, N_trunc]."""
    pts = [(225, nt) for nt in (7, 15, 31, 63, 127)]
    pts += [(n, 31) for n in (16, 49, 100, 400)]
    return pts
