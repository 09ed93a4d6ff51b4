"""ctypes wrapper around oracle/nspt_oracle.c plus the parts of the oracle that are plain numpy.

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).  Nothing here imports the CUDA package.

What is defined here, with the passage each follows:

* ``series_mul(A, B)``      -- eq. 2.5: C^(k) = sum_{l<=k} A^(l) B^(k-l)   (C code)
* ``dagger(A)``             -- coefficient-wise conjugate transpose; g is real, PAPER.md:48   (C code)
* ``staple(U, z)``          -- eq. 2.3, written out literally (52 star-products):
      S_mu = U_mu * [ sum_{nu != mu} ( z_mu,nu  U_nu * U_mu^+ * U_nu^+
                                       - z_mu,nu^*  U_nu^+ * U_mu^+ * U_nu ) ]
  left-to-right association, truncation after every product (readings c6, c9).
* ``series_exp(X)``         -- exp(X) = sum_{m>=0} X^{*m} / m!  of a series with X^(0) = 0, every power a chain of
  star-products of eq. 2.5 (the link update U <- exp(i eps P) * U of the NSPT integrator,
  PAPER.md:50-55; readings c15, c17).  The sum stops at m = Ntrunc exactly because
  X^{*m} starts at g^m.
* ``force(S, c)``           -- F^(k) = i c [ S^(k) - S^(k)+ - Tr(S^(k) - S^(k)+)/N ], PAPER.md:50 (eq. 2.3),
  with the coefficient c ("beta" after the paper's time rescaling, reading c10) left to the caller.
* ``product_bound`` / ``staple_bound`` / ``per_order_error`` -- the error metric of the north
  star: per order k, ||C_test^(k) - C_oracle^(k)||_F / bound_k with
  bound_k = sum_{j<=k} ||A^(j)||_F ||B^(k-j)||_F   (readings c11, c12).

Arrays are numpy complex128, C-contiguous, shape (Ntrunc+1, N, N): X[k, i, j] = X^(k)_{ij}.
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import platform
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "nspt_oracle.c"
_LIB = None


def _cpu_tag() -> str:
    """A short tag of this host's ISA so a library built on another box is never reused."""
    flags = ""
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    flags = line
                    break
    except OSError:
        pass
    return hashlib.sha1((platform.machine() + flags).encode()).hexdigest()[:10]


def build(force: bool = False) -> Path:
    """Compile nspt_oracle.c with gcc (-O3 -march=native -fopenmp) into oracle/_build/."""
    src = _SRC.read_bytes()
    tag = hashlib.sha1(src).hexdigest()[:10] + "-" + _cpu_tag()
    out_dir = _HERE / "_build"
    out = out_dir / f"libnspt_oracle-{tag}.so"
    if out.exists() and not force:
        return out
    out_dir.mkdir(exist_ok=True)
    tmp = out_dir / f".tmp-{os.getpid()}-{tag}.so"
    cmd = ["gcc", "-O3", "-march=native", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-std=c11", "-o", str(tmp), str(_SRC)]
    subprocess.run(cmd, check=True)
    os.replace(tmp, out)
    return out


def _lib():
    global _LIB
    if _LIB is None:
        lib = ctypes.CDLL(str(build()))
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        lib.oracle_series_mul.argtypes = [dp, dp, dp, ctypes.c_int, ctypes.c_int]
        lib.oracle_series_mul.restype = ctypes.c_int
        lib.oracle_series_mul_rows.argtypes = [dp, dp, dp, ctypes.c_int, ctypes.c_int, ip, ctypes.c_int]
        lib.oracle_series_mul_rows.restype = ctypes.c_int
        lib.oracle_dagger.argtypes = [dp, dp, ctypes.c_int, ctypes.c_int]
        lib.oracle_dagger.restype = ctypes.c_int
        lib.oracle_num_threads.restype = ctypes.c_int
        _LIB = lib
    return _LIB


def num_threads() -> int:
    """OpenMP threads the C oracle uses (omp_get_max_threads)."""
    return int(_lib().oracle_num_threads())


def _as_series(X, name: str) -> np.ndarray:
    X = np.ascontiguousarray(X, dtype=np.complex128)
    if X.ndim != 3 or X.shape[1] != X.shape[2]:
        raise ValueError(f"{name}: expected shape (Ntrunc+1, N, N), got {X.shape}")
    return X


def _dptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def series_mul(A, B) -> np.ndarray:
    """C = A * B truncated at the common order (eq. 2.5)."""
    A = _as_series(A, "A")
    B = _as_series(B, "B")
    if A.shape != B.shape:
        raise ValueError("A and B must have the same shape")
    n, N, _ = A.shape
    C = np.empty_like(A)
    rc = _lib().oracle_series_mul(_dptr(A), _dptr(B), _dptr(C), N, n - 1)
    if rc != 0:
        raise RuntimeError("oracle_series_mul failed")
    return C


def series_mul_rows(A, B, rows) -> np.ndarray:
    """Rows ``rows`` of every order of A * B: out[k, r, :] = (A*B)^(k)[rows[r], :]."""
    A = _as_series(A, "A")
    B = _as_series(B, "B")
    n, N, _ = A.shape
    rows = np.ascontiguousarray(rows, dtype=np.int32)
    out = np.empty((n, len(rows), N), dtype=np.complex128)
    rc = _lib().oracle_series_mul_rows(_dptr(A), _dptr(B), _dptr(out), N, n - 1,
                                       rows.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), len(rows))
    if rc != 0:
        raise RuntimeError("oracle_series_mul_rows failed")
    return out


def dagger(A) -> np.ndarray:
    """(A^+)^(k) = (A^(k))^+ (reading c9)."""
    A = _as_series(A, "A")
    n, N, _ = A.shape
    out = np.empty_like(A)
    rc = _lib().oracle_dagger(_dptr(A), _dptr(out), N, n - 1)
    if rc != 0:
        raise RuntimeError("oracle_dagger failed")
    return out


def staple(U, z):
    """Literal eq. 2.3.  U: four series; z: 4x4 complex, z[mu, nu] = z_{mu nu}.

    Returns [S_0, S_1, S_2, S_3].  52 star-products; the second term uses conj(z[mu, nu])
    exactly as the equation prints it.  The diagonal of z is ignored (sum over nu != mu)."""
    U = [_as_series(u, "U") for u in U]
    if len(U) != 4:
        raise ValueError("the TEK model has four directions")
    z = np.asarray(z, dtype=np.complex128).reshape(4, 4)
    Ud = [dagger(u) for u in U]
    S = []
    for mu in range(4):
        X = np.zeros_like(U[mu])
        for nu in range(4):
            if nu == mu:
                continue
            t1 = series_mul(series_mul(U[nu], Ud[mu]), Ud[nu])      # U_nu * U_mu^+ * U_nu^+
            t2 = series_mul(series_mul(Ud[nu], Ud[mu]), U[nu])      # U_nu^+ * U_mu^+ * U_nu
            X += z[mu, nu] * t1 - np.conj(z[mu, nu]) * t2
        S.append(series_mul(U[mu], X))
    return S


def series_exp(X) -> np.ndarray:
    """exp(X) = sum_{m=0}^{Ntrunc} X^{*m} / m!  for a series with X^(0) = 0 (a non-zero X^(0) is an error).

    Written out as the definition: the powers X^{*m} = X * X^{*(m-1)} are formed one after the other
    with the star-product of eq. 2.5 and added with weight 1/m!.  X^{*m} has no orders below g^m, so
    the sum ends at m = Ntrunc with nothing dropped."""
    X = _as_series(X, "X")
    n, N, _ = X.shape
    if np.any(X[0] != 0):
        raise ValueError("series_exp needs X^(0) = 0")
    E = np.zeros_like(X)
    E[0] = np.eye(N)
    power = E.copy()          # X^{*0} = 1
    fact = 1.0
    for m in range(1, n):
        power = series_mul(X, power)
        fact *= m
        E += power / fact
    return E


def exp_bound(X) -> np.ndarray:
    """Tolerance denominator for series_exp: the scalar series exp(x), x_k = ||X^(k)||_F, which
    majorises every term of the definition (sub-multiplicativity of the Frobenius norm), plus
    sqrt(N) at order 0 for the identity."""
    x = _order_norms(X)
    n = len(x)
    e = np.zeros(n)
    e[0] = 1.0
    power = e.copy()
    fact = 1.0
    for m in range(1, n):
        power = _scalar_conv(x, power)
        fact *= m
        e += power / fact
    e[0] = np.sqrt(np.asarray(X).shape[1])
    return e


def force(S, c: float) -> np.ndarray:
    """F^(k) = i c [ S^(k) - S^(k)+ - Tr(S^(k) - S^(k)+)/N 1 ]   (eq. 2.3; c real)."""
    S = _as_series(S, "S")
    n, N, _ = S.shape
    F = np.empty_like(S)
    for k in range(n):
        D = S[k] - S[k].conj().T
        F[k] = 1j * c * (D - (np.trace(D) / N) * np.eye(N))
    return F


# ----------------------------------------------------------------------------- error metric

def _order_norms(X) -> np.ndarray:
    X = np.asarray(X)
    return np.sqrt((np.abs(X.reshape(X.shape[0], -1)) ** 2).sum(axis=1))


def _scalar_conv(a: np.ndarray, b: np.ndarray) -> np.ndarray:
    n = len(a)
    return np.array([sum(a[j] * b[k - j] for j in range(k + 1)) for k in range(n)])


def product_bound(A, B) -> np.ndarray:
    """bound_k = sum_{j<=k} ||A^(j)||_F ||B^(k-j)||_F  (north star tolerance denominator)."""
    return _scalar_conv(_order_norms(A), _order_norms(B))


def staple_bound(U) -> list:
    """Reading c12: propagate the product bound through eq. 2.3 with |z| = 1:
    bound(S_mu) = u_mu * sum_{nu != mu} 2 (u_nu * u_mu * u_nu), u = per-order Frobenius norms."""
    u = [_order_norms(x) for x in U]
    out = []
    for mu in range(4):
        acc = np.zeros_like(u[mu])
        for nu in range(4):
            if nu != mu:
                acc += 2.0 * _scalar_conv(_scalar_conv(u[nu], u[mu]), u[nu])
        out.append(_scalar_conv(u[mu], acc))
    return out


def per_order_error(C_test, C_ref, bound) -> np.ndarray:
    """err_k = ||C_test^(k) - C_ref^(k)||_F / max(bound_k, 1e-3 max_k' bound_k')  (reading c11)."""
    d = _order_norms(np.asarray(C_test) - np.asarray(C_ref))
    bound = np.asarray(bound, dtype=np.float64)
    floor = 1e-3 * bound.max() if bound.size else 0.0
    den = np.maximum(bound, floor)
    den = np.where(den > 0, den, 1.0)
    return d / den
