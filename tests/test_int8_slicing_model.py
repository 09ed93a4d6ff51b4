"""Error model of the INT8-sliced mode-wise product, in numpy, against the oracle.

csrc/nspt_ozaki.cu replaces the FP64 matrix product of FFT-CONV's Step 3 (eq. 2.8) by exact integer
products of int8 digit planes.  This test restates the number format in numpy -- fixed point relative to the largest
element of a mode, balanced base-256 digits, digit pairs with s + t < S kept, 3-multiplication complex product -- and
answers the design question "how many slices does the north-star tolerance need?" on series shaped like the paper's
(unitary order by order, norms growing with the order): S = 7 meets 1e-11 with two orders of magnitude to spare, S = 5
does not.  The integer matrix products are exact in float64 here (|entries| <= 2^7, K <= 2^8), as they are in INT32 on
the tensor core.
"""
import numpy as np
import pytest

import oracle
from paper_2001_02835_b200 import workloads as wl


def digits(y, S):
    """y real, |y| < 1  ->  S integer arrays q_s, y ~ sum_s q_s 2^(-6 - 8 s); q_0 in [-64, 64], the others in [-128, 127]."""
    v = np.rint(y * 2.0 ** (6 + 8 * (S - 1)))
    out = []
    for _ in range(S - 1):
        q = (v + 128) % 256 - 128          # balanced digit of weight 256^j
        out.append(q)
        v = (v - q) / 256
    out.append(v)
    assert np.abs(out[-1]).max() <= 64 and all(np.abs(q).max() <= 128 for q in out)
    return out[::-1]                        # most significant first


def sliced_real_product(X, Y, S):
    qx, qy = digits(X, S), digits(Y, S)
    acc = [0.0] * S
    for s in range(S):
        for t in range(S - s):
            acc[s + t] = acc[s + t] + qx[s] @ qy[t]      # exact integers
    h = acc[S - 1]
    for d in range(S - 2, -1, -1):
        h = h / 256 + acc[d]
    return h * 2.0 ** -12


def sliced_fft_conv(A, B, S):
    n = A.shape[0]
    L = 1
    while L < 2 * n - 1:
        L *= 2
    FA = np.fft.ifft(A, n=L, axis=0) * L        # forward transform with the paper's sign (eq. 2.7)
    FB = np.fft.ifft(B, n=L, axis=0) * L
    FC = np.empty_like(FA)
    for p in range(L):
        out = []
        ea = np.frexp(max(np.abs(FA[p].real).max(), np.abs(FA[p].imag).max()))[1]
        eb = np.frexp(max(np.abs(FB[p].real).max(), np.abs(FB[p].imag).max()))[1]
        a, b = FA[p] * 2.0 ** -ea, FB[p] * 2.0 ** -eb
        p1 = sliced_real_product(a.real, b.real, S)
        p2 = sliced_real_product(a.imag, b.imag, S)
        p3 = sliced_real_product((a.real + a.imag) / 2, (b.real + b.imag) / 2, S)
        FC[p] = 2.0 ** (ea + eb) * ((p1 - p2) + 1j * (4 * p3 - p1 - p2))
    return (np.fft.fft(FC, axis=0) / L)[:n]


@pytest.fixture(scope="module")
def case():
    A, B = wl.config_product(24, 31, seed=[9, 24, 31])
    return A, B, oracle.series_mul(A, B), oracle.product_bound(A, B)


def test_seven_slices_meet_the_tolerance_with_margin(case):
    A, B, ref, bound = case
    err = oracle.per_order_error(sliced_fft_conv(A, B, 7), ref, bound).max()
    assert err < 1e-13, err


def test_five_slices_do_not(case):
    A, B, ref, bound = case
    err = oracle.per_order_error(sliced_fft_conv(A, B, 5), ref, bound).max()
    assert err > 1e-11, err


def test_digits_reconstruct_exactly_to_the_last_kept_bit():
    rng = np.random.default_rng(1)
    y = rng.uniform(-1, 1, 1000) * (1 - 2.0 ** -40)
    q = digits(y, 7)
    back = sum(q[s] * 2.0 ** (-6 - 8 * s) for s in range(7))
    assert np.abs(back - y).max() <= 2.0 ** -55


def test_integer_inputs_stay_exact():
    # small-integer series: the sliced product must round to the oracle's integers (north-star bit-exact criterion)
    rng = np.random.default_rng(2)
    A, B = wl.integer_series(6, 7, rng), wl.integer_series(6, 7, rng)
    got = sliced_fft_conv(A, B, 7)
    ref = oracle.series_mul(A, B)
    assert np.array_equal(np.round(got.real), ref.real) and np.array_equal(np.round(got.imag), ref.imag)
