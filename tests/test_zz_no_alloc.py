"""nspt_series_mul_noalloc (include/nspt.h): the ⋆-product with its scratch in the library's static device array, for callers
that must not allocate.  Checked against the existing path (nspt_series_mul, workspace from cudaMalloc) on the same inputs, at
the tolerance of tests/test_gpu_parity.py (per order k: ||dC^(k)||_F <= 1e-11 * sum_j ||A^(j)||_F ||B^(k-j)||_F), on calls in
a row that share the array.  Collected last on purpose (pytest -x): a failure here hides nothing else.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-11


@pytest.fixture(scope="module")
def nspt():
    import torch
    assert torch.cuda.is_available()
    from paper_2001_02835_b200 import build
    build.build()
    from paper_2001_02835_b200 import binding
    binding.use_current_stream()
    binding.nspt_set_order_scale(1.0)
    binding.nspt_set_gemm_variant(1)
    binding.nspt_set_conv_algorithm(1)      # the existing path as FFT-CONV too (the new entry point has no Naive-CONV branch)
    yield binding
    binding.nspt_set_order_scale(1.0)
    binding.nspt_set_gemm_variant(1)
    binding.nspt_set_conv_algorithm(0)


def series(N, Ntrunc, seed):
    import torch
    from paper_2001_02835_b200 import workloads as wl
    rng = np.random.default_rng([seed, N, Ntrunc])
    return torch.from_numpy(np.ascontiguousarray(wl.gaussian_series(N, Ntrunc, rng))).cuda()


def per_order_error(got, ref, A, B):
    """max_k ||got^(k) - ref^(k)||_F / sum_{j<=k} ||A^(j)||_F ||B^(k-j)||_F, on the device tensors"""
    import torch
    na = torch.linalg.matrix_norm(A).cpu().numpy()
    nb = torch.linalg.matrix_norm(B).cpu().numpy()
    bound = np.array([sum(na[j] * nb[k - j] for j in range(k + 1)) for k in range(len(na))])
    diff = torch.linalg.matrix_norm(got - ref).cpu().numpy()
    return float((diff / bound).max())


def test_two_calls_in_a_row_match_the_existing_path(nspt):
    import torch
    # near the limit of the static array (N = 104 at N_trunc = 31), several tiles and a ragged edge
    A1, B1 = series(97, 31, 1), series(97, 31, 2)
    A2, B2 = series(97, 31, 3), series(97, 31, 4)
    C1, C2 = torch.empty_like(A1), torch.empty_like(A2)
    launches0 = nspt.nspt_launch_count()
    nspt.nspt_series_mul_noalloc(A1, B1, C1)      # two calls back to back on one stream: the second reuses the array
    nspt.nspt_series_mul_noalloc(A2, B2, C2)
    assert nspt.nspt_launch_count() - launches0 == 6
    ref1 = nspt.nspt_series_mul(A1, B1)
    ref2 = nspt.nspt_series_mul(A2, B2)
    torch.cuda.synchronize()
    for got, ref, A, B in ((C1, ref1, A1, B1), (C2, ref2, A2, B2)):
        assert torch.isfinite(got.real).all() and torch.isfinite(got.imag).all()
        assert per_order_error(got, ref, A, B) <= TOL
    assert not torch.equal(C1, C2)


def test_shape_change_order_scale_and_aliased_output(nspt):
    import torch
    # a different transform length after the calls above (the tables in the array are rewritten), with the order scale on,
    # then the first shape again with the output in place of the left factor
    A, B = series(50, 12, 5), series(50, 12, 6)
    nspt.nspt_set_order_scale(0.75)
    try:
        C = nspt.nspt_series_mul_noalloc(A, B, torch.empty_like(A))
        ref = nspt.nspt_series_mul(A, B)
        torch.cuda.synchronize()
        assert per_order_error(C, ref, A, B) <= TOL
    finally:
        nspt.nspt_set_order_scale(1.0)
    A1, B1 = series(97, 31, 7), series(97, 31, 8)
    ref = nspt.nspt_series_mul(A1, B1)
    X = A1.clone()
    nspt.nspt_series_mul_noalloc(X, B1, X)
    torch.cuda.synchronize()
    assert per_order_error(X, ref, A1, B1) <= TOL


def test_sizes_beyond_the_static_array_are_rejected(nspt):
    import torch
    # 3 * 16 * 64 * 105^2 + 16640 bytes > 32 MiB: a clear error, the output untouched
    A = torch.zeros((32, 105, 105), dtype=torch.complex128, device="cuda")
    C = torch.full_like(A, 7.0)
    with pytest.raises(nspt.NsptError) as e:
        nspt.nspt_series_mul_noalloc(A, A, C)
    assert e.value.code == nspt.NSPT_ETOOBIG
    assert "static scratch" in str(e.value)
    torch.cuda.synchronize()
    assert bool((C == 7.0).all())
    # the largest N that fits at this order does run
    A = series(104, 31, 9)
    C = nspt.nspt_series_mul_noalloc(A, A, torch.empty_like(A))
    ref = nspt.nspt_series_mul(A, A)
    torch.cuda.synchronize()
    assert per_order_error(C, ref, A, A) <= TOL
