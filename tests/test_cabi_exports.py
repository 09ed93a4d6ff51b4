"""CPU-side checks of the C-ABI library: it builds, loads, and exports every symbol that
include/nspt.h declares.  No compute call is made here (no GPU in this container); argument
validation that happens before any CUDA call is exercised."""
import ctypes
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lib():
    from paper_2001_02835_b200 import build
    path = build.build()
    return ctypes.CDLL(str(path))


def declared_functions(headers=("nspt.h", "nspt_debug.h")):
    names = set()
    for h in headers:
        text = (ROOT / "include" / h).read_text()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        names |= set(re.findall(r"\b(nspt_[a-z0-9_]+)\s*\(", text))
    return sorted(names)


def test_header_declares_the_north_star_calls():
    names = declared_functions(("nspt.h",))
    for must in ("nspt_series_mul", "nspt_series_mul_batched", "nspt_staple"):
        assert must in names
    # diagnostics are kept out of the method's boundary
    for dbg in ("nspt_set_gemm_variant", "nspt_profile", "nspt_profile_read", "nspt_probe_fp64_peak", "nspt_launch_count"):
        assert dbg not in names and dbg in declared_functions(("nspt_debug.h",))


def test_library_exports_every_declared_symbol(lib):
    for name in declared_functions():
        assert hasattr(lib, name), f"libnspt.so does not export {name}"


def test_binding_lists_every_declared_symbol():
    from paper_2001_02835_b200 import binding
    assert sorted(binding.EXPORTS) == declared_functions()
    for name in binding.EXPORTS:
        assert hasattr(binding, name), f"binding lacks a wrapper named {name}"


def test_argument_validation_without_a_gpu(lib):
    lib.nspt_strerror.restype = ctypes.c_char_p
    lib.nspt_workspace_bytes.argtypes = [ctypes.c_int] * 4 + [ctypes.POINTER(ctypes.c_size_t)]
    out = ctypes.c_size_t(0)
    assert lib.nspt_workspace_bytes(225, 63, 1, 0, ctypes.byref(out)) == 0
    # three spectra of L=128 modes x 225 x 225 interleaved complex128
    assert out.value >= 3 * 128 * 225 * 225 * 16
    assert lib.nspt_workspace_bytes(225, 31, 1, 1, ctypes.byref(out)) == 0 and out.value > 0
    assert lib.nspt_workspace_bytes(0, 3, 1, 0, ctypes.byref(out)) == -1
    assert lib.nspt_workspace_bytes(4, 128, 1, 0, ctypes.byref(out)) == -1
    assert lib.nspt_workspace_bytes(4, 3, 1, 7, ctypes.byref(out)) == -1
    assert lib.nspt_series_mul(None, None, None, 4, 3) == -1
    assert lib.nspt_series_mul_batched(None, None, None, 4, 3, 2) == -1
    assert lib.nspt_staple(None, None, None, 4, 3) == -1
    assert lib.nspt_series_exp(None, None, 4, 3) == -1
    assert lib.nspt_series_exp_batched(None, None, 4, 3, 2) == -1
    assert lib.nspt_series_mul_batched(None, None, None, 4, 3, 70000) == -1
    lib.nspt_force.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_double, ctypes.c_int, ctypes.c_int]
    assert lib.nspt_force(None, None, 1.0, 4, 3) == -1
    assert lib.nspt_set_gemm_variant(1) == 0     # FP64 tensor pipe: spectra only
    assert lib.nspt_workspace_bytes(225, 31, 5, 2, ctypes.byref(out)) == 0 and out.value == 5 * 12 * 64 * 225 * 225 * 16 + 256   # Paterson-Stockmeyer: 6 powers + 6 block polynomials, + pad
    fp64_bytes = out.value
    assert lib.nspt_set_gemm_variant(-1) == 0    # automatic: INT8 tensor cores at this size, the int8 slice store comes on top
    assert lib.nspt_workspace_bytes(225, 31, 5, 2, ctypes.byref(out)) == 0 and out.value > fp64_bytes
    assert lib.nspt_workspace_bytes(100, 31, 1, 0, ctypes.byref(out)) == 0 and out.value == 3 * 64 * 100 * 100 * 16 + 256      # below N = 192: FP64 pipe
    assert lib.nspt_set_order_scale(ctypes.c_double(-1.0)) == -1
    assert lib.nspt_set_gemm_variant(9) == -1 and lib.nspt_set_gemm_variant(-2) == -1 and lib.nspt_set_gemm_variant(1) == 0
    assert b"invalid" in lib.nspt_strerror(-1)
    assert lib.nspt_version() >= 100


def test_product_path_has_no_cpu_fallback():
    # the binding must refuse to import without the CUDA library instead of falling back, and the
    # oracle and the CUDA package must not import each other
    src = (ROOT / "paper_2001_02835_b200" / "binding.py").read_text()
    assert "raise ImportError" in src
    imp = re.compile(r"^\s*(import|from)\s+oracle\b", re.M)
    for f in (ROOT / "paper_2001_02835_b200").rglob("*.py"):
        assert not imp.search(f.read_text()), f"{f} imports the oracle"
    for f in (ROOT / "paper_2001_02835_b200" / "csrc").glob("*"):
        assert "oracle" not in f.read_text().replace("the oracle shares nothing with this", ""), f
    imp2 = re.compile(r"^\s*(import|from)\s+paper_2001_02835_b200\b", re.M)
    for f in (ROOT / "oracle").glob("*.py"):
        assert not imp2.search(f.read_text()), f"{f} imports the CUDA package"
    assert "include" not in (ROOT / "oracle" / "nspt_oracle.c").read_text().split("*/", 1)[1].replace(
        "#include <stdlib.h>", "").replace("#include <string.h>", "").replace("#include <omp.h>", "")


def test_binding_rejects_mismatched_host_operands():
    # the C ABI takes N, Ntrunc and batch once; a short second operand or output would be overrun silently, so the
    # wrappers check every array before the call (no CUDA call is reached here)
    import numpy as np
    from paper_2001_02835_b200 import binding
    A = np.zeros((4, 3, 3), dtype=np.complex128)
    small = np.zeros((3, 3, 3), dtype=np.complex128)
    with pytest.raises(ValueError):
        binding.nspt_series_mul_host(A, A, small)
    with pytest.raises(ValueError):
        binding.nspt_series_mul_host(A, small, A)
    with pytest.raises(ValueError):
        binding.nspt_series_mul_batched_host(A[None], A[None], small[None])
    with pytest.raises(ValueError):
        binding.nspt_staple_host([A, A, A, small], np.ones((4, 4)), [A, A, A, A])
    with pytest.raises(ValueError):
        binding.nspt_staple_host([A, A, A, A], np.ones((4, 4)), [A, A, small, A])
    with pytest.raises(ValueError):
        binding.nspt_staple_host([A, A, A], np.ones((4, 4)), [A, A, A])
