"""Thin ctypes binding of libnspt.so with the names of include/nspt.h.

Argument marshalling only: every step of the path runs in the library's CUDA kernels.
Importing this module loads the library and fails loudly if it is missing (build it with
``python -m paper_2001_02835_b200.build``); there is no CPU fallback of any kind.

Device entry points take torch CUDA tensors (complex128, contiguous, shape
(Ntrunc+1, N, N) or (batch, Ntrunc+1, N, N)); host entry points take numpy arrays or torch
CPU tensors of the same shape.  torch is used for device memory and streams only.
"""
from __future__ import annotations

import ctypes
from pathlib import Path

import numpy as np

_PKG = Path(__file__).resolve().parent
_LIB_PATH = _PKG / "libnspt.so"

NSPT_OK, NSPT_EINVAL, NSPT_ENOMEM, NSPT_ECUDA, NSPT_EARCH = 0, -1, -2, -3, -4
NSPT_OP_SERIES_MUL, NSPT_OP_STAPLE, NSPT_OP_SERIES_EXP = 0, 1, 2
STAGES = {"fft_forward": 0, "zgemm_modes": 1, "fft_inverse": 2, "fft_retruncate": 3, "other": 4, "freq_block_polys": 5,
          "int8_slicing": 6}

EXPORTS = [
    "nspt_series_mul", "nspt_series_mul_batched", "nspt_series_mul_noalloc", "nspt_staple", "nspt_staple_dir", "nspt_series_exp", "nspt_series_exp_batched", "nspt_link_update", "nspt_link_update_batched", "nspt_force",
    "nspt_series_mul_host", "nspt_series_mul_batched_host", "nspt_staple_host",
    "nspt_set_stream", "nspt_set_order_scale", "nspt_workspace_bytes", "nspt_set_workspace",
    "nspt_set_gemm_variant", "nspt_set_conv_algorithm", "nspt_probe_fp64_peak", "nspt_profile", "nspt_profile_read", "nspt_launch_count",
    "nspt_release", "nspt_strerror", "nspt_version",
]


class NsptError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where} failed with code {code}: {strerror(code)}")


if not _LIB_PATH.exists():
    raise ImportError(
        f"{_LIB_PATH} is missing: build the CUDA library first (python -m paper_2001_02835_b200.build). "
        "There is no CPU fallback.")

_lib = ctypes.CDLL(str(_LIB_PATH))
_vp, _int, _dbl = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
_lib.nspt_series_mul.argtypes = [_vp, _vp, _vp, _int, _int]
_lib.nspt_series_mul_batched.argtypes = [_vp, _vp, _vp, _int, _int, _int]
_lib.nspt_series_mul_noalloc.argtypes = [_vp, _vp, _vp, _int, _int]
_lib.nspt_staple.argtypes = [ctypes.POINTER(_vp), _vp, ctypes.POINTER(_vp), _int, _int]
_lib.nspt_staple_dir.argtypes = [ctypes.POINTER(_vp), _vp, _int, _vp, _int, _int]
_lib.nspt_series_exp.argtypes = [_vp, _vp, _int, _int]
_lib.nspt_series_exp_batched.argtypes = [_vp, _vp, _int, _int, _int]
_lib.nspt_link_update.argtypes = [_vp, _vp, _dbl, _vp, _int, _int]
_lib.nspt_link_update_batched.argtypes = [_vp, _vp, _dbl, _vp, _int, _int, _int]
_lib.nspt_force.argtypes = [_vp, _vp, _dbl, _int, _int]
_lib.nspt_series_mul_host.argtypes = [_vp, _vp, _vp, _int, _int]
_lib.nspt_series_mul_batched_host.argtypes = [_vp, _vp, _vp, _int, _int, _int]
_lib.nspt_staple_host.argtypes = [ctypes.POINTER(_vp), _vp, ctypes.POINTER(_vp), _int, _int]
_lib.nspt_set_stream.argtypes = [_vp]
_lib.nspt_set_order_scale.argtypes = [_dbl]
_lib.nspt_workspace_bytes.argtypes = [_int, _int, _int, _int, ctypes.POINTER(ctypes.c_size_t)]
_lib.nspt_set_workspace.argtypes = [_vp, ctypes.c_size_t]
_lib.nspt_set_gemm_variant.argtypes = [_int]
_lib.nspt_set_conv_algorithm.argtypes = [_int]
_lib.nspt_probe_fp64_peak.argtypes = [ctypes.POINTER(_dbl)]
_lib.nspt_profile.argtypes = [_int]
_lib.nspt_profile_read.argtypes = [_int, ctypes.POINTER(_dbl), ctypes.POINTER(ctypes.c_longlong)]
_lib.nspt_launch_count.restype = ctypes.c_longlong
_lib.nspt_strerror.argtypes = [_int]
_lib.nspt_strerror.restype = ctypes.c_char_p
for _name in EXPORTS:
    if _name not in ("nspt_launch_count", "nspt_strerror"):
        getattr(_lib, _name).restype = _int


def library_path() -> Path:
    return _LIB_PATH


def strerror(code: int) -> str:
    return _lib.nspt_strerror(int(code)).decode()


def _check(code: int, where: str):
    if code != 0:
        raise NsptError(code, where)


def _torch():
    import torch
    return torch


def _dev_series(x, name):
    torch = _torch()
    if not isinstance(x, torch.Tensor) or not x.is_cuda:
        raise TypeError(f"{name}: expected a CUDA torch tensor")
    if x.dtype != torch.complex128 or not x.is_contiguous():
        raise TypeError(f"{name}: expected contiguous complex128")
    return x


def _match(x, ref, name):
    """Every operand and output of a call must have the shape of the first one (the C ABI takes N, Ntrunc and batch
    once and cannot see a short buffer), and, for device tensors, live on the same device."""
    if tuple(x.shape) != tuple(ref.shape):
        raise ValueError(f"{name}: shape {tuple(x.shape)} does not match {tuple(ref.shape)}")
    if getattr(ref, "is_cuda", False) and x.device != ref.device:
        raise ValueError(f"{name}: on {x.device}, expected {ref.device}")
    return x


def _shape(x, batched):
    if batched:
        if x.ndim != 4 or x.shape[2] != x.shape[3]:
            raise ValueError("expected shape (batch, Ntrunc+1, N, N)")
        return int(x.shape[0]), int(x.shape[1]) - 1, int(x.shape[2])
    if x.ndim != 3 or x.shape[1] != x.shape[2]:
        raise ValueError("expected shape (Ntrunc+1, N, N)")
    return 1, int(x.shape[0]) - 1, int(x.shape[1])


def use_current_stream():
    """Point the library at torch's current CUDA stream."""
    nspt_set_stream(_torch().cuda.current_stream().cuda_stream)


# ------------------------------------------------------------------------------ device calls

def nspt_series_mul(A, B, C=None):
    """C = A * B (eq. 2.5) on the device.  Asynchronous on the library stream."""
    torch = _torch()
    A, B = _dev_series(A, "A"), _dev_series(B, "B")
    if A.shape != B.shape:
        raise ValueError("A and B must have the same shape")
    _, Ntrunc, N = _shape(A, False)
    if C is None:
        C = torch.empty_like(A)
    _match(_dev_series(B, "B"), A, "B")
    _match(_dev_series(C, "C"), A, "C")
    _check(_lib.nspt_series_mul(A.data_ptr(), B.data_ptr(), C.data_ptr(), N, Ntrunc), "nspt_series_mul")
    return C


NSPT_NOALLOC_SCRATCH_BYTES = 32 << 20
NSPT_ETOOBIG = -5


def nspt_series_mul_noalloc(A, B, C):
    """C = A * B with the scratch in the library's static device array: no allocation anywhere, so the caller passes C.
    Raises NsptError (code NSPT_ETOOBIG) when 3 * 16 * L * N * N + 16640 bytes exceed NSPT_NOALLOC_SCRATCH_BYTES."""
    A, B, C = _dev_series(A, "A"), _dev_series(B, "B"), _dev_series(C, "C")
    _, Ntrunc, N = _shape(A, False)
    _match(B, A, "B")
    _match(C, A, "C")
    _check(_lib.nspt_series_mul_noalloc(A.data_ptr(), B.data_ptr(), C.data_ptr(), N, Ntrunc), "nspt_series_mul_noalloc")
    return C


def nspt_series_mul_batched(A, B, C=None):
    torch = _torch()
    A, B = _dev_series(A, "A"), _dev_series(B, "B")
    if A.shape != B.shape:
        raise ValueError("A and B must have the same shape")
    batch, Ntrunc, N = _shape(A, True)
    if C is None:
        C = torch.empty_like(A)
    _match(_dev_series(B, "B"), A, "B")
    _match(_dev_series(C, "C"), A, "C")
    _check(_lib.nspt_series_mul_batched(A.data_ptr(), B.data_ptr(), C.data_ptr(), N, Ntrunc, batch),
           "nspt_series_mul_batched")
    return C


def _z_array(z):
    z = np.ascontiguousarray(np.asarray(z, dtype=np.complex128).reshape(4, 4))
    return z


def nspt_staple(U, z, S=None):
    """S_mu of eq. 2.3 for mu = 0..3.  U: four device series; z: 4x4 complex (host)."""
    torch = _torch()
    U = [_dev_series(u, "U") for u in U]
    if len(U) != 4:
        raise ValueError("four link series expected")
    _, Ntrunc, N = _shape(U[0], False)
    if S is None:
        S = [torch.empty_like(u) for u in U]
    S = [_dev_series(s, "S") for s in S]
    if len(S) != 4:
        raise ValueError("four staple series expected")
    for t in U[1:]:
        _match(t, U[0], "U")
    for t in S:
        _match(t, U[0], "S")
    zz = _z_array(z)
    Up = (_vp * 4)(*[u.data_ptr() for u in U])
    Sp = (_vp * 4)(*[s.data_ptr() for s in S])
    _check(_lib.nspt_staple(Up, zz.ctypes.data, Sp, N, Ntrunc), "nspt_staple")
    return S


def nspt_staple_dir(U, z, mu: int, S_mu=None):
    """S_mu of eq. 2.3 for ONE direction (the per-GPU unit of the paper's direction split)."""
    torch = _torch()
    U = [_dev_series(u, "U") for u in U]
    if len(U) != 4:
        raise ValueError("four link series expected")
    if not 0 <= int(mu) <= 3:
        raise ValueError("mu must be 0..3")
    _, Ntrunc, N = _shape(U[0], False)
    for t in U[1:]:
        _match(t, U[0], "U")
    if S_mu is None:
        S_mu = torch.empty_like(U[0])
    _match(_dev_series(S_mu, "S_mu"), U[0], "S_mu")
    if any(S_mu.data_ptr() == u.data_ptr() for u in U):
        raise ValueError("S_mu must not alias a link series")
    zz = _z_array(z)
    Up = (_vp * 4)(*[u.data_ptr() for u in U])
    _check(_lib.nspt_staple_dir(Up, zz.ctypes.data, int(mu), S_mu.data_ptr(), N, Ntrunc), "nspt_staple_dir")
    return S_mu


def nspt_series_exp(X, E=None):
    """E = exp(X) = sum_m X^{*m}/m! for a series with X^(0) = 0 (X^(0) is not read).  Device tensors."""
    torch = _torch()
    X = _dev_series(X, "X")
    _, Ntrunc, N = _shape(X, False)
    if E is None:
        E = torch.empty_like(X)
    _match(_dev_series(E, "E"), X, "E")
    _check(_lib.nspt_series_exp(X.data_ptr(), E.data_ptr(), N, Ntrunc), "nspt_series_exp")
    return E


def nspt_series_exp_batched(X, E=None):
    """E_b = exp(X_b) for a stack of series, shape (batch, Ntrunc+1, N, N)."""
    torch = _torch()
    X = _dev_series(X, "X")
    batch, Ntrunc, N = _shape(X, True)
    if E is None:
        E = torch.empty_like(X)
    _match(_dev_series(E, "E"), X, "E")
    _check(_lib.nspt_series_exp_batched(X.data_ptr(), E.data_ptr(), N, Ntrunc, batch), "nspt_series_exp_batched")
    return E


def nspt_link_update(P, U, eps: float, Unew=None):
    """Unew = exp(i eps P) * U; P^(0) is not read.  Device tensors, shape (Ntrunc+1, N, N); Unew may alias
    U or P.  (A stack of links, shape (batch, Ntrunc+1, N, N), is forwarded to nspt_link_update_batched.)"""
    torch = _torch()
    P, U = _dev_series(P, "P"), _dev_series(U, "U")
    if P.dim() == 4:
        return nspt_link_update_batched(P, U, eps, Unew)
    _match(U, P, "U")
    _, Ntrunc, N = _shape(P, False)
    if Unew is None:
        Unew = torch.empty_like(U)
    _match(_dev_series(Unew, "Unew"), P, "Unew")
    _check(_lib.nspt_link_update(P.data_ptr(), U.data_ptr(), float(eps), Unew.data_ptr(), N, Ntrunc), "nspt_link_update")
    return Unew


def nspt_link_update_batched(P, U, eps: float, Unew=None):
    """Unew_b = exp(i eps P_b) * U_b for a stack of links (the four directions), shape (batch, Ntrunc+1, N, N)."""
    torch = _torch()
    P, U = _dev_series(P, "P"), _dev_series(U, "U")
    _match(U, P, "U")
    batch, Ntrunc, N = _shape(P, True)
    if Unew is None:
        Unew = torch.empty_like(U)
    _match(_dev_series(Unew, "Unew"), P, "Unew")
    _check(_lib.nspt_link_update_batched(P.data_ptr(), U.data_ptr(), float(eps), Unew.data_ptr(), N, Ntrunc, batch),
           "nspt_link_update_batched")
    return Unew


def nspt_force(S, c: float, F=None):
    """F^(k) = i c [S^(k) - S^(k)+ - Tr(S^(k) - S^(k)+)/N] (eq. 2.3).  Device tensors; F must not alias S."""
    torch = _torch()
    S = _dev_series(S, "S")
    _, Ntrunc, N = _shape(S, False)
    if F is None:
        F = torch.empty_like(S)
    _match(_dev_series(F, "F"), S, "F")
    _check(_lib.nspt_force(S.data_ptr(), F.data_ptr(), float(c), N, Ntrunc), "nspt_force")
    return F


# ------------------------------------------------------------------------------ host calls

def _host_ptr(x, name):
    """numpy array or torch CPU tensor -> (address, keepalive)."""
    if isinstance(x, np.ndarray):
        if x.dtype != np.complex128 or not x.flags.c_contiguous:
            raise TypeError(f"{name}: expected C-contiguous complex128")
        return x.ctypes.data, x
    torch = _torch()
    if isinstance(x, torch.Tensor) and not x.is_cuda:
        if x.dtype != torch.complex128 or not x.is_contiguous():
            raise TypeError(f"{name}: expected contiguous complex128")
        return x.data_ptr(), x
    raise TypeError(f"{name}: expected a numpy array or a torch CPU tensor")


def nspt_series_mul_host(A, B, C):
    _, Ntrunc, N = _shape(A, False)
    _match(B, A, "B")
    _match(C, A, "C")
    pa, _a = _host_ptr(A, "A")
    pb, _b = _host_ptr(B, "B")
    pc, _c = _host_ptr(C, "C")
    _check(_lib.nspt_series_mul_host(pa, pb, pc, N, Ntrunc), "nspt_series_mul_host")
    return C


def nspt_series_mul_batched_host(A, B, C):
    batch, Ntrunc, N = _shape(A, True)
    _match(B, A, "B")
    _match(C, A, "C")
    pa, _a = _host_ptr(A, "A")
    pb, _b = _host_ptr(B, "B")
    pc, _c = _host_ptr(C, "C")
    _check(_lib.nspt_series_mul_batched_host(pa, pb, pc, N, Ntrunc, batch), "nspt_series_mul_batched_host")
    return C


def nspt_staple_host(U, z, S):
    if len(U) != 4 or len(S) != 4:
        raise ValueError("four link series and four staple series expected")
    _, Ntrunc, N = _shape(U[0], False)
    for t in list(U[1:]) + list(S):
        _match(t, U[0], "U/S")
    up = [_host_ptr(u, "U") for u in U]
    sp = [_host_ptr(s, "S") for s in S]
    zz = _z_array(z)
    Up = (_vp * 4)(*[p for p, _ in up])
    Sp = (_vp * 4)(*[p for p, _ in sp])
    _check(_lib.nspt_staple_host(Up, zz.ctypes.data, Sp, N, Ntrunc), "nspt_staple_host")
    return S


# ------------------------------------------------------------------------------ context calls

def nspt_set_stream(stream_ptr):
    _check(_lib.nspt_set_stream(_vp(stream_ptr)), "nspt_set_stream")


def nspt_set_order_scale(s: float):
    _check(_lib.nspt_set_order_scale(float(s)), "nspt_set_order_scale")


def nspt_workspace_bytes(N: int, Ntrunc: int, batch: int = 1, op: int = NSPT_OP_SERIES_MUL) -> int:
    out = ctypes.c_size_t(0)
    _check(_lib.nspt_workspace_bytes(N, Ntrunc, batch, op, ctypes.byref(out)), "nspt_workspace_bytes")
    return int(out.value)


def nspt_set_workspace(dptr, nbytes: int):
    _check(_lib.nspt_set_workspace(_vp(dptr), nbytes), "nspt_set_workspace")


def nspt_set_gemm_variant(variant: int):
    _check(_lib.nspt_set_gemm_variant(int(variant)), "nspt_set_gemm_variant")


def nspt_set_conv_algorithm(algorithm: int):
    """0 = automatic, 1 = FFT-CONV, 2 = Naive-CONV (include/nspt_debug.h)."""
    _check(_lib.nspt_set_conv_algorithm(int(algorithm)), "nspt_set_conv_algorithm")


def nspt_profile(enable: bool):
    _check(_lib.nspt_profile(1 if enable else 0), "nspt_profile")


def nspt_profile_read(stage):
    """(milliseconds, launches) accumulated for a stage since the last read."""
    if isinstance(stage, str):
        stage = STAGES[stage]
    ms, n = _dbl(0.0), ctypes.c_longlong(0)
    _check(_lib.nspt_profile_read(int(stage), ctypes.byref(ms), ctypes.byref(n)), "nspt_profile_read")
    return float(ms.value), int(n.value)


def nspt_probe_fp64_peak() -> float:
    """Measured FP64 tensor-pipe (DMMA) peak of the current device in TFLOP/s."""
    out = _dbl(0.0)
    _check(_lib.nspt_probe_fp64_peak(ctypes.byref(out)), "nspt_probe_fp64_peak")
    return float(out.value)


def nspt_launch_count() -> int:
    return int(_lib.nspt_launch_count())


def nspt_release():
    _check(_lib.nspt_release(), "nspt_release")


def nspt_strerror(code: int) -> str:
    return strerror(code)


def nspt_version() -> int:
    return int(_lib.nspt_version())


def raw():
    """The ctypes library handle (for tests that call the C ABI with raw pointers)."""
    return _lib
