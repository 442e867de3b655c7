"""Thin ctypes binding of libplspec.so -- same names as include/plspec.h.

Argument marshalling only: every step of the path (sc16 conversion, decode, FFT, |X|^2,
accumulation, write-out) runs in the CUDA kernels behind the C ABI.  There is no CPU
fallback: if the library is missing or fails to load, importing callers get an exception.

Buffers may be torch tensors (CUDA or CPU, pinned or not) or numpy arrays (host); the
binding passes their raw pointers.  PyTorch is used for device memory and streams only.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

PLSPEC_CF32 = 0
PLSPEC_SC16 = 1

PLSPEC_OK = 0
PLSPEC_ERR_INVALID_ARG = -1
PLSPEC_ERR_ALLOC = -2
PLSPEC_ERR_CUDA = -3
PLSPEC_ERR_UNSUPPORTED = -4

PLSPEC_OPT_KERNEL = 1
PLSPEC_OPT_IPP_CHUNKS = 2
PLSPEC_OPT_H2D_BATCH = 3
PLSPEC_OPT_BPSK_PACK = 4
PLSPEC_OPT_STAGE = 5
PLSPEC_OPT_SPLIT = 6
PLSPEC_OPT_SHARED_CODE = 7
PLSPEC_OPT_DEFER = 8
PLSPEC_OPT_RING_DEPTH = 9
PLSPEC_OPT_RING_AHEAD = 10
KERNEL_AUTO, KERNEL_GENERIC, KERNEL_FUSED = 0, 1, 2

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libplspec.so")

# every symbol include/plspec.h declares (tests check the library exports each one)
EXPORTED_SYMBOLS = (
    "plspec_create", "plspec_accumulate", "plspec_finalize", "plspec_reset", "plspec_destroy",
    "plspec_configure", "plspec_get_stats", "plspec_last_cuda_error", "plspec_profile", "plspec_mean_spectrum",
    "plspec_diag_fp32_peak", "plspec_diag_mem_bandwidth", "plspec_finalize_products", "plspec_profile_static",
    "plspec_strerror",
    "plspec_version",
)
_INT_STATUS = EXPORTED_SYMBOLS[:-2]          # every call but strerror / version returns an int status


class plspec_stats_t(ctypes.Structure):
    _fields_ = [
        ("kernel_launches", ctypes.c_longlong),
        ("h2d_bytes", ctypes.c_longlong),
        ("d2h_bytes", ctypes.c_longlong),
        ("ipps_accumulated", ctypes.c_longlong),
        ("kernel_kind", ctypes.c_int),
        ("ipp_chunks_last", ctypes.c_int),
    ]


class plspec_products_t(ctypes.Structure):
    _fields_ = [
        ("n_ipp", ctypes.c_int), ("centred", ctypes.c_int), ("P_out", ctypes.c_void_p),
        ("k_min", ctypes.c_int), ("guard", ctypes.c_int),
        ("k_up", ctypes.c_void_p), ("p_up", ctypes.c_void_p), ("k_dn", ctypes.c_void_p), ("p_dn", ctypes.c_void_p),
        ("noise", ctypes.c_void_p),
    ]


class PlspecError(RuntimeError):
    def __init__(self, status: int, where: str, cuda_error: int = 0):
        self.status = status
        self.cuda_error = cuda_error
        msg = f"{where}: {strerror(status)} (status {status}"
        msg += f", cudaError {cuda_error})" if cuda_error else ")"
        super().__init__(msg)


_lib = None


def lib() -> ctypes.CDLL:
    """Load libplspec.so (built in-tree by paper_2311_18737_b200.build). Fails loudly."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(
                f"{LIB_PATH} is missing: build it with `python -m paper_2311_18737_b200.build` "
                "(nvcc, sm_100a). There is no CPU fallback.")
        L = ctypes.CDLL(LIB_PATH)
        vp, ci = ctypes.c_void_p, ctypes.c_int
        L.plspec_create.argtypes = [ci, ci, ci, ci, ci, ci, ci, ctypes.POINTER(vp)]
        L.plspec_accumulate.argtypes = [vp, vp, vp, ci, vp]
        L.plspec_finalize.argtypes = [vp, vp]
        L.plspec_reset.argtypes = [vp]
        L.plspec_destroy.argtypes = [vp]
        L.plspec_configure.argtypes = [vp, ci, ci]
        L.plspec_get_stats.argtypes = [vp, ctypes.POINTER(plspec_stats_t)]
        L.plspec_last_cuda_error.argtypes = [vp]
        L.plspec_strerror.argtypes = [ci]
        L.plspec_strerror.restype = ctypes.c_char_p
        L.plspec_version.restype = ctypes.c_char_p
        L.plspec_profile.argtypes = [vp, ci, ci, ci, ci, ci, vp, vp, vp, vp, vp, vp]
        L.plspec_profile_static.argtypes = [vp, ci, ci, ci, ci, ci, vp, vp, vp, vp, vp, vp]
        L.plspec_mean_spectrum.argtypes = [vp, vp, ci, ci, ci, ci, vp]
        L.plspec_finalize_products.argtypes = [vp, vp, ctypes.POINTER(plspec_products_t)]
        L.plspec_diag_mem_bandwidth.argtypes = [ci, ctypes.c_longlong, ci, ci, ctypes.POINTER(ctypes.c_double), vp]
        L.plspec_diag_fp32_peak.argtypes = [ci, ci, ci, ctypes.POINTER(ctypes.c_double),
                                            ctypes.POINTER(ctypes.c_double), vp]
        for name in _INT_STATUS:
            getattr(L, name).restype = ci
        _lib = L
    return _lib


def strerror(status: int) -> str:
    try:
        return lib().plspec_strerror(int(status)).decode()
    except Exception:
        return f"status {status}"


def _ptr(buf) -> int:
    """Raw address of a torch tensor / numpy array / int; contiguity is the caller's duty."""
    if buf is None:
        return 0
    if isinstance(buf, int):
        return buf
    if hasattr(buf, "data_ptr"):
        if not buf.is_contiguous():
            raise ValueError("tensor must be contiguous")
        return int(buf.data_ptr())
    if isinstance(buf, np.ndarray):
        if not buf.flags.c_contiguous:
            raise ValueError("array must be C-contiguous")
        return int(buf.ctypes.data)
    raise TypeError(f"unsupported buffer type {type(buf)}")


def _stream_ptr(stream) -> int:
    if stream is None:
        return 0
    if isinstance(stream, int):
        return stream
    return int(stream.cuda_stream)          # torch.cuda.Stream


# ---- the C calls, one to one -----------------------------------------------------------------
def plspec_create(N, code_len, n_ranges, r0, stride, ipp_len, dtype) -> int:
    h = ctypes.c_void_p()
    rc = lib().plspec_create(N, code_len, n_ranges, r0, stride, ipp_len, dtype, ctypes.byref(h))
    if rc != PLSPEC_OK:
        raise PlspecError(rc, "plspec_create")
    return h.value


def _check(h, rc, where):
    if rc != PLSPEC_OK:
        raise PlspecError(rc, where, lib().plspec_last_cuda_error(h) if h else 0)


def plspec_accumulate(h, voltages, codes, n_ipp, stream=None) -> None:
    _check(h, lib().plspec_accumulate(h, _ptr(voltages), _ptr(codes), int(n_ipp), _stream_ptr(stream)),
           "plspec_accumulate")


def plspec_finalize(h, S_out) -> None:
    _check(h, lib().plspec_finalize(h, _ptr(S_out)), "plspec_finalize")


def plspec_finalize_products(h, S_out, n_ipp, P_out=None, centred=False, k_min=1, guard=0, k_up=None, p_up=None,
                             k_dn=None, p_dn=None, noise=None) -> None:
    prod = plspec_products_t(int(n_ipp), int(bool(centred)), _ptr(P_out) or None, int(k_min), int(guard),
                             _ptr(k_up) or None, _ptr(p_up) or None, _ptr(k_dn) or None, _ptr(p_dn) or None,
                             _ptr(noise) or None)
    _check(h, lib().plspec_finalize_products(h, _ptr(S_out), ctypes.byref(prod)), "plspec_finalize_products")


def plspec_profile(S, n_ranges, N, n_ipp, k_min, guard, k_up, p_up, k_dn, p_dn, noise, stream=None) -> None:
    _check(None, lib().plspec_profile(_ptr(S), int(n_ranges), int(N), int(n_ipp), int(k_min), int(guard), _ptr(k_up),
                                      _ptr(p_up), _ptr(k_dn), _ptr(p_dn), _ptr(noise), _stream_ptr(stream)),
           "plspec_profile")


STATIC_MAX_GATES = 8192                       # PLSPEC_STATIC_MAX_GATES of include/plspec.h


def plspec_profile_static(S, n_ranges, N, n_ipp, k_min, guard, k_up, p_up, k_dn, p_dn, noise, stream=None) -> None:
    """plspec_profile without any device allocation (file-scope workspace, n_ranges <= STATIC_MAX_GATES; calls that
    overlap on the GPU race on it -- include/plspec.h)."""
    _check(None, lib().plspec_profile_static(_ptr(S), int(n_ranges), int(N), int(n_ipp), int(k_min), int(guard),
                                             _ptr(k_up), _ptr(p_up), _ptr(k_dn), _ptr(p_dn), _ptr(noise),
                                             _stream_ptr(stream)), "plspec_profile_static")


def plspec_mean_spectrum(S, P_out, n_ranges, N, n_ipp, centred=False, stream=None) -> None:
    _check(None, lib().plspec_mean_spectrum(_ptr(S), _ptr(P_out), int(n_ranges), int(N), int(n_ipp), int(bool(centred)),
                                            _stream_ptr(stream)), "plspec_mean_spectrum")


def plspec_diag_fp32_peak(packed=True, iters=1 << 16, reps=10, stream=None) -> dict:
    """Measured FP32 multiply-add rate of the current device in TFLOP/s (best launch, mean over launches)."""
    best, mean = ctypes.c_double(), ctypes.c_double()
    _check(None, lib().plspec_diag_fp32_peak(int(bool(packed)), int(iters), int(reps), ctypes.byref(best),
                                             ctypes.byref(mean), _stream_ptr(stream)), "plspec_diag_fp32_peak")
    return {"tflops_best": best.value, "tflops_mean": mean.value}


def plspec_diag_mem_bandwidth(kind, n_bytes, n_ctas, passes=8, stream=None) -> float:
    """Streaming bandwidth in GB/s (kind: 0 read, 1 write, 2 copy, 3 TMA bulk stores); see include/plspec.h."""
    gbs = ctypes.c_double()
    _check(None, lib().plspec_diag_mem_bandwidth(int(kind), int(n_bytes), int(n_ctas), int(passes), ctypes.byref(gbs),
                                                 _stream_ptr(stream)), "plspec_diag_mem_bandwidth")
    return gbs.value


def plspec_reset(h) -> None:
    _check(h, lib().plspec_reset(h), "plspec_reset")


def plspec_destroy(h) -> None:
    lib().plspec_destroy(h)


def plspec_configure(h, option, value) -> None:
    _check(h, lib().plspec_configure(h, int(option), int(value)), "plspec_configure")


def plspec_get_stats(h) -> dict:
    st = plspec_stats_t()
    _check(h, lib().plspec_get_stats(h, ctypes.byref(st)), "plspec_get_stats")
    return {k: getattr(st, k) for k, _ in plspec_stats_t._fields_}


def plspec_version() -> str:
    return lib().plspec_version().decode()


# ---- convenience wrapper (lifetime only; no arithmetic) ---------------------------------------
class Integrator:
    """Owns one plspec handle.  `accumulate` / `finalize` forward to the C calls."""

    def __init__(self, N, code_len, n_ranges, r0=0, stride=1, ipp_len=0, dtype=PLSPEC_CF32,
                 kernel=KERNEL_AUTO, ipp_chunks=0, h2d_batch=0, bpsk_pack=1, stage=1, split=1, shared_code=0, defer=1, ring_depth=0, ring_ahead=0):
        self.N, self.n_ranges = N, n_ranges
        self.h = plspec_create(N, code_len, n_ranges, r0, stride, ipp_len, dtype)
        try:
            if kernel:
                plspec_configure(self.h, PLSPEC_OPT_KERNEL, kernel)
            if ipp_chunks:
                plspec_configure(self.h, PLSPEC_OPT_IPP_CHUNKS, ipp_chunks)
            if h2d_batch:
                plspec_configure(self.h, PLSPEC_OPT_H2D_BATCH, h2d_batch)
            if not bpsk_pack:
                plspec_configure(self.h, PLSPEC_OPT_BPSK_PACK, 0)
            if stage != 1:
                plspec_configure(self.h, PLSPEC_OPT_STAGE, stage)
            if split != 1:
                plspec_configure(self.h, PLSPEC_OPT_SPLIT, split)
            if shared_code:
                plspec_configure(self.h, PLSPEC_OPT_SHARED_CODE, 1)
            if not defer:
                plspec_configure(self.h, PLSPEC_OPT_DEFER, 0)
            if ring_depth:
                plspec_configure(self.h, PLSPEC_OPT_RING_DEPTH, ring_depth)
            if ring_ahead:
                plspec_configure(self.h, PLSPEC_OPT_RING_AHEAD, ring_ahead)
        except Exception:
            self.close()
            raise

    @classmethod
    def for_workload(cls, w, **kw):
        return cls(w.N, w.code_len, w.n_ranges, w.r0, w.stride, w.ipp_len, w.dtype, **kw)

    def accumulate(self, voltages, codes, n_ipp=None, stream=None):
        if n_ipp is None:
            n_ipp = int(codes.shape[0])
        plspec_accumulate(self.h, voltages, codes, n_ipp, stream)

    def finalize(self, S_out):
        plspec_finalize(self.h, S_out)
        return S_out

    def finalize_products(self, S_out, n_ipp, **products):
        plspec_finalize_products(self.h, S_out, n_ipp, **products)
        return S_out

    def reset(self):
        plspec_reset(self.h)

    def stats(self):
        return plspec_get_stats(self.h)

    def close(self):
        if getattr(self, "h", None):
            plspec_destroy(self.h)
            self.h = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
