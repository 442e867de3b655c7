"""ctypes loader for the float64 C oracle (``plspec_oracle.c``).

TEST INFRASTRUCTURE, NOT PRODUCT CODE (see ``oracle/__init__.py``).  Argument
marshalling only; all arithmetic is in the C file, which cites the paper.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

CF32 = 0  # voltages are interleaved float32 (re, im)
SC16 = 1  # voltages are interleaved int16 (I, Q), no scaling (reading A12)

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "plspec_oracle.c")
_LIB = os.path.join(_HERE, "libplspec_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no CUDA involved). Returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.plspec_oracle_fft.argtypes = [ctypes.c_void_p, ctypes.c_int]
        lib.plspec_oracle_fft.restype = ctypes.c_int
        lib.plspec_oracle_accumulate.argtypes = [
            ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
            ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int,
            ctypes.c_void_p, ctypes.c_int,
        ]
        lib.plspec_oracle_accumulate.restype = ctypes.c_int
        lib.plspec_oracle_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(_load().plspec_oracle_max_threads())


def fft(x: np.ndarray) -> np.ndarray:
    """The oracle's own radix-2 forward FFT of a complex128 vector (for pinning it)."""
    x = np.ascontiguousarray(x, dtype=np.complex128).copy()
    rc = _load().plspec_oracle_fft(x.ctypes.data, x.shape[0])
    if rc != 0:
        raise ValueError(f"plspec_oracle_fft failed ({rc})")
    return x


def spectra(voltages: np.ndarray, codes: np.ndarray, *, N: int, n_ranges: int,
            r0: int = 0, stride: int = 1, S: np.ndarray | None = None,
            n_threads: int = 0) -> np.ndarray:
    """S[r][f] (+)= sum_p |FFT_N(V[p][r0+r*stride+t] * conj(C[p][t]))[f]|^2, float64.

    voltages: [P][ipp_len] complex64, or [P][ipp_len][2] int16 (sc16).
    codes:    [P][code_len] complex64.
    S:        optional float64 [n_ranges][N] to accumulate into (else zeros).
    """
    codes = np.ascontiguousarray(codes)
    if codes.dtype != np.complex64 or codes.ndim != 2:
        raise TypeError("codes must be complex64 [P][code_len]")
    voltages = np.ascontiguousarray(voltages)
    if voltages.dtype == np.complex64 and voltages.ndim == 2:
        dtype = CF32
    elif voltages.dtype == np.int16 and voltages.ndim == 3 and voltages.shape[2] == 2:
        dtype = SC16
    else:
        raise TypeError("voltages must be complex64 [P][M] or int16 [P][M][2]")
    P, ipp_len = voltages.shape[0], voltages.shape[1]
    if codes.shape[0] != P:
        raise ValueError("codes and voltages disagree on the number of IPPs")
    if S is None:
        S = np.zeros((n_ranges, N), dtype=np.float64)
    if S.dtype != np.float64 or S.shape != (n_ranges, N) or not S.flags.c_contiguous:
        raise TypeError("S must be C-contiguous float64 [n_ranges][N]")
    rc = _load().plspec_oracle_accumulate(
        N, codes.shape[1], n_ranges, r0, stride, ipp_len, dtype,
        voltages.ctypes.data, codes.ctypes.data, P, S.ctypes.data, n_threads)
    if rc != 0:
        raise ValueError(f"plspec_oracle_accumulate rejected its arguments ({rc})")
    return S
