"""Seeded synthetic radar inputs shaped like BASELINE.json's configs.

This module serves BOTH the oracle tests and the CUDA path's tests / bench.  It holds
none of the method's arithmetic (no decode, no FFT of decoded windows, no |X|^2, no
accumulation): it only draws transmit codes and simulates received voltages with the
paper's measurement model, Eq. 2-3:

    V[p][n] = xi[n] + sum_g a_{p,g} * C[p][n - d_g] * m_{p,g}[n - d_g],   d_g = r0 + g*stride

with xi ~ CN(0, sigma^2), a_{p,g} ~ CN(0, SNR*sigma^2) redrawn every pulse ("does change
from pulse to pulse") and m a tone (or a narrow Lorentzian line) at the
plasma-line offset f_p(g) of a Chapman-layer profile.  The paper used SciPy-simulated
data and no public dataset; these inputs stand in for it.

Arrays are produced in *storage* dtype (complex64, or int16 pairs for sc16) so that the
oracle and the GPU read bit-identical bytes.  numpy only; importing this module does
not load the CUDA library.
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import numpy as np

CF32 = 0
SC16 = 1
FS_HZ = 25.0e6  # sample rate: 250 000 samples per 10 ms IPP (configs[4])


@dataclass(frozen=True)
class Workload:
    """Problem shape; field names follow plspec_create (include/plspec.h)."""
    name: str
    N: int
    code_len: int
    n_ranges: int
    r0: int
    stride: int
    ipp_len: int
    n_ipp: int
    dtype: int              # CF32 | SC16 (voltages only; codes are always complex64)
    code: str               # "bpsk" | "chirp"
    echo: str               # "tone1" | "tone" | "tone2" | "lorentz"
    echo_every: int = 1     # echoes injected at every k-th gate
    sigma: float = 1.0      # total noise std (per complex sample)
    snr: float = 0.01       # per-sample echo/noise power ratio
    seed: int = 0

    @property
    def span(self) -> int:
        return self.r0 + (self.n_ranges - 1) * self.stride + self.code_len

    @property
    def windows(self) -> int:
        return self.n_ipp * self.n_ranges

    @property
    def data_seconds(self) -> float:
        return self.n_ipp * self.ipp_len / FS_HZ

    @property
    def fft_flops(self) -> float:
        """Nominal 5*N*log2(N) per decoded window (BASELINE.json north_star)."""
        return 5.0 * self.N * np.log2(self.N) * self.windows


# BASELINE.json configs[0..4] (1-based cfg ids as in SURVEY.md section 8) + the paper's own
# workload (Table 1) as "paper".
CONFIGS = {
    "cfg1": Workload("cfg1", 1024, 1024, 64, 0, 1, 2048, 16, CF32, "bpsk", "tone1", seed=1000),
    "cfg2": Workload("cfg2", 4096, 4096, 500, 0, 1, 8192, 100, CF32, "bpsk", "tone", seed=2000),
    "cfg3": Workload("cfg3", 16384, 16384, 1000, 0, 1, 32768, 200, SC16, "bpsk", "tone2",
                     echo_every=4, sigma=1000.0, seed=3000),
    "cfg4": Workload("cfg4", 65536, 65536, 800, 0, 4, 131072, 50, CF32, "chirp", "lorentz",
                     echo_every=8, seed=4000),
    "cfg5": Workload("cfg5", 8192, 8192, 2000, 0, 1, 250000, 1000, SC16, "bpsk", "tone2",
                     echo_every=8, sigma=1000.0, seed=5000),
    "paper": Workload("paper", 16384, 16384, 4096, 0, 25, 250000, 100, CF32, "bpsk", "tone",
                      echo_every=16, seed=6000),
}


def scaled(w: Workload, *, n_ranges: int | None = None, n_ipp: int | None = None,
           ipp_len: int | None = None) -> Workload:
    """Same recipe with fewer gates / pulses (parity cases the oracle finishes quickly)."""
    n_ranges = w.n_ranges if n_ranges is None else n_ranges
    n_ipp = w.n_ipp if n_ipp is None else n_ipp
    span = w.r0 + (n_ranges - 1) * w.stride + w.code_len
    if ipp_len is None:
        ipp_len = max(span, min(w.ipp_len, 2 * span))
    return replace(w, n_ranges=n_ranges, n_ipp=n_ipp, ipp_len=ipp_len,
                   name=f"{w.name}[R={n_ranges},P={n_ipp}]")


def chapman_bins(n_ranges_full: int, N: int, gates: np.ndarray) -> np.ndarray:
    """Plasma-line offset (in FFT bins, real valued) per gate: sqrt of a Chapman-alpha
    layer, spanning bins 200..1800 at N = 4096 and scaled with N (configs[1])."""
    g = np.asarray(gates, dtype=np.float64)
    gpk, H = 0.45 * n_ranges_full, n_ranges_full / 6.0
    def c(x):
        z = (x - gpk) / H
        return np.exp(0.25 * (1.0 - z - np.exp(-z)))
    allg = np.arange(n_ranges_full, dtype=np.float64)
    cmin = c(allg).min()
    k_lo, k_hi = 200.0 * N / 4096.0, 1800.0 * N / 4096.0
    return k_lo + (k_hi - k_lo) * (c(g) - cmin) / (1.0 - cmin)


def make_codes(w: Workload, rng: np.random.Generator) -> np.ndarray:
    """codes[P][code_len] complex64: fresh random BPSK (+-1+0j) per IPP, or one linear-FM
    chirp sweeping +-0.4 of the sample rate repeated for every IPP (configs[3])."""
    if w.code == "bpsk":
        bits = rng.integers(0, 2, size=(w.n_ipp, w.code_len), dtype=np.int8)
        return (2.0 * bits - 1.0).astype(np.float32).astype(np.complex64)
    if w.code == "chirp":
        t = np.arange(w.code_len, dtype=np.float64)
        phase = -0.4 * t + 0.4 * t * t / w.code_len          # cycles; inst. freq -0.4..+0.4
        phase -= np.floor(phase)
        c = np.exp(2j * np.pi * phase).astype(np.complex64)
        return np.ascontiguousarray(np.broadcast_to(c, (w.n_ipp, w.code_len)))
    raise ValueError(w.code)


def _cn(rng, shape, var=1.0):
    s = np.sqrt(var / 2.0)
    out = rng.standard_normal(shape, dtype=np.float32).astype(np.complex64)
    out *= s
    out += 1j * (s * rng.standard_normal(shape, dtype=np.float32))
    return out


def make_inputs(w: Workload, full_ranges: int | None = None):
    """Returns (voltages, codes).  voltages: complex64 [P][ipp_len] or int16 [P][ipp_len][2]."""
    full_ranges = full_ranges or max(w.n_ranges, CONFIGS.get(w.name.split("[")[0], w).n_ranges)
    rng_code = np.random.default_rng(w.seed + 0)
    rng_noise = np.random.default_rng(w.seed + 1)
    rng_amp = np.random.default_rng(w.seed + 2)
    codes = make_codes(w, rng_code)
    L, N, P = w.code_len, w.N, w.n_ipp
    t = np.arange(L, dtype=np.float64)

    if w.echo == "tone1":                       # configs[0]: one echo, gate 20, bin 100, amp 0.5
        gates = np.array([min(20, w.n_ranges - 1)])
        mods = [np.exp(2j * np.pi * 100.0 * t / N).astype(np.complex64)]
    else:
        gates = np.arange(0, w.n_ranges, w.echo_every)
        k = chapman_bins(full_ranges, N, gates)
        mods = None                              # built per gate below
    delays = w.r0 + gates * w.stride
    amp_var = w.snr * w.sigma ** 2

    V = np.empty((P, w.ipp_len), dtype=np.complex64)
    for p in range(P):
        v = _cn(rng_noise, w.ipp_len, w.sigma ** 2)
        V[p] = v
    if w.echo == "tone1":
        for p in range(P):
            V[p, delays[0]:delays[0] + L] += np.complex64(0.5) * codes[p] * mods[0]
    else:
        for gi, g in enumerate(gates):
            d = int(delays[gi])
            if w.echo == "tone":
                a = _cn(rng_amp, P, amp_var)
                m = np.exp(2j * np.pi * k[gi] * t / N).astype(np.complex64)
                V[:, d:d + L] += (a[:, None] * m[None, :]) * codes
            elif w.echo == "tone2":             # up- and down-shifted lines (configs[2])
                a1, a2 = _cn(rng_amp, P, amp_var), _cn(rng_amp, P, amp_var)
                m = np.exp(2j * np.pi * k[gi] * t / N).astype(np.complex64)
                V[:, d:d + L] += (a1[:, None] * m[None, :] + a2[:, None] * np.conj(m)[None, :]) * codes
            elif w.echo == "lorentz":           # narrow line, FWHM 2 bins (configs[3])
                kk = np.arange(-32, 33)
                kc = int(round(k[gi]))
                ell = 1.0 / (1.0 + (kk / 1.0) ** 2)
                ell /= ell.sum()
                for p in range(P):
                    A = np.zeros(N, dtype=np.complex128)
                    A[(kc + kk) % N] = _cn(rng_amp, kk.size, 1.0) * np.sqrt(amp_var * ell)
                    m = (np.fft.ifft(A)[:L] * N).astype(np.complex64)   # sum_k A_k e^{2 pi i k t/N}
                    V[p, d:d + L] += m * codes[p]
            else:
                raise ValueError(w.echo)
    if w.dtype == CF32:
        return V, codes
    out = np.empty((P, w.ipp_len, 2), dtype=np.int16)
    out[..., 0] = np.clip(np.rint(V.real), -32768, 32767).astype(np.int16)
    out[..., 1] = np.clip(np.rint(V.imag), -32768, 32767).astype(np.int16)
    return out, codes
