"""Oracle for the post-integration products: per range gate, the mean
power spectrum and the position of the up- and down-shifted plasma lines.

TEST INFRASTRUCTURE, NOT PRODUCT CODE (see ``oracle/__init__.py``).  Plain numpy, one gate at a time,
written from the definitions:

  P[r][f]   = S[r][f] / n_ipp                       -- the average <|x|^2> of Eq. 8; the hot
                                                       path accumulates the plain sum (reading A2)
  k_up[r]   = arg max_{k_min <= f < N/2} S[r][f]    -- up-shifted line at +f_r (Eq. 1: the
  k_dn[r]   = arg max_{N/2 < f <= N-k_min} S[r][f]     plasma line sits at +-f_r from the ion line; bins
                                                       above N/2 are negative frequencies, reading A9);
                                                       the first (lowest) bin wins a tie
  p_up, p_dn = P at those bins (float32 division, as the GPU does it: the inputs are float32)
  noise[r]  = mean of P[r][f] over k_min <= f <= N-k_min, f != N/2, leaving out the bins within `guard`
              of either line; float64 accumulation
k_min keeps the ion line and DC (|f| < k_min bins, "relatively narrow") out of the search.
The arg max is an integer decided by float32 values that both sides hold exactly, so it is compared exactly.
"""
from __future__ import annotations

import numpy as np


def profile(S, n_ipp: int, k_min: int, guard: int):
    S = np.asarray(S)
    if S.dtype != np.float32 or S.ndim != 2:
        raise ValueError("S must be float32 [n_ranges][N]")
    R, N = S.shape
    if not (1 <= k_min < N // 2) or guard < 0 or n_ipp < 1:
        raise ValueError("bad arguments")
    k_up = np.zeros(R, np.int32); k_dn = np.zeros(R, np.int32)
    p_up = np.zeros(R, np.float32); p_dn = np.zeros(R, np.float32)
    noise = np.zeros(R, np.float32)
    for r in range(R):
        row = S[r]
        ku = k_min + int(np.argmax(row[k_min:N // 2]))                 # numpy: first maximum
        kd = N // 2 + 1 + int(np.argmax(row[N // 2 + 1:N - k_min + 1]))
        k_up[r], k_dn[r] = ku, kd
        p_up[r] = row[ku] / np.float32(n_ipp)
        p_dn[r] = row[kd] / np.float32(n_ipp)
        acc, cnt = 0.0, 0
        for f in range(k_min, N - k_min + 1):
            if f == N // 2 or abs(f - ku) <= guard or abs(f - kd) <= guard:
                continue
            acc += float(row[f])
            cnt += 1
        noise[r] = np.float32(acc / cnt / n_ipp) if cnt else np.float32(0)
    return k_up, p_up, k_dn, p_dn, noise


def mean_spectrum(S, n_ipp: int, centred: bool = False):
    """Mean power spectrum, Eq. 8: P[r][f] = S[r][f] / n_ipp, written out bin by bin; with
    ``centred`` bin f goes to column (f + N/2) mod N, so that DC sits at column N/2 and the negative
    frequencies (bins above N/2, reading A9) to its left -- the usual centred display of a spectrum.  float32
    division, as the GPU does it: the inputs are float32."""
    S = np.asarray(S)
    if S.dtype != np.float32 or S.ndim != 2 or n_ipp < 1:
        raise ValueError("S must be float32 [n_ranges][N], n_ipp >= 1")
    R, N = S.shape
    P = np.zeros((R, N), np.float32)
    for r in range(R):
        for f in range(N):
            g = (f + N // 2) % N if centred else f
            P[r, g] = S[r, f] / np.float32(n_ipp)
    return P
