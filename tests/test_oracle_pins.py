"""Pins for the float64 oracle (CPU only; no CUDA involved).

The paper prints no spectra values (tests/golden/README.md), so the oracle is pinned to
what the mathematics fixes -- each pin chosen so that a plausible mistake (dropped term,
wrong sign, wrong index, conj on the wrong factor, missing zero-pad, 1/N scaling) fails
at least one.  Pin names follow SURVEY.md section 8(c).
"""
import os

import numpy as np
import pytest

import oracle
from paper_2311_18737_b200 import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
rng = np.random.default_rng(20231118)


def crandn(*shape):
    return (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)).astype(np.complex64)


def qpsk(*shape):
    return np.exp(0.5j * np.pi * rng.integers(0, 4, size=shape)).astype(np.complex64)


def brute_dft(x):
    """O(N^2) definition X[f] = sum_t x[t] exp(-2 pi i f t / N), in long double."""
    N = x.shape[0]
    t = np.arange(N)
    ang = (-2.0 * np.pi * ((t[:, None] * t[None, :]) % N).astype(np.longdouble) / N)
    Wr, Wi = np.cos(ang), np.sin(ang)
    xr, xi = x.real.astype(np.longdouble), x.imag.astype(np.longdouble)
    Xr = Wr @ xr - Wi @ xi
    Xi = Wr @ xi + Wi @ xr
    return Xr.astype(np.float64) + 1j * Xi.astype(np.float64)


# ---- I1: FFT core vs brute force ------------------------------------------------------
@pytest.mark.parametrize("N", [2, 4, 8, 16, 64, 256])
def test_I1_fft_matches_bruteforce_dft(N):
    x = rng.standard_normal(N) + 1j * rng.standard_normal(N)
    X = oracle.fft(x)
    ref = brute_dft(x)
    assert np.max(np.abs(X - ref)) <= 1e-12 * np.max(np.abs(ref))


def test_I1_fft_sign_convention_forward():
    # exp(+2 pi i k t/N) must land in bin k (reading A1), not N-k.
    N, k = 64, 5
    x = np.exp(2j * np.pi * k * np.arange(N) / N)
    X = oracle.fft(x)
    assert abs(X[k] - N) < 1e-10 and abs(X[N - k]) < 1e-10


def test_I1_spectra_bruteforce_tiny():
    # whole path, tiny: complex code, stride 3, r0 2, code_len < N, against the definition.
    N, L, R, r0, s, P = 16, 11, 4, 2, 3, 3
    M = r0 + (R - 1) * s + L + 5
    V, C = crandn(P, M), crandn(P, L)
    S = oracle.spectra(V, C, N=N, n_ranges=R, r0=r0, stride=s)
    ref = np.zeros((R, N))
    for p in range(P):
        for r in range(R):
            d = np.zeros(N, dtype=np.complex128)
            for t in range(L):
                d[t] = complex(V[p, r0 + r * s + t]) * np.conj(complex(C[p, t]))
            ref[r] += np.abs(brute_dft(d)) ** 2
    assert np.max(np.abs(S - ref)) <= 1e-12 * ref.max()


# ---- I2: Parseval ----------------------------------------------------------------------
@pytest.mark.parametrize("L", [64, 40])
def test_I2_parseval(L):
    N, R, r0, s, P = 64, 7, 3, 2, 5
    M = r0 + (R - 1) * s + L
    V, C = crandn(P, M), crandn(P, L)
    S = oracle.spectra(V, C, N=N, n_ranges=R, r0=r0, stride=s)
    for r in range(R):
        w = V[:, r0 + r * s: r0 + r * s + L].astype(np.complex128)
        energy = np.sum(np.abs(w) ** 2 * np.abs(C.astype(np.complex128)) ** 2)
        assert abs(S[r].sum() - N * energy) <= 1e-12 * N * energy


# ---- I3: single tone, closed form (+ golden value for config 1) -------------------------
def test_I3_single_tone_config1_golden():
    row = [l for l in open(os.path.join(GOLDEN, "config1_tone.txt")) if not l.startswith("#")][0]
    N, L, P, A, gate, k, expected = row.split()
    N, L, P, gate, k = int(N), int(L), int(P), int(gate), int(k)
    A, expected = float(A), float(expected)
    R, M = 64, 2048
    C = (2.0 * rng.integers(0, 2, size=(P, L)) - 1.0).astype(np.complex64)
    V = np.zeros((P, M), dtype=np.complex64)
    tone = np.exp(2j * np.pi * k * np.arange(L) / N)
    V[:, gate:gate + L] = (A * C * tone).astype(np.complex64)
    S = oracle.spectra(V, C, N=N, n_ranges=R)
    assert abs(S[gate, k] - expected) <= 1e-6 * expected        # complex64 rounding of the input
    others = np.delete(S[gate], k)
    assert others.max() <= 1e-9 * expected                       # no leakage when L = N
    assert int(np.argmax(S.max(axis=1))) == gate                  # lands at the right range gate
    assert abs(P * A * A * L * L - expected) == 0


def test_I3_tone_with_complex_code_lands_in_bin_k_not_N_minus_k():
    N = L = 128
    P, k, d = 2, 9, 4
    C = qpsk(P, L)
    V = np.zeros((P, 200), dtype=np.complex64)
    V[:, d:d + L] = C * np.exp(2j * np.pi * k * np.arange(L) / N).astype(np.complex64)
    S = oracle.spectra(V, C, N=N, n_ranges=8)
    assert int(np.argmax(S[d])) == k
    assert abs(S[d, k] - P * L * L) <= 1e-5 * P * L * L
    assert S[d, N - k] <= 1e-9 * S[d, k]


def test_I3_zero_padding_gives_dirichlet_kernel():
    N, L, k, A = 64, 24, 7, 1.5
    C = qpsk(1, L)
    t = np.arange(L)
    V = (A * C * np.exp(2j * np.pi * k * t / N)).astype(np.complex64)
    S = oracle.spectra(V, C, N=N, n_ranges=1)[0]
    f = np.arange(N)
    with np.errstate(invalid="ignore", divide="ignore"):
        dk = np.where(f == k, float(L), np.sin(np.pi * (f - k) * L / N) / np.sin(np.pi * (f - k) / N))
    ref = A * A * dk ** 2
    assert np.max(np.abs(S - ref)) <= 2e-6 * ref.max()


# ---- I4: identity code reduces to a library periodogram ----------------------------------
def test_I4_identity_code_is_periodogram():
    N, R, s, P = 256, 5, 4, 3
    M = (R - 1) * s + N
    V = crandn(P, M)
    C = np.ones((P, N), dtype=np.complex64)
    S = oracle.spectra(V, C, N=N, n_ranges=R, stride=s)
    for r in range(R):
        ref = sum(np.abs(np.fft.fft(V[p, r * s: r * s + N].astype(np.complex128))) ** 2 for p in range(P))
        assert np.max(np.abs(S[r] - ref)) <= 1e-10 * ref.max()


@pytest.mark.parametrize("N,R,r0,s,ipp_len,sc16", [
    (65536, 3, 0, 4, 131072, False),      # cfg4's geometry: r0, stride, row pitch (BASELINE.json configs[3])
    (16384, 3, 5, 1, 32768, True),        # cfg3's geometry, sc16 input, a non-zero first sample
    (8192, 2, 0, 1, 250000, True),        # cfg5's row pitch: offsets p * ipp_len beyond 2^17
])
def test_I4_identity_code_is_periodogram_at_the_sizes_the_oracle_judges(N, R, r0, s, ipp_len, sc16):
    """The oracle is the checker at N = 8192 ... 65536 with large row pitches: pin its twiddle indexing
    (k * step), bit reversal and p * ipp_len offsets there, against numpy's complex128 FFT.  The last
    gate is moved to the far end of the row so that a wrong pitch or an int overflow cannot go unseen."""
    P = 2
    if sc16:
        V = rng.integers(-3000, 3000, size=(P, ipp_len, 2)).astype(np.int16)
        Vc = V[..., 0].astype(np.float64) + 1j * V[..., 1].astype(np.float64)
    else:
        V = crandn(P, ipp_len)
        Vc = V.astype(np.complex128)
    C = np.ones((P, N), dtype=np.complex64)
    S = oracle.spectra(V, C, N=N, n_ranges=R, r0=r0, stride=s)
    far = ipp_len - N                                           # one more gate flush with the end of the row
    S_far = oracle.spectra(V, C, N=N, n_ranges=1, r0=far, stride=1)
    for r, off in [(r, r0 + r * s) for r in range(R)] + [(-1, far)]:
        ref = sum(np.abs(np.fft.fft(Vc[p, off: off + N])) ** 2 for p in range(P))
        got = S_far[0] if r < 0 else S[r]
        assert np.max(np.abs(got - ref)) <= 1e-10 * ref.max()


def test_I3_tone_closed_form_at_N65536_with_the_chirp_code():
    """Single tone through cfg4's complex chirp at full length: lands in bin k of the right gate with
    P A^2 L^2 (conj on the code, forward sign, stride-4 gate indexing), nothing at N - k."""
    w = synth.CONFIGS["cfg4"]
    N, P, k, g, A = w.N, 2, 12345, 2, 0.25
    C = synth.make_codes(synth.scaled(w, n_ranges=1, n_ipp=P), np.random.default_rng(0))
    assert np.abs(C.imag).max() > 0.5 and np.allclose(np.abs(C), 1.0, atol=1e-6)
    V = np.zeros((P, w.ipp_len), dtype=np.complex64)
    d = w.r0 + g * w.stride
    V[:, d:d + N] = (A * C.astype(np.complex128) * np.exp(2j * np.pi * k * np.arange(N) / N)).astype(np.complex64)
    S = oracle.spectra(V, C, N=N, n_ranges=4, r0=w.r0, stride=w.stride)
    expected = P * A * A * N * N
    assert int(np.argmax(S[g])) == k and abs(S[g, k] - expected) <= 2e-6 * expected
    assert S[g, N - k] <= 1e-9 * expected
    assert S[g].sum() - S[g, k] <= 1e-9 * expected * N         # no leakage: L = N, unit-modulus code


# ---- I5: zero in, zero out ---------------------------------------------------------------
def test_I5_zero_input_zero_output():
    C = qpsk(2, 32)
    S = oracle.spectra(np.zeros((2, 64), dtype=np.complex64), C, N=32, n_ranges=9)
    assert np.all(S == 0.0)
    S16 = oracle.spectra(np.zeros((2, 64, 2), dtype=np.int16), C, N=32, n_ranges=9)
    assert np.all(S16 == 0.0)


# ---- I6: modulation theorem (sign, and that conj sits on the code) ------------------------
def test_I6_modulating_the_code_shifts_bins():
    N, R, P, m = 64, 4, 3, 5
    V, C = crandn(P, N + R), crandn(P, N)
    S = oracle.spectra(V, C, N=N, n_ranges=R)
    mod = np.exp(2j * np.pi * m * np.arange(N) / N)
    C2 = (C.astype(np.complex128) * mod).astype(np.complex64)
    S2 = oracle.spectra(V, C2, N=N, n_ranges=R)
    assert np.max(np.abs(S2 - np.roll(S, -m, axis=1))) <= 1e-5 * S.max()   # S'[f] = S[(f+m) mod N]


# ---- I7: conjugation symmetry ---------------------------------------------------------------
def test_I7_conjugating_both_mirrors_bins():
    N, R, P = 64, 4, 3
    V, C = crandn(P, N + R), crandn(P, N)
    S = oracle.spectra(V, C, N=N, n_ranges=R)
    S2 = oracle.spectra(np.conj(V), np.conj(C), N=N, n_ranges=R)
    mirror = S[:, (-np.arange(N)) % N]
    assert np.max(np.abs(S2 - mirror)) <= 1e-12 * S.max()
    # conjugating only the code is NOT the same thing for a complex code
    S3 = oracle.spectra(V, np.conj(C), N=N, n_ranges=R)
    assert np.max(np.abs(S3 - S)) > 1e-3 * S.max()


# ---- I8: invariances (scaling, code phase, gate shift, split / permuted accumulation) -----
def test_I8_invariances():
    N, R, P, r0, s = 64, 6, 4, 1, 2
    M = r0 + (R - 1) * s + N + 3
    V, C = crandn(P, M), crandn(P, N)
    S = oracle.spectra(V, C, N=N, n_ranges=R, r0=r0, stride=s)
    # V -> a V  =>  S -> |a|^2 S   (a = 2: exact in binary floating point)
    S2 = oracle.spectra((2 * V).astype(np.complex64), C, N=N, n_ranges=R, r0=r0, stride=s)
    assert np.array_equal(S2, 4 * S)
    # C -> -i C (exact in fp) leaves S unchanged up to rounding order
    S3 = oracle.spectra(V, (-1j * C).astype(np.complex64), N=N, n_ranges=R, r0=r0, stride=s)
    assert np.max(np.abs(S3 - S)) <= 1e-13 * S.max()
    # gate r of (r0, s) == gate 0 of (r0 + r s, .)
    for r in (1, R - 1):
        Sr = oracle.spectra(V, C, N=N, n_ranges=1, r0=r0 + r * s, stride=1)
        assert np.array_equal(Sr[0], S[r])
    # splitting the pulses over several calls, and permuting them
    Sa = oracle.spectra(V[:1], C[:1], N=N, n_ranges=R, r0=r0, stride=s)
    Sa = oracle.spectra(V[1:], C[1:], N=N, n_ranges=R, r0=r0, stride=s, S=Sa)
    assert np.max(np.abs(Sa - S)) <= 1e-13 * S.max()
    perm = rng.permutation(P)
    Sp = oracle.spectra(V[perm], C[perm], N=N, n_ranges=R, r0=r0, stride=s)
    assert np.max(np.abs(Sp - S)) <= 1e-13 * S.max()


def test_I8_sc16_equals_cf32_of_same_integers():
    N, R, P = 32, 5, 2
    Vi = rng.integers(-32768, 32768, size=(P, N + R, 2)).astype(np.int16)
    Vi[0, 0] = (-32768, 32767)
    C = qpsk(P, N)
    Vf = (Vi[..., 0].astype(np.float32) + 1j * Vi[..., 1].astype(np.float32)).astype(np.complex64)
    assert np.array_equal(oracle.spectra(Vi, C, N=N, n_ranges=R), oracle.spectra(Vf, C, N=N, n_ranges=R))


# ---- argument checking ---------------------------------------------------------------------
def test_bad_arguments_rejected():
    V, C = crandn(1, 40), crandn(1, 32)
    with pytest.raises(ValueError):
        oracle.spectra(V, C, N=32, n_ranges=10)          # span 41 > ipp_len 40
    with pytest.raises(ValueError):
        oracle.spectra(V, C, N=24, n_ranges=1)           # not a power of two
    with pytest.raises(ValueError):
        oracle.spectra(V, crandn(1, 33), N=32, n_ranges=1)  # code_len > N


# ---- I9: generator sanity (statistics, loose) + peak positions ---------------------------------
def test_I9_config1_statistics_and_tone():
    w = synth.CONFIGS["cfg1"]
    V, C = synth.make_inputs(w)
    assert V.shape == (16, 2048) and V.dtype == np.complex64 and C.shape == (16, 1024)
    assert np.all(C.imag == 0) and np.all(np.abs(C.real) == 1)
    S = oracle.spectra(V, C, N=w.N, n_ranges=w.n_ranges)
    # noise floor: E S = P * L * sigma^2 (+25% from the misaligned echo) ; tone at (20, 100)
    floor = np.median(S)
    assert 0.6 * 16 * 1024 < floor < 1.4 * 16 * 1024 * 1.25
    r, f = np.unravel_index(np.argmax(S), S.shape)
    assert (r, f) == (20, 100)
    assert abs(S[20, 100] / 4194304.0 - 1.0) < 0.1     # closed form +- noise cross-term


def test_I9_chapman_profile_and_peaks_cfg2_small():
    w = synth.scaled(synth.CONFIGS["cfg2"], n_ranges=40, n_ipp=12)
    k = synth.chapman_bins(500, 4096, np.arange(500))
    assert abs(k.min() - 200) < 1e-9 and abs(k.max() - 1800) < 1.0
    V, C = synth.make_inputs(w)
    S = oracle.spectra(V, C, N=w.N, n_ranges=w.n_ranges)
    kk = synth.chapman_bins(500, 4096, np.arange(w.n_ranges))
    hits = sum(abs(int(np.argmax(S[g])) - kk[g]) <= 1.0 for g in range(w.n_ranges))
    assert hits >= 0.9 * w.n_ranges


def test_realtime_factor_definition_matches_table1():
    # "Speed ratio" of Table 1 = 1 s of data (100 pulses x 10 ms) / time
    for line in open(os.path.join(GOLDEN, "table1_speed_ratio.txt")):
        if line.startswith("#") or not line.strip():
            continue
        _, t, ratio, _ = [c.strip() for c in line.split("|")]
        assert abs(100 * 0.010 / float(t) - float(ratio)) <= 6e-4
    w = synth.CONFIGS["paper"]
    assert abs(w.data_seconds - 1.0) < 1e-12
