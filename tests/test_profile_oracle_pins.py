"""Pins of the NEXT-2 oracle (oracle/profile_oracle.py) against things other than itself: closed forms on
constructed spectra, tie-breaking, exclusion windows, and recovery of the Chapman-layer line positions the
synthetic generator put in (the generator is independent of the oracle)."""
import numpy as np
import pytest

import oracle
from paper_2311_18737_b200 import synth


def flat(R, N, b):
    return np.full((R, N), b, dtype=np.float32)


def test_constructed_spectrum_closed_form():
    R, N, P = 3, 256, 8
    S = flat(R, N, 16.0)
    S[0, 40] = 400.0; S[0, N - 37] = 240.0
    S[1, 100] = 80.0; S[1, 200] = 96.0
    S[2, 5] = 1e6                                     # inside the excluded ion-line region: must be ignored
    S[2, 127] = 32.0; S[2, 129] = 48.0                # the edge bins of both halves count
    ku, pu, kd, pd, nz = oracle.profile(S, P, k_min=8, guard=2)
    assert ku.tolist() == [40, 100, 127] and kd.tolist() == [N - 37, 200, 129]
    assert pu.tolist() == [50.0, 10.0, 4.0] and pd.tolist() == [30.0, 12.0, 6.0]
    assert nz.tolist() == [2.0, 2.0, 2.0]             # floor 16 / 8 everywhere once the lines are cut out


def test_ties_take_the_first_bin_and_nyquist_is_skipped():
    N = 64
    S = flat(1, N, 1.0)
    S[0, 10] = S[0, 20] = 5.0
    S[0, 40] = S[0, 50] = 7.0
    S[0, N // 2] = 100.0                              # Nyquist belongs to neither half
    ku, _, kd, _, nz = oracle.profile(S, 1, k_min=2, guard=0)
    assert (ku[0], kd[0]) == (10, 40)
    # the floor keeps the second copies of the tied maxima: (5 + 7 + (61 - 2 - 4) * 1) bins ...
    bins = [f for f in range(2, N - 1) if f != 32 and f not in (10, 40)]
    assert nz[0] == np.float32(sum(float(S[0, f]) for f in bins) / len(bins))


def test_guard_window_removes_a_broad_line_from_the_floor():
    N = 512
    S = flat(1, N, 2.0)
    S[0, 98:103] = [3, 6, 50, 6, 3]
    S[0, 400] = 9.0
    _, _, _, _, n0 = oracle.profile(S, 1, k_min=4, guard=0)
    _, _, _, _, n2 = oracle.profile(S, 1, k_min=4, guard=2)
    assert n2[0] == 2.0 and n0[0] > 2.0


def test_bad_arguments():
    S = flat(2, 64, 1.0)
    for kw in (dict(n_ipp=0, k_min=2, guard=0), dict(n_ipp=1, k_min=0, guard=0), dict(n_ipp=1, k_min=32, guard=0),
               dict(n_ipp=1, k_min=2, guard=-1)):
        with pytest.raises(ValueError):
            oracle.profile(S, **kw)
    with pytest.raises(ValueError):
        oracle.profile(S.astype(np.float64), 1, 2, 0)


def test_recovers_the_chapman_profile_of_the_generator():
    """cfg 2 scaled down: every gate carries a tone at the Chapman-layer bin the generator chose; integrate
    with the hot-path oracle, then the profile oracle must find those bins (+-1: the profile is real-valued)."""
    from dataclasses import replace
    w = replace(synth.scaled(synth.CONFIGS["cfg2"], n_ranges=24, n_ipp=24), snr=0.5)
    V, C = synth.make_inputs(w)
    S = oracle.spectra(V, C, N=w.N, n_ranges=w.n_ranges, r0=w.r0, stride=w.stride).astype(np.float32)
    ku, pu, _, _, nz = oracle.profile(S, w.n_ipp, k_min=16, guard=3)
    want = synth.chapman_bins(synth.CONFIGS["cfg2"].n_ranges, w.N, np.arange(w.n_ranges))
    assert np.abs(ku - np.rint(want)).max() <= 1
    assert np.all(pu > 5 * nz)
    # floor per bin and IPP: L sigma^2 from the noise (pin I9) plus the other 23 gates' echoes (power snr each,
    # windows overlapping almost fully) decoded to noise: L (1 + 23 snr), amplitudes redrawn per IPP
    expect = w.code_len * (1.0 + (w.n_ranges - 1) * w.snr)
    assert np.all(nz > 0.6 * expect) and np.all(nz < 1.5 * expect)


def test_mean_spectrum_pins():
    """oracle.mean_spectrum against things other than itself: numpy's fftshift (library special case, n_ipp = 1),
    a hand-placed spectrum (where DC, Nyquist and bins +-1 must land), exact halving, and the centred frequency
    axis: column g holds frequency g - N/2 in cycles per N samples."""
    rng = np.random.default_rng(5)
    S = rng.random((4, 64), dtype=np.float32)
    assert np.array_equal(oracle.mean_spectrum(S, 1, centred=True), np.fft.fftshift(S, axes=1))
    assert np.array_equal(oracle.mean_spectrum(S, 1, centred=False), S)
    assert np.array_equal(oracle.mean_spectrum(S, 2, centred=False), S * np.float32(0.5))
    N = 16
    T = np.zeros((1, N), np.float32)
    T[0, 0] = 8.0; T[0, 1] = 16.0; T[0, N - 1] = 24.0; T[0, N // 2] = 32.0
    P = oracle.mean_spectrum(T, 8, centred=True)[0]
    want = np.zeros(N, np.float32)
    want[N // 2] = 1.0; want[N // 2 + 1] = 2.0; want[N // 2 - 1] = 3.0; want[0] = 4.0    # Nyquist = most negative
    assert np.array_equal(P, want)
    # a tone at signed frequency k shows at column k + N/2 of the centred periodogram
    N = 128
    for k in (-40, -1, 0, 7, 63):
        x = np.exp(2j * np.pi * k * np.arange(N) / N)
        per = (np.abs(np.fft.fft(x)) ** 2).astype(np.float32)[None, :]
        assert int(np.argmax(oracle.mean_spectrum(per, 1, centred=True)[0])) == k + N // 2
    with pytest.raises(ValueError):
        oracle.mean_spectrum(S, 0)
