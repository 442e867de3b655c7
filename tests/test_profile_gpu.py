"""GPU parity of plspec_profile (post-integration products, NEXT-2) against oracle/profile_oracle.py on the
same float32 spectra: line bins and powers bit-exact (integer decisions on values both sides hold exactly,
one IEEE float32 division), noise floor to 1e-6 relative (float64 sums in a different order)."""
import numpy as np
import pytest

import oracle
from paper_2311_18737_b200 import synth
from paper_2311_18737_b200 import binding as pl

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def run(S, n_ipp, k_min, guard, stream=None):
    R, N = S.shape
    Sd = torch.from_numpy(np.ascontiguousarray(S)).cuda()
    ku = torch.full((R,), -7, dtype=torch.int32, device="cuda"); kd = torch.full_like(ku, -7)
    pu = torch.full((R,), -1.0, dtype=torch.float32, device="cuda"); pd = torch.full_like(pu, -1.0)
    nz = torch.full_like(pu, -1.0)
    pl.plspec_profile(Sd, R, N, n_ipp, k_min, guard, ku, pu, kd, pd, nz, stream)
    torch.cuda.synchronize()
    return [t.cpu().numpy() for t in (ku, pu, kd, pd, nz)]


def compare(S, n_ipp, k_min, guard):
    got = run(S, n_ipp, k_min, guard)
    ref = oracle.profile(S, n_ipp, k_min, guard)
    for g, r, name in zip(got[:4], ref[:4], ("k_up", "p_up", "k_dn", "p_dn")):
        assert np.array_equal(g, r), name
    assert np.allclose(got[4], ref[4], rtol=1e-6, atol=0)
    return got


@pytest.mark.parametrize("N", [16, 64, 1024, 4096, 65536])
def test_random_spectra_with_ties(N):
    rng = np.random.default_rng(N)
    R = 37 if N <= 4096 else 5
    S = rng.integers(0, 50, size=(R, N)).astype(np.float32) * 0.25       # few distinct values: many ties
    compare(S, 7, k_min=1, guard=0)
    compare(S, 3, k_min=min(5, N // 2 - 1), guard=2)
    S2 = rng.random((R, N)).astype(np.float32) * 1e6
    compare(S2, 1000, k_min=min(3, N // 2 - 1), guard=1)


def test_edges_of_both_halves_and_all_bins_guarded():
    N = 32
    S = np.ones((2, N), np.float32)
    S[0, N // 2 - 1] = 9; S[0, N // 2 + 1] = 8; S[0, N // 2] = 100       # Nyquist ignored
    S[1, 1] = 5; S[1, N - 1] = 6
    got = compare(S, 1, k_min=1, guard=0)
    assert got[0].tolist() == [15, 1] and got[2].tolist() == [17, 31]
    got = compare(S, 1, k_min=1, guard=N)                                 # every bin within the guard
    assert got[4].tolist() == [0.0, 0.0]


def test_after_an_integration_recovers_the_chapman_profile():
    from dataclasses import replace
    w = replace(synth.scaled(synth.CONFIGS["cfg2"], n_ranges=24, n_ipp=24), snr=0.5)
    V, C = synth.make_inputs(w)
    S = torch.empty((w.n_ranges, w.N), dtype=torch.float32, device="cuda")
    with pl.Integrator.for_workload(w) as it:
        it.accumulate(torch.from_numpy(V).cuda(), torch.from_numpy(C).cuda(), w.n_ipp)
        it.finalize(S)
    got = compare(S.cpu().numpy(), w.n_ipp, k_min=16, guard=3)            # oracle on the very same float32 S
    want = synth.chapman_bins(synth.CONFIGS["cfg2"].n_ranges, w.N, np.arange(w.n_ranges))
    assert np.abs(got[0] - np.rint(want)).max() <= 1
    # and against the float64 path end to end: same bins from the oracle's own spectra
    S64 = oracle.spectra(V, C, N=w.N, n_ranges=w.n_ranges, r0=w.r0, stride=w.stride).astype(np.float32)
    ref = oracle.profile(S64, w.n_ipp, 16, 3)
    assert np.array_equal(got[0], ref[0]) and np.allclose(got[1], ref[1], rtol=1e-4)
    assert np.allclose(got[4], ref[4], rtol=1e-4)


def test_user_stream_and_argument_errors():
    S = np.ones((3, 64), np.float32); S[:, 9] = 4; S[:, 50] = 3
    st = torch.cuda.Stream()
    got = run(S, 2, 2, 1, stream=st)
    assert got[0].tolist() == [9, 9, 9] and got[3].tolist() == [1.5, 1.5, 1.5]
    Sd = torch.ones((3, 64), dtype=torch.float32, device="cuda")
    ki = torch.zeros(3, dtype=torch.int32, device="cuda"); pf = torch.zeros(3, dtype=torch.float32, device="cuda")
    bad = [dict(N=48), dict(N=8), dict(n_ranges=0), dict(n_ipp=0), dict(k_min=0), dict(k_min=32), dict(guard=-1)]
    base = dict(n_ranges=3, N=64, n_ipp=1, k_min=2, guard=0)
    for b in bad:
        a = {**base, **b}
        with pytest.raises(pl.PlspecError) as e:
            pl.plspec_profile(Sd, a["n_ranges"], a["N"], a["n_ipp"], a["k_min"], a["guard"], ki, pf, ki, pf, pf)
        assert e.value.status == pl.PLSPEC_ERR_INVALID_ARG
    with pytest.raises(pl.PlspecError):                                   # host pointer
        pl.plspec_profile(np.ones((3, 64), np.float32), 3, 64, 1, 2, 0, ki, pf, ki, pf, pf)
    with pytest.raises(pl.PlspecError):
        pl.plspec_profile(Sd, 3, 64, 1, 2, 0, None, pf, ki, pf, pf)


@pytest.mark.parametrize("N,R", [(16, 1), (64, 37), (1024, 13), (4096, 301), (65536, 7)])
@pytest.mark.parametrize("centred", [False, True])
def test_mean_spectrum_parity(N, R, centred):
    """plspec_mean_spectrum against oracle.mean_spectrum: bit-exact (one IEEE float32 division per bin on both
    sides, the rest is addressing).  Shapes span one vector per thread to several grid-stride rounds."""
    rng = np.random.default_rng(N + R)
    S = (rng.random((R, N), dtype=np.float32) * np.float32(1e6)).astype(np.float32)
    Sd = torch.from_numpy(S).cuda()
    for n_ipp in (1, 7, 1000):
        Pd = torch.full_like(Sd, -1.0)
        pl.plspec_mean_spectrum(Sd, Pd, R, N, n_ipp, centred)
        torch.cuda.synchronize()
        assert np.array_equal(Pd.cpu().numpy(), oracle.mean_spectrum(S, n_ipp, centred)), (n_ipp,)
        assert np.array_equal(Sd.cpu().numpy(), S)                      # the input is left alone


def test_mean_spectrum_of_an_integration():
    """End to end on cfg 1: accumulate -> finalize -> centred mean; the injected tone (bin 100, gate 20) shows at
    column 100 + N/2 and the values equal the oracle's product of the same finalized spectrum."""
    w = synth.CONFIGS["cfg1"]
    V, C = synth.make_inputs(w)
    S = torch.empty((w.n_ranges, w.N), dtype=torch.float32, device="cuda")
    with pl.Integrator.for_workload(w) as it:
        it.accumulate(torch.from_numpy(V).cuda(), torch.from_numpy(C).cuda(), w.n_ipp)
        it.finalize(S)
    P = torch.empty_like(S)
    pl.plspec_mean_spectrum(S, P, w.n_ranges, w.N, w.n_ipp, True)
    torch.cuda.synchronize()
    Ph = P.cpu().numpy()
    assert np.array_equal(Ph, oracle.mean_spectrum(S.cpu().numpy(), w.n_ipp, True))
    assert int(np.argmax(Ph[20])) == 100 + w.N // 2


def test_mean_spectrum_argument_errors():
    Sd = torch.ones((3, 64), dtype=torch.float32, device="cuda"); Pd = torch.empty_like(Sd)
    bad = [dict(N=48), dict(N=8), dict(n_ranges=0), dict(n_ipp=0)]
    for b in bad:
        a = dict(n_ranges=3, N=64, n_ipp=1); a.update(b)
        with pytest.raises(pl.PlspecError):
            pl.plspec_mean_spectrum(Sd, Pd, a["n_ranges"], a["N"], a["n_ipp"], False)
    with pytest.raises(pl.PlspecError):
        pl.plspec_mean_spectrum(Sd, Sd, 3, 64, 1, True)                 # aliased
    with pytest.raises(pl.PlspecError):
        pl.plspec_mean_spectrum(np.ones((3, 64), np.float32), Pd, 3, 64, 1, False)   # host pointer
    with pytest.raises(pl.PlspecError):
        pl.plspec_mean_spectrum(Sd.view(-1)[1:65], Pd, 1, 64, 1, False)  # misaligned


def test_products_on_a_user_stream_and_misaligned_profile_input():
    """Both product calls enqueue on the caller's stream without synchronising; plspec_profile refuses a spectrum
    that is not 16-byte aligned (its rows are read in 128-bit loads)."""
    rng = np.random.default_rng(77)
    S = rng.random((9, 256), dtype=np.float32)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        Sd = torch.from_numpy(S).cuda()
        Pd = torch.empty_like(Sd)
    st.synchronize()
    pl.plspec_mean_spectrum(Sd, Pd, 9, 256, 3, True, st)
    got = run(S, 3, 4, 1, stream=st)
    st.synchronize()
    assert np.array_equal(Pd.cpu().numpy(), oracle.mean_spectrum(S, 3, True))
    ref = oracle.profile(S, 3, 4, 1)
    assert np.array_equal(got[0], ref[0]) and np.array_equal(got[2], ref[2])
    buf = torch.ones(64 * 3 + 4, dtype=torch.float32, device="cuda")
    ki = torch.zeros(3, dtype=torch.int32, device="cuda"); pf = torch.zeros(3, dtype=torch.float32, device="cuda")
    with pytest.raises(pl.PlspecError):
        pl.plspec_profile(buf[1:], 3, 64, 1, 2, 0, ki, pf, ki, pf, pf)


# ---- the products folded into the write-out: plspec_finalize_products ------------------------------------------------
@pytest.mark.parametrize("N,R,dtype,kernel", [(1024, 19, synth.CF32, pl.KERNEL_FUSED), (4096, 11, synth.SC16, pl.KERNEL_FUSED),
                                              (16384, 5, synth.SC16, pl.KERNEL_FUSED), (65536, 3, synth.CF32, pl.KERNEL_FUSED),
                                              (32768, 3, synth.SC16, pl.KERNEL_FUSED), (256, 9, synth.CF32, pl.KERNEL_GENERIC),
                                              (2048, 7, synth.CF32, pl.KERNEL_GENERIC), (32768, 2, synth.CF32, pl.KERNEL_GENERIC)])
def test_finalize_products_equals_finalize_then_products(N, R, dtype, kernel):
    """One pass: S_out must be the spectrum the oracle computes, and the mean spectrum / line search must be exactly
    what their oracles give ON THAT S_out (bins, powers, mean bit for bit; noise floor to summation order)."""
    rng = np.random.default_rng(N + R)
    P, L = 4, N
    M = 2 + (R - 1) * 3 + L
    C = (2.0 * rng.integers(0, 2, size=(P, L)) - 1.0).astype(np.complex64)
    if dtype == synth.CF32:
        V = (rng.standard_normal((P, M)) + 1j * rng.standard_normal((P, M))).astype(np.complex64)
    else:
        V = rng.integers(-2000, 2000, size=(P, M, 2)).astype(np.int16)
    S_ref = oracle.spectra(V, C, N=N, n_ranges=R, r0=2, stride=3)
    v, c = torch.from_numpy(V).cuda(), torch.from_numpy(C).cuda()
    k_min, guard = max(1, N // 256), 2
    with pl.Integrator(N, L, R, 2, 3, M, dtype, kernel=kernel) as it:
        for centred, with_mean, with_prof in ((True, True, True), (False, True, False), (False, False, True)):
            S = torch.full((R, N), -1.0, dtype=torch.float32, device="cuda")
            Pm = torch.full((R, N), -1.0, dtype=torch.float32, device="cuda")
            ki = torch.full((2, R), -7, dtype=torch.int32, device="cuda")
            pf = torch.full((3, R), -1.0, dtype=torch.float32, device="cuda")
            it.accumulate(v, c, P)
            kw = {}
            if with_mean:
                kw.update(P_out=Pm, centred=centred)
            if with_prof:
                kw.update(k_min=k_min, guard=guard, k_up=ki[0], p_up=pf[0], k_dn=ki[1], p_dn=pf[1], noise=pf[2])
            it.finalize_products(S, P, **kw)
            S_h = S.cpu().numpy()
            m = np.abs(S_h.astype(np.float64) - S_ref).max(axis=1) / S_ref.mean(axis=1)
            assert m.max() <= 1e-4
            if with_mean:
                assert np.array_equal(Pm.cpu().numpy(), oracle.mean_spectrum(S_h, P, centred))
            else:
                assert float(Pm.min()) == -1.0 and float(Pm.max()) == -1.0
            if with_prof:
                ref = oracle.profile(S_h, P, k_min, guard)
                assert np.array_equal(ki[0].cpu().numpy(), ref[0]) and np.array_equal(ki[1].cpu().numpy(), ref[2])
                assert np.array_equal(pf[0].cpu().numpy(), ref[1]) and np.array_equal(pf[1].cpu().numpy(), ref[3])
                assert np.allclose(pf[2].cpu().numpy(), ref[4], rtol=1e-6, atol=0)
            it.finalize(S)                                        # the accumulators were zeroed by the fused call
            assert float(S.abs().max()) == 0.0


def test_finalize_products_argument_errors():
    with pl.Integrator(1024, 1024, 4) as it:
        S = torch.zeros((4, 1024), dtype=torch.float32, device="cuda")
        ki = torch.zeros((2, 4), dtype=torch.int32, device="cuda")
        pf = torch.zeros((3, 4), dtype=torch.float32, device="cuda")
        bad = [dict(n_ipp=0), dict(n_ipp=1, P_out=S),                                        # aliasing
               dict(n_ipp=1, k_up=ki[0]),                                                    # some but not all outputs
               dict(n_ipp=1, k_min=0, k_up=ki[0], p_up=pf[0], k_dn=ki[1], p_dn=pf[1], noise=pf[2]),
               dict(n_ipp=1, k_min=512, k_up=ki[0], p_up=pf[0], k_dn=ki[1], p_dn=pf[1], noise=pf[2]),
               dict(n_ipp=1, P_out=np.zeros((4, 1024), np.float32))]                          # host pointer
        for kw in bad:
            n = kw.pop("n_ipp")
            with pytest.raises(pl.PlspecError) as e:
                it.finalize_products(S, n, **kw)
            assert e.value.status == pl.PLSPEC_ERR_INVALID_ARG
        with pytest.raises(pl.PlspecError):
            it.finalize_products(np.zeros((4, 1024), np.float32), 1)                          # host S_out
