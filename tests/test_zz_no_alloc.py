"""plspec_profile_static (include/plspec.h; csrc/plspec_static.cu): the entry point that allocates nothing -- its
per-gate workspace is a file-scope array in device memory of PLSPEC_STATIC_MAX_GATES entries -- against the existing
path, plspec_profile, on the same float32 spectra: line bins and powers bit-exact (integer decisions on values both
sides hold exactly, one IEEE float32 division), noise floor to 1e-6 relative (float64 sums in a different order), the
tolerances of tests/test_profile_gpu.py.  Every case makes two calls in a row on DIFFERENT spectra, the second with
smaller values and other line positions, so that anything left in the shared workspace by the first call would show.

The file sorts last on purpose (pytest collects in name order; the suite runs with pytest -x)."""
import numpy as np
import pytest

from paper_2311_18737_b200 import binding as pl

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def outputs(R):
    ku = torch.full((R,), -7, dtype=torch.int32, device="cuda"); kd = torch.full_like(ku, -7)
    pu = torch.full((R,), -1.0, dtype=torch.float32, device="cuda"); pd = torch.full_like(pu, -1.0)
    return [ku, pu, kd, pd, torch.full_like(pu, -1.0)]


def both(Sd, n_ipp, k_min, guard, stream=None):
    R, N = Sd.shape
    old, new = outputs(R), outputs(R)
    pl.plspec_profile(Sd, R, N, n_ipp, k_min, guard, *old, stream)
    pl.plspec_profile_static(Sd, R, N, n_ipp, k_min, guard, *new, stream)
    torch.cuda.synchronize()
    return [t.cpu().numpy() for t in old], [t.cpu().numpy() for t in new]


def check(Sd, n_ipp, k_min, guard, stream=None):
    old, new = both(Sd, n_ipp, k_min, guard, stream)
    for o, n, name in zip(old[:4], new[:4], ("k_up", "p_up", "k_dn", "p_dn")):
        assert np.array_equal(o, n), name
    assert np.all(np.isfinite(new[4])) and np.allclose(new[4], old[4], rtol=1e-6, atol=0), "noise"
    return new


def spectra(rng, R, N, scale, ties):
    if ties:
        S = rng.integers(0, 50, size=(R, N)).astype(np.float32) * np.float32(0.25 * scale)   # few distinct values
    else:
        S = (rng.random((R, N)) * scale).astype(np.float32)
    rows = np.arange(R)
    if N >= 1024:
        # a line in each half, a few times the floor as plasma lines are.  Both paths add a thread's <= 16 bins in
        # float32 before going to float64, so a line L rounds the row sum by ~2^-24 L, and the noise floor (that sum
        # less the bins around the lines, over ~N bins) is good to 1e-6 only while L / (N x floor) stays small: no
        # planted lines in the tiny rows, whose arg maxima are the maxima of the floor itself
        S[rows, rng.integers(1, N // 2, size=R)] += np.float32(14.0 * scale)
        S[rows, rng.integers(N // 2 + 1, N, size=R)] += np.float32(13.0 * scale)
    return torch.from_numpy(S).cuda()


@pytest.mark.parametrize("N,R", [(16, 8192), (64, 37), (1024, 300), (4096, 129), (8192, 50), (16384, 1000), (65536, 33)])
def test_two_calls_in_a_row_equal_the_existing_path(N, R):
    rng = np.random.default_rng(1000 * N + R)
    first = spectra(rng, R, N, 1.0e6, ties=False)
    second = spectra(rng, R, N, 1.0, ties=True)             # smaller everywhere: stale maxima or sums would win
    a = check(first, 1000, k_min=min(3, N // 2 - 1), guard=1)
    b = check(second, 7, k_min=1, guard=0)
    assert not np.array_equal(a[0], b[0]) or R < 4           # the two inputs really differ
    check(second, 3, k_min=min(5, N // 2 - 1), guard=2)      # and a third time, on the same input
    check(first, 1, k_min=1, guard=N)                        # every bin within the guard: noise 0 on both paths


def test_user_stream_and_fewer_gates_than_the_call_before():
    rng = np.random.default_rng(5)
    st = torch.cuda.Stream()
    big = spectra(rng, 700, 16384, 10.0, ties=False)
    small = spectra(rng, 3, 16384, 1.0, ties=False)
    st.wait_stream(torch.cuda.current_stream())
    check(big, 50, 16, 3, stream=st)
    check(small, 50, 16, 3, stream=st)
    check(big, 50, 16, 3)


def test_sizes_beyond_the_static_workspace_and_bad_arguments_are_rejected():
    assert pl.STATIC_MAX_GATES == 8192
    R = pl.STATIC_MAX_GATES + 1
    Sd = torch.ones((R, 16), dtype=torch.float32, device="cuda")
    out = outputs(R)
    with pytest.raises(pl.PlspecError) as e:
        pl.plspec_profile_static(Sd, R, 16, 1, 1, 0, *out)
    assert e.value.status == pl.PLSPEC_ERR_INVALID_ARG
    torch.cuda.synchronize()
    assert out[0][0].item() == -7                            # nothing was enqueued
    ok = outputs(4)
    for args in [(4, 24, 1, 1, 0), (4, 16, 0, 1, 0), (4, 16, 1, 0, 0), (4, 16, 1, 8, 0), (4, 16, 1, 1, -1), (0, 16, 1, 1, 0)]:
        with pytest.raises(pl.PlspecError):
            pl.plspec_profile_static(Sd, *args, *ok)
    with pytest.raises(pl.PlspecError):                      # host pointer
        pl.plspec_profile_static(np.ones((4, 16), np.float32), 4, 16, 1, 1, 0, *ok)
    with pytest.raises(pl.PlspecError):                      # misaligned S
        pl.plspec_profile_static(Sd.view(-1)[1:], 4, 16, 1, 1, 0, *ok)
