"""Randomised parity: seeded random problem shapes, code families, buffer kinds and library options through the C ABI
against the float64 oracle on every gate (bar 1e-4, BASELINE.json north_star).  The default run is a few dozen cases
(about a minute on a B200); PLSPEC_FUZZ_CASES=<n> widens it for a soak run, PLSPEC_FUZZ_SEED / PLSPEC_FUZZ_BUDGET / PLSPEC_FUZZ_MAX_IPP vary the
sequence and the problem sizes (profiles/r02_fuzz.md)."""
import os

import numpy as np
import pytest

import oracle
from paper_2311_18737_b200 import binding as pl
from paper_2311_18737_b200 import synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL = 1e-4
N_CASES = int(os.environ.get("PLSPEC_FUZZ_CASES", "48"))
SEED = int(os.environ.get("PLSPEC_FUZZ_SEED", "20260105"))
BUDGET = float(os.environ.get("PLSPEC_FUZZ_BUDGET", "3.0e7"))   # decoded samples per case (P * R * N): keeps the oracle at a fraction of a second
MAX_IPP = int(os.environ.get("PLSPEC_FUZZ_MAX_IPP", "8"))


def draw_case(rng):
    logN = int(rng.integers(4, 17))                             # 16 ... 65536
    N = 1 << logN
    L = int(N if rng.random() < 0.5 else rng.integers(1, N + 1))
    stride = int(rng.choice([1, 1, 2, 3, 4, 7, 25, 64]))
    r0 = int(rng.integers(0, 9))
    P = int(rng.integers(1, MAX_IPP + 1))
    r_max = max(1, int(BUDGET / (P * N)))
    R = int(rng.integers(1, min(r_max, 300 if BUDGET <= 3.0e7 else 2000) + 1))
    pad = int(rng.choice([0, 0, 1, 5, 100]))
    M = r0 + (R - 1) * stride + L + pad
    dtype = int(rng.integers(0, 2))
    code = str(rng.choice(["bpsk", "complex", "shared"]))
    if code == "bpsk":
        C = (2.0 * rng.integers(0, 2, size=(P, L)) - 1.0).astype(np.complex64)
    else:
        C = (np.exp(2j * np.pi * rng.random((P, L))) * (0.5 + rng.random((P, L)))).astype(np.complex64)
        if code == "shared":
            C[:] = C[0]
    if dtype == synth.CF32:
        V = (rng.standard_normal((P, M)) + 1j * rng.standard_normal((P, M))).astype(np.complex64)
    else:
        V = rng.integers(-4000, 4000, size=(P, M, 2)).astype(np.int16)
    opts = dict(
        kernel=int(rng.choice([pl.KERNEL_AUTO, pl.KERNEL_AUTO, pl.KERNEL_GENERIC] if N <= 16384 or R * P <= 8
                              else [pl.KERNEL_AUTO])),
        ipp_chunks=int(rng.choice([0, 0, 0, 1, 2, 3])),
        h2d_batch=int(rng.choice([0, 0, 1, 3])),
        bpsk_pack=int(rng.random() < 0.8),
        stage=int(rng.choice([1, 1, 0, 2])),
        split=int(rng.choice([1, 1, 2, 0])),
        shared_code=int(code == "shared" and rng.random() < 0.7),
        defer=int(rng.random() < 0.7),
    )
    if opts["kernel"] == pl.KERNEL_AUTO and N < 1024:
        opts["kernel"] = pl.KERNEL_GENERIC if rng.random() < 0.5 else pl.KERNEL_AUTO
    where = str(rng.choice(["device", "pinned", "pageable"]))
    out = str(rng.choice(["device", "device", "pinned", "pageable"]))
    n_calls = int(rng.integers(1, min(P, 3) + 1))
    cuts = sorted(rng.choice(np.arange(1, P), size=n_calls - 1, replace=False).tolist()) if n_calls > 1 else []
    return dict(N=N, L=L, R=R, r0=r0, stride=stride, P=P, M=M, dtype=dtype, C=C, V=V, opts=opts, where=where, out=out,
                bounds=[0] + cuts + [P])


def describe(c):
    return (f"N={c['N']} L={c['L']} R={c['R']} r0={c['r0']} stride={c['stride']} P={c['P']} M={c['M']} dtype={c['dtype']} "
            f"opts={c['opts']} where={c['where']} out={c['out']} bounds={c['bounds']}")


def run_case(c):
    N, L, R, P = c["N"], c["L"], c["R"], c["P"]
    S_ref = oracle.spectra(c["V"], c["C"], N=N, n_ranges=R, r0=c["r0"], stride=c["stride"])
    if c["out"] == "device":
        S = torch.full((R, N), -1.0, dtype=torch.float32, device="cuda")
    else:
        S = torch.full((R, N), -1.0, dtype=torch.float32)
        if c["out"] == "pinned":
            S = S.pin_memory()
    keep = []
    with pl.Integrator(N, L, R, c["r0"], c["stride"], c["M"], c["dtype"], **c["opts"]) as it:
        for a, b in zip(c["bounds"][:-1], c["bounds"][1:]):
            v = np.ascontiguousarray(c["V"][a:b])
            cc = np.ascontiguousarray(c["C"][0] if c["opts"]["shared_code"] else c["C"][a:b])
            if c["where"] == "device":
                v, cc = torch.from_numpy(v).cuda(), torch.from_numpy(cc).cuda()
            elif c["where"] == "pinned":
                v, cc = torch.from_numpy(v).pin_memory(), torch.from_numpy(cc).pin_memory()
            keep.append((v, cc))
            it.accumulate(v, cc, b - a)
        it.finalize(S)
    S_h = S.cpu().numpy().astype(np.float64)
    mean = S_ref.mean(axis=1)
    if not np.all(mean > 0):                                     # cannot happen with these inputs; exact zero otherwise
        return float(np.abs(S_h - S_ref).max())
    return float((np.abs(S_h - S_ref).max(axis=1) / mean).max())


def test_random_cases_against_the_oracle():
    rng = np.random.default_rng(SEED)
    worst, worst_case = 0.0, ""
    for k in range(N_CASES):
        c = draw_case(rng)
        m = run_case(c)
        assert np.isfinite(m) and m <= TOL, f"case {k}: metric {m:.3e}: {describe(c)}"
        if m > worst:
            worst, worst_case = m, describe(c)
    print(f"\nFUZZ {N_CASES} cases: worst metric {worst:.3e} ({worst_case})")
