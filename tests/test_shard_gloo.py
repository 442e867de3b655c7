"""N > 1 host logic on CPU: two processes, gloo backend.  Each rank takes its shard of a tiny workload (IPP
sharding with one sum all-reduce; gate sharding with no reduction), computes it with the float64 oracle
(the CUDA library needs a GPU), and the exchanged result must equal the unsharded integration."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

import oracle  # noqa: E402
from paper_2311_18737_b200 import shard, synth  # noqa: E402


def test_split_covers_range_exactly():
    for n in (0, 1, 7, 200, 1001):
        for world in (1, 2, 3, 8):
            parts = [shard.split(n, k, world) for k in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(parts[:-1], parts[1:]))
            sizes = [b - a for a, b in parts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.split(4, 2, 2)


def test_gate_shard_geometry():
    gs = [shard.gate_shard(1000, 3, 4, 4096, k, 3) for k in range(3)]
    assert [g.n_ranges for g in gs] == [334, 333, 333] and gs[1].r0 == 3 + 334 * 4
    assert all(g.span == (g.n_ranges - 1) * 4 + 4096 for g in gs)
    # the shards' sample ranges lie inside the unsharded span
    assert gs[-1].r0 + gs[-1].span == 3 + 999 * 4 + 4096


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = synth.scaled(synth.CONFIGS["cfg1"], n_ranges=9, n_ipp=5)
        V, C = synth.make_inputs(w)                       # same seeded inputs on every rank
        full = oracle.spectra(V, C, N=w.N, n_ranges=w.n_ranges, r0=w.r0, stride=w.stride)
        # --- by IPP: private partial sums, one all-reduce
        a, b = shard.split(w.n_ipp, rank, world)
        part = oracle.spectra(V[a:b], C[a:b], N=w.N, n_ranges=w.n_ranges, r0=w.r0, stride=w.stride) if b > a \
            else np.zeros_like(full)
        S = shard.sum_spectra(torch.from_numpy(part.copy()))
        ok_ipp = np.allclose(S.numpy(), full, rtol=1e-12, atol=0)
        # --- by gate: no reduction, concatenate
        g = shard.gate_shard(w.n_ranges, w.r0, w.stride, w.code_len, rank, world)
        loc = oracle.spectra(V, C, N=w.N, n_ranges=g.n_ranges, r0=g.r0, stride=w.stride)
        G = shard.gather_gates(torch.from_numpy(loc.copy()), w.n_ranges)
        ok_gate = G.shape == full.shape and np.array_equal(G.numpy(), full)
        # --- timing rule
        mx = shard.max_over_ranks([1.0 + rank, 5.0 - rank])
        ok_max = mx == [float(world), 5.0]
        out[rank] = (ok_ipp, ok_gate, ok_max)
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_rank_gloo_sharding_matches_unsharded():
    world = 2
    oracle.build()
    ctx = mp.get_context("spawn")
    out = ctx.Manager().dict()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(240)
        assert p.exitcode == 0
    assert dict(out) == {0: (True, True, True), 1: (True, True, True)}
