"""Host-side plans for running one integration on several GPUs.

Pulses and range gates are independent, so the path shards two ways:

* by IPP   -- rank k integrates IPPs [begin, end) into its own S; ONE exchange step at the end, a sum
              all-reduce of S over the ranks (`sum_spectra`).  Inputs are split, not replicated.
* by gate  -- rank k owns gates [g0, g1); it needs samples r0 + g0*stride ... of every IPP and all codes;
              no reduction, the outputs are concatenated (`gather_gates`).

This module holds index arithmetic and torch.distributed calls only -- none of the method's arithmetic --
and works on any backend (NCCL on GPUs; gloo in the CPU tests).  bench.py --gpus N uses the third,
collective-free arrangement: N independent integrations ("replicas", weak scaling).
"""
from __future__ import annotations

from dataclasses import dataclass


def split(n: int, rank: int, world: int):
    """Contiguous near-equal split of range(n): sizes differ by at most one, earlier ranks get the extra."""
    if world < 1 or not 0 <= rank < world or n < 0:
        raise ValueError("bad split arguments")
    q, rem = divmod(n, world)
    begin = rank * q + min(rank, rem)
    return begin, begin + q + (1 if rank < rem else 0)


@dataclass(frozen=True)
class GateShard:
    g0: int          # first global gate of this rank
    g1: int          # one past the last
    r0: int          # first sample of gate g0 within an IPP: the `r0` to create this rank's handle with
    n_ranges: int    # g1 - g0
    span: int        # samples from r0 on that this rank reads of each IPP


def gate_shard(n_ranges: int, r0: int, stride: int, code_len: int, rank: int, world: int) -> GateShard:
    g0, g1 = split(n_ranges, rank, world)
    n = g1 - g0
    return GateShard(g0, g1, r0 + g0 * stride, n, (n - 1) * stride + code_len if n > 0 else 0)


def sum_spectra(S, group=None):
    """IPP sharding: in-place sum of the per-rank partial spectra (the path's only exchange step)."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(S, op=dist.ReduceOp.SUM, group=group)
    return S


def gather_gates(S_local, n_ranges: int, group=None):
    """Gate sharding: concatenate the ranks' gate blocks (split() order) into S[n_ranges][N] on every rank."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return S_local
    world = dist.get_world_size(group)
    sizes = [split(n_ranges, k, world) for k in range(world)]
    rows = max(b - a for a, b in sizes)
    pad = torch.zeros((rows, S_local.shape[1]), dtype=S_local.dtype, device=S_local.device)
    pad[: S_local.shape[0]] = S_local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad, group=group)
    return torch.cat([p[: b - a] for p, (a, b) in zip(parts, sizes)], dim=0)


def max_over_ranks(values, device=None, group=None):
    """Timing rule: every multi-GPU number is the MAX over ranks of device-measured times."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return [float(x) for x in t.cpu()]
