"""Multi-GPU plan of the batched solver: accounts are independent programs that share only the
read-only universe ("each account instantiates Equation (1) with its own data"; "close accounts
in parallel"), so a batch SHARDS BY ACCOUNT: rank r solves the contiguous block `account_range(A, world, r)` with the
universe (B, f, d, group ids) replicated, there is NO collective on the data path, and the only exchange is the gather
of the per-account outputs at the end (plus the barrier / max-reduction of the timings in bench.py).

Host-side logic only (no arithmetic of the method): the plan, the slicing of an instance, and the gather, written
against `torch.distributed` so that the same code runs over NCCL on GPUs and over gloo in the CPU tests.
"""
from __future__ import annotations

import dataclasses

import numpy as np

# per-account fields of instances.gen.Instance (first axis = account); everything else is the shared universe
PER_ACCOUNT = ("mu", "gamma", "w0", "w_b", "lo", "hi", "hi_full", "excl", "tau", "kappa", "band_lo", "band_hi", "c_buy",
               "lot_slope", "lot_width", "lot_count", "witness", "tau_drawn")


def account_range(A: int, world: int, rank: int) -> tuple[int, int]:
    """Contiguous block [start, stop) of rank `rank`: the first A % world ranks hold one account more.
    Every account belongs to exactly one rank; ranks beyond A hold an empty block."""
    if A < 0 or world < 1 or not (0 <= rank < world):
        raise ValueError(f"bad shard request A={A} world={world} rank={rank}")
    base, rem = divmod(A, world)
    start = rank * base + min(rank, rem)
    return start, start + base + (1 if rank < rem else 0)


def plan(A: int, world: int) -> list[tuple[int, int]]:
    """The blocks of all ranks, in rank order."""
    return [account_range(A, world, r) for r in range(world)]


def slice_instance(inst, start: int, stop: int):
    """The accounts [start, stop) of a batch as a batch of their own (shared universe by reference, no copy)."""
    if not (0 <= start <= stop <= inst.A):
        raise ValueError(f"bad slice [{start}, {stop}) of {inst.A} accounts")
    kw = {}
    for f in dataclasses.fields(inst):
        v = getattr(inst, f.name)
        if f.name in PER_ACCOUNT and v is not None:
            v = v[start:stop]
        kw[f.name] = v
    kw["A"] = stop - start
    return type(inst)(**kw)


def gather_accounts(local, A: int, group=None):
    """All ranks' per-account rows in account order.  `local`: torch tensor (n_local, ...) of this rank's block
    (CPU tensor for gloo, CUDA tensor for NCCL); returns a tensor (A, ...) on every rank."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    blocks = plan(A, world)
    nmax = max(b - a for a, b in blocks)
    pad = torch.zeros((nmax,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    pad[: local.shape[0]] = local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad, group=group)
    return torch.cat([parts[r][: b - a] for r, (a, b) in enumerate(blocks)], dim=0)


def solve_sharded(inst, solve_block, group=None):
    """Strong-scaling driver: rank r solves its block of `inst` with `solve_block(sub_instance) -> dict of torch
    tensors with one row per account` and every rank receives the whole batch's rows.  On a GPU box `solve_block`
    wraps `Problem(sub).solve()`; the CPU tests pass a stand-in, because the plan and the gather are what they cover."""
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    start, stop = account_range(inst.A, world, rank)
    out = solve_block(slice_instance(inst, start, stop)) if stop > start else None
    keys = [None]
    if rank == 0:
        keys = [sorted(out.keys())] if out is not None else [[]]
    dist.broadcast_object_list(keys, src=0, group=group)
    if out is None:
        raise ValueError("more ranks than accounts: give every rank at least one account")
    return {k: gather_accounts(out[k], inst.A, group) for k in keys[0]}
