"""Multi-GPU sharding of the chain ensemble.

Chains are independent and interact only through two sums: the accumulation buffer and tourCount.
Each rank owns a contiguous range of GLOBAL chain ids (RNG streams are keyed by global id, so the sharded run draws
the same numbers as the unsharded one), a replica of the scene and a private accumulation buffer.  The only exchange
is one all-reduce(sum) of the buffer and the counters per resolve.  Backend-agnostic: NCCL on GPUs, gloo in the CPU tests.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard_offset(n_local: int, rank: int) -> int:
    """Weak scaling: every rank runs n_local chains; global id of its chain 0."""
    return n_local * rank


def shard_range(n_total: int, rank: int, world: int) -> tuple[int, int]:
    """Strong scaling: contiguous [begin, end) of n_total chains for `rank` (sizes differ by at most one)."""
    base, rem = divmod(n_total, world)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def allreduce_totals(accum: torch.Tensor, tours: int, mutations: int):
    """Sum of the per-shard accumulation buffers (new tensor) and of the counters over all ranks."""
    acc = accum.clone()
    cnt = torch.tensor([int(tours), int(mutations)], dtype=torch.int64, device=accum.device)
    if dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(acc, op=dist.ReduceOp.SUM)
        dist.all_reduce(cnt, op=dist.ReduceOp.SUM)
    return acc, int(cnt[0].item()), int(cnt[1].item())


def resolve_frame(chains):
    """One sharded frame's exchange: dr_pack_frame, ONE all-reduce(sum), dr_resolve_image_packed.  No host synchronisation:
    the counters travel as 16-bit limbs in the tail of the same fp32 buffer (exact for up to 256 ranks)."""
    buf = chains.pack_frame()
    if dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(buf, op=dist.ReduceOp.SUM)
    return chains.resolve_packed(buf)


def limbs(value: int) -> list:
    """The four 16-bit limbs of a counter, as the floats k_pack_frame writes (host mirror for the tests)."""
    return [float((int(value) >> (16 * k)) & 0xFFFF) for k in range(4)]


def from_limbs(t) -> int:
    return sum(int(round(float(v))) << (16 * k) for k, v in enumerate(t))
