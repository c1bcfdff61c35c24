"""Multi-GPU plumbing of the sharded build: one process per GPU,
``torch.distributed`` for the exchange.  Nothing here computes distances or sorts edges - the
shards' keys come out of ``tcrnet_build_shard`` and go into ``tcrnet_assemble``; this module
only moves them between ranks.

The all-pairs path shards by work items (tiles of one length-bucket pair): every rank loads the
same N sequences (13-80 MB, replicated), evaluates the items  rank + k * world  and emits its
own edge keys.  The one exchange step is an all-gather of the keys (8 B per edge, a few tens of
MB at N = 800,000) - over NVLink 5 / NVSwitch this is microseconds against milliseconds of
distance work - after which every rank assembles the same CSR + degrees.
"""
from __future__ import annotations

from typing import List, Optional

import torch
import torch.distributed as dist


def all_gather_v(t: torch.Tensor, group: Optional["dist.ProcessGroup"] = None) -> torch.Tensor:
    """Concatenation, in rank order, of every rank's 1-D tensor `t` (lengths may differ, 0 allowed).
    Works for CUDA tensors over NCCL and CPU tensors over gloo.  Two collectives, one host synchronisation: the
    counts (one all_gather_into_tensor, read back once), then the keys padded to the longest shard (one
    all_gather_into_tensor into a single buffer; shards of interleaved work items differ by a few percent)."""
    assert t.dim() == 1
    world = dist.get_world_size(group)
    if world == 1:
        return t
    counts = torch.empty(world, dtype=torch.int64, device=t.device)
    dist.all_gather_into_tensor(counts, torch.tensor([t.numel()], dtype=torch.int64, device=t.device), group=group)
    sizes = counts.tolist()  # the one host synchronisation
    width = max(max(sizes), 1)
    padded = t if t.numel() == width else torch.cat([t, t.new_zeros(width - t.numel())])
    parts = torch.empty(world * width, dtype=t.dtype, device=t.device)
    dist.all_gather_into_tensor(parts, padded, group=group)
    if all(s == width for s in sizes):
        return parts
    return torch.cat([parts[r * width: r * width + s] for r, s in enumerate(sizes)])


def build_distributed(net, l_max: int, group: Optional["dist.ProcessGroup"] = None) -> int:
    """Sharded tcrnet_build: every rank must have loaded the same sequences into `net`.
    Rank r evaluates the work items r, r + world, ...; the keys are all-gathered; every rank
    assembles the full CSR + degrees (identical on all ranks).  Returns |E|."""
    rank, world = (dist.get_rank(group), dist.get_world_size(group)) if dist.is_initialized() else (0, 1)
    keys = net.build_shard(l_max, rank, world)
    if world > 1:
        keys = all_gather_v(keys, group)
    return net.assemble(keys)


def sum_degrees(deg_partial: torch.Tensor, group: Optional["dist.ProcessGroup"] = None) -> torch.Tensor:
    """Alternative exchange when the CSR stays rank-partitioned: degrees of the union of the
    shards' edge sets = element-wise sum of the shards' degree vectors (d(u) = sum_v A_uv
    is linear in A)."""
    out = deg_partial.clone()
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(out, op=dist.ReduceOp.SUM, group=group)
    return out
