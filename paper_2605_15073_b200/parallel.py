"""Host-side sharding of the hot path over ranks (one process per GPU, torch.distributed).

The paper's implementation is single-GPU; DESIGN.md "Multi-GPU" derives the split:

* on-site (Eq.(1)): atoms are independent -> split the batch, no collective;
* message passing (Eq.(2)): the receiver-sorted edge list is cut into contiguous
  receiver ranges balanced by work; every rank owns the node features, the in-edges and the output
  rows of its range.  A sender may live on any rank, so the one exchange step is an all-gather of
  the node features (NCCL over NVLink on GPUs) before `cgtp_message_bipartite`; outputs need no
  reduction.

Only index arithmetic and the collective live here; the arithmetic of the method stays in the CUDA
kernels (`compute` defaults to binding.cgtp_message_bipartite).
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Callable, Optional, Sequence

import numpy as np
import torch
import torch.distributed as dist


# ------------------------------------------------------------------------------------------ on-site
def shard_batch(batch: int, world: int, rank: int) -> tuple[int, int]:
    """[start, stop) of the atoms rank `rank` owns: contiguous, sizes differ by at most one."""
    if world < 1 or not 0 <= rank < world or batch < 0:
        raise ValueError("bad shard_batch arguments")
    q, r = divmod(batch, world)
    start = rank * q + min(rank, r)
    return start, start + q + (1 if rank < r else 0)


# ---------------------------------------------------------------------------------- message passing
def row_ptr_from_receivers(receivers: np.ndarray, nodes: int) -> np.ndarray:
    """CSR offsets of a receiver-sorted edge list (host copy of what cgtp_build_segments computes)."""
    receivers = np.asarray(receivers, np.int64)
    if receivers.size and (np.any(np.diff(receivers) < 0) or receivers[0] < 0 or receivers[-1] >= nodes):
        raise ValueError("edge list is not receiver-sorted or has a receiver outside [0, nodes)")
    return np.searchsorted(receivers, np.arange(nodes + 1, dtype=np.int64), side="left").astype(np.int64)


def shard_receivers(row_ptr: np.ndarray, world: int, node_cost: float = 4.0) -> np.ndarray:
    """Cuts [0, nodes) into `world` contiguous receiver ranges of near-equal cost.

    cost(range) = edges in the range + node_cost * nodes in the range (the per-receiver analysis and
    projections are not free).  Returns bounds int64 [world+1], bounds[0] = 0, bounds[-1] = nodes,
    non-decreasing; the same on every rank (a pure function of row_ptr)."""
    row_ptr = np.asarray(row_ptr, np.int64)
    nodes = row_ptr.shape[0] - 1
    if world < 1 or nodes < 0:
        raise ValueError("bad shard_receivers arguments")
    cum = row_ptr.astype(np.float64) + node_cost * np.arange(nodes + 1, dtype=np.float64)
    total = cum[-1]
    targets = total * np.arange(1, world, dtype=np.float64) / world
    cuts = np.searchsorted(cum, targets, side="left")
    # choose the nearer of the two neighbouring node boundaries
    for k, (c, t) in enumerate(zip(cuts, targets)):
        if 0 < c <= nodes and abs(cum[c - 1] - t) <= abs(cum[min(c, nodes)] - t):
            cuts[k] = c - 1
    bounds = np.concatenate([[0], np.clip(cuts, 0, nodes), [nodes]]).astype(np.int64)
    return np.maximum.accumulate(bounds)


def local_edge_slice(row_ptr: np.ndarray, lo: int, hi: int) -> tuple[int, int]:
    """[e0, e1) of the receiver-sorted edge list whose receivers lie in [lo, hi)."""
    return int(row_ptr[lo]), int(row_ptr[hi])


@dataclass
class MessageShard:
    """What one rank holds: its receiver range, its in-edges (global sender ids, receivers rebased to
    the range) and the features of its own nodes."""
    lo: int
    hi: int
    edge_index: torch.Tensor   # int64 [2, E_local]; row 0 global sender, row 1 receiver - lo
    edge_vec: torch.Tensor     # [E_local, 3]
    edge_radial: torch.Tensor  # [E_local, C]
    node_feats: torch.Tensor   # [hi - lo, N, (lmax+1)^2]


def row_ptr_on_device(receivers: torch.Tensor, nodes: int) -> torch.Tensor:
    """CSR offsets of a receiver-sorted edge list, computed where the list lives (no host copy)."""
    probe = torch.arange(nodes + 1, dtype=torch.int64, device=receivers.device)
    return torch.searchsorted(receivers.contiguous(), probe, right=False)


def make_shard(node_feats: torch.Tensor, edge_index: torch.Tensor, edge_vec: torch.Tensor,
               edge_radial: torch.Tensor, bounds: Sequence[int], rank: int, row_ptr=None) -> MessageShard:
    """Cuts rank `rank`'s shard out of a full (replicated) problem; used by tests and by callers that
    load the whole graph on every rank.  `row_ptr` (device or host, int64 [nodes+1]) is reused when given; otherwise the
    two offsets the shard needs are found on the device the edge list lives on."""
    nodes = node_feats.shape[0]
    lo, hi = int(bounds[rank]), int(bounds[rank + 1])
    if row_ptr is None:
        probe = torch.tensor([lo, hi], dtype=torch.int64, device=edge_index.device)
        e0, e1 = (int(v) for v in torch.searchsorted(edge_index[1].contiguous(), probe, right=False).tolist())
    else:
        e0, e1 = int(row_ptr[lo]), int(row_ptr[hi])
    if not (0 <= lo <= hi <= nodes):
        raise ValueError("receiver bounds outside [0, nodes]")
    ei = edge_index[:, e0:e1].clone()
    ei[1] -= lo
    return MessageShard(lo, hi, ei.contiguous(), edge_vec[e0:e1].contiguous(), edge_radial[e0:e1].contiguous(),
                        node_feats[lo:hi].contiguous())


def all_gather_node_feats(local: torch.Tensor, bounds: Sequence[int], group=None, out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """All-gather of the per-rank node-feature blocks into [nodes, N, L^2] (the one exchange step).

    The blocks land directly in their rows of the result: one all_gather_into_tensor when every range has the same
    length (the balanced case), else one all_gather over views of the result with per-rank lengths (NCCL moves uneven
    blocks as grouped broadcasts).  Only the gloo backend (CPU tests) needs equal blocks and goes through a padded
    staging copy.  A single process (no process group) has nothing to exchange."""
    if not (dist.is_available() and dist.is_initialized()):
        if local.shape[0] != int(bounds[-1] - bounds[0]):
            raise ValueError("local block does not match the receiver bounds")
        return local
    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    sizes = [int(bounds[r + 1] - bounds[r]) for r in range(world)]
    if local.shape[0] != sizes[rank]:
        raise ValueError("local block does not match the receiver bounds")
    tail = tuple(local.shape[1:])
    if out is None:
        out = local.new_empty((sum(sizes),) + tail)
    if len(set(sizes)) == 1:
        dist.all_gather_into_tensor(out, local.contiguous(), group=group)
        return out
    if dist.get_backend(group) != "gloo":
        dist.all_gather(list(out.split(sizes, dim=0)), local.contiguous(), group=group)
        return out
    longest = max(max(sizes), 1)
    send = local.new_zeros((longest,) + tail)
    send[: sizes[rank]] = local
    recv = local.new_empty((world * longest,) + tail)
    dist.all_gather_into_tensor(recv, send, group=group)
    recv = recv.view((world, longest) + tail)
    off = 0
    for r in range(world):
        out[off: off + sizes[r]] = recv[r, : sizes[r]]
        off += sizes[r]
    return out


def message_sharded(shard: MessageShard, bounds: Sequence[int], W_node: torch.Tensor, W_out: torch.Tensor,
                    lmax: int, lmax_out: int, N: int, C: int, parity_mask, group=None,
                    compute: Optional[Callable] = None) -> torch.Tensor:
    """out rows [lo, hi) of the message-passing layer on this rank: all-gather node features, then the
    bipartite kernel path over the local in-edges.  `compute(node_feats_all, edge_index, edge_vec,
    edge_radial, W_node, W_out, lmax, lmax_out, N, C, parity_mask, n_recv)` defaults to the CUDA path."""
    if compute is None:
        from . import binding
        compute = binding.cgtp_message_bipartite
    feats = all_gather_node_feats(shard.node_feats, bounds, group)
    return compute(feats, shard.edge_index, shard.edge_vec, shard.edge_radial, W_node, W_out, lmax, lmax_out, N, C,
                   parity_mask, shard.hi - shard.lo)


# ------------------------------------------------------------------ two feature fields, Eq.(28)
@dataclass
class FieldShard:
    """One rank's part of the two-field coupling: its receiver range, its in-edges with their edge feature field
    (global sender ids, receivers rebased) and the features of its own nodes."""
    lo: int
    hi: int
    edge_index: torch.Tensor   # int64 [2, E_local]
    edge_feats: torch.Tensor   # [E_local, Ne, (lmax+1)^2]
    node_feats: torch.Tensor   # [hi - lo, N, (lmax+1)^2]


def make_field_shard(node_feats: torch.Tensor, edge_index: torch.Tensor, edge_feats: torch.Tensor,
                     bounds: Sequence[int], rank: int) -> FieldShard:
    lo, hi = int(bounds[rank]), int(bounds[rank + 1])
    probe = torch.tensor([lo, hi], dtype=torch.int64, device=edge_index.device)
    e0, e1 = (int(v) for v in torch.searchsorted(edge_index[1].contiguous(), probe, right=False).tolist())
    ei = edge_index[:, e0:e1].clone()
    ei[1] -= lo
    return FieldShard(lo, hi, ei.contiguous(), edge_feats[e0:e1].contiguous(), node_feats[lo:hi].contiguous())


def message_field_sharded(shard: FieldShard, bounds: Sequence[int], W_edge: torch.Tensor, W_node: torch.Tensor,
                          W_out: torch.Tensor, lmax: int, lmax_out: int, N: int, Ne: int, C: int, parity_mask, group=None,
                          compute: Optional[Callable] = None) -> torch.Tensor:
    """out rows [lo, hi) of the two-field coupling on this rank: the edge feature field is local to the receiver's rank,
    so the one exchange step is again the all-gather of the node features.  `compute(node_feats_all, edge_index,
    edge_feats, W_edge, W_node, W_out, lmax, lmax_out, N, Ne, C, parity_mask, n_recv)` defaults to the CUDA path."""
    if compute is None:
        from . import binding
        compute = binding.cgtp_message_field_bipartite
    feats = all_gather_node_feats(shard.node_feats, bounds, group)
    return compute(feats, shard.edge_index, shard.edge_feats, W_edge, W_node, W_out, lmax, lmax_out, N, Ne, C, parity_mask,
                   shard.hi - shard.lo)
