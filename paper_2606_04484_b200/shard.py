"""Host-side logic for running the path data-parallel, one process per GPU.

The path shards with no data-path collective:
  * merge — timelines are only ever compared inside one `traj_ids` group (reading M-4), so whole groups go to
    ranks (balanced by token count) and every rank runs `ajt_merge_timelines` on its own groups;
  * loss  — rows are independent given the per-trajectory normalisers N_s and the count S' (reading L-4).  When
    the rows of one trajectory can land on several ranks, N_s ([S] floats) is all-reduced before the loss calls
    and the scalar partials (one double per rank) after them.  Both messages are bytes to kilobytes.

Nothing here computes any step of the method: it is index bookkeeping plus `torch.distributed` calls (NCCL on GPUs,
gloo in the CPU tests).  Arrays are numpy on the host; the collectives take torch tensors on whatever device the
process group uses.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional, Sequence, Tuple

import numpy as np
import torch
import torch.distributed as dist


# ------------------------------------------------------------------------------------------- merge: groups -> ranks


def group_token_counts(offsets: np.ndarray, traj_ids: np.ndarray) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Returns (keys, tokens_per_key, key_index_of_timeline): the distinct `traj_ids` in ascending order, the number
    of tokens each holds, and for every timeline the position of its key in `keys`."""
    lens = np.diff(np.asarray(offsets, dtype=np.int64))
    keys, inv = np.unique(np.asarray(traj_ids), return_inverse=True)
    tok = np.bincount(inv, weights=lens.astype(np.float64), minlength=keys.shape[0]).astype(np.int64)
    return keys, tok, inv.astype(np.int64)


def assign_groups(offsets: np.ndarray, traj_ids: np.ndarray, world: int) -> np.ndarray:
    """rank_of_timeline int32 [n].  Longest-processing-time greedy: groups in descending token count (ties: smaller
    key first) each go to the currently lightest rank (ties: lowest rank).  Deterministic, so every rank computes the
    same assignment from the same metadata without talking to the others."""
    if world < 1:
        raise ValueError("world must be >= 1")
    keys, tok, inv = group_token_counts(offsets, traj_ids)
    order = np.lexsort((keys, -tok))
    load = np.zeros(world, dtype=np.int64)
    rank_of_key = np.zeros(keys.shape[0], dtype=np.int32)
    for g in order:
        r = int(np.argmin(load))       # first minimum = lowest rank among the lightest
        rank_of_key[g] = r
        load[r] += tok[g]
    return rank_of_key[inv]


@dataclass
class MergeShard:
    """The timelines one rank owns, in input order (so the in-group order Algorithm 1 relies on is kept)."""
    index: np.ndarray        # int64 [n_local] global timeline index of each local timeline, ascending
    tokens: np.ndarray       # int32 [N_local]
    offsets: np.ndarray      # int64 [n_local + 1]
    traj_ids: np.ndarray     # int32 [n_local]
    resp_start: Optional[np.ndarray]
    mask_in: Optional[np.ndarray]
    old_logp: Optional[np.ndarray]


def _gather_segments(values: np.ndarray, offsets: np.ndarray, idx: np.ndarray, new_offsets: np.ndarray) -> np.ndarray:
    out = np.empty(int(new_offsets[-1]), dtype=values.dtype)
    for k, j in enumerate(idx):
        out[new_offsets[k]:new_offsets[k + 1]] = values[offsets[j]:offsets[j + 1]]
    return out


def shard_merge_inputs(tokens, offsets, traj_ids, resp_start=None, mask_in=None, old_logp=None, *, rank: int, world: int,
                       assignment: Optional[np.ndarray] = None) -> MergeShard:
    offsets = np.asarray(offsets, dtype=np.int64)
    assignment = assign_groups(offsets, traj_ids, world) if assignment is None else assignment
    idx = np.nonzero(assignment == rank)[0].astype(np.int64)
    lens = np.diff(offsets)[idx]
    no = np.zeros(idx.shape[0] + 1, dtype=np.int64)
    np.cumsum(lens, out=no[1:])
    take = lambda a: None if a is None else _gather_segments(np.asarray(a), offsets, idx, no)
    return MergeShard(idx, take(tokens), no, np.asarray(traj_ids)[idx].astype(np.int32),
                      None if resp_start is None else np.asarray(resp_start)[idx].astype(np.int32), take(mask_in), take(old_logp))


def to_global_indices(shard: MergeShard, merged_origin: np.ndarray, merged_src: np.ndarray) -> Tuple[np.ndarray, np.ndarray]:
    """Local timeline indices in a rank's merge output -> global timeline indices (-1 stays -1)."""
    go = shard.index[np.asarray(merged_origin, dtype=np.int64)]
    src = np.asarray(merged_src, dtype=np.int64)
    gs = np.where(src >= 0, shard.index[np.maximum(src, 0)], -1)
    return go.astype(np.int64), gs.astype(np.int64)


def gather_counts(M: int, N_out: int, group=None, device="cpu") -> np.ndarray:
    """All-gather of every rank's {M, N_out}: int64 [world, 2].  Enough to place each rank's merged sequences in a
    global packed layout (exclusive prefix over ranks)."""
    world = dist.get_world_size(group)
    mine = torch.tensor([M, N_out], dtype=torch.int64, device=device)
    out = [torch.zeros(2, dtype=torch.int64, device=device) for _ in range(world)]
    dist.all_gather(out, mine, group=group)
    return torch.stack(out).cpu().numpy()


# ------------------------------------------------------------------------------------------- loss: rows -> ranks


def split_rows(T: int, world: int) -> np.ndarray:
    """Row boundaries int64 [world + 1] of an even contiguous split of T packed rows (token-budget sharding: the
    rows of one trajectory may straddle two ranks, which is what `allreduce_seg_denom` is for)."""
    return (np.arange(world + 1, dtype=np.int64) * int(T)) // world


def allreduce_seg_denom(seg_denom: torch.Tensor, group=None) -> torch.Tensor:
    """In-place SUM over ranks of the per-trajectory masked-token counts N_s ([S] fp32, integers < 2^24, so the sum
    is exact in any order).  Call between `ajt_segment_counts` and the loss calls."""
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(seg_denom, op=dist.ReduceOp.SUM, group=group)
    return seg_denom


def inv_num_segs(seg_denom: torch.Tensor) -> float:
    """1/S' with S' = #{s : N_s > 0} (reading L-3), as the fp32 value the C ABI takes."""
    live = int((seg_denom > 0).sum().item())
    return float(np.float32(1.0) / np.float32(live)) if live > 0 else 0.0


def allreduce_loss(partials: Sequence[torch.Tensor], group=None) -> float:
    """Batch loss = sum over this rank's calls and over ranks of the per-call partials sum_t w_t L_t, added in
    fp64 (each partial is the fp32 value `ajt_policy_loss_fwd_bwd` wrote)."""
    dev = partials[0].device if len(partials) else "cpu"
    tot = torch.zeros(1, dtype=torch.float64, device=dev)
    for p in partials:
        tot += p.reshape(-1)[:1].to(torch.float64)
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(tot, op=dist.ReduceOp.SUM, group=group)
    return float(tot.item())
