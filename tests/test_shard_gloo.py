"""CPU, world_size 2, gloo: the host logic of the data-parallel path (paper_2606_04484_b200/shard.py).

Each rank plays one GPU; the oracle stands in for the kernels (tests may use it).  Checked: sharding whole trajectory
groups across ranks and merging locally gives exactly the unsharded merge (no data-path collective is needed), and
splitting the loss rows across ranks with an all-reduce of N_s before and of the scalar after gives the single-call
loss (readings M-4 and L-4)."""
import os
import socket
import sys
import tempfile

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_04484_b200 import shard as SH          # noqa: E402
from paper_2606_04484_b200 import workloads as W       # noqa: E402


def _free_port() -> int:
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _loss_case():
    T, V, S = 96, 40, 5
    lv = W.loss_sweep_vectors(T, V, S, 0.6, seed=31)
    logits = W.small_logits(T, V, 2.0, seed=31)
    old = (-np.abs(W.rng_for(31, 7).standard_normal(T)) - 3.0).astype(np.float32)
    return T, V, S, lv, logits, old


def _worker(rank: int, world: int, port: int, outdir: str):
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # ---- merge: whole groups per rank, merged locally
        mi = W.merge_workload("c1")
        asg = SH.assign_groups(mi.offsets, mi.traj_ids, world)
        sh = SH.shard_merge_inputs(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp, rank=rank, world=world,
                                   assignment=asg)
        res = {}
        for rule in (oracle.OWNER_LONGEST, oracle.OWNER_PAPER):
            r = oracle.merge_timelines(sh.tokens, sh.offsets, sh.traj_ids, sh.resp_start, None, sh.old_logp, rule)
            go, gs = SH.to_global_indices(sh, r.merged_origin, r.merged_src)
            counts = SH.gather_counts(r.M, r.N_out)
            res[rule] = dict(origin=go, src=gs, tokens=r.merged_tokens, mask=r.merged_mask, logp=r.merged_old_logp,
                             offsets=r.merged_offsets, owner_global=go[r.owner], index=sh.index, counts=counts)
        # ---- loss: contiguous row split; N_s all-reduced before, scalar after
        T, V, S, lv, logits, old = _loss_case()
        b = SH.split_rows(T, world)
        lo, hi = int(b[rank]), int(b[rank + 1])
        Ns_local = np.bincount(lv.seg_ids[lo:hi], weights=lv.mask[lo:hi].astype(np.float64), minlength=S).astype(np.float32)
        Ns = SH.allreduce_seg_denom(torch.from_numpy(Ns_local.copy()))
        inv = SH.inv_num_segs(Ns)
        rid = np.arange(lo, hi, dtype=np.int64)
        part = oracle.policy_loss(logits[lo:hi], lv.targets, old, lv.adv, lv.mask, lv.seg_ids, S, 0.2, 0.28,
                                  seg_denom=Ns.numpy(), inv_num_segs=inv, row_ids=rid)
        total = SH.allreduce_loss([torch.tensor([np.float32(part.loss)])])
        np.savez(os.path.join(outdir, f"rank{rank}.npz"), total=total, Ns=Ns.numpy(), inv=inv, dl=part.dlogits, lo=lo, hi=hi,
                 **{f"m{rule}_{k}": v for rule, d in res.items() for k, v in d.items()})
    finally:
        dist.destroy_process_group()


@pytest.fixture(scope="module")
def two_rank_run():
    d = tempfile.mkdtemp(prefix="ajt_gloo_")
    mp.spawn(_worker, args=(2, _free_port(), d), nprocs=2, join=True)
    return [np.load(os.path.join(d, f"rank{r}.npz")) for r in range(2)]


def test_assignment_is_balanced_and_keeps_groups_whole():
    mi = W.merge_workload("c2")
    for world in (2, 3, 8):
        asg = SH.assign_groups(mi.offsets, mi.traj_ids, world)
        for key in np.unique(mi.traj_ids):
            assert np.unique(asg[mi.traj_ids == key]).size == 1          # a group never straddles ranks
        lens = np.diff(mi.offsets)
        load = np.array([lens[asg == r].sum() for r in range(world)])
        _, tok, _ = SH.group_token_counts(mi.offsets, mi.traj_ids)
        assert load.sum() == mi.n_tokens
        assert load.max() - load.min() <= tok.max()                       # the LPT bound
        assert np.array_equal(asg, SH.assign_groups(mi.offsets, mi.traj_ids, world))   # deterministic


def test_shard_keeps_input_order_and_content():
    mi = W.merge_workload("c1")
    parts = [SH.shard_merge_inputs(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp, rank=r, world=3)
             for r in range(3)]
    allidx = np.concatenate([p.index for p in parts])
    assert np.array_equal(np.sort(allidx), np.arange(mi.n))
    for p in parts:
        assert np.all(np.diff(p.index) > 0)
        for k, j in enumerate(p.index):
            assert np.array_equal(p.tokens[p.offsets[k]:p.offsets[k + 1]], mi.tokens[mi.offsets[j]:mi.offsets[j + 1]])
            assert p.resp_start[k] == mi.resp_start[j] and p.traj_ids[k] == mi.traj_ids[j]



def test_sharded_merge_equals_unsharded(two_rank_run):
    import oracle
    mi = W.merge_workload("c1")
    for rule in (oracle.OWNER_LONGEST, oracle.OWNER_PAPER):
        ref = oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp, rule)
        seen = {}
        owner_global = np.full(mi.n, -1, dtype=np.int64)
        for rk in two_rank_run:
            origin, off = rk[f"m{rule}_origin"], rk[f"m{rule}_offsets"]
            owner_global[rk[f"m{rule}_index"]] = rk[f"m{rule}_owner_global"]
            for m, o in enumerate(origin):
                sl = slice(off[m], off[m + 1])
                seen[int(o)] = (rk[f"m{rule}_tokens"][sl], rk[f"m{rule}_mask"][sl], rk[f"m{rule}_src"][sl], rk[f"m{rule}_logp"][sl])
            c = rk[f"m{rule}_counts"]
            assert c[:, 0].sum() == ref.M and c[:, 1].sum() == ref.N_out       # the all-gathered layout
        assert sorted(seen) == [int(x) for x in ref.merged_origin]
        for m, o in enumerate(ref.merged_origin):
            sl = slice(ref.merged_offsets[m], ref.merged_offsets[m + 1])
            t, k, s, l = seen[int(o)]
            assert np.array_equal(t, ref.merged_tokens[sl]) and np.array_equal(k, ref.merged_mask[sl])
            assert np.array_equal(s, ref.merged_src[sl]) and np.array_equal(l, ref.merged_old_logp[sl])
        assert np.array_equal(owner_global, ref.merged_origin[ref.owner])


def test_row_sharded_loss_equals_single_call(two_rank_run):
    import oracle
    T, V, S, lv, logits, old = _loss_case()
    ref = oracle.policy_loss(logits, lv.targets, old, lv.adv, lv.mask, lv.seg_ids, S, 0.2, 0.28)
    Ns = np.bincount(lv.seg_ids, weights=lv.mask.astype(np.float64), minlength=S)
    for rk in two_rank_run:
        assert np.array_equal(rk["Ns"], Ns.astype(np.float32))
        assert abs(float(rk["total"]) - ref.loss) <= 2e-7 * max(1.0, abs(ref.loss))
        lo, hi = int(rk["lo"]), int(rk["hi"])
        assert np.allclose(rk["dl"], ref.dlogits[lo:hi], rtol=1e-6, atol=1e-12)     # inv is fp32: 6e-8 relative
    assert two_rank_run[0]["total"] == two_rank_run[1]["total"]
