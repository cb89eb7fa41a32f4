"""GPU: the data-parallel decomposition of DESIGN.md "Multi-GPU" run with the CUDA calls, on one
GPU — every "rank" is executed in turn by the same process, so the kernels never wait on one another.

  * merge: trajectory groups -> ranks (shard.assign_groups), ajt_merge_timelines per shard, indices mapped back
    (shard.to_global_indices): the union of the shards' merged sequences equals the unsharded GPU merge bit for bit;
  * loss: rows split across ranks, ajt_segment_counts accumulated over the shards (what the all-reduce of N_s gives),
    ajt_policy_loss_fwd_bwd per shard: dlogits rows identical to the single call, scalars sum to it;
  * token-budget packing: ajt_pack_microbatches against oracle.pack_microbatches, and a loss call per micro-batch."""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_04484_b200 as ajt
from paper_2606_04484_b200 import shard as SH
from paper_2606_04484_b200 import workloads as W
from helpers import assert_merge_equal, gpu_merge, harness_old_logp

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("cfg,world", [("c1", 2), ("c2", 2), ("c2", 3), ("c4A", 4)])
def test_group_sharded_merge_equals_unsharded(cfg, world):
    mi = W.merge_workload_c4()["A"] if cfg == "c4A" else W.merge_workload(cfg)
    full, st = gpu_merge(mi, ajt.OWNER_LONGEST)
    assert st == 0
    seqs = []   # (global origin, tokens, mask, global src, logp, traj)
    owner_tl = np.full(mi.n, -1, np.int64)   # global index of the survivor owning each timeline
    for rank in range(world):
        sh = SH.shard_merge_inputs(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp, rank=rank, world=world)
        if sh.index.shape[0] == 0:
            continue
        smi = W.MergeInputs(sh.tokens, sh.offsets, sh.traj_ids, sh.resp_start, sh.old_logp)
        g, st = gpu_merge(smi, ajt.OWNER_LONGEST)
        assert st == 0
        go, gsrc = SH.to_global_indices(sh, g.merged_origin.cpu().numpy(), g.merged_src.cpu().numpy())
        off = g.merged_offsets.cpu().numpy()
        tok, mk, lp = g.merged_tokens.cpu().numpy(), g.merged_mask.cpu().numpy(), g.merged_old_logp.cpu().numpy()
        tr = g.merged_traj.cpu().numpy()
        for m in range(g.M):
            a, b = int(off[m]), int(off[m + 1])
            seqs.append((int(go[m]), tok[a:b], mk[a:b], gsrc[a:b], lp[a:b], int(tr[m])))
        owner_tl[sh.index] = go[g.owner.cpu().numpy()]
    seqs.sort(key=lambda s: s[0])   # survivors in original order over the whole batch (reading M-8)
    assert len(seqs) == full.M
    cat = lambda k: np.concatenate([s[k] for s in seqs])
    assert np.array_equal(np.array([s[0] for s in seqs]), full.merged_origin.cpu().numpy())
    assert np.array_equal(cat(1), full.merged_tokens.cpu().numpy())
    assert np.array_equal(cat(2), full.merged_mask.cpu().numpy())
    assert np.array_equal(cat(3), full.merged_src.cpu().numpy().astype(np.int64))
    assert np.array_equal(cat(4).view(np.uint32), full.merged_old_logp.cpu().numpy().view(np.uint32))
    assert np.array_equal(np.array([s[5] for s in seqs]), full.merged_traj.cpu().numpy())
    assert np.array_equal(owner_tl, full.merged_origin.cpu().numpy().astype(np.int64)[full.owner.cpu().numpy()])


@pytest.mark.parametrize("world", [2, 3])
def test_row_sharded_loss_equals_single_call(world):
    T, V, S = 6000, 32000, 24
    lv = W.loss_sweep_vectors(T, V, S, 0.5, seed=11)
    gen = torch.Generator(device="cuda").manual_seed(3)
    logits = (torch.randn((T, V), generator=gen, device="cuda") * 3.0).to(torch.bfloat16)
    dev = lambda a: torch.from_numpy(a).cuda()
    targets, adv, mask, seg = dev(lv.targets), dev(lv.adv), dev(lv.mask), dev(lv.seg_ids)
    old = harness_old_logp(logits, targets, lv.noise)
    one = ajt.policy_loss_fwd_bwd(logits, targets, old, adv, mask, seg, S, 0.2, 0.28, want_logp=True, want_stats=True)
    torch.cuda.synchronize()
    # N_s: every "rank" counts its rows, the counts are summed (= the all-reduce); then the loss per shard
    bounds = SH.split_rows(T, world)
    Ns = torch.zeros(S, dtype=torch.float32, device="cuda")
    for r in range(world):
        a, b = int(bounds[r]), int(bounds[r + 1])
        ajt.segment_counts(mask[a:b], seg[a:b], S, out=Ns, accumulate=r > 0)
    dl = torch.empty_like(one.dlogits)
    parts, stats, logp = [], torch.zeros(4, dtype=torch.float64), torch.empty(T, dtype=torch.float32, device="cuda")
    for r in range(world):
        a, b = int(bounds[r]), int(bounds[r + 1])
        o = ajt.policy_loss_fwd_bwd(logits[a:b], targets[a:b], old[a:b], adv[a:b], mask[a:b], seg[a:b], S, 0.2, 0.28, seg_denom=Ns,
                                    inv_num_segs=0.0, dlogits=dl[a:b], want_logp=True, want_stats=True)
        torch.cuda.synchronize()
        assert ajt.last_status(o.workspace) == 0
        parts.append(o.loss.clone())
        stats += o.stats.double().cpu()
        logp[a:b] = o.logp
    assert torch.equal(dl.view(torch.int16), one.dlogits.view(torch.int16))     # rows are independent given N_s: bit-identical
    assert torch.equal(logp, one.logp)
    tot = SH.allreduce_loss(parts)
    l1 = float(np.abs(lv.adv).mean()) + 1e-9
    assert abs(tot - float(one.loss[0])) <= 2e-6 * l1 + 1e-6 * abs(float(one.loss[0]))
    assert stats[0] == one.stats[0].item() and stats[1] == one.stats[1].item() and stats[2] == one.stats[2].item()


@pytest.mark.parametrize("budget", [300, 4096, 10**7])
def test_microbatch_table_and_loss_per_microbatch(budget):
    mi = W.merge_workload("c1")
    dev = lambda a: torch.from_numpy(a).cuda()
    mo = ajt.merge_timelines(dev(mi.tokens), dev(mi.offsets), dev(mi.traj_ids), dev(mi.resp_start), None, dev(mi.old_logp))
    mb_seq, mb_row, n_mb = ajt.pack_microbatches(mo, budget)
    fin = mo.finalize()
    off = fin.merged_offsets.cpu().numpy()
    ref = oracle.pack_microbatches(np.diff(off).tolist(), budget)
    k = int(n_mb.item())
    assert k == len(ref)
    seq, row = mb_seq.cpu().numpy()[:k + 1], mb_row.cpu().numpy()[:k + 1]
    assert [(int(seq[i]), int(seq[i + 1])) for i in range(k)] == ref
    assert np.array_equal(row, off[seq])
    # one loss call per micro-batch (row ranges of the packed arrays) sums to the single call over all rows
    uniq, tl_seg = np.unique(mi.traj_ids, return_inverse=True)
    S = int(uniq.shape[0])
    pk = ajt.pack_loss_inputs(mo, dev(tl_seg.astype(np.int32)), S, dev(W.advantages_pm1(W.BASE_SEED, 0, S).astype(np.float32)))
    T, V = fin.N_out, 1024
    logits = dev(W.small_logits(T, V, 2.0, 5))
    old = harness_old_logp(logits, pk.targets[:T], (np.random.default_rng(1).standard_normal(T) * 0.05).astype(np.float32))
    Ns = ajt.segment_counts(pk.mask[:T], pk.seg_ids[:T], S)
    one = ajt.policy_loss_fwd_bwd(logits, pk.targets[:T], old, pk.adv[:T], pk.mask[:T], pk.seg_ids[:T], S, 0.2, 0.2, seg_denom=Ns)
    parts = []
    dl = torch.empty_like(one.dlogits)
    for i in range(k):
        a, b = int(row[i]), int(row[i + 1])
        o = ajt.policy_loss_fwd_bwd(logits[a:b], pk.targets[a:b], old[a:b], pk.adv[a:b], pk.mask[a:b], pk.seg_ids[a:b], S, 0.2, 0.2,
                                    seg_denom=Ns, dlogits=dl[a:b])
        parts.append(o.loss.clone())
    torch.cuda.synchronize()
    assert torch.equal(dl.view(torch.int16), one.dlogits.view(torch.int16))
    assert abs(SH.allreduce_loss(parts) - float(one.loss[0])) <= 1e-5 * max(1.0, abs(float(one.loss[0])))
