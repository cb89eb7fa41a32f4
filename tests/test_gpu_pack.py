"""GPU parity: ajt_pack_loss_inputs (merge outputs -> per-token loss inputs on the device) vs oracle.pack_loss_inputs, bit-exact;
and the whole device-resident chain merge -> pack -> segment counts -> loss against the oracle chain."""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_04484_b200 as ajt
from paper_2606_04484_b200 import workloads as W
from helpers import check_loss, harness_old_logp

pytestmark = pytest.mark.gpu


def device_merge(mi, rule=ajt.OWNER_LONGEST):
    d = lambda a: torch.from_numpy(a).cuda()
    return ajt.merge_timelines(d(mi.tokens), d(mi.offsets), d(mi.traj_ids), d(mi.resp_start), None, d(mi.old_logp), owner_rule=rule)


@pytest.mark.parametrize("config,n_traj", [("c1", None), ("c2", None), ("c3", 12)])
def test_pack_matches_oracle(config, n_traj):
    mi = W.merge_workload(config, n_traj=n_traj)
    uniq, tl_seg = np.unique(mi.traj_ids, return_inverse=True)
    S = int(uniq.shape[0])
    adv = W.advantages_group_zscore(W.BASE_SEED, 1, S)
    mo = device_merge(mi)                                     # not finalized: counts stay on the device
    pk = ajt.pack_loss_inputs(mo, torch.from_numpy(tl_seg.astype(np.int32)).cuda(), S, torch.from_numpy(adv).cuda())
    torch.cuda.synchronize()
    assert int(pk.status[0]) == 0
    r = oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp)
    t, m, o, s, a = oracle.pack_loss_inputs(r.merged_tokens, r.merged_mask, r.merged_old_logp, r.merged_offsets, r.merged_origin,
                                            tl_seg.astype(np.int32), adv)
    N = r.N_out
    assert np.array_equal(pk.targets[:N].cpu().numpy(), t) and np.array_equal(pk.mask[:N].cpu().numpy(), m)
    assert np.array_equal(pk.old_logp[:N].cpu().numpy().view(np.uint32), o.view(np.uint32))
    assert np.array_equal(pk.seg_ids[:N].cpu().numpy(), s) and np.array_equal(pk.adv[:N].cpu().numpy().view(np.uint32), a.view(np.uint32))


def test_pack_without_optional_arrays_and_bad_segment():
    mi = W.merge_workload("c1")
    d = lambda a: torch.from_numpy(a).cuda()
    mo = ajt.merge_timelines(d(mi.tokens), d(mi.offsets), d(mi.traj_ids), d(mi.resp_start))
    uniq, tl_seg = np.unique(mi.traj_ids, return_inverse=True)
    pk = ajt.pack_loss_inputs(mo, d(tl_seg.astype(np.int32)), int(uniq.shape[0]))
    torch.cuda.synchronize()
    assert pk.old_logp is None and pk.adv is None and int(pk.status[0]) == 0
    bad = tl_seg.astype(np.int32).copy()
    bad[:] = 99999
    pk = ajt.pack_loss_inputs(mo, d(bad), int(uniq.shape[0]))
    torch.cuda.synchronize()
    assert int(pk.status[0]) & ajt.STATUS_BAD_SEG


def test_pack_after_block_merge():
    bi = W.block_workload("b1")
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    mo = ajt.merge_blocks(d(bi.block_ids), d(bi.block_offsets), d(bi.traj_ids), d(bi.author), d(bi.tok_off), d(bi.tokens), d(bi.logp))
    uniq, tl_seg = np.unique(bi.traj_ids, return_inverse=True)
    pk = ajt.pack_loss_inputs(mo, d(tl_seg.astype(np.int32)), int(uniq.shape[0]))
    torch.cuda.synchronize()
    r = oracle.merge_blocks(bi.block_ids, bi.block_offsets, bi.traj_ids, bi.author, bi.tok_off, bi.tokens, bi.logp)
    t, m, o, s, _ = oracle.pack_loss_inputs(r.merged_tokens, r.merged_mask, r.merged_logp, r.merged_offsets, r.merged_origin,
                                            tl_seg.astype(np.int32))
    N = r.N_out
    assert np.array_equal(pk.targets[:N].cpu().numpy(), t) and np.array_equal(pk.mask[:N].cpu().numpy(), m)
    assert np.array_equal(pk.old_logp[:N].cpu().numpy().view(np.uint32), o.view(np.uint32))
    assert np.array_equal(pk.seg_ids[:N].cpu().numpy(), s)


def test_device_resident_chain_c1():
    """configs[0] end to end with no host round trip between the stages: merge -> pack -> segment counts -> loss."""
    mi = W.merge_workload("c1")
    uniq, tl_seg = np.unique(mi.traj_ids, return_inverse=True)
    S = int(uniq.shape[0])
    advt = W.advantages_pm1(W.BASE_SEED, 0, S)
    mo = device_merge(mi)
    pk = ajt.pack_loss_inputs(mo, torch.from_numpy(tl_seg.astype(np.int32)).cuda(), S, torch.from_numpy(advt).cuda())
    N = int(mo.counts.cpu()[1])              # only to size the synthetic logits of this test
    V = 1024
    g = torch.Generator(device="cuda").manual_seed(W.BASE_SEED)
    logits = torch.randn((N, V), generator=g, device="cuda") * 2.0
    noise = (W.rng_for(W.BASE_SEED, 0, 99).standard_normal(N) * 0.05).astype(np.float32)
    old = harness_old_logp(logits, pk.targets[:N], noise)
    Ns = ajt.segment_counts(pk.mask[:N], pk.seg_ids[:N], S)
    out = ajt.policy_loss_fwd_bwd(logits, pk.targets[:N], old, pk.adv[:N], pk.mask[:N], pk.seg_ids[:N], S, 0.2, 0.2, seg_denom=Ns,
                                  want_logp=True, want_stats=True)
    torch.cuda.synchronize()
    # oracle chain
    r = oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp)
    t, m, _, s, a = oracle.pack_loss_inputs(r.merged_tokens, r.merged_mask, r.merged_old_logp, r.merged_offsets, r.merged_origin,
                                            tl_seg.astype(np.int32), advt)
    ref = oracle.policy_loss(logits.cpu().numpy(), t, old.cpu().numpy(), a, m, s, S, float(np.float32(0.2)), float(np.float32(0.2)))
    check_loss(out, ref, m, 0.2, 0.2, a, old.cpu().numpy(), 1.0, V)


def test_fatal_merge_status_leaves_zero_counts_and_pack_does_nothing():
    mi = W.merge_workload("c1")
    off = mi.offsets.copy()
    off[5] = off[4]                      # a zero-length timeline
    d = lambda a: torch.from_numpy(a).cuda()
    mo = ajt.merge_timelines(d(mi.tokens), d(off), d(mi.traj_ids), d(mi.resp_start), None, d(mi.old_logp))
    assert ajt.last_status(mo.workspace) & (ajt.STATUS_ZERO_LEN | ajt.STATUS_BAD_OFFSETS)
    assert mo.counts.cpu().tolist() == [0, 0]
    uniq, tl_seg = np.unique(mi.traj_ids, return_inverse=True)
    pk = ajt.pack_loss_inputs(mo, d(tl_seg.astype(np.int32)), int(uniq.shape[0]))
    torch.cuda.synchronize()
    assert int(pk.status[0]) == 0


def test_hbm_probe_modes():
    # the measurement helper really moves the bytes it is timed on: write zeros, copy, memset; read leaves everything alone
    n = 1 << 20
    a = torch.arange(n, dtype=torch.int32, device="cuda")
    b = torch.full((n,), 7, dtype=torch.int32, device="cuda")
    sink = torch.zeros(4, dtype=torch.int32, device="cuda")
    ajt.hbm_probe(sink, a, 4 * n, 0)
    ajt.hbm_probe(b, a, 4 * n, 2)
    torch.cuda.synchronize()
    assert torch.equal(a, torch.arange(n, dtype=torch.int32, device="cuda")) and torch.equal(b, a) and int(sink.sum()) == 0
    ajt.hbm_probe(b, None, 4 * n, 1)
    ajt.hbm_probe(a, None, 4 * n, 3)
    torch.cuda.synchronize()
    assert not bool(b.any()) and not bool(a.any())
    with pytest.raises(ajt.AjtError):
        ajt.hbm_probe(b, None, 4 * n + 4, 1)      # not a multiple of 16 bytes


def test_chain_captured_in_a_cuda_graph_replays_bit_exactly():
    """include/ajt.h: the device-pointer calls only enqueue on the caller's stream (no synchronisation, no cooperative launch;
    kernels 2.. of a call are programmatic dependents of their predecessor), so merge -> pack -> segment counts -> loss can be
    captured once and replayed.  The replay on NEW inputs of the same shapes must equal the eager calls on them bit for bit."""
    mi = W.merge_workload("c2")
    uniq, tl_seg = np.unique(mi.traj_ids, return_inverse=True)
    S = int(uniq.shape[0])
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    tokens, offsets, traj, rs, lp = d(mi.tokens), d(mi.offsets), d(mi.traj_ids), d(mi.resp_start), d(mi.old_logp)
    tls, adv = d(tl_seg.astype(np.int32)), d(W.advantages_group_zscore(W.BASE_SEED, 1, S))
    T, V = 1500, 4096
    gen = torch.Generator(device="cuda").manual_seed(5)
    logits = (torch.randn((T, V), generator=gen, device="cuda") * 2).to(torch.bfloat16)
    old = torch.full((T,), -8.5, device="cuda")
    stream = torch.cuda.Stream()
    st = {}

    def chain():
        st["mo"] = ajt.merge_timelines(tokens, offsets, traj, rs, None, lp, out=st.get("mo"), stream=stream)
        st["pk"] = ajt.pack_loss_inputs(st["mo"], tls, S, adv, out=st.get("pk"), stream=stream)
        pk = st["pk"]
        st["Ns"] = ajt.segment_counts(pk.mask[:T], pk.seg_ids[:T], S, out=st.get("Ns"), stream=stream)
        st["lo"] = ajt.policy_loss_fwd_bwd(logits, pk.targets[:T], old, pk.adv[:T], pk.mask[:T], pk.seg_ids[:T], S, 0.2, 0.28,
                                           seg_denom=st["Ns"], out=st.get("lo"), stream=stream)

    with torch.cuda.stream(stream):
        chain()                      # eager once: allocates every output and workspace
        stream.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=stream):
            chain()
        # new inputs, same shapes: the token values go through a bijection (same prefix structure, other contents), the
        # log-probs are halved, the logits redrawn
        tok2 = (mi.tokens.astype(np.int64) * 7 + 3) % 151939   # 151939 is prime: a bijection on [0, 151939)
        mi2 = W.MergeInputs(tok2.astype(np.int32), mi.offsets, mi.traj_ids, mi.resp_start, (mi.old_logp * 0.5).astype(np.float32))
        tokens.copy_(d(mi2.tokens)); lp.copy_(d(mi2.old_logp))
        logits.copy_((torch.randn((T, V), generator=gen, device="cuda") * 2).to(torch.bfloat16))
        g.replay()
        stream.synchronize()
        got = {k: v.clone() for k, v in dict(tok=st["mo"].merged_tokens, mask=st["mo"].merged_mask, src=st["mo"].merged_src,
                                             cnt=st["mo"].counts, dl=st["lo"].dlogits, loss=st["lo"].loss, tg=st["pk"].targets).items()}
        st.clear()
        chain()                      # eager on the same new inputs
        stream.synchronize()
    want = dict(tok=st["mo"].merged_tokens, mask=st["mo"].merged_mask, src=st["mo"].merged_src, cnt=st["mo"].counts,
                dl=st["lo"].dlogits, loss=st["lo"].loss, tg=st["pk"].targets)
    N = int(want["cnt"][1])
    assert N > 0 and torch.equal(got["cnt"], want["cnt"])
    for k in ("tok", "mask", "src", "tg"):
        assert torch.equal(got[k][:N], want[k][:N]), k
    assert torch.equal(got["dl"], want["dl"]) and torch.equal(got["loss"], want["loss"])
    r = oracle.merge_timelines(mi2.tokens, mi2.offsets, mi2.traj_ids, mi2.resp_start, None, mi2.old_logp)
    assert N == r.N_out and np.array_equal(got["tok"][:N].cpu().numpy(), r.merged_tokens)
