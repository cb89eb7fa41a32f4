"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.

The oracle cannot produce [T,V] fp64 gradients for 40k-131k rows of a 151,936-wide vocabulary, so at these sizes:
  * sampled rows (first, last, random unmasked, random masked) are checked element by element against the oracle,
    computed one by one (`row_ids`);
  * the scalar is checked against the oracle over ALL rows where that takes seconds (the bench micro-batch), else
    through properties that hold at any size: masked rows are exactly zero, every dlogits row sums to ~0, the big
    call's loss equals the sum of smaller chunked calls (reading L-4) one of which is oracle-checked in full.
Merge at full size (configs[2], configs[3]) is bit-exact against the brute-force oracle in tests/test_gpu_merge.py.
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_04484_b200 as ajt
from paper_2606_04484_b200 import harness as H
from paper_2606_04484_b200 import workloads as W
from helpers import bf16_bits, check_loss, seg_ids_from_merged, shift_for_next_token

pytestmark = pytest.mark.gpu

EPS = (0.2, 0.28)
E32 = (float(np.float32(EPS[0])), float(np.float32(EPS[1])))


def sample_rows(mask_np, n, seed):
    rng = np.random.default_rng(seed)
    T = mask_np.shape[0]
    on, off = np.nonzero(mask_np)[0], np.nonzero(mask_np == 0)[0]
    pick = [0, T - 1]
    if on.size:
        pick += list(rng.choice(on, size=min(n, on.size), replace=False)) + [on[0], on[-1]]
    if off.size:
        pick += list(rng.choice(off, size=min(n // 4 + 1, off.size), replace=False))
    return np.unique(np.array(pick, dtype=np.int64))


def check_sampled(out, logits, vec, S, rows, Ns=None, inv=0.0, grad_scale=1.0):
    """Element-by-element on `rows`; returns the oracle result for them."""
    tg, old, adv, mask, seg = vec
    V = logits.shape[1]
    bits = bf16_bits(logits[torch.from_numpy(rows).to(logits.device)])
    ref = oracle.policy_loss(bits, tg, old, adv, mask, seg, S, E32[0], E32[1], seg_denom=Ns, inv_num_segs=inv, row_ids=rows,
                             grad_scale=grad_scale, logits_is_bf16_bits=True)
    check_loss(out, ref, mask, EPS[0], EPS[1], adv, old, grad_scale, V, row_ids=rows, check_scalar=False)
    return ref


def anysize_properties(out, mask_t, V, slab=4096):
    """Masked rows exactly zero; unmasked rows sum to ~0 (sum_v (1[v=y] - p_v) = 0; bf16 rounding leaves at most
    V half-ulps of the row's largest entry, in practice far less)."""
    T = out.dlogits.shape[0]
    for a in range(0, T, slab):
        d = out.dlogits[a:a + slab, :V]
        m = mask_t[a:a + slab] != 0
        assert not bool(d[~m].any()), f"masked rows not zero in slab {a}"
        df = d[m].float()
        if df.numel():
            rs = df.sum(dim=1).abs()
            bound = df.abs().amax(dim=1) * (2.0 ** -8) * 64 + 1e-12
            assert bool((rs <= bound).all()), f"row sums in slab {a}: {float(rs.max())}"


def oracle_scalar_all_rows(logits, vec, S, Ns, inv, slab=2048):
    """sum_t w_t L_t and sum_t w_t |L_t| over ALL rows, oracle fp64, streamed device -> host in slabs."""
    tg, old, adv, mask, seg = vec
    T = logits.shape[0]
    tot = l1 = 0.0
    stats = np.zeros(4)
    for a in range(0, T, slab):
        b = min(T, a + slab)
        if not mask[a:b].any():
            continue
        r = oracle.policy_loss(bf16_bits(logits[a:b]), tg, old, adv, mask, seg, S, E32[0], E32[1], seg_denom=Ns, inv_num_segs=inv,
                               row_ids=np.arange(a, b, dtype=np.int64), want_dlogits=False, logits_is_bf16_bits=True)
        tot += r.loss
        l1 += float(np.sum(r.w * np.abs(r.Lt)))
        stats += r.stats
    return tot, l1, stats


def test_bench_microbatch_c2_full():
    """configs[1] exactly as bench.py runs it: merge on the GPU, one [40960,151936] bf16 micro-batch of the merged
    tokens with batch-wide normalisers; scalar vs the oracle over all rows, dlogits on sampled rows."""
    seed = W.BASE_SEED + 1
    mi = W.merge_workload("c2", seed=seed)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    mo = ajt.merge_timelines(d(mi.tokens), d(mi.offsets), d(mi.traj_ids), d(mi.resp_start), None, d(mi.old_logp))
    assert ajt.last_status(mo.workspace) == 0
    fin = mo.finalize()
    r = oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp)
    assert fin.N_out == r.N_out and np.array_equal(fin.merged_tokens.cpu().numpy(), r.merged_tokens)
    targets, mask, _ = shift_for_next_token(r.merged_tokens, r.merged_mask, r.merged_old_logp, r.merged_offsets)
    seg, S, _ = seg_ids_from_merged(r.merged_offsets, r.merged_traj)
    adv = W.advantages_group_zscore(seed, 1, S)[seg].astype(np.float32)
    T, V = 40960, 151936
    Ns_t = ajt.segment_counts(d(mask), d(seg), S)
    Ns = Ns_t.cpu().numpy()
    assert np.array_equal(Ns, np.bincount(seg, weights=mask.astype(np.float64), minlength=S).astype(np.float32))
    logits = torch.empty((T, V), dtype=torch.bfloat16, device="cuda")
    H.fill_logits(logits, seed * 7)
    tg, mk, sg, av = targets[:T].copy(), mask[:T].copy(), seg[:T].copy(), adv[:T].copy()
    noise = (W.rng_for(seed, 1, 99).standard_normal(T) * 0.05).astype(np.float32)
    old_t = H.harness_old_logp(logits, d(tg), noise)
    old = old_t.cpu().numpy()
    out = ajt.policy_loss_fwd_bwd(logits, d(tg), old_t, d(av), d(mk), d(sg), S, EPS[0], EPS[1], seg_denom=Ns_t, inv_num_segs=0.0,
                                  want_logp=True, want_stats=True)
    torch.cuda.synchronize()
    assert ajt.last_status(out.workspace) == 0
    vec = (tg, old, av, mk, sg)
    inv = float(np.float32(1.0) / np.float32((Ns > 0).sum()))
    check_sampled(out, logits, vec, S, sample_rows(mk, 40, 1), Ns=Ns, inv=inv)
    anysize_properties(out, d(mk), V)
    tot, l1, stats = oracle_scalar_all_rows(logits, vec, S, Ns, inv)
    dlt = abs(float(out.loss[0]) - tot)
    assert dlt <= 1e-5 * l1 + 1e-7 * abs(tot), (float(out.loss[0]), tot, l1)      # reading L-8 gate (ii)
    if abs(tot) >= 1e-2 * l1:
        assert dlt <= 1e-5 * abs(tot)
    st = out.stats.cpu().numpy()
    assert st[0] == stats[0] and abs(st[1] - stats[1]) <= 2 and abs(st[2] - stats[2]) <= 2


def _sweep_cell(T, V, S, rho, cell):
    lv = W.loss_sweep_vectors(T, V, S, rho, cell=cell)
    logits = torch.empty((T, V), dtype=torch.bfloat16, device="cuda")
    H.fill_logits(logits, 5000 + cell)
    d = lambda a: torch.from_numpy(a).cuda()
    tg = d(lv.targets)
    old_t = H.harness_old_logp(logits, tg, lv.noise)
    return lv, logits, (tg, old_t, d(lv.adv), d(lv.mask), d(lv.seg_ids))


@pytest.mark.parametrize("T,V,S,rho", [
    (131072, 151936, 64, 0.7),     # configs[4] largest cell: 39.8 GB in, 39.8 GB out
    (65536, 151936, 512, 0.3),     # the chunk shape of configs[2] / configs[3] model A
    (65536, 128256, 8, 0.7),       # configs[3] model B vocabulary
    (131072, 32000, 64, 0.3),      # single-CTA rows
])
def test_sweep_cells_full_size(T, V, S, rho):
    lv, logits, (tg, old_t, adv_t, mask_t, seg_t) = _sweep_cell(T, V, S, rho, cell=3)
    out = ajt.policy_loss_fwd_bwd(logits, tg, old_t, adv_t, mask_t, seg_t, lv.S, EPS[0], EPS[1], want_logp=True, want_stats=True)
    torch.cuda.synchronize()
    assert ajt.last_status(out.workspace) == 0
    old = old_t.cpu().numpy()
    vec = (lv.targets, old, lv.adv, lv.mask, lv.seg_ids)
    ref = check_sampled(out, logits, vec, lv.S, sample_rows(lv.mask, 32, 2))
    anysize_properties(out, mask_t, V)
    assert float(out.stats[0]) == float(lv.mask.sum())
    # chunked = unchunked: the same rows through 8 smaller calls with batch-wide normalisers give the same dlogits rows
    # bit for bit and the same scalar; the first chunk's first 2048 rows are oracle-checked in full, scalar included.
    Ns_t = ajt.segment_counts(mask_t, seg_t, lv.S)
    Ns = Ns_t.cpu().numpy()
    inv = float(np.float32(1.0) / np.float32((Ns > 0).sum()))
    step = T // 8
    tot = l1 = 0.0
    buf = torch.empty((step, V), dtype=torch.bfloat16, device="cuda")
    for a in range(0, T, step):
        c = ajt.policy_loss_fwd_bwd(logits[a:a + step], tg[a:a + step], old_t[a:a + step], adv_t[a:a + step], mask_t[a:a + step],
                                    seg_t[a:a + step], lv.S, EPS[0], EPS[1], seg_denom=Ns_t, inv_num_segs=0.0, dlogits=buf)
        tot += float(c.loss[0])
        l1 += abs(float(c.loss[0]))
        assert torch.equal(buf, out.dlogits[a:a + step])
    # every call accumulates in fp64 and rounds its scalar to fp32 once (half an ulp = 2^-24 relative, of each chunk's
    # partial and of the big call's total): that rounding is all that may separate the two
    assert abs(tot - float(out.loss[0])) <= 2.0 ** -23 * (l1 + abs(float(out.loss[0]))) + 1e-12
    R = 2048
    small = ajt.policy_loss_fwd_bwd(logits[:R], tg[:R], old_t[:R], adv_t[:R], mask_t[:R], seg_t[:R], lv.S, EPS[0], EPS[1],
                                    seg_denom=Ns_t, inv_num_segs=0.0, want_logp=True, want_stats=True)
    torch.cuda.synchronize()
    full_ref = oracle.policy_loss(bf16_bits(logits[:R]), lv.targets, old, lv.adv, lv.mask, lv.seg_ids, lv.S, E32[0], E32[1],
                                  seg_denom=Ns, inv_num_segs=inv, row_ids=np.arange(R, dtype=np.int64), logits_is_bf16_bits=True)
    check_loss(small, full_ref, lv.mask, EPS[0], EPS[1], lv.adv, old, 1.0, V, row_ids=np.arange(R))
    assert torch.equal(small.dlogits, out.dlogits[:R])


def test_c3_chunk_with_real_merge_vectors():
    """configs[2]: a 64k-row chunk whose targets / mask / segments come from the GPU merge of the long-horizon batch."""
    mi = W.merge_workload("c3")
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    mo = ajt.merge_timelines(d(mi.tokens), d(mi.offsets), d(mi.traj_ids), d(mi.resp_start), None, d(mi.old_logp))
    assert ajt.last_status(mo.workspace) == 0
    fin = mo.finalize()
    cpu = lambda t: t.cpu().numpy()
    targets, mask, _ = shift_for_next_token(cpu(fin.merged_tokens), cpu(fin.merged_mask), cpu(fin.merged_old_logp),
                                              cpu(fin.merged_offsets))
    seg, S, _ = seg_ids_from_merged(cpu(fin.merged_offsets), cpu(fin.merged_traj))
    adv = W.advantages_group_zscore(W.BASE_SEED + 2, 2, S)[seg].astype(np.float32)
    Ns_t = ajt.segment_counts(d(mask), d(seg), S)
    Ns = Ns_t.cpu().numpy()
    inv = float(np.float32(1.0) / np.float32((Ns > 0).sum()))
    T, V, k = 65536, 151936, 5
    sl = slice(k * T, (k + 1) * T)
    tg, mk, sg, av = targets[sl].copy(), mask[sl].copy(), seg[sl].copy(), adv[sl].copy()
    logits = torch.empty((T, V), dtype=torch.bfloat16, device="cuda")
    H.fill_logits(logits, 77)
    noise = (W.rng_for(W.BASE_SEED + 2, 2, 99).standard_normal(T) * 0.05).astype(np.float32)
    old_t = H.harness_old_logp(logits, d(tg), noise)
    out = ajt.policy_loss_fwd_bwd(logits, d(tg), old_t, d(av), d(mk), d(sg), S, 0.2, 0.2, seg_denom=Ns_t, inv_num_segs=0.0,
                                  want_logp=True)
    torch.cuda.synchronize()
    assert ajt.last_status(out.workspace) == 0
    rows = sample_rows(mk, 32, 3)
    bits = bf16_bits(logits[torch.from_numpy(rows).cuda()])
    old = old_t.cpu().numpy()
    e = float(np.float32(0.2))
    ref = oracle.policy_loss(bits, tg, old, av, mk, sg, S, e, e, seg_denom=Ns, inv_num_segs=inv, row_ids=rows, logits_is_bf16_bits=True)
    check_loss(out, ref, mk, 0.2, 0.2, av, old, 1.0, V, row_ids=rows, check_scalar=False)
    anysize_properties(out, d(mk), V)


@pytest.mark.parametrize("model,V", [("A", 151936), ("B", 128256)])
def test_c4_chunks_with_real_merge_vectors(model, V):
    """configs[3]: each model's own merge (GPU) -> ajt_pack_loss_inputs (GPU, checked against the oracle's pack over the WHOLE
    batch) -> one 64k-row chunk [65536, V] with eps 0.2 / 0.2 and batch-wide normalisers; sampled rows against the oracle."""
    seed = W.BASE_SEED + 3
    mi = W.merge_workload_c4(seed=seed)[model]
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    mo = ajt.merge_timelines(d(mi.tokens), d(mi.offsets), d(mi.traj_ids), d(mi.resp_start), None, d(mi.old_logp))
    assert ajt.last_status(mo.workspace) == 0
    uniq, tl_seg = np.unique(mi.traj_ids, return_inverse=True)
    S = int(uniq.shape[0])
    seg_adv = W.advantages_group_zscore(seed, 3, S).astype(np.float32)
    pk = ajt.pack_loss_inputs(mo, d(tl_seg.astype(np.int32)), S, d(seg_adv))
    fin = mo.finalize()
    r = oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp)
    targets, mask, olp, seg, adv = oracle.pack_loss_inputs(r.merged_tokens, r.merged_mask, r.merged_old_logp, r.merged_offsets,
                                                           r.merged_origin, tl_seg.astype(np.int32), seg_adv)
    No = r.N_out
    cpu = lambda t: t.cpu().numpy()
    assert fin.N_out == No and np.array_equal(cpu(pk.targets[:No]), targets) and np.array_equal(cpu(pk.mask[:No]), mask)
    assert np.array_equal(cpu(pk.seg_ids[:No]), seg) and np.array_equal(cpu(pk.adv[:No]), adv)
    Ns_t = ajt.segment_counts(pk.mask[:No], pk.seg_ids[:No], S)
    Ns = Ns_t.cpu().numpy()
    assert np.array_equal(Ns, np.bincount(seg, weights=mask.astype(np.float64), minlength=S).astype(np.float32))
    inv = float(np.float32(1.0) / np.float32((Ns > 0).sum()))
    T, k = 65536, 3
    sl = slice(k * T, (k + 1) * T)
    logits = torch.empty((T, V), dtype=torch.bfloat16, device="cuda")
    H.fill_logits(logits, 91 + V % 7)
    noise = (W.rng_for(seed, 3, 99).standard_normal(T) * 0.05).astype(np.float32)
    old_t = H.harness_old_logp(logits, pk.targets[sl], noise)
    out = ajt.policy_loss_fwd_bwd(logits, pk.targets[sl], old_t, pk.adv[sl], pk.mask[sl], pk.seg_ids[sl], S, 0.2, 0.2,
                                  seg_denom=Ns_t, inv_num_segs=0.0, want_logp=True)
    torch.cuda.synchronize()
    assert ajt.last_status(out.workspace) == 0
    tg, mk, sg, av, old = targets[sl], mask[sl], seg[sl], adv[sl], old_t.cpu().numpy()
    rows = sample_rows(mk, 32, 3)
    e = float(np.float32(0.2))
    ref = oracle.policy_loss(bf16_bits(logits[torch.from_numpy(rows).cuda()]), tg, old, av, mk, sg, S, e, e, seg_denom=Ns,
                             inv_num_segs=inv, row_ids=rows, logits_is_bf16_bits=True)
    check_loss(out, ref, mk, 0.2, 0.2, av, old, 1.0, V, row_ids=rows, check_scalar=False)
    anysize_properties(out, pk.mask[sl], V)


@pytest.mark.parametrize("T", [4096, 16384, 65536, 131072])
@pytest.mark.parametrize("V", [32000, 128256, 151936])
@pytest.mark.parametrize("rho", [0.3, 0.7])
def test_every_sweep_cell_sampled(T, V, rho):
    """configs[4], all 24 (T, V, mask density) cells (S rotates over 8 / 64 / 512): sampled rows element by element against
    the oracle, masked rows exactly zero, every gradient row sums to zero, the masked-token count."""
    cell = (T // 4096) % 5 + (V // 1000) % 7 + int(rho * 10)
    S = (8, 64, 512)[cell % 3]
    lv, logits, (tg, old_t, adv_t, mask_t, seg_t) = _sweep_cell(T, V, S, rho, cell=cell)
    out = ajt.policy_loss_fwd_bwd(logits, tg, old_t, adv_t, mask_t, seg_t, lv.S, EPS[0], EPS[1], want_logp=True, want_stats=True)
    torch.cuda.synchronize()
    assert ajt.last_status(out.workspace) == 0
    vec = (lv.targets, old_t.cpu().numpy(), lv.adv, lv.mask, lv.seg_ids)
    check_sampled(out, logits, vec, lv.S, sample_rows(lv.mask, 16, 7))
    anysize_properties(out, mask_t, V)
    assert float(out.stats[0]) == float(lv.mask.sum())


def test_lm_head_full_size_sampled_rows():
    """ajt_lm_head_logp at the size bench.py's LM-head record times (40,960 x 4,096 x 151,936: CTA pairs, 9 waves of row blocks, 4 vocabulary
    ranges of 149 tiles): sampled rows against the fp64 oracle computed row by row; every row finite and a valid log-prob."""
    T, d, V = 40960, 4096, 151936
    g = torch.Generator(device="cuda").manual_seed(41)
    Hh = torch.randn((T, d), generator=g, device="cuda").to(torch.bfloat16)
    Ww = (torch.randn((V, d), generator=g, device="cuda") * 0.02).to(torch.bfloat16)
    y = torch.randint(0, V, (T,), generator=g, device="cuda", dtype=torch.int32)
    logp, ent = ajt.lm_head_logp(Hh, Ww, y)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(logp).all()) and bool(torch.isfinite(ent).all())
    assert float(logp.max()) <= 1e-6 and float(ent.min()) >= 0.0 and float(ent.max()) <= np.log(V) + 1e-4
    rng = np.random.default_rng(2)
    rows = np.unique(np.concatenate([[0, 127, 128, 255, 256, T - 1], rng.choice(T, size=48, replace=False)]))
    rt = torch.from_numpy(rows).cuda()
    wb = bf16_bits(Ww)
    rl, re = oracle.lm_head_logp(bf16_bits(Hh[rt]), wb, y[rt].cpu().numpy())
    # |z| ~ 1.3 here and d = 4096: fp32 accumulation error ~ sqrt(d) 2^-24 |z| ~ 5e-6; 5e-5 absolute leaves room for the tails
    assert np.abs(logp[rt].cpu().numpy().astype(np.float64) - rl).max() <= 5e-5
    assert np.abs(ent[rt].cpu().numpy().astype(np.float64) - re).max() <= 5e-5


def test_lm_head_loss_bwd_full_width_against_oracle():
    """ajt_lm_head_loss_bwd at the full hidden size and vocabulary (d = 4,096, V = 151,936: 594 vocabulary tiles, 4 ranges, CTA
    pairs) on 512 rows, where the fp64 oracle (O-HB) still computes everything: loss, dH and dW element by element."""
    T, d, V, S = 512, 4096, 151936, 6
    g = torch.Generator(device="cuda").manual_seed(5)
    rng = np.random.default_rng(5)
    Hh = torch.randn((T, d), generator=g, device="cuda").to(torch.bfloat16)
    Ww = (torch.randn((V, d), generator=g, device="cuda") * 0.02).to(torch.bfloat16)
    y = torch.randint(0, V, (T,), generator=g, device="cuda", dtype=torch.int32)
    adv = torch.from_numpy(rng.standard_normal(T).astype(np.float32)).cuda()
    mask = torch.from_numpy((rng.random(T) < 0.6).astype(np.uint8)).cuda()
    seg = torch.from_numpy(np.sort(rng.integers(0, S, size=T)).astype(np.int32)).cuda()
    lp, _ = ajt.lm_head_logp(Hh, Ww, y)
    old = (lp + torch.from_numpy((rng.standard_normal(T) * 0.1).astype(np.float32)).cuda()).contiguous()
    out = ajt.lm_head_loss_bwd(Hh, Ww, y, old, adv, mask, seg, S, 0.2, 0.28)
    torch.cuda.synchronize()
    assert ajt.last_status(out["workspace"]) == 0
    e = (float(np.float32(0.2)), float(np.float32(0.28)))
    ref = oracle.lm_head_loss_bwd(bf16_bits(Hh), bf16_bits(Ww), y.cpu().numpy(), old.cpu().numpy(), adv.cpu().numpy(),
                                  mask.cpu().numpy(), seg.cpu().numpy(), S, e[0], e[1], round_dz_bf16=True)
    l1 = float(np.sum(ref["w"] * np.abs(ref["Lt"])))
    assert abs(float(out["loss"][0]) - ref["loss"]) <= 1e-5 * l1 + 1e-7 * abs(ref["loss"])
    dH, dW = out["dH"].float().cpu().numpy().astype(np.float64), out["dW"].cpu().numpy().astype(np.float64)
    sH, sW = np.abs(ref["dH"]).max(), np.abs(ref["dW"]).max()
    assert np.abs(dH - ref["dH"]).max() <= 2.0 ** -7 * sH
    assert np.abs(dW - ref["dW"]).max() <= 2e-3 * sW


def test_lm_head_loss_bwd_bench_size_properties():
    """The size bench.py's LM-head record times (40,960 x 4,096 x 151,936, mask density ~0.34: 4 chunks of staged dZ): sampled dH rows against
    the oracle computed row by row (the row's own 151,936 logits in fp64), masked rows exactly zero, and two identities of
    the exact gradients that tie dW to them at any size: sum_v dW_v = 0 (every dZ row sums to zero) and <dW, W> = sum_t <dH_t, h_t>."""
    T, d, V, S = 40960, 4096, 151936, 64
    g = torch.Generator(device="cuda").manual_seed(6)
    rng = np.random.default_rng(6)
    Hh = torch.randn((T, d), generator=g, device="cuda").to(torch.bfloat16)
    Ww = (torch.randn((V, d), generator=g, device="cuda") * 0.02).to(torch.bfloat16)
    lv = W.loss_sweep_vectors(T, V, S, 0.35, cell=9)
    dd = lambda a: torch.from_numpy(a).cuda()
    y, adv, mask, seg = dd(lv.targets), dd(lv.adv), dd(lv.mask), dd(lv.seg_ids)
    lp, _ = ajt.lm_head_logp(Hh, Ww, y, mask)
    old = (lp + dd(lv.noise)).contiguous()
    out = ajt.lm_head_loss_bwd(Hh, Ww, y, old, adv, mask, seg, S, 0.2, 0.28)
    torch.cuda.synchronize()
    assert ajt.last_status(out["workspace"]) == 0
    dH, dW = out["dH"], out["dW"]
    assert bool(torch.isfinite(dW).all()) and bool(torch.isfinite(dH.float()).all())
    assert not bool(dH[mask == 0].any())
    # identities of the exact gradients
    colsum = dW.double().sum(dim=0)
    assert float(colsum.abs().max()) <= 1e-3 * float(dW.double().abs().sum(dim=0).max())
    lhs = float((dW.double() * Ww.double()).sum())
    rhs = float((dH.double() * Hh.double()).sum())
    scale = float((dH.double().abs() * Hh.double().abs()).sum())
    assert abs(lhs - rhs) <= 2.0 ** -8 * scale
    # sampled rows, oracle row by row: z_t = W h_t in fp64, steps 1-6, dH_t = dZ_t W
    Ns = np.bincount(lv.seg_ids, weights=lv.mask.astype(np.float64), minlength=S)
    inv = 1.0 / max(1, int((Ns > 0).sum()))
    Wf = Ww.double().cpu().numpy()
    oldh, e = old.cpu().numpy().astype(np.float64), (float(np.float32(0.2)), float(np.float32(0.28)))
    on = np.nonzero(lv.mask)[0]
    for t in [int(on[0]), int(on[-1])] + [int(x) for x in rng.choice(on, size=6, replace=False)]:
        h = Hh[t].double().cpu().numpy()
        z = Wf @ h
        lse = z.max() + np.log(np.exp(z - z.max()).sum())
        logp = z[lv.targets[t]] - lse
        r = np.exp(logp - oldh[t])
        A = float(lv.adv[t])
        passes = not ((A > 0 and r > 1 + e[1]) or (A < 0 and r < 1 - e[0]))
        w = inv / Ns[lv.seg_ids[t]]
        gt = w * (-A * r) if passes else 0.0
        dz = -gt * np.exp(z - lse)
        dz[lv.targets[t]] += gt
        ref = oracle.round_bf16(dz) @ Wf
        got = dH[t].double().cpu().numpy()
        assert np.abs(got - ref).max() <= 2.0 ** -7 * np.abs(ref).max() + 1e-30, t


def test_merge_blocks_full_size_b3():
    """ajt_merge_blocks on the full b3 workload (7,805 timelines, 253,556 blocks, 145.6 M tokens), bit-exact in every output."""
    from test_gpu_blocks import as_dict, run
    bi = W.block_workload("b3")
    g, r, _ = run(as_dict(bi))
    assert g.N_out > 20_000_000 and g.M < bi.n // 5
