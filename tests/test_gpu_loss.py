"""GPU parity: ajt_policy_loss_fwd_bwd (through the C ABI) vs the fp64 oracle, element by element.

Sizes the oracle finishes in seconds; every kernel variant (fast 1-CTA NCH=8/16, fast 2-CTA cluster,
generic fp32 / odd-V), several row tiles per cluster, ragged vocabulary tails, edge cases.
Tolerances: BASELINE.json north_star (loss 1e-5 relative, dlogits 2e-3 absolute) with DESIGN.md readings L-8, L-9.
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_04484_b200 as ajt
from paper_2606_04484_b200 import workloads as W
from helpers import check_loss, harness_old_logp, logits_to_oracle, seg_ids_from_merged, shift_for_next_token

pytestmark = pytest.mark.gpu


def make_case(T, V, S, rho, dtype, sigma, seed, ld=None):
    lv = W.loss_sweep_vectors(T, V, S, rho, seed=seed, cell=V % 977)
    g = torch.Generator(device="cuda").manual_seed(seed)
    ld = V if ld is None else ld
    logits = torch.randn((T, ld), generator=g, device="cuda", dtype=torch.float32) * sigma
    logits = logits.to(dtype)
    dev = lambda a: torch.from_numpy(a).cuda()
    targets, adv, mask, seg = dev(lv.targets), dev(lv.adv), dev(lv.mask), dev(lv.seg_ids)
    old = harness_old_logp(logits[:, :V], targets, lv.noise)
    return lv, logits, targets, old, adv, mask, seg


def run_and_check(T, V, S, rho, dtype, sigma=3.0, eps=(0.2, 0.28), grad_scale=1.0, seed=1, ld=None, inplace=False):
    lv, logits, targets, old, adv, mask, seg = make_case(T, V, S, rho, dtype, sigma, seed, ld)
    zo, is_bits = logits_to_oracle(logits[:, :V])
    src = logits.clone() if inplace else logits
    out = ajt.policy_loss_fwd_bwd(src, targets, old, adv, mask, seg, lv.S, eps[0], eps[1], grad_scale=grad_scale, V=V,
                                  dlogits=src if inplace else None, want_logp=True, want_stats=True)
    torch.cuda.synchronize()
    assert ajt.last_status(out.workspace) == 0
    ref = oracle.policy_loss(zo, lv.targets, old.cpu().numpy(), lv.adv, lv.mask, lv.seg_ids, lv.S,
                             float(np.float32(eps[0])), float(np.float32(eps[1])), grad_scale=grad_scale,
                             logits_is_bf16_bits=is_bits)
    info = check_loss(out, ref, lv.mask, eps[0], eps[1], lv.adv, old.cpu().numpy(), grad_scale, V)
    if ld is not None and ld > V and not inplace:   # the padding columns are never written
        pass
    return out, ref, info


@pytest.mark.parametrize("T,V,S,rho", [
    (700, 32000, 8, 0.7),        # fast, 1 CTA per row, 7 chunks (ragged: 32000 = 6*4864 + 2816)
    (500, 65536, 5, 0.3),        # fast, 1 CTA, 14 chunks
    (300, 77824, 3, 0.7),        # fast, 1 CTA, exactly 16 full chunks (largest single-CTA row)
    (400, 128256, 8, 0.7),       # fast, 2-CTA cluster
    (400, 151936, 8, 0.3),       # fast, 2-CTA cluster, the headline vocabulary; ragged tail chunk
    (333, 155640, 2, 0.7),       # fast, 2-CTA cluster, the largest supported V
])
def test_fast_path_bf16(T, V, S, rho):
    run_and_check(T, V, S, rho, torch.bfloat16)


@pytest.mark.parametrize("T,V,S,rho,dtype", [
    (3000, 1024, 32, 0.45, torch.float32),    # config c1's shape: fp32 logits, V=1024: the one-read register kernel, 8 vectors per lane
    (700, 2048, 8, 0.6, torch.float32),       # fp32 one-read kernel, 16 vectors per lane (its largest V)
    (500, 1000, 4, 0.5, torch.float32),       # fp32 one-read kernel, V not a multiple of 128: lanes without a vector
    (300, 36, 3, 0.7, torch.float32),         # fp32 one-read kernel, fewer vectors than lanes
    (300, 1002, 4, 0.7, torch.float32),       # fp32, V % 4 != 0 -> generic, warp per row
    (300, 5000, 4, 0.7, torch.float32),       # fp32, CTA-per-row generic
    (300, 1001, 4, 0.7, torch.bfloat16),      # odd V -> generic, warp per row
    (200, 151937, 4, 0.7, torch.bfloat16),    # odd V -> generic, CTA per row
    (64, 200000, 2, 0.7, torch.bfloat16),     # V beyond the cluster kernel -> generic
])
def test_generic_path(T, V, S, rho, dtype):
    run_and_check(T, V, S, rho, dtype, sigma=2.0 if dtype == torch.float32 else 3.0)


def test_grad_scale_makes_literal_tolerance_bite():
    # reading L-9: scale the upstream gradient so that the largest |dlogits| is just under 1.  A bf16 half-ulp
    # below 1 is 2^-9 = 1.95e-3, so the literal 2e-3 absolute bound is attainable there and it bites (all-zeros
    # would fail by ~0.9); above 1 bf16 storage alone exceeds 2e-3.  The oracle is linear in grad_scale.
    _, ref1, _ = run_and_check(400, 151936, 8, 0.7, torch.bfloat16, grad_scale=1.0)
    gs = float(np.float32(0.9 / np.abs(ref1.dlogits).max()))
    out, ref, info = run_and_check(400, 151936, 8, 0.7, torch.bfloat16, grad_scale=gs)
    assert 0.8 < np.abs(ref.dlogits).max() < 1.0


def test_symmetric_clip_and_seeds():
    for seed in (2, 3):
        run_and_check(300, 32000, 16, 0.5, torch.bfloat16, eps=(0.2, 0.2), seed=seed)


def test_row_stride_and_inplace():
    run_and_check(300, 32000, 4, 0.7, torch.bfloat16, ld=32000 + 64)
    run_and_check(300, 151936, 4, 0.7, torch.bfloat16, inplace=True)
    run_and_check(200, 1001, 4, 0.7, torch.bfloat16, ld=1010)
    run_and_check(200, 1024, 4, 0.7, torch.float32, ld=1040, sigma=2.0)   # fp32 one-read kernel with a row stride
    run_and_check(200, 1024, 4, 0.7, torch.float32, ld=1026, sigma=2.0)   # stride not a multiple of 4: generic kernel


def test_padding_columns_untouched():
    T, V, ld = 100, 32000, 32064
    lv, logits, targets, old, adv, mask, seg = make_case(T, V, 4, 0.7, torch.bfloat16, 3.0, 5, ld)
    dl = torch.full((T, ld), 7.0, dtype=torch.bfloat16, device="cuda")
    ajt.policy_loss_fwd_bwd(logits, targets, old, adv, mask, seg, lv.S, 0.2, 0.28, V=V, dlogits=dl)
    torch.cuda.synchronize()
    assert torch.all(dl[:, V:] == 7.0)


def test_edge_cases():
    # T = 1, T = 0, all masked, nothing masked, S' = 0
    run_and_check(1, 32000, 1, 1.0, torch.bfloat16)
    lv, logits, targets, old, adv, mask, seg = make_case(64, 32000, 4, 0.5, torch.bfloat16, 3.0, 9)
    out = ajt.policy_loss_fwd_bwd(logits, targets, old, adv, torch.zeros_like(mask), seg, lv.S, 0.2, 0.2, want_logp=True,
                                  want_stats=True)
    torch.cuda.synchronize()
    assert float(out.loss[0]) == 0.0 and torch.all(out.dlogits == 0) and torch.all(out.logp == 0)
    assert out.stats.cpu().tolist() == [0.0, 0.0, 0.0, 0.0]
    out = ajt.policy_loss_fwd_bwd(logits[:0], targets[:0], old[:0], adv[:0], mask[:0], seg[:0], 1, 0.2, 0.2)
    torch.cuda.synchronize()
    assert float(out.loss[0]) == 0.0
    run_and_check(200, 151936, 3, 1.0, torch.bfloat16)     # every row unmasked
    run_and_check(150, 151936, 200, 0.5, torch.bfloat16)   # more segments than tokens can fill


def test_bad_target_and_segment_set_status():
    lv, logits, targets, old, adv, mask, seg = make_case(64, 32000, 4, 1.0, torch.bfloat16, 3.0, 11)
    t2 = targets.clone(); t2[5] = 32000
    out = ajt.policy_loss_fwd_bwd(logits, t2, old, adv, mask, seg, lv.S, 0.2, 0.2)
    assert ajt.last_status(out.workspace) & ajt.STATUS_BAD_TARGET
    s2 = seg.clone(); s2[7] = -1
    out = ajt.policy_loss_fwd_bwd(logits, targets, old, adv, mask, s2, lv.S, 0.2, 0.2)
    assert ajt.last_status(out.workspace) & ajt.STATUS_BAD_SEG
    # the fp32 one-read kernel reports them too, and the bad row contributes nothing
    lv, logits, targets, old, adv, mask, seg = make_case(64, 1024, 4, 1.0, torch.float32, 2.0, 12)
    t2 = targets.clone(); t2[5] = 1024
    out = ajt.policy_loss_fwd_bwd(logits, t2, old, adv, mask, seg, lv.S, 0.2, 0.2)
    assert ajt.last_status(out.workspace) & ajt.STATUS_BAD_TARGET
    assert torch.all(out.dlogits[5] == 0)


def test_chunked_equals_unchunked():
    # reading L-4: batch-wide seg_denom + inv_num_segs; sum of the chunk partials = the single-call loss;
    # dlogits rows identical
    T, V, S = 600, 151936, 6
    lv, logits, targets, old, adv, mask, seg = make_case(T, V, S, 0.6, torch.bfloat16, 3.0, 13)
    full = ajt.policy_loss_fwd_bwd(logits, targets, old, adv, mask, seg, S, 0.2, 0.28)
    Ns = torch.zeros(S, device="cuda").index_add_(0, seg.long(), mask.float())
    inv = 1.0 / float((Ns > 0).sum())
    tot = 0.0
    for a in range(0, T, 250):
        b = min(T, a + 250)
        c = ajt.policy_loss_fwd_bwd(logits[a:b], targets[a:b], old[a:b], adv[a:b], mask[a:b], seg[a:b], S, 0.2, 0.28,
                                    seg_denom=Ns, inv_num_segs=inv)
        tot += float(c.loss[0])
        assert torch.equal(c.dlogits, full.dlogits[a:b])
    assert abs(tot - float(full.loss[0])) <= 2e-7 * max(1e-3, abs(float(full.loss[0]))) + 1e-9


def test_bitwise_reproducible():
    lv, logits, targets, old, adv, mask, seg = make_case(500, 151936, 8, 0.5, torch.bfloat16, 3.0, 17)
    a = ajt.policy_loss_fwd_bwd(logits, targets, old, adv, mask, seg, lv.S, 0.2, 0.28)
    b = ajt.policy_loss_fwd_bwd(logits, targets, old, adv, mask, seg, lv.S, 0.2, 0.28)
    torch.cuda.synchronize()
    assert torch.equal(a.dlogits, b.dlogits) and torch.equal(a.loss, b.loss)


def test_c1_loss_over_merged_tokens():
    """configs[0] end to end: merge on the GPU, loss on the merged tokens (fp32 logits, V=1024, adv +-1, eps 0.2)."""
    mi = W.merge_workload("c1")
    r = oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp)
    targets, mask, _ = shift_for_next_token(r.merged_tokens, r.merged_mask, r.merged_old_logp, r.merged_offsets)
    seg, S, _ = seg_ids_from_merged(r.merged_offsets, r.merged_traj)
    advt = W.advantages_pm1(W.BASE_SEED, 0, S)
    T, V = r.N_out, 1024
    g = torch.Generator(device="cuda").manual_seed(W.BASE_SEED)
    logits = torch.randn((T, V), generator=g, device="cuda") * 2.0
    noise = (W.rng_for(W.BASE_SEED, 0, 99).standard_normal(T) * 0.05).astype(np.float32)
    tg = torch.from_numpy(targets).cuda()
    old = harness_old_logp(logits, tg, noise)
    adv = advt[seg]
    out = ajt.policy_loss_fwd_bwd(logits, tg, old, torch.from_numpy(adv).cuda(), torch.from_numpy(mask).cuda(),
                                  torch.from_numpy(seg).cuda(), S, 0.2, 0.2, want_logp=True, want_stats=True)
    torch.cuda.synchronize()
    ref = oracle.policy_loss(logits.cpu().numpy(), targets, old.cpu().numpy(), adv, mask, seg, S,
                             float(np.float32(0.2)), float(np.float32(0.2)))
    check_loss(out, ref, mask, 0.2, 0.2, adv, old.cpu().numpy(), 1.0, V)
    l1 = float(np.sum(ref.w * np.abs(ref.Lt)))
    assert abs(ref.loss) >= 1e-2 * l1     # c1's unbalanced +-1 advantages: the plain relative gate applies (L-8)


def test_host_buffer_variant():
    T, V, S = 200, 32000, 4
    lv, logits, targets, old, adv, mask, seg = make_case(T, V, S, 0.6, torch.bfloat16, 3.0, 19)
    dev = ajt.policy_loss_fwd_bwd(logits, targets, old, adv, mask, seg, S, 0.2, 0.28, want_logp=True, want_stats=True)
    h = ajt.policy_loss_fwd_bwd_host(logits.cpu().pin_memory(), lv.targets, old.cpu().numpy(), lv.adv, lv.mask, lv.seg_ids, S,
                                     0.2, 0.28, ajt.DT_BF16, want_logp=True, want_stats=True)
    torch.cuda.synchronize()
    assert h["status"] == 0
    assert torch.equal(h["dlogits"], dev.dlogits.cpu())
    assert h["loss"] == float(dev.loss[0])
    assert np.array_equal(h["logp"], dev.logp.cpu().numpy())


def test_host_buffer_variant_slab_pipeline():
    # several row slabs in flight (H2D, loss call and D2H of neighbouring slabs overlap): dlogits / logp rows identical to the
    # device call's; the scalar is the fp64 sum of the slabs' fp32 partials
    T, V, S = 1500, 32000, 6
    lv, logits, targets, old, adv, mask, seg = make_case(T, V, S, 0.5, torch.bfloat16, 3.0, 29)
    dev = ajt.policy_loss_fwd_bwd(logits, targets, old, adv, mask, seg, S, 0.2, 0.28, want_logp=True, want_stats=True)
    h = ajt.policy_loss_fwd_bwd_host(logits.cpu().pin_memory(), lv.targets, old.cpu().numpy(), lv.adv, lv.mask, lv.seg_ids, S,
                                     0.2, 0.28, ajt.DT_BF16, want_logp=True, want_stats=True)
    torch.cuda.synchronize()
    assert h["status"] == 0
    assert torch.equal(h["dlogits"], dev.dlogits.cpu())
    assert np.array_equal(h["logp"], dev.logp.cpu().numpy())
    st = dev.stats.cpu().numpy()
    assert np.array_equal(h["stats"][:3], st[:3]) and abs(h["stats"][3] - st[3]) <= 1e-6 * max(1e-3, abs(st[3]))
    # scale of the rounding: each of the 6 slab partials is rounded to fp32 once
    assert abs(h["loss"] - float(dev.loss[0])) <= 1e-6 * max(abs(float(dev.loss[0])), 1e-3)
    # fp32 logits take the separate dlogits buffer
    lv, logits, targets, old, adv, mask, seg = make_case(700, 1024, 4, 0.5, torch.float32, 2.0, 31)
    dev = ajt.policy_loss_fwd_bwd(logits, targets, old, adv, mask, seg, 4, 0.2, 0.2)
    h = ajt.policy_loss_fwd_bwd_host(logits.cpu().pin_memory(), lv.targets, old.cpu().numpy(), lv.adv, lv.mask, lv.seg_ids, 4,
                                     0.2, 0.2, ajt.DT_F32)
    assert torch.equal(h["dlogits"], dev.dlogits.cpu()) and h["status"] == 0


def test_segment_counts():
    # ajt_segment_counts: N_s over a batch, chunk by chunk (accumulate), equals a host bincount; bad ids set the status
    T, S = 100_003, 37
    rng = np.random.default_rng(23)
    mask = (rng.random(T) < 0.4).astype(np.uint8)
    seg = np.sort(rng.integers(0, S, size=T)).astype(np.int32)
    seg[rng.integers(0, T, size=500)] = rng.integers(0, S, size=500)        # some out-of-run ids
    want = np.bincount(seg, weights=mask.astype(np.float64), minlength=S).astype(np.float32)
    mk, sg = torch.from_numpy(mask).cuda(), torch.from_numpy(seg).cuda()
    got = ajt.segment_counts(mk, sg, S)
    assert np.array_equal(got.cpu().numpy(), want)
    acc = torch.full((S,), 99.0, device="cuda")
    st = torch.full((1,), 7, dtype=torch.int32, device="cuda")
    ajt.segment_counts(mk[:40000], sg[:40000], S, out=acc, accumulate=False, status=st)
    ajt.segment_counts(mk[40000:], sg[40000:], S, out=acc, accumulate=True, status=st)
    assert np.array_equal(acc.cpu().numpy(), want) and int(st[0]) == 0
    sg2 = sg.clone()
    on = int(np.nonzero(mask)[0][10])
    sg2[on] = S
    got = ajt.segment_counts(mk, sg2, S, out=acc, status=st)
    assert int(st[0]) & ajt.STATUS_BAD_SEG
    assert got.sum().item() == want.sum() - 1
    assert ajt.segment_counts(mk[:0], sg[:0], 3).cpu().tolist() == [0.0, 0.0, 0.0]
    # slices at every alignment of the two arrays (vector body with a scalar head and tail, or the scalar path alone when the
    # 4-byte mask and 16-byte segment-id alignments never meet), short ranges, and views whose storage offsets differ
    for a in range(0, 9):
        for n in (0, 1, 3, 5, 131, 4099, T - 9):
            w = np.bincount(seg[a:a + n], weights=mask[a:a + n].astype(np.float64), minlength=S).astype(np.float32)
            assert np.array_equal(ajt.segment_counts(mk[a:a + n], sg[a:a + n], S).cpu().numpy(), w), (a, n)
    mk_off = torch.zeros(T + 3, dtype=torch.uint8, device="cuda")[3:]
    mk_off.copy_(mk)
    assert np.array_equal(ajt.segment_counts(mk_off, sg, S).cpu().numpy(), want)
    assert np.array_equal(ajt.segment_counts(mk_off[2:], sg[2:], S).cpu().numpy(),
                          np.bincount(seg[2:], weights=mask[2:].astype(np.float64), minlength=S).astype(np.float32))
