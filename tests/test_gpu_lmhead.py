"""GPU parity: ajt_lm_head_logp (tcgen05 GEMM tiles reduced on the fly) vs oracle.lm_head_logp (fp64 from the same bf16 inputs).
Tolerance: the logits are fp32 sums of d exact bf16 products (relative error ~ d 2^-24 in the worst case, ~ sqrt(d) 2^-24
typically) and the reductions are fp32: 3e-5 absolute on logp and on the entropy at these sizes (|z| of order 1-10)."""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_04484_b200 as ajt

pytestmark = pytest.mark.gpu


def bits(t):
    return t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


def run(T, d, V, seed=0, mask_frac=None, wscale=0.05):
    g = torch.Generator(device="cuda").manual_seed(seed)
    H = torch.randn((T, d), generator=g, device="cuda").to(torch.bfloat16)
    W = (torch.randn((V, d), generator=g, device="cuda") * wscale).to(torch.bfloat16)
    y = torch.randint(0, V, (T,), generator=g, device="cuda", dtype=torch.int32)
    mask = None
    if mask_frac is not None:
        mask = (torch.rand(T, generator=g, device="cuda") < mask_frac).to(torch.uint8)
    logp, ent = ajt.lm_head_logp(H, W, y, mask)
    torch.cuda.synchronize()
    rl, re = oracle.lm_head_logp(bits(H), bits(W), y.cpu().numpy(), None if mask is None else mask.cpu().numpy())
    el = np.abs(logp.cpu().numpy().astype(np.float64) - rl).max()
    ee = np.abs(ent.cpu().numpy().astype(np.float64) - re).max()
    # fp32 accumulation error of a logit ~ sqrt(d) 2^-24 |z| with |z| ~ wscale sqrt(d) (a few times that in the tails, which
    # is where the maximum and usually the target sit): 3e-5 absolute while wscale sqrt(d) <= 2, proportionally more above
    tol = 3e-5 * max(1.0, wscale * np.sqrt(d) / 2.0)
    assert el <= tol and ee <= tol, (el, ee, tol)
    if mask is not None:
        off = mask.cpu().numpy() == 0
        assert np.all(logp.cpu().numpy()[off] == 0) and np.all(ent.cpu().numpy()[off] == 0)
    return el, ee


@pytest.mark.parametrize("T,d,V", [
    (128, 64, 256),        # one row block, one K slab, one tile
    (1, 64, 8),            # a single row, a vocabulary smaller than any tile (TMA boxes larger than the tensors)
    (50, 64, 100),         # one CTA, ragged everywhere
    (129, 128, 257),       # CTA pair with one live row in the second CTA, one column in the second tile
    (300, 256, 1000),      # ragged rows and columns, a single vocabulary range
    (257, 128, 5000),      # four vocabulary ranges, ragged last tile
    (1000, 1024, 32000),   # 8 row blocks x 4 ranges, 16 K slabs: the smem ring and both accumulators wrap many times
])
def test_matches_oracle(T, d, V):
    run(T, d, V, seed=T + V)


def test_masked_rows_and_many_row_blocks():
    run(148 * 128 // 4 + 200, 128, 2048, seed=5, mask_frac=0.4)      # more row blocks than one wave holds


def test_peaked_rows():
    run(256, 256, 4096, seed=9, wscale=0.5)                          # |z| up to ~30: the online re-basing matters


def test_row_lse_output():
    g = torch.Generator(device="cuda").manual_seed(3)
    H = torch.randn((200, 128), generator=g, device="cuda").to(torch.bfloat16)
    W = (torch.randn((3000, 128), generator=g, device="cuda") * 0.1).to(torch.bfloat16)
    y = torch.randint(0, 3000, (200,), generator=g, device="cuda", dtype=torch.int32)
    logp, ent, lse = ajt.lm_head_logp(H, W, y, want_lse=True)
    torch.cuda.synchronize()
    z = H.double() @ W.double().T
    want = torch.logsumexp(z, dim=-1)
    assert float((lse.double() - want).abs().max()) <= 3e-5
    zy = z.gather(1, y.long()[:, None])[:, 0]
    assert float((logp.double() - (zy - want)).abs().max()) <= 3e-5


def test_rounded_logits_agree_with_the_loss_call_on_stored_logits():
    # AJT_LM_ROUND_LOGITS_BF16: log-probs from hidden states == log-probs the loss call computes from the bf16 logits a forward
    # pass would store (same rounded values, fp32 reductions in a different order)
    g = torch.Generator(device="cuda").manual_seed(11)
    T, d, V = 300, 256, 32000
    H = torch.randn((T, d), generator=g, device="cuda").to(torch.bfloat16)
    W = (torch.randn((V, d), generator=g, device="cuda") * 0.1).to(torch.bfloat16)
    y = torch.randint(0, V, (T,), generator=g, device="cuda", dtype=torch.int32)
    logp, ent = ajt.lm_head_logp(H, W, y, round_logits_bf16=True)
    rl, re = oracle.lm_head_logp(bits(H), bits(W), y.cpu().numpy(), round_logits_bf16=True)
    # a logit whose fp32 value lies within rounding error of a bf16 tie may round the other way: compare in bulk, not per row
    el = np.abs(logp.cpu().numpy().astype(np.float64) - rl)
    assert np.median(el) <= 3e-6 and np.quantile(el, 0.99) <= 2e-3
    logits = (H.float() @ W.float().T).to(torch.bfloat16)
    one = torch.ones(T, device="cuda")
    out = ajt.policy_loss_fwd_bwd(logits, y, torch.zeros(T, device="cuda"), one, torch.ones(T, dtype=torch.uint8, device="cuda"),
                                  torch.zeros(T, dtype=torch.int32, device="cuda"), 1, 0.2, 0.2, want_logp=True)
    torch.cuda.synchronize()
    dl = (logp - out.logp).abs().cpu().numpy()
    assert np.median(dl) <= 3e-6 and np.quantile(dl, 0.99) <= 2e-3


def test_unsupported_shapes_are_rejected():
    H = torch.zeros((8, 48), dtype=torch.bfloat16, device="cuda")
    W = torch.zeros((16, 48), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(ajt.AjtError):
        ajt.lm_head_logp(H, W, torch.zeros(8, dtype=torch.int32, device="cuda"))


def test_bad_target_sets_status_word():
    # an out-of-range target must not silently give logp = -inf; the status word reports it, the row returns 0
    g = torch.Generator(device="cuda").manual_seed(9)
    T, d, V = 200, 128, 1000
    Hh = torch.randn((T, d), generator=g, device="cuda").to(torch.bfloat16)
    Ww = (torch.randn((V, d), generator=g, device="cuda") * 0.05).to(torch.bfloat16)
    y = torch.randint(0, V, (T,), generator=g, device="cuda", dtype=torch.int32)
    ws = torch.empty(int(ajt.lib().ajt_lm_head_workspace_bytes(T, d, V)) + 256, dtype=torch.uint8, device="cuda")
    lp, en = ajt.lm_head_logp(Hh, Ww, y, workspace=ws)
    torch.cuda.synchronize()
    assert ajt.last_status(ws) == 0 and bool(torch.isfinite(lp).all())
    y2 = y.clone()
    y2[17] = V + 5
    y2[150] = -1
    lp2, en2 = ajt.lm_head_logp(Hh, Ww, y2, workspace=ws)
    torch.cuda.synchronize()
    assert ajt.last_status(ws) & ajt.STATUS_BAD_TARGET
    assert float(lp2[17]) == 0.0 and float(lp2[150]) == 0.0 and bool(torch.isfinite(lp2).all())
    keep = torch.ones(T, dtype=torch.bool, device="cuda")
    keep[17] = keep[150] = False
    assert torch.equal(lp2[keep], lp[keep])


def _bwd_inputs(T, d, V, S, seed, rho=0.7, wscale=0.05):
    g = torch.Generator(device="cuda").manual_seed(seed)
    rng = np.random.default_rng(seed)
    Hh = torch.randn((T, d), generator=g, device="cuda").to(torch.bfloat16)
    Ww = (torch.randn((V, d), generator=g, device="cuda") * wscale).to(torch.bfloat16)
    y = torch.randint(0, V, (T,), generator=g, device="cuda", dtype=torch.int32)
    adv = torch.from_numpy(rng.standard_normal(T).astype(np.float32)).cuda()
    mask = torch.from_numpy((rng.random(T) < rho).astype(np.uint8)).cuda()
    seg = torch.from_numpy(np.sort(rng.integers(0, S, size=T)).astype(np.int32)).cuda()
    lp, _ = ajt.lm_head_logp(Hh, Ww, y)
    old = (lp + torch.from_numpy((rng.standard_normal(T) * 0.2).astype(np.float32)).cuda()).contiguous()
    return Hh, Ww, y, old, adv, mask, seg


@pytest.mark.parametrize("T,d,V,S,use_mask", [(300, 128, 1000, 4, True), (300, 128, 1000, 4, False), (700, 256, 5000, 9, True),
                                               (5000, 64, 777, 3, True)])
def test_loss_bwd_matches_oracle(T, d, V, S, use_mask):
    """ajt_lm_head_loss_bwd vs oracle.lm_head_loss_bwd (O-HB) element by element: loss, log-probs, dH, dW.  The kernel feeds dZ
    to the tensor cores in bf16 (reading H-4), so it is compared with the oracle's rounded-operand variant (fp32 accumulation
    and rare bf16 ties are all that is left), and its distance to the unrounded definition is bounded by the operand rounding."""
    Hh, Ww, y, old, adv, mask, seg = _bwd_inputs(T, d, V, S, seed=T + V)
    out = ajt.lm_head_loss_bwd(Hh, Ww, y, old, adv, mask if use_mask else None, seg, S, 0.2, 0.28)
    torch.cuda.synchronize()
    assert ajt.last_status(out["workspace"]) == 0
    b16 = lambda t: t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
    mk = mask.cpu().numpy() if use_mask else np.ones(T, np.uint8)
    e = (float(np.float32(0.2)), float(np.float32(0.28)))
    args = (b16(Hh), b16(Ww), y.cpu().numpy(), old.cpu().numpy(), adv.cpu().numpy(), mk, seg.cpu().numpy(), S, e[0], e[1])
    ref = oracle.lm_head_loss_bwd(*args, round_dz_bf16=True)
    exact = oracle.lm_head_loss_bwd(*args)
    l1 = float(np.sum(ref["w"] * np.abs(ref["Lt"])))
    assert abs(float(out["loss"][0]) - ref["loss"]) <= 1e-5 * l1 + 1e-7 * abs(ref["loss"])
    assert np.abs(out["logp"].cpu().numpy() - ref["logp"]).max() <= 3e-5
    dH, dW = out["dH"].float().cpu().numpy().astype(np.float64), out["dW"].cpu().numpy().astype(np.float64)
    # rows whose ratio sits on a clip bound may take the other branch in fp32: excluded (as in the loss tests)
    r = np.exp(exact["logp"] - old.cpu().numpy())
    A = adv.cpu().numpy()
    near = ((A > 0) & (np.abs(r - (1 + e[1])) < 1e-4)) | ((A < 0) & (np.abs(r - (1 - e[0])) < 1e-4))
    assert not near.any() or near.sum() < 3
    ok = ~near
    sH = np.abs(ref["dH"]).max() + 1e-30
    assert not dH[mk == 0].any()                                    # masked rows: exactly zero
    assert np.abs(dH[ok] - ref["dH"][ok]).max() <= 2.0 ** -7 * sH   # bf16 output rounding (2^-9 relative) + fp32 accumulation
    if not near.any():
        sW = np.abs(ref["dW"]).max() + 1e-30
        assert np.abs(dW - ref["dW"]).max() <= 2e-3 * sW
        assert np.abs(dW - exact["dW"]).max() <= 2.0 ** -6 * sW       # the operand rounding itself (reading H-4)
    assert np.abs(dH[ok] - exact["dH"][ok]).max() <= 2.0 ** -6 * sH


def test_loss_bwd_accumulates_dw_and_takes_batch_normalisers():
    T, d, V, S = 600, 128, 2000, 5
    Hh, Ww, y, old, adv, mask, seg = _bwd_inputs(T, d, V, S, seed=77)
    one = ajt.lm_head_loss_bwd(Hh, Ww, y, old, adv, mask, seg, S, 0.2, 0.28)
    Ns = ajt.segment_counts(mask, seg, S)
    dW = torch.zeros((V, d), dtype=torch.float32, device="cuda")
    tot = 0.0
    dH = torch.empty((T, d), dtype=torch.bfloat16, device="cuda")
    for a, b in ((0, 256), (256, 600)):       # two micro-batches of the same batch: row ranges + batch-wide N_s (reading L-4)
        o = ajt.lm_head_loss_bwd(Hh[a:b], Ww, y[a:b], old[a:b], adv[a:b], mask[a:b], seg[a:b], S, 0.2, 0.28, seg_denom=Ns, dW=dW,
                                 accumulate_dw=True)
        tot += float(o["loss"][0])
        dH[a:b] = o["dH"]
    torch.cuda.synchronize()
    assert abs(tot - float(one["loss"][0])) <= 1e-5 * max(1.0, abs(tot))
    assert torch.equal(dH, one["dH"])
    assert float((dW - one["dW"]).abs().max()) <= 1e-5 * float(one["dW"].abs().max())
