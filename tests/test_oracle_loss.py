"""Pins for the loss oracle (CPU only).  DESIGN.md pins P-L1..P-L5 and P-M4.

The oracle follows BASELINE.json north_star's sentence (the paper prints no formula: PAPER.md:91, 136, 531).
It is pinned against: torch's cross-entropy backward (library routine, special case), the clip closed form at
ratio = 1 +- eps, central finite differences, torch fp64 autograd of an independently written graph, and
invariants that hold for any input.
"""
import numpy as np
import pytest
import torch

import oracle
from helpers import seg_ids_from_merged, shift_for_next_token
from paper_2606_04484_b200 import workloads as W


def rand_case(rng, T, V, S, sigma=2.0, rho=0.7):
    z = (rng.standard_normal((T, V)) * sigma).astype(np.float32)
    y = rng.integers(0, V, size=T).astype(np.int32)
    seg = np.sort(rng.integers(0, S, size=T)).astype(np.int32)
    mask = (rng.random(T) < rho).astype(np.uint8)
    adv = rng.standard_normal(T).astype(np.float32)
    zt = torch.tensor(z, dtype=torch.float64)
    lp = torch.log_softmax(zt, -1).gather(1, torch.tensor(y, dtype=torch.int64)[:, None])[:, 0].numpy()
    old = (lp + rng.standard_normal(T) * 0.2).astype(np.float32)
    return z, y, old, adv, mask, seg


# ------------------------------------------------------------------ P-L1 library special case


def test_reduces_to_mean_cross_entropy():
    rng = np.random.default_rng(0)
    T, V = 13, 37
    z = (rng.standard_normal((T, V)) * 2).astype(np.float32)
    y = rng.integers(0, V, size=T).astype(np.int32)
    zt = torch.tensor(z, dtype=torch.float64, requires_grad=True)
    ce = torch.nn.functional.cross_entropy(zt, torch.tensor(y, dtype=torch.int64), reduction="mean")
    ce.backward()
    lp = -torch.nn.functional.cross_entropy(zt.detach(), torch.tensor(y, dtype=torch.int64), reduction="none").numpy()
    # A = +1, old_logp = logp (r = 1), all masks 1, one segment  =>  loss = -1, dlogits = d(mean CE)/dz
    old = lp.astype(np.float32)
    r = oracle.policy_loss(z, y, old, np.ones(T, np.float32), np.ones(T, np.uint8), np.zeros(T, np.int32), 1, 0.2, 0.2)
    # old_logp is stored in fp32, so r = exp(logp - fl32(logp)) = 1 + O(1e-7)
    assert abs(r.loss - (-1.0)) < 1e-6
    np.testing.assert_allclose(r.logp, lp, rtol=0, atol=1e-12)
    ratio = np.exp(r.logp - old.astype(np.float64))
    np.testing.assert_allclose(r.dlogits, zt.grad.numpy() * ratio[:, None], rtol=1e-12, atol=1e-15)
    np.testing.assert_allclose(r.dlogits, zt.grad.numpy(), rtol=1e-6, atol=1e-9)
    # sign: the gradient pushes the target logit up for positive advantage
    assert np.all(r.dlogits[np.arange(T), y] < 0)


# ------------------------------------------------------------------ P-L2 clip closed form at ratio = 1 +- eps


@pytest.mark.parametrize("eps_lo,eps_hi", [(0.2, 0.2), (0.2, 0.28)])
def test_clip_closed_form(eps_lo, eps_hi):
    rng = np.random.default_rng(1)
    V = 11
    d = 1e-3
    rstars = [1 - eps_lo - d, 1 - eps_lo + d, 1 + eps_hi - d, 1 + eps_hi + d, 1.0]
    rows = [(rs, A) for rs in rstars for A in (+1.5, -0.5)]
    T = len(rows)
    z = (rng.standard_normal((T, V)) * 2).astype(np.float32)
    y = rng.integers(0, V, size=T).astype(np.int32)
    lp = torch.log_softmax(torch.tensor(z, dtype=torch.float64), -1).numpy()[np.arange(T), y]
    old = np.array([lp[i] - np.log(rs) for i, (rs, _) in enumerate(rows)]).astype(np.float32)
    adv = np.array([A for _, A in rows], np.float32)
    # one token per segment so w_t = 1/T and L_t can be read back
    res = oracle.policy_loss(z, y, old, adv, np.ones(T, np.uint8), np.arange(T, dtype=np.int32), T, eps_lo, eps_hi)
    for i, (rs, A) in enumerate(rows):
        rr = np.exp(lp[i] - float(old[i]))          # the ratio the oracle sees (old is fp32-rounded)
        assert abs(rr - rs) < 1e-6
        want = -A * min(rr, 1 + eps_hi) if A >= 0 else -A * max(rr, 1 - eps_lo)   # closed form
        assert abs(res.Lt[i] - want) < 1e-12
        clipped = (A > 0 and rs > 1 + eps_hi) or (A < 0 and rs < 1 - eps_lo)      # exactly two quadrants
        if clipped:
            assert res.g[i] == 0.0 and np.all(res.dlogits[i] == 0.0)
        else:
            assert abs(res.g[i] - (1.0 / T) * (-A * rr)) < 1e-12
            assert np.any(res.dlogits[i] != 0.0)
    assert abs(res.loss - res.Lt.mean()) < 1e-12
    n_hi = sum(1 for rs, A in rows if A > 0 and rs > 1 + eps_hi)
    n_lo = sum(1 for rs, A in rows if A < 0 and rs < 1 - eps_lo)
    assert res.stats[0] == T and res.stats[1] == n_hi == 1 and res.stats[2] == n_lo == 1


def test_zero_advantage_and_boundary():
    rng = np.random.default_rng(2)
    z, y, old, adv, mask, seg = rand_case(rng, 6, 9, 2)
    adv[:] = 0
    res = oracle.policy_loss(z, y, old, adv, np.ones(6, np.uint8), seg, 2, 0.2, 0.2)
    assert res.loss == 0.0 and np.all(res.dlogits == 0.0)      # reading L-5


# ------------------------------------------------------------------ P-L3 finite differences


def test_finite_differences():
    rng = np.random.default_rng(3)
    for trial in range(6):
        T, V, S = 6, 12, 3
        z, y, old, adv, mask, seg = rand_case(rng, T, V, S)
        mask[:2] = 1
        base = oracle.policy_loss(z, y, old, adv, mask, seg, S, 0.2, 0.28, grad_scale=1.0)
        # stay away from the clip kinks
        ratio = np.exp(base.logp - old)
        if np.any(np.abs(ratio - 0.8) < 1e-2) or np.any(np.abs(ratio - 1.28) < 1e-2):
            continue
        h = 2.0 ** -7   # exactly representable step on fp32 logits
        fd = np.zeros((T, V))
        for t in range(T):
            for v in range(V):
                zp = z.copy(); zp[t, v] += h
                zm = z.copy(); zm[t, v] -= h
                lp_ = oracle.policy_loss(zp, y, old, adv, mask, seg, S, 0.2, 0.28, want_dlogits=False).loss
                lm_ = oracle.policy_loss(zm, y, old, adv, mask, seg, S, 0.2, 0.28, want_dlogits=False).loss
                fd[t, v] = (lp_ - lm_) / (2 * h)
        np.testing.assert_allclose(base.dlogits, fd, rtol=2e-3, atol=2e-5)


# ------------------------------------------------------------------ P-L4 torch fp64 autograd, written independently


def torch_loss(z, y, old, adv, mask, seg, S, eps_lo, eps_hi, seg_denom=None, inv_num_segs=0.0):
    zt = torch.tensor(z, dtype=torch.float64, requires_grad=True)
    lp = torch.log_softmax(zt, dim=-1).gather(1, torch.tensor(y, dtype=torch.int64)[:, None]).squeeze(1)
    ratio = torch.exp(lp - torch.tensor(old, dtype=torch.float64))
    A = torch.tensor(adv, dtype=torch.float64)
    surr = torch.minimum(ratio * A, torch.clamp(ratio, 1 - eps_lo, 1 + eps_hi) * A)
    m = torch.tensor(mask, dtype=torch.float64)
    sg = torch.tensor(seg, dtype=torch.int64)
    Ns = torch.zeros(S, dtype=torch.float64).index_add_(0, sg, m)
    if seg_denom is not None:
        Ns = torch.tensor(seg_denom, dtype=torch.float64)
    num = torch.zeros(S, dtype=torch.float64).index_add(0, sg, -surr * m)
    live = Ns > 0
    per_seg = num[live] / Ns[live]
    loss = per_seg.sum() * inv_num_segs if inv_num_segs else (per_seg.mean() if live.any() else zt.sum() * 0)
    loss.backward()
    return float(loss.detach()), zt.grad.numpy(), lp.detach().numpy()


@pytest.mark.parametrize("T,V,S", [(5, 7, 1), (40, 33, 4), (64, 257, 9)])
def test_against_torch_autograd(T, V, S):
    rng = np.random.default_rng(T * V)
    z, y, old, adv, mask, seg = rand_case(rng, T, V, S)
    if S > 3:
        mask[seg == 1] = 0        # a trajectory with no masked token is dropped from numerator and count (L-3)
    want_loss, want_grad, want_lp = torch_loss(z, y, old, adv, mask, seg, S, 0.2, 0.28)
    r = oracle.policy_loss(z, y, old, adv, mask, seg, S, 0.2, 0.28)
    assert abs(r.loss - want_loss) < 1e-13
    np.testing.assert_allclose(r.dlogits, want_grad, rtol=1e-10, atol=1e-16)
    np.testing.assert_allclose(r.logp[mask == 1], want_lp[mask == 1], rtol=0, atol=1e-12)
    r2 = oracle.policy_loss(z, y, old, adv, mask, seg, S, 0.2, 0.28, grad_scale=37.5)
    np.testing.assert_allclose(r2.dlogits, 37.5 * want_grad, rtol=1e-10, atol=1e-15)


def test_bf16_input_is_read_exactly():
    rng = np.random.default_rng(5)
    T, V, S = 9, 64, 2
    z, y, old, adv, mask, seg = rand_case(rng, T, V, S, sigma=3.0)
    zb = torch.tensor(z).to(torch.bfloat16)
    bits = zb.view(torch.int16).numpy().view(np.uint16)
    a = oracle.policy_loss(bits, y, old, adv, mask, seg, S, 0.2, 0.2, logits_is_bf16_bits=True)
    b = oracle.policy_loss(zb.to(torch.float32).numpy(), y, old, adv, mask, seg, S, 0.2, 0.2)
    assert a.loss == b.loss and np.array_equal(a.dlogits, b.dlogits)


def test_round_bf16_matches_library():
    rng = np.random.default_rng(6)
    x = np.concatenate([rng.standard_normal(5000) * 10.0 ** rng.integers(-12, 3, size=5000),
                        [0.0, 1.0, 1.00390625, 1.01171875, -1.00390625, 2.0 ** -130, 3.0 * 2.0 ** -134]])
    want = torch.tensor(x, dtype=torch.float64).to(torch.float32)   # go via fp32 only where exact
    exact32 = want.to(torch.float64).numpy() == x
    got = oracle.round_bf16(x)
    lib = torch.tensor(x[exact32], dtype=torch.float32).to(torch.bfloat16).to(torch.float64).numpy()
    assert np.array_equal(got[exact32], lib)
    # ties to even on hand-picked points: 1 + 2^-8 is halfway between 1 and 1 + 2^-7 -> 1 ; 1 + 3*2^-8 -> 1 + 2^-6
    assert oracle.round_bf16(np.array([1.00390625]))[0] == 1.0
    assert oracle.round_bf16(np.array([1.01171875]))[0] == 1.015625
    err = np.abs(got - x)
    nz = np.abs(x) > 1e-30
    assert np.all(err[nz] <= np.abs(x[nz]) * 2.0 ** -8)


# ------------------------------------------------------------------ P-L5 invariants


def test_invariants():
    rng = np.random.default_rng(8)
    T, V, S = 48, 50, 5
    z, y, old, adv, mask, seg = rand_case(rng, T, V, S)
    z = (np.round(z * 1024) / 1024).astype(np.float32)          # so that z + 4 is exact in fp32
    r = oracle.policy_loss(z, y, old, adv, mask, seg, S, 0.2, 0.28)
    assert np.all(np.abs(r.dlogits.sum(1)) < 1e-15)             # rows sum to zero
    assert np.all(r.dlogits[mask == 0] == 0.0)                   # masked rows exactly zero
    assert np.all(r.logp[mask == 0] == 0.0)
    # shift invariance (power-of-two shift is exact in fp32)
    z2 = z.copy(); z2[::2] += 4.0
    r2 = oracle.policy_loss(z2, y, old, adv, mask, seg, S, 0.2, 0.28)
    assert abs(r2.loss - r.loss) < 1e-13
    np.testing.assert_allclose(r2.dlogits, r.dlogits, rtol=1e-9, atol=1e-16)
    # uniform row: logp = -log V, p = 1/V
    zu = np.zeros((T, V), np.float32)
    ru = oracle.policy_loss(zu, y, np.full(T, -np.log(V), np.float32), np.ones(T, np.float32),
                            np.ones(T, np.uint8), np.zeros(T, np.int32), 1, 0.2, 0.2)
    np.testing.assert_allclose(ru.logp, -np.log(V), rtol=0, atol=1e-14)
    offdiag = ru.dlogits.copy(); offdiag[np.arange(T), y] = np.nan
    np.testing.assert_allclose(offdiag[~np.isnan(offdiag)], ru.g[0] * (-1.0 / V), rtol=1e-12)
    # permuting tokens leaves the loss unchanged, permutes dlogits
    perm = rng.permutation(T)
    rp = oracle.policy_loss(z[perm], y[perm], old[perm], adv[perm], mask[perm], seg[perm], S, 0.2, 0.28)
    assert abs(rp.loss - r.loss) < 1e-14
    np.testing.assert_allclose(rp.dlogits, r.dlogits[perm], rtol=1e-12, atol=1e-18)
    # weights: sum over tokens of w_t = 1 when some segment is live
    assert abs(r.w[mask == 1].sum() - 1.0) < 1e-12


def test_chunked_equals_unchunked():
    # reading L-4: batch-wide seg_denom + inv_num_segs; each chunk returns its partial sum
    rng = np.random.default_rng(9)
    T, V, S = 60, 21, 6
    z, y, old, adv, mask, seg = rand_case(rng, T, V, S)
    full = oracle.policy_loss(z, y, old, adv, mask, seg, S, 0.2, 0.28)
    Ns = np.bincount(seg[mask == 1], minlength=S).astype(np.float32)
    inv = 1.0 / float((Ns > 0).sum())
    tot, parts = 0.0, []
    for a in range(0, T, 17):
        b = min(T, a + 17)
        c = oracle.policy_loss(z[a:b], y[a:b], old[a:b], adv[a:b], mask[a:b], seg[a:b], S, 0.2, 0.28,
                               seg_denom=Ns, inv_num_segs=inv)
        tot += c.loss
        parts.append(c.dlogits)
    assert abs(tot - full.loss) < 1e-14
    np.testing.assert_allclose(np.concatenate(parts), full.dlogits, rtol=1e-12, atol=1e-18)
    # row subset API = same rows of the full call
    rows = np.array([3, 17, 18, 59], np.int64)
    sub = oracle.policy_loss(z[rows], y, old, adv, mask, seg, S, 0.2, 0.28, row_ids=rows)
    np.testing.assert_array_equal(sub.dlogits, full.dlogits[rows])
    np.testing.assert_array_equal(sub.logp, full.logp[rows])


def test_no_live_segment():
    rng = np.random.default_rng(10)
    z, y, old, adv, mask, seg = rand_case(rng, 7, 5, 2)
    r = oracle.policy_loss(z, y, old, adv, np.zeros(7, np.uint8), seg, 2, 0.2, 0.2)
    assert r.loss == 0.0 and np.all(r.dlogits == 0.0)


def test_out_of_range_target_rejected():
    rng = np.random.default_rng(11)
    z, y, old, adv, mask, seg = rand_case(rng, 7, 5, 2)
    mask[:] = 1
    y[3] = 5
    with pytest.raises(ValueError):
        oracle.policy_loss(z, y, old, adv, mask, seg, 2, 0.2, 0.2)


# ------------------------------------------------------------------ P-M4 loss over merged == loss over unmerged


@pytest.mark.parametrize("rule", [oracle.OWNER_LONGEST, oracle.OWNER_PAPER])
def test_loss_merged_equals_unmerged(rule):
    mi = W.merge_workload("c1", n_traj=6)
    r = oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp, rule)
    V = 24
    rng = np.random.default_rng(12)
    # one logits row per MERGED token; targets = the token itself folded into V; adv per trajectory
    zm = (rng.standard_normal((r.N_out, V)) * 2).astype(np.float32)
    seg_m, S, uniq = seg_ids_from_merged(r.merged_offsets, r.merged_traj)
    adv_traj = rng.standard_normal(S).astype(np.float32)
    ym = (r.merged_tokens % V).astype(np.int32)
    # give the merged old_logp values a plausible scale: old = (random row logp) - handled by using carried values
    lm = oracle.policy_loss(zm, ym, r.merged_old_logp, adv_traj[seg_m], r.merged_mask, seg_m, S, 0.2, 0.28)
    # unmerged layout through the index map: timeline j, position p  <-  merged row merged_offsets[owner[j]] + p
    rows = np.concatenate([r.merged_offsets[r.owner[j]] + np.arange(mi.offsets[j + 1] - mi.offsets[j])
                           for j in range(mi.n)])
    zu = zm[rows]
    yu = (mi.tokens % V).astype(np.int32)
    mask_u = W.explicit_mask(mi)
    traj_to_seg = {int(t): i for i, t in enumerate(uniq)}
    seg_u = np.repeat(np.array([traj_to_seg[int(t)] for t in mi.traj_ids], np.int32), np.diff(mi.offsets))
    lu = oracle.policy_loss(zu, yu, mi.old_logp, adv_traj[seg_u], mask_u, seg_u, S, 0.2, 0.28)
    assert lm.stats[0] == lu.stats[0] == mask_u.sum() == r.merged_mask.sum()   # every response token once
    assert abs(lm.loss - lu.loss) < 1e-12 * max(1.0, abs(lu.loss))
    # and the gradient scattered back through the index map agrees
    gm = np.zeros_like(lm.dlogits)
    np.add.at(gm, rows, lu.dlogits)
    np.testing.assert_allclose(gm, lm.dlogits, rtol=1e-9, atol=1e-15)


# ------------------------------------------------------------------ P-L6..P-L8: steps 8-9 (KL vs reference policy, entropy)


def test_k3_closed_forms():
    """Step 8 (PAPER.md:531 `low_var_kl`, reading L-16): k3(d) = exp(d) - d - 1 with d = ref_logp - logp, clamped at 10."""
    V, T = 7, 5
    z = np.zeros((T, V), np.float32)                    # uniform rows: logp = -log V exactly representable enough
    y = np.arange(T, dtype=np.int32) % V
    lp = -np.log(V)
    ds = np.array([0.0, np.log(2.0), -1.0, 1e-3, 3.0])   # k3: 0, 1 - log 2, e^-1, ~d^2/2, clamped (e^3 - 4 = 16.09 > 10)
    ref = (lp + ds).astype(np.float32)
    old = np.full(T, lp, np.float32)
    r = oracle.policy_loss(z, y, old, np.zeros(T, np.float32), np.ones(T, np.uint8), np.zeros(T, np.int32), 1, 0.2, 0.2,
                           ref_logp=ref, kl_coef=1.0)
    d = ref.astype(np.float64) - r.logp
    np.testing.assert_allclose(r.k3[0], 0.0, atol=1e-7)
    np.testing.assert_allclose(r.k3[1], 1.0 - np.log(2.0), atol=1e-6)
    np.testing.assert_allclose(r.k3[2], np.exp(-1.0), atol=1e-6)
    np.testing.assert_allclose(r.k3[3], d[3] ** 2 / 2, rtol=1e-3)
    assert r.k3[4] == 10.0
    assert np.all(r.k3 >= 0)
    # A = 0: the loss is the KL term alone, = kl_coef * mean over the segment's tokens
    np.testing.assert_allclose(r.loss, r.k3.mean(), rtol=1e-12)
    np.testing.assert_allclose(r.ext[0], r.k3.mean(), rtol=1e-12)
    # the clamped token has no KL gradient (A = 0 kills the policy-gradient part): its dlogits row is zero
    assert np.all(r.dlogits[4] == 0.0) and np.any(r.dlogits[1] != 0.0)


def test_k3_is_unbiased_for_kl():
    """E_{y~pi} k3(y) = KL(pi || pi_ref) exactly (sum_y pi_y [pi_ref_y/pi_y - log(pi_ref_y/pi_y) - 1] = KL): enumerate y."""
    from scipy.special import rel_entr
    rng = np.random.default_rng(21)
    V = 9
    z = rng.standard_normal(V).astype(np.float32)
    zr = (z + 0.3 * rng.standard_normal(V)).astype(np.float32)
    pi = torch.softmax(torch.tensor(z, dtype=torch.float64), -1).numpy()
    pr = torch.softmax(torch.tensor(zr, dtype=torch.float64), -1).numpy()
    logits = np.tile(z, (V, 1))                          # one row per possible target
    y = np.arange(V, dtype=np.int32)
    ref = np.log(pr).astype(np.float32)
    r = oracle.policy_loss(logits, y, np.log(pi).astype(np.float32), np.zeros(V, np.float32), np.ones(V, np.uint8),
                           np.zeros(V, np.int32), 1, 0.2, 0.2, ref_logp=ref, kl_coef=1.0)
    kl = rel_entr(pi, pr).sum()
    np.testing.assert_allclose((pi * r.k3).sum(), kl, rtol=2e-6)   # ref_logp is stored in fp32


def test_entropy_matches_library():
    """Step 9: H = lse - sum_v p_v z_v = -sum_v p_v log p_v (torch.distributions / scipy), uniform row -> log V."""
    from scipy.stats import entropy as sp_entropy
    rng = np.random.default_rng(22)
    T, V = 6, 33
    z = (rng.standard_normal((T, V)) * 3).astype(np.float32)
    z[0] = 1.25
    y = rng.integers(0, V, T).astype(np.int32)
    r = oracle.policy_loss(z, y, np.full(T, -3.0, np.float32), np.ones(T, np.float32), np.ones(T, np.uint8),
                           np.zeros(T, np.int32), 1, 0.2, 0.2, extended=True)
    H = torch.distributions.Categorical(logits=torch.tensor(z, dtype=torch.float64)).entropy().numpy()
    np.testing.assert_allclose(r.ent, H, rtol=1e-12, atol=1e-12)
    p = torch.softmax(torch.tensor(z, dtype=torch.float64), -1).numpy()
    np.testing.assert_allclose(r.ent, [sp_entropy(row) for row in p], rtol=1e-10)
    np.testing.assert_allclose(r.ent[0], np.log(V), rtol=1e-12)
    np.testing.assert_allclose(r.ext[1], H.mean(), rtol=1e-12)
    # steps 1-7 are untouched by the extended entry point when kl_coef = 0
    r0 = oracle.policy_loss(z, y, np.full(T, -3.0, np.float32), np.ones(T, np.float32), np.ones(T, np.uint8),
                            np.zeros(T, np.int32), 1, 0.2, 0.2)
    assert r.loss == r0.loss and np.array_equal(r.dlogits, r0.dlogits)


@pytest.mark.parametrize("T,V,S", [(9, 14, 3), (20, 40, 4)])
def test_extended_against_torch_autograd(T, V, S):
    """Whole extended definition (steps 1-8) vs an independently written torch fp64 graph."""
    rng = np.random.default_rng(23 + T)
    z, y, old, adv, mask, seg = rand_case(rng, T, V, S)
    ref = (old + rng.standard_normal(T) * 0.3).astype(np.float32)
    kl_coef, eps_lo, eps_hi = 0.37, 0.2, 0.28
    zt = torch.tensor(z, dtype=torch.float64, requires_grad=True)
    lp = torch.log_softmax(zt, -1).gather(1, torch.tensor(y, dtype=torch.int64)[:, None])[:, 0]
    ratio = torch.exp(lp - torch.tensor(old, dtype=torch.float64))
    A = torch.tensor(adv, dtype=torch.float64)
    pg = -torch.minimum(ratio * A, torch.clamp(ratio, 1 - eps_lo, 1 + eps_hi) * A)
    d = torch.tensor(ref, dtype=torch.float64) - lp
    k3 = torch.clamp(torch.exp(d) - d - 1, max=10.0)
    m = torch.tensor(mask, dtype=torch.float64)
    total = torch.zeros((), dtype=torch.float64)
    live = 0
    for s_ in range(S):
        sel = torch.tensor(seg == s_, dtype=torch.float64) * m
        if sel.sum() > 0:
            total = total + ((pg + kl_coef * k3) * sel).sum() / sel.sum()
            live += 1
    total = total / max(live, 1)
    total.backward()
    r = oracle.policy_loss(z, y, old, adv, mask, seg, S, eps_lo, eps_hi, ref_logp=ref, kl_coef=kl_coef)
    np.testing.assert_allclose(r.loss, float(total), rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(r.dlogits, zt.grad.numpy(), rtol=1e-9, atol=1e-14)


# ---- step 3b: the three-parameter dual-clip bound c (reading L-18)


def _dual_clip_case(rstar, A, c, eps=(0.2, 0.28)):
    """One token, one segment, ratio set exactly: old_logp = logp - log r*."""
    V = 7
    z = np.linspace(-1.0, 1.5, V).astype(np.float32)[None, :]
    y = np.array([3], np.int32)
    lse = np.log(np.exp(z.astype(np.float64)).sum())
    logp = float(z[0, 3]) - lse
    old = np.array([logp - np.log(rstar)], np.float32)
    return oracle.policy_loss(z, y, old, np.array([A], np.float32), np.ones(1, np.uint8), np.zeros(1, np.int32), 1, eps[0], eps[1],
                              clip_c=c), float(np.exp(logp - float(old[0])))


def test_dual_clip_closed_form():
    # P-L10: for A < 0 the loss is -A min(max(r, 1 - eps_lo), c); the gradient vanishes exactly where r > c (and where r < 1 - eps_lo);
    # for A >= 0 the bound changes nothing
    c = 3.0
    for rstar in (0.5, 0.9, 1.5, 2.9, 3.1, 6.0):
        res, r = _dual_clip_case(rstar, -2.0, c)
        assert abs(res.Lt[0] - 2.0 * min(max(r, 0.8), c)) < 1e-12
        assert (res.g[0] == 0.0) == (r > c or r < 0.8)
        plain, _ = _dual_clip_case(rstar, -2.0, 0.0)
        if r <= c:
            assert res.Lt[0] == plain.Lt[0] and res.g[0] == plain.g[0]
        pos, _ = _dual_clip_case(rstar, 2.0, c)
        pos0, _ = _dual_clip_case(rstar, 2.0, 0.0)
        assert pos.Lt[0] == pos0.Lt[0] and pos.g[0] == pos0.g[0]


def test_dual_clip_against_torch_autograd():
    # P-L11: an independent torch fp64 graph of the published form: max(-A r, -A clip(r)) capped by -A c where A < 0
    rng = np.random.default_rng(12)
    T, V, S, c = 40, 11, 3, 2.5
    z = rng.standard_normal((T, V)).astype(np.float32) * 2
    y = rng.integers(0, V, size=T).astype(np.int32)
    adv = rng.standard_normal(T).astype(np.float32)
    mask = (rng.random(T) < 0.8).astype(np.uint8)
    seg = rng.integers(0, S, size=T).astype(np.int32)
    zt = torch.tensor(z, dtype=torch.float64, requires_grad=True)
    lp = torch.log_softmax(zt, dim=-1).gather(1, torch.tensor(y, dtype=torch.int64)[:, None])[:, 0]
    old = (lp.detach().numpy() + rng.standard_normal(T) * 0.8).astype(np.float32)     # wide ratios: the cap fires
    r = torch.exp(lp - torch.tensor(old, dtype=torch.float64))
    A = torch.tensor(adv, dtype=torch.float64)
    l1 = torch.maximum(-A * r, -A * torch.clamp(r, 1 - 0.2, 1 + 0.28))
    l = torch.where(A < 0, torch.minimum(l1, -A * c), l1)
    m = torch.tensor(mask, dtype=torch.float64)
    sg = torch.tensor(seg, dtype=torch.int64)
    Ns = torch.zeros(S, dtype=torch.float64).index_add_(0, sg, m)
    live = (Ns > 0).sum()
    w = torch.where(Ns[sg] > 0, m / (Ns[sg] * live), torch.zeros_like(m))
    loss = (w * l).sum()
    loss.backward()
    res = oracle.policy_loss(z, y, old, adv, mask, seg, S, 0.2, 0.28, clip_c=c)
    assert abs(res.loss - float(loss)) < 1e-12
    assert np.abs(res.dlogits - zt.grad.numpy()).max() < 1e-12
    assert (np.exp(res.logp - old) > c)[(adv < 0) & (mask > 0)].any()      # the case is exercised
