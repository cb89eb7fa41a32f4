"""Pins for oracle.lm_head_logp: torch fp64 log_softmax / Categorical entropy on the same bf16 inputs, the
W = 0 closed form (uniform distribution), and consistency with the loss oracle's own log-prob on the materialised logits."""
import numpy as np
import torch

import oracle


def bf16_bits(x):
    return torch.from_numpy(np.asarray(x, np.float32)).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)


def test_against_torch_fp64():
    rng = np.random.default_rng(1)
    T, d, V = 37, 64, 301
    hb, wb = bf16_bits(rng.standard_normal((T, d))), bf16_bits(rng.standard_normal((V, d)) * 0.3)
    y = rng.integers(0, V, size=T)
    logp, ent = oracle.lm_head_logp(hb, wb, y)
    H = torch.from_numpy(hb.view(np.int16)).view(torch.bfloat16).double()
    W = torch.from_numpy(wb.view(np.int16)).view(torch.bfloat16).double()
    z = H @ W.T
    ls = torch.log_softmax(z, dim=-1)
    np.testing.assert_allclose(logp, ls[torch.arange(T), torch.from_numpy(y)].numpy(), rtol=0, atol=1e-12)
    np.testing.assert_allclose(ent, torch.distributions.Categorical(logits=z).entropy().numpy(), rtol=0, atol=1e-12)


def test_zero_weights_uniform():
    T, d, V = 5, 32, 1000
    hb, wb = bf16_bits(np.ones((T, d))), bf16_bits(np.zeros((V, d)))
    logp, ent = oracle.lm_head_logp(hb, wb, np.arange(T), mask=np.array([1, 1, 0, 1, 1]))
    on = np.array([1, 1, 0, 1, 1], bool)
    np.testing.assert_allclose(logp[on], -np.log(V), atol=1e-13)
    np.testing.assert_allclose(ent[on], np.log(V), atol=1e-13)
    assert logp[2] == 0.0 and ent[2] == 0.0


def test_consistent_with_the_loss_oracle():
    # materialise the logits in fp32, hand them to the loss oracle with A = 0: its logp and entropy are the same quantities
    rng = np.random.default_rng(3)
    T, d, V = 16, 32, 200
    hb, wb = bf16_bits(rng.standard_normal((T, d))), bf16_bits(rng.standard_normal((V, d)) * 0.2)
    y = rng.integers(0, V, size=T).astype(np.int32)
    logp, ent = oracle.lm_head_logp(hb, wb, y)
    H = torch.from_numpy(hb.view(np.int16)).view(torch.bfloat16).double()
    W = torch.from_numpy(wb.view(np.int16)).view(torch.bfloat16).double()
    z32 = (H @ W.T).float().numpy()
    r = oracle.policy_loss(z32, y, np.zeros(T, np.float32), np.zeros(T, np.float32), np.ones(T, np.uint8), np.zeros(T, np.int32), 1,
                           0.2, 0.2, extended=True)
    np.testing.assert_allclose(logp, r.logp, atol=2e-6)       # fp32 rounding of the materialised logits
    np.testing.assert_allclose(ent, r.ent, atol=2e-6)


def test_rounded_logits_match_the_loss_oracle_on_stored_bf16_logits():
    # with the logits rounded to bf16 first, lm_head_logp is exactly the loss oracle's log-prob of the stored bf16 matrix
    rng = np.random.default_rng(5)
    T, d, V = 12, 64, 150
    hb, wb = bf16_bits(rng.standard_normal((T, d))), bf16_bits(rng.standard_normal((V, d)) * 0.3)
    y = rng.integers(0, V, size=T).astype(np.int32)
    logp, ent = oracle.lm_head_logp(hb, wb, y, round_logits_bf16=True)
    H = torch.from_numpy(hb.view(np.int16)).view(torch.bfloat16).double()
    W = torch.from_numpy(wb.view(np.int16)).view(torch.bfloat16).double()
    zb = bf16_bits((H @ W.T).numpy())            # torch's own fp64 -> bf16 rounding of the same products
    r = oracle.policy_loss(zb, y, np.zeros(T, np.float32), np.zeros(T, np.float32), np.ones(T, np.uint8), np.zeros(T, np.int32), 1,
                           0.2, 0.2, extended=True, logits_is_bf16_bits=True)
    np.testing.assert_allclose(logp, r.logp, atol=1e-12)
    np.testing.assert_allclose(ent, r.ent, atol=1e-12)


# ---- O-HB: loss from hidden states and its gradients w.r.t. H and W (backward half)


def _bwd_case(seed=3, T=24, d=16, V=40, S=3):
    rng = np.random.default_rng(seed)
    Hb = bf16_bits_of(rng.standard_normal((T, d)).astype(np.float32))
    Wb = bf16_bits_of((rng.standard_normal((V, d)) * 0.3).astype(np.float32))
    y = rng.integers(0, V, size=T).astype(np.int32)
    adv = rng.standard_normal(T).astype(np.float32)
    mask = (rng.random(T) < 0.8).astype(np.uint8)
    seg = rng.integers(0, S, size=T).astype(np.int32)
    return Hb, Wb, y, adv, mask, seg, S


def bf16_bits_of(x32):
    t = torch.from_numpy(np.ascontiguousarray(x32)).to(torch.bfloat16)
    return t.view(torch.int16).numpy().view(np.uint16)


def bits_to_f64(b):
    return (b.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def test_bwd_against_torch_autograd():
    # P-HB1: an independent torch fp64 graph (linear -> log_softmax -> gather -> ratio -> clamp -> minimum -> segment means)
    Hb, Wb, y, adv, mask, seg, S = _bwd_case()
    lp0, _ = oracle.lm_head_logp(Hb, Wb, y)
    old = (lp0 + np.random.default_rng(1).standard_normal(len(y)) * 0.3).astype(np.float32)
    res = oracle.lm_head_loss_bwd(Hb, Wb, y, old, adv, mask, seg, S, 0.2, 0.28)
    Ht = torch.tensor(bits_to_f64(Hb), requires_grad=True)
    Wt = torch.tensor(bits_to_f64(Wb), requires_grad=True)
    lp = torch.log_softmax(Ht @ Wt.T, dim=-1).gather(1, torch.tensor(y, dtype=torch.int64)[:, None])[:, 0]
    r = torch.exp(lp - torch.tensor(old, dtype=torch.float64))
    A = torch.tensor(adv, dtype=torch.float64)
    L = -torch.minimum(r * A, torch.clamp(r, 0.8, 1.28) * A)
    m = torch.tensor(mask, dtype=torch.float64)
    sg = torch.tensor(seg, dtype=torch.int64)
    Ns = torch.zeros(S, dtype=torch.float64).index_add_(0, sg, m)
    w = torch.where(Ns[sg] > 0, m / (Ns[sg] * (Ns > 0).sum()), torch.zeros_like(m))
    loss = (w * L).sum()
    loss.backward()
    assert abs(res["loss"] - float(loss)) < 1e-12
    assert np.abs(res["dH"] - Ht.grad.numpy()).max() < 1e-12
    assert np.abs(res["dW"] - Wt.grad.numpy()).max() < 1e-12


def test_bwd_consistent_with_the_loss_oracle_and_finite_differences():
    # P-HB2: dZ of O-HB is the dlogits of the loss oracle on the same logits (here exactly representable in fp32: small integers),
    # so dH = dlogits W and dW = dlogits^T H; P-HB3: central differences of the loss w.r.t. single entries of H and W
    rng = np.random.default_rng(5)
    T, d, V, S = 10, 4, 9, 2
    Hf = rng.integers(-2, 3, size=(T, d)).astype(np.float32)
    Wf = rng.integers(-2, 3, size=(V, d)).astype(np.float32) * 0.5
    Hb, Wb = bf16_bits_of(Hf), bf16_bits_of(Wf)
    y = rng.integers(0, V, size=T).astype(np.int32)
    adv = rng.standard_normal(T).astype(np.float32)
    mask = np.ones(T, np.uint8)
    seg = rng.integers(0, S, size=T).astype(np.int32)
    z = (Hf.astype(np.float64) @ Wf.astype(np.float64).T).astype(np.float32)     # exact
    lp0, _ = oracle.lm_head_logp(Hb, Wb, y)
    old = (lp0 + 0.05).astype(np.float32)
    res = oracle.lm_head_loss_bwd(Hb, Wb, y, old, adv, mask, seg, S, 0.2, 0.28)
    ref = oracle.policy_loss(z, y, old, adv, mask, seg, S, 0.2, 0.28)
    assert abs(res["loss"] - ref.loss) < 1e-13
    assert np.abs(res["dH"] - ref.dlogits @ Wf.astype(np.float64)).max() < 1e-13
    assert np.abs(res["dW"] - ref.dlogits.T @ Hf.astype(np.float64)).max() < 1e-13

    def loss_at(Hx, Wx):   # the oracle's own scalar on perturbed (fp64) inputs, through the loss oracle's fp32 logits is too
        zz = Hx @ Wx.T     # coarse: restate the scalar with numpy on fp64 logits
        lse = np.log(np.exp(zz - zz.max(1, keepdims=True)).sum(1)) + zz.max(1)
        lp = zz[np.arange(T), y] - lse
        r = np.exp(lp - old.astype(np.float64))
        L = -np.minimum(r * adv, np.clip(r, 0.8, 1.28) * adv)
        return float(np.sum(res["w"] * L))
    H64, W64, e = Hf.astype(np.float64), Wf.astype(np.float64), 1e-6
    for (i, j) in ((0, 0), (3, 2), (9, 3)):
        Hp, Hm = H64.copy(), H64.copy()
        Hp[i, j] += e
        Hm[i, j] -= e
        assert abs((loss_at(Hp, W64) - loss_at(Hm, W64)) / (2 * e) - res["dH"][i, j]) < 1e-7
    for (v, j) in ((0, 0), (4, 1), (8, 3)):
        Wp, Wm = W64.copy(), W64.copy()
        Wp[v, j] += e
        Wm[v, j] -= e
        assert abs((loss_at(H64, Wp) - loss_at(H64, Wm)) / (2 * e) - res["dW"][v, j]) < 1e-7


def test_bwd_rounded_operand_variant_is_close():
    # reading H-4: rounding dZ to bf16 before the two products moves every gradient entry by at most 2^-9 sum |dZ| |operand|
    Hb, Wb, y, adv, mask, seg, S = _bwd_case(seed=8, T=64, d=32, V=200)
    lp0, _ = oracle.lm_head_logp(Hb, Wb, y)
    old = (lp0 + 0.1).astype(np.float32)
    a = oracle.lm_head_loss_bwd(Hb, Wb, y, old, adv, mask, seg, S, 0.2, 0.28)
    b = oracle.lm_head_loss_bwd(Hb, Wb, y, old, adv, mask, seg, S, 0.2, 0.28, round_dz_bf16=True)
    assert a["loss"] == b["loss"]
    scale = np.abs(a["dH"]).max()
    assert 0 < np.abs(a["dH"] - b["dH"]).max() <= 2.0 ** -8 * scale * 4
