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
