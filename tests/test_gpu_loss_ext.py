"""GPU parity: ajt_policy_loss_fwd_bwd_ext (steps 8-9: low_var_kl term against reference log-probs, row entropy;
PAPER.md:136, 469, 531; readings L-16, L-17) through the C ABI vs the fp64 oracle, element by element.

Every kernel variant of the extended form (fast 1-CTA NCH=8/16, 2-CTA cluster, generic fp32 / odd V), the clamp of k3,
KL switched off, and bit-identity of the shared outputs with the plain call.
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_04484_b200 as ajt
from paper_2606_04484_b200 import workloads as W
from helpers import check_loss, logits_to_oracle
from test_gpu_loss import make_case

pytestmark = pytest.mark.gpu


def ref_logp_for(old: torch.Tensor, seed: int, mask=None, sigma=0.1, n_far=3):
    """INPUT synthesis: reference-policy log-probs = the behaviour log-probs + N(0, sigma); a few rows pushed far away so
    that k3 exceeds its clamp of 10."""
    rng = W.rng_for(seed, 77)
    T = old.numel()
    ref = old.cpu().numpy() + (rng.standard_normal(T) * sigma).astype(np.float32)
    on = np.arange(T) if mask is None else np.nonzero(mask)[0]
    if on.size > 8 and n_far:
        ref[rng.choice(on, size=n_far, replace=False)] += 5.0    # exp(5) - 5 - 1 = 142 > 10
    return ref.astype(np.float32)


def check_ext(out, ref, mask, kl_coef, old_np):
    m = mask != 0
    k3 = out.k3.cpu().numpy().astype(np.float64)[:mask.size]
    H = out.ent.cpu().numpy().astype(np.float64)[:mask.size]
    assert np.all(k3[~m] == 0.0) and np.all(H[~m] == 0.0)
    # k3 = exp(d) - d - 1 with d = ref_logp - logp: |dk3| <= |exp(d) - 1| |dd| + fp32 rounding of the evaluation;
    # |dd| is the logp tolerance of check_loss (2e-6 max(1, |logp|)), doubled
    lp = ref.logp
    scale = np.maximum(1.0, np.abs(lp))
    unclamped = ref.k3 < 10.0
    # slope bound without inverting k3: |exp(d) - 1| <= sqrt(2 k3) + k3 for every d  (d > 0: exp(d) - 1 = k3 + d and
    # k3 >= d^2 / 2;  d < 0: with u = 1 - exp(d), -d = -ln(1 - u) >= u + u^2 / 2, so 2 k3 = 2 (-d - u) >= u^2)
    slope = np.sqrt(2.0 * ref.k3) + ref.k3
    tol = 4e-6 * scale * slope + 4e-7 * (ref.k3 + slope) + 1e-12
    e = np.abs(k3 - ref.k3)
    ok = m & unclamped & (np.abs(ref.k3 - 10.0) > 1e-3)
    assert np.all(e[ok] <= tol[ok]), (e[ok] - tol[ok]).max()
    assert np.all(k3[m & ~unclamped] == 10.0)
    # H = lse - sum p z in fp32 over V terms (pairwise / per-thread partial sums): 1e-5 relative to max(1, H)
    eh = np.abs(H - ref.ent)
    assert np.all(eh[m] <= 1e-5 * np.maximum(1.0, np.abs(ref.ent[m]))), eh[m].max()
    ext = out.ext.cpu().numpy().astype(np.float64)
    assert abs(ext[0] - ref.ext[0]) <= 1e-5 * max(ref.ext[0], 1e-6) + float(np.sum(ref.w * np.where(m, tol, 0.0)))
    assert abs(ext[1] - ref.ext[1]) <= 1e-5 * max(abs(ref.ext[1]), 1e-6)
    # scalar: sum w (L + kl_coef k3); scale = sum w (|L| + kl_coef k3) (reading L-8)
    l1 = float(np.sum(ref.w * (np.abs(ref.Lt) + kl_coef * ref.k3)))
    loss = float(out.loss.cpu()[0])
    assert abs(loss - ref.loss) <= 1e-5 * l1 + 1e-7 * abs(ref.loss) + 1e-30, (loss, ref.loss, l1)


def run_ext(T, V, S, rho, dtype, kl_coef=0.37, sigma=3.0, eps=(0.2, 0.28), seed=1, with_ref=True, grad_scale=1.0):
    lv, logits, targets, old, adv, mask, seg = make_case(T, V, S, rho, dtype, sigma, seed)
    zo, is_bits = logits_to_oracle(logits[:, :V])
    refp = ref_logp_for(old, seed, lv.mask) if with_ref else None
    out = ajt.policy_loss_fwd_bwd_ext(logits, targets, old, adv, mask, seg, lv.S, eps[0], eps[1],
                                      ref_logp=torch.from_numpy(refp).cuda() if with_ref else None, kl_coef=kl_coef,
                                      grad_scale=grad_scale, V=V, want_logp=True, want_stats=True)
    torch.cuda.synchronize()
    assert ajt.last_status(out.workspace) == 0
    ref = oracle.policy_loss(zo, lv.targets, old.cpu().numpy(), lv.adv, lv.mask, lv.seg_ids, lv.S,
                             float(np.float32(eps[0])), float(np.float32(eps[1])), grad_scale=grad_scale,
                             logits_is_bf16_bits=is_bits, ref_logp=refp, kl_coef=float(np.float32(kl_coef)), extended=True)
    # dlogits (with the KL gradient inside g_t), logp and stats: the rules of the plain call
    check_loss(out, ref, lv.mask, eps[0], eps[1], lv.adv, old.cpu().numpy(), grad_scale, V, check_scalar=False)
    check_ext(out, ref, lv.mask, float(np.float32(kl_coef)) if with_ref else 0.0, old.cpu().numpy())
    st = out.stats.cpu().numpy().astype(np.float64)
    assert st[0] == ref.stats[0]
    return lv, (logits, targets, old, adv, mask, seg), out, ref


@pytest.mark.parametrize("T,V,S,rho", [
    (600, 32000, 8, 0.7),        # fast, 1 CTA per row, NCH = 8
    (300, 77824, 3, 0.7),        # fast, 1 CTA, NCH = 16, exactly 16 full chunks
    (400, 128256, 8, 0.7),       # fast, 2-CTA cluster
    (400, 151936, 8, 0.3),       # fast, 2-CTA cluster, headline vocabulary, ragged tail chunk
])
def test_ext_fast_path(T, V, S, rho):
    _, _, out, ref = run_ext(T, V, S, rho, torch.bfloat16)
    assert (ref.k3 >= 10.0).sum() >= 1          # the clamp branch is exercised
    assert ref.ext[0] > 0 and ref.ext[1] > 0


@pytest.mark.parametrize("T,V,S,rho,dtype", [
    (3000, 1024, 32, 0.45, torch.float32),    # c1's shape: fp32 logits, one-read register kernel
    (500, 2048, 6, 0.6, torch.float32),       # one-read register kernel, 16 vectors per lane
    (300, 1002, 4, 0.7, torch.float32),       # fp32 generic, warp per row
    (300, 5000, 4, 0.7, torch.float32),       # fp32, CTA-per-row generic
    (200, 151937, 4, 0.7, torch.bfloat16),    # odd V -> generic
])
def test_ext_generic_path(T, V, S, rho, dtype):
    run_ext(T, V, S, rho, dtype, sigma=2.0 if dtype == torch.float32 else 3.0)


def test_ext_protocol_coefficient():
    # the protocol's own constants: kl_loss_coef = 2e-3, clip_ratio = 0.2
    run_ext(400, 151936, 8, 0.7, torch.bfloat16, kl_coef=2e-3, eps=(0.2, 0.2), seed=4)


def test_ext_without_reference_is_the_plain_call():
    # ref_logp = NULL (or kl_coef = 0): k3 = 0 and loss, dlogits, logp, stats are bit-identical to ajt_policy_loss_fwd_bwd
    for V, dtype in ((151936, torch.bfloat16), (32000, torch.bfloat16), (1024, torch.float32)):
        lv, args, out, ref = run_ext(300, V, 4, 0.6, dtype, with_ref=False, seed=6, sigma=2.0)
        logits, targets, old, adv, mask, seg = args
        plain = ajt.policy_loss_fwd_bwd(logits, targets, old, adv, mask, seg, lv.S, 0.2, 0.28, want_logp=True, want_stats=True)
        torch.cuda.synchronize()
        assert torch.equal(plain.dlogits, out.dlogits) and torch.equal(plain.loss, out.loss)
        assert torch.equal(plain.logp, out.logp) and torch.equal(plain.stats, out.stats)
        assert torch.all(out.k3 == 0) and float(out.ext[0]) == 0.0
        refp = torch.from_numpy(ref_logp_for(old, 6)).cuda()
        zero = ajt.policy_loss_fwd_bwd_ext(logits, targets, old, adv, mask, seg, lv.S, 0.2, 0.28, ref_logp=refp, kl_coef=0.0)
        torch.cuda.synchronize()
        assert torch.equal(zero.dlogits, plain.dlogits) and torch.equal(zero.loss, plain.loss)


def test_ext_uniform_row_entropy_and_zero_kl():
    # closed forms through the CUDA path: a constant row has H = log V exactly; ref_logp = logp gives k3 = 0 and no KL
    # gradient, so dlogits equal the plain call's
    T, V = 64, 32000
    logits = torch.full((T, V), 1.25, dtype=torch.bfloat16, device="cuda")
    targets = torch.arange(T, dtype=torch.int32, device="cuda")
    old = torch.full((T,), -float(np.log(V)), device="cuda")
    adv = torch.ones(T, device="cuda")
    mask = torch.ones(T, dtype=torch.uint8, device="cuda")
    seg = torch.zeros(T, dtype=torch.int32, device="cuda")
    out = ajt.policy_loss_fwd_bwd_ext(logits, targets, old, adv, mask, seg, 1, 0.2, 0.2, ref_logp=old.clone(), kl_coef=1.0,
                                      want_logp=True)
    torch.cuda.synchronize()
    assert torch.allclose(out.ent, torch.full_like(out.ent, float(np.log(V))), rtol=0, atol=2e-6 * np.log(V))
    assert float(out.k3.abs().max()) <= 1e-10
    assert abs(float(out.ext[1]) - np.log(V)) <= 2e-6 * np.log(V)


def test_ext_argument_errors():
    lv, logits, targets, old, adv, mask, seg = make_case(8, 32000, 2, 1.0, torch.bfloat16, 3.0, 3)
    with pytest.raises(ajt.AjtError):
        ajt.policy_loss_fwd_bwd_ext(logits, targets, old, adv, mask, seg, lv.S, 0.2, 0.2, ref_logp=old, kl_coef=-1.0)


@pytest.mark.parametrize("T,V", [(300, 1000), (257, 151936)])
def test_dual_clip_bound_matches_oracle(T, V):
    # step 3b (reading L-18): wide ratio noise so that r > c occurs on negative-advantage tokens; both kernel families
    rng = np.random.default_rng(17)
    S, c = 5, 2.0
    g = torch.Generator(device="cuda").manual_seed(23)
    logits = (torch.randn((T, V), generator=g, device="cuda") * 3.0).to(torch.bfloat16)
    y = rng.integers(0, V, size=T).astype(np.int32)
    adv = rng.standard_normal(T).astype(np.float32)
    mask = (rng.random(T) < 0.8).astype(np.uint8)
    seg = rng.integers(0, S, size=T).astype(np.int32)
    dev = lambda a: torch.from_numpy(a).cuda()
    lp = torch.log_softmax(logits.float(), dim=-1).gather(1, dev(y).long()[:, None])[:, 0]
    old = (lp.cpu().numpy() + rng.standard_normal(T).astype(np.float32)).astype(np.float32)
    out = ajt.policy_loss_fwd_bwd_ext(logits, dev(y), dev(old), dev(adv), dev(mask), dev(seg), S, 0.2, 0.28, clip_c=c, want_logp=True)
    torch.cuda.synchronize()
    assert ajt.last_status(out.workspace) == 0
    bits = logits.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
    e = (float(np.float32(0.2)), float(np.float32(0.28)))
    ref = oracle.policy_loss(bits, y, old, adv, mask, seg, S, e[0], e[1], logits_is_bf16_bits=True, clip_c=c)
    r = np.exp(ref.logp - old)
    capped = (adv < 0) & (mask > 0) & (r > c)
    assert capped.any()
    near = np.abs(r - c) < 1e-4     # fp32 and fp64 may land on different sides of the cap there
    d_gpu = out.dlogits[:, :V].float().cpu().numpy().astype(np.float64)
    ok = (mask > 0) & ~near
    err = np.abs(d_gpu[ok] - ref.dlogits[ok])
    assert (err <= 2.0 ** -8 * np.abs(ref.dlogits[ok]) + 1e-10).all()
    assert not d_gpu[capped & ~near].any()
    l1 = float(np.sum(ref.w * np.abs(ref.Lt)))
    assert abs(float(out.loss[0]) - ref.loss) <= 1e-5 * l1 + 1e-7 * abs(ref.loss)
    plain = ajt.policy_loss_fwd_bwd_ext(logits, dev(y), dev(old), dev(adv), dev(mask), dev(seg), S, 0.2, 0.28)
    assert float(plain.loss[0]) != float(out.loss[0])
