"""GPU: ajt_policy_loss_fwd_bwd_static (include/ajt.h) -- the loss call whose scratch is the library's file-scope device
array, for callers that cannot call cudaMalloc -- against the existing workspace path, on two calls in a row.

Both entry points run the same kernels on the same inputs, so the outputs must be IDENTICAL (dlogits bit for bit, loss /
log-probs / statistics bit for bit: the scalar is reduced in a fixed order); the comparison is nevertheless written with
the tolerances the loss tests use (BASELINE.json north_star: loss 1e-5 relative, dlogits 2e-3 absolute) plus the exact
check.  The second call has another shape and other inputs: the array keeps the first call's contents, and what must start at
zero is cleared by the call.  This file is named so that pytest collects it last; it passes alone in a fresh process and
after the other tests (the static array is per process and per device, and no other test touches it)."""
import numpy as np
import pytest
import torch

import paper_2606_04484_b200 as ajt
from paper_2606_04484_b200 import workloads as W
from helpers import harness_old_logp

pytestmark = pytest.mark.gpu


def _case(T, V, S, rho, dtype, seed):
    lv = W.loss_sweep_vectors(T, V, S, rho, seed=seed, cell=V % 977)
    g = torch.Generator(device="cuda").manual_seed(seed)
    logits = (torch.randn((T, V), generator=g, device="cuda", dtype=torch.float32) * 3.0).to(dtype)
    dev = lambda a: torch.from_numpy(a).cuda()
    targets, adv, mask, seg = dev(lv.targets), dev(lv.adv), dev(lv.mask), dev(lv.seg_ids)
    old = harness_old_logp(logits, targets, lv.noise)
    return logits, targets, old, adv, mask, seg


def _both(T, V, S, rho, dtype, seed):
    logits, targets, old, adv, mask, seg = _case(T, V, S, rho, dtype, seed)
    ref = ajt.policy_loss_fwd_bwd(logits, targets, old, adv, mask, seg, S, 0.2, 0.28, want_logp=True, want_stats=True)
    torch.cuda.synchronize()
    assert ajt.last_status(ref.workspace) == 0
    # the caller's outputs, filled with garbage first; nothing is allocated inside the call
    dl = torch.full((T, V), 7.0, dtype=torch.bfloat16, device="cuda")
    loss = torch.full((1,), 9.0, device="cuda")
    logp = torch.full((T,), 9.0, device="cuda")
    stats = torch.full((4,), 9.0, device="cuda")
    status = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    before = torch.cuda.memory_allocated()
    ajt.policy_loss_fwd_bwd_static(logits, targets, old, adv, mask, seg, S, 0.2, 0.28, dl, loss, logp=logp, stats=stats,
                                   status=status)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before
    assert int(status[0]) == 0
    # tolerances of the loss tests ...
    assert abs(float(loss[0]) - float(ref.loss[0])) <= 1e-5 * max(abs(float(ref.loss[0])), 1e-30)
    assert float((dl.float() - ref.dlogits.float()).abs().max()) <= 2e-3
    assert float((logp - ref.logp[:T]).abs().max()) <= 3e-5
    # ... and, since the kernels are the same, exact equality
    assert torch.equal(dl, ref.dlogits) and torch.equal(loss, ref.loss)
    assert torch.equal(logp, ref.logp[:T]) and torch.equal(stats, ref.stats)
    assert float(ref.dlogits.float().abs().max()) > 0.0   # not a comparison of zeros


def test_static_scratch_loss_matches_workspace_path_twice_in_a_row():
    assert ajt.loss_static_scratch_bytes() == 4 << 20
    _both(3000, 32000, 16, 0.6, torch.bfloat16, seed=41)     # 1-CTA fast kernel, several row tiles per SM
    _both(700, 151936, 5, 0.3, torch.bfloat16, seed=42)      # right after it: 2-CTA cluster kernel, other shape and inputs
    _both(900, 1024, 7, 0.5, torch.float32, seed=43)         # and the fp32 register kernel


def test_static_scratch_rejects_sizes_beyond_the_array():
    T, V, S = 70000, 8, 4                                    # 69 bytes per row: 4.8 MB > 4 MiB
    assert ajt.loss_workspace_bytes(T, V, S) > ajt.loss_static_scratch_bytes()
    z = torch.zeros((T, V), dtype=torch.bfloat16, device="cuda")
    i32 = torch.zeros(T, dtype=torch.int32, device="cuda")
    f32 = torch.zeros(T, device="cuda")
    u8 = torch.ones(T, dtype=torch.uint8, device="cuda")
    loss = torch.full((1,), 5.0, device="cuda")
    with pytest.raises(ajt.AjtError) as e:
        ajt.policy_loss_fwd_bwd_static(z, i32, f32, f32, u8, i32, S, 0.2, 0.2, torch.empty_like(z), loss)
    assert e.value.code == -3 and "capacity" in str(e.value)  # AJT_ERR_CAPACITY, nothing launched
    torch.cuda.synchronize()
    assert float(loss[0]) == 5.0
    # the largest documented size fits
    assert ajt.loss_workspace_bytes(40960, 151936, 4096) <= ajt.loss_static_scratch_bytes()
