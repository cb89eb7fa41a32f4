"""Shared test helpers: run the CUDA path through the binding, run the oracle, compare.

The comparison rules are those of DESIGN.md "Tolerances" (BASELINE.json north_star + readings L-8, L-9)."""
import numpy as np
import torch

import oracle
import paper_2606_04484_b200 as ajt

MERGE_FIELDS = ("merged_tokens", "merged_mask", "merged_src", "merged_old_logp", "merged_offsets", "merged_origin",
                "merged_traj", "owner")


def gpu_merge(mi, owner_rule, use_explicit_mask=False, flags=0, with_logp=True, pad=0, mask_in=None):
    """Runs ajt_merge_timelines on cuda:0.  `pad` shifts the token array by `pad` elements to test unaligned bases."""
    dev = "cuda"
    tok_full = torch.zeros(mi.n_tokens + pad, dtype=torch.int32, device=dev)
    tok_full[pad:] = torch.from_numpy(mi.tokens).to(dev)
    tokens = tok_full[pad:]
    offsets = torch.from_numpy(mi.offsets).to(dev)
    traj = torch.from_numpy(mi.traj_ids).to(dev)
    rs = None if use_explicit_mask else torch.from_numpy(mi.resp_start).to(dev)
    mk = torch.from_numpy(mask_in).to(dev) if use_explicit_mask else None
    lp = torch.from_numpy(mi.old_logp).to(dev) if with_logp else None
    out = ajt.merge_timelines(tokens, offsets, traj, rs, mk, lp, owner_rule=owner_rule, flags=flags)
    status = ajt.last_status(out.workspace)
    fatal = ajt.STATUS_PROBE_CAPACITY | ajt.STATUS_BAD_OFFSETS | ajt.STATUS_ZERO_LEN
    return (None if status & fatal else out.finalize()), status


def assert_merge_equal(g, r):
    """Bit-exact in all nine outputs (pin P-M6)."""
    assert g.M == r.M and g.N_out == r.N_out, (g.M, r.M, g.N_out, r.N_out)
    for f in MERGE_FIELDS:
        a = getattr(g, f)
        b = getattr(r, f)
        if b is None:
            assert a is None
            continue
        a = a.cpu().numpy()
        if f == "merged_old_logp":
            a, b = a.view(np.uint32), b.view(np.uint32)
        if not np.array_equal(a, b):
            bad = np.nonzero(a != b)[0]
            raise AssertionError(f"{f}: {bad.size} mismatches, first at {bad[:5]}: gpu {a[bad[:5]]} oracle {b[bad[:5]]}")


def harness_old_logp(logits_t: torch.Tensor, targets_t: torch.Tensor, noise: np.ndarray) -> torch.Tensor:
    """INPUT synthesis (not the method): old_logp = (library log-softmax of the row at the target) + noise."""
    T = logits_t.shape[0]
    out = torch.empty(T, dtype=torch.float32, device=logits_t.device)
    step = max(1, (1 << 27) // max(1, logits_t.shape[1]))
    for a in range(0, T, step):
        z = logits_t[a:a + step].float()
        lse = torch.logsumexp(z, dim=-1)
        out[a:a + step] = z.gather(1, targets_t[a:a + step].long().clamp_(0, z.shape[1] - 1)[:, None])[:, 0] - lse
    return out + torch.from_numpy(noise).to(out.device)


def bf16_bits(t: torch.Tensor) -> np.ndarray:
    return t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


def logits_to_oracle(t: torch.Tensor):
    if t.dtype == torch.bfloat16:
        return bf16_bits(t), True
    return t.float().cpu().numpy(), False


def check_loss(out, ref: "oracle.LossResult", logits_rows_mask, eps_lo, eps_hi, adv, old_logp, grad_scale, V, row_ids=None,
               check_scalar=True, stats=True):
    """out: binding LossOutput (device).  ref: oracle result for rows `row_ids` (all rows if None)."""
    T = out.dlogits.shape[0]
    rows = np.arange(T) if row_ids is None else np.asarray(row_ids)
    d_gpu = out.dlogits[torch.from_numpy(rows).to(out.dlogits.device), :V].float().cpu().numpy().astype(np.float64)
    d_ref = ref.dlogits
    m = logits_rows_mask[rows] != 0
    # masked rows: exactly zero (bit-exact)
    assert np.all(d_gpu[~m] == 0.0)
    # rows whose ratio sits on a clip bound may take either branch in fp32 vs fp64: excluded from dlogits compare
    ratio = np.exp(ref.logp - old_logp[rows].astype(np.float64))
    A = adv[rows].astype(np.float64)
    near = ((A > 0) & (np.abs(ratio - (1 + float(np.float32(eps_hi)))) < 1e-5)) | \
           ((A < 0) & (np.abs(ratio - (1 - float(np.float32(eps_lo)))) < 1e-5))
    ok = m & ~near
    err = np.abs(d_gpu[ok] - d_ref[ok])
    # (a) the literal north_star bound, where bf16 storage can meet it at all: |dlogits| < 1 (a bf16 half-ulp is 2^-9 = 1.95e-3
    # just below 1 and doubles with every binade above it; reading L-9)
    lit = err[np.abs(d_ref[ok]) < 1.0]
    assert lit.size == 0 or lit.max() <= 2e-3, lit.max()
    # (b) the bound with teeth (reading L-9): half-ulp bf16 rounding + fp32 slack, relative
    tol = 2.0 ** -8 * np.abs(d_ref[ok]) + 1e-10 * max(1.0, abs(grad_scale))
    if err.size:
        worst = (err - tol).max()
        assert worst <= 0, f"dlogits: worst excess {worst:.3e}, max err {err.max():.3e}"
    if out.logp is not None:
        lp = out.logp.cpu().numpy()[rows].astype(np.float64)
        assert np.all(lp[~m] == 0.0)
        assert np.all(np.abs(lp[m] - ref.logp[m]) <= 2e-6 * np.maximum(1.0, np.abs(ref.logp[m])))
    if check_scalar:
        loss_gpu = float(out.loss.cpu()[0])
        l1 = float(np.sum(ref.w * np.abs(ref.Lt)))
        d = abs(loss_gpu - ref.loss)
        # fp32 output of an fp64 accumulation: allow half an fp32 ulp of the result on top of 1e-5
        assert d <= 1e-5 * l1 + 1e-7 * abs(ref.loss) + 1e-30, (loss_gpu, ref.loss, l1)
        if abs(ref.loss) >= 1e-2 * l1 and l1 > 0:
            assert d <= 1e-5 * abs(ref.loss), (loss_gpu, ref.loss)
        if stats and out.stats is not None:
            st = out.stats.cpu().numpy().astype(np.float64)
            assert st[0] == ref.stats[0]
            n_near = int(near.sum())
            assert abs(st[1] - ref.stats[1]) <= n_near and abs(st[2] - ref.stats[2]) <= n_near
            # sum_t w_t (-(logp_t - old_t)): every log-ratio carries the fp32 error of logp_t itself (the 2e-6 max(1, |logp|)
            # bound checked above), which does not average out when few rows are unmasked
            tol3 = float(np.sum(ref.w * 2e-6 * np.maximum(1.0, np.abs(ref.logp)))) + \
                1e-5 * max(1e-3, float(np.sum(ref.w * np.abs(ref.logp - old_logp[rows]))))
            assert abs(st[3] - ref.stats[3]) <= tol3, (st[3], ref.stats[3], tol3)
    return dict(max_err=float(err.max()) if err.size else 0.0, n_near=int(near.sum()))


# ---- pin P-K2 of oracle.pack_loss_inputs: a second formulation of reading L-12 as one global shift (lives with the tests:
# the product package holds none of the method's arithmetic outside its kernels)


def shift_for_next_token(merged_tokens: np.ndarray, merged_mask: np.ndarray, merged_old_logp: np.ndarray,
                         merged_offsets: np.ndarray):
    """inside each merged sequence targets[q] = tokens[q+1], mask[q] = mask[q+1],
    old_logp[q] = old_logp[q+1]; the last position of every sequence is masked out.  Pure index plumbing."""
    N = merged_tokens.shape[0]
    targets = np.zeros(N, dtype=np.int32)
    mask = np.zeros(N, dtype=np.uint8)
    olp = np.zeros(N, dtype=np.float32)
    if N > 1:
        targets[:-1] = merged_tokens[1:]
        mask[:-1] = merged_mask[1:]
        olp[:-1] = merged_old_logp[1:]
    last = merged_offsets[1:] - 1
    last = last[last >= 0]
    mask[last] = 0
    targets[last] = 0
    olp[last] = 0
    return targets, mask, olp


def seg_ids_from_merged(merged_offsets: np.ndarray, merged_traj: np.ndarray):
    """Segment = trajectory: dense ids 0..S-1 in order of first appearance."""
    uniq, inv = np.unique(merged_traj, return_inverse=True)
    lens = np.diff(merged_offsets)
    return np.repeat(inv.astype(np.int32), lens), int(uniq.shape[0]), uniq
