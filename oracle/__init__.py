"""ORACLE — test infrastructure, not the product.

ctypes wrapper around oracle/ajt_oracle.c (plain C: brute-force merge, fp64 loss).  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import this package.
It never imports paper_2606_04484_b200 and shares nothing with its CUDA sources.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ajt_oracle.c")
# AJT_ORACLE_SANITIZE=1 (tests/test_oracle_sanitize.py): a second build with -fsanitize=address,undefined next to the normal one
_SAN = os.environ.get("AJT_ORACLE_SANITIZE") == "1"
_SO = os.path.join(_HERE, "libajt_oracle_san.so" if _SAN else "libajt_oracle.so")

OWNER_LONGEST = 0   # BASELINE.json north_star: longest surviving extender, then lowest index
OWNER_PAPER = 1     # Algorithm 1 taken literally: the latest extender
DT_BF16 = 0
DT_F32 = 1

_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        flags = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-omit-frame-pointer"] if _SAN else ["-O2"]
        subprocess.check_call(["gcc"] + flags + ["-fopenmp", "-shared", "-fPIC", "-o", _SO, _SRC, "-lm"])
    return _SO


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_SO)
        _lib.ajt_oracle_merge.restype = C.c_int
        _lib.ajt_oracle_merge_blocks.restype = C.c_int
        _lib.ajt_oracle_loss.restype = C.c_int
        _lib.ajt_oracle_loss_ex.restype = C.c_int
        _lib.ajt_oracle_round_bf16.restype = C.c_double
        _lib.ajt_oracle_round_bf16.argtypes = [C.c_double]
        _lib.ajt_oracle_num_threads.restype = C.c_int
        _lib.ajt_oracle_set_threads.argtypes = [C.c_int]
    return _lib


def num_threads() -> int:
    return int(lib().ajt_oracle_num_threads())


def set_threads(n: int) -> None:
    lib().ajt_oracle_set_threads(int(n))


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _c(a, dtype):
    if a is None:
        return None
    a = np.ascontiguousarray(a, dtype=dtype)
    return a


@dataclass
class MergeResult:
    merged_tokens: np.ndarray    # int32 [N_out]
    merged_mask: np.ndarray      # uint8 [N_out]
    merged_src: np.ndarray       # int32 [N_out]
    merged_old_logp: Optional[np.ndarray]  # float32 [N_out]
    merged_offsets: np.ndarray   # int64 [M+1]
    merged_origin: np.ndarray    # int32 [M]
    merged_traj: np.ndarray      # int32 [M]
    owner: np.ndarray            # int32 [n]
    M: int
    N_out: int


def merge_timelines(tokens, offsets, traj_ids, resp_start=None, mask_in=None, old_logp_in=None,
                    owner_rule: int = OWNER_LONGEST) -> MergeResult:
    """Definition of the merge (DESIGN.md O-M; Algorithm 1) by brute force."""
    tokens = _c(tokens, np.int32)
    offsets = _c(offsets, np.int64)
    traj_ids = _c(traj_ids, np.int32)
    resp_start = _c(resp_start, np.int32)
    mask_in = _c(mask_in, np.uint8)
    old_logp_in = _c(old_logp_in, np.float32)
    n = int(traj_ids.shape[0])
    assert offsets.shape[0] == n + 1
    N = int(tokens.shape[0])
    assert n == 0 or int(offsets[-1]) == N
    mt = np.zeros(max(N, 1), np.int32)
    mm = np.zeros(max(N, 1), np.uint8)
    ms = np.zeros(max(N, 1), np.int32)
    ml = np.zeros(max(N, 1), np.float32) if old_logp_in is not None else None
    mo = np.zeros(n + 1, np.int64)
    mor = np.zeros(max(n, 1), np.int32)
    mtr = np.zeros(max(n, 1), np.int32)
    ow = np.zeros(max(n, 1), np.int32)
    cnt = np.zeros(2, np.int64)
    rc = lib().ajt_oracle_merge(_p(tokens), _p(offsets), _p(traj_ids), _p(resp_start), _p(mask_in), _p(old_logp_in),
                                C.c_int32(n), C.c_int32(owner_rule), _p(mt), _p(mm), _p(ms), _p(ml), _p(mo),
                                _p(mor), _p(mtr), _p(ow), _p(cnt))
    if rc != 0:
        raise ValueError(f"ajt_oracle_merge: invalid input (rc={rc})")
    M, No = int(cnt[0]), int(cnt[1])
    return MergeResult(mt[:No].copy(), mm[:No].copy(), ms[:No].copy(), None if ml is None else ml[:No].copy(),
                       mo[:M + 1].copy(), mor[:M].copy(), mtr[:M].copy(), ow[:n].copy(), M, No)


AUTHOR_ENV, AUTHOR_USER, AUTHOR_LLM = 0, 1, 2   # author labels of eq. (1)
MATCH_TEXT = 0    # "text (default)"
MATCH_TOKEN = 1   # "token"


@dataclass
class BlockMergeResult:
    merged_tokens: np.ndarray         # int32 [N_out]
    merged_mask: np.ndarray           # uint8 [N_out]
    merged_logp: Optional[np.ndarray]  # float32 [N_out]
    merged_tok_src: np.ndarray        # int32 [N_out]
    merged_offsets: np.ndarray        # int64 [M+1]   tokens
    merged_block_offsets: np.ndarray  # int64 [M+1]   blocks
    merged_block_src: np.ndarray      # int32 [B_out]
    merged_block_author: np.ndarray   # uint8 [B_out]
    merged_block_tok_off: np.ndarray  # int64 [B_out+1]
    merged_origin: np.ndarray         # int32 [M]
    merged_traj: np.ndarray           # int32 [M]
    owner: np.ndarray                 # int32 [n]
    M: int
    B_out: int
    N_out: int


def merge_blocks(block_ids, block_offsets, traj_ids, author, tok_off, tokens, logp=None, tok_mask=None,
                 match: int = MATCH_TEXT) -> BlockMergeResult:
    """Algorithm 1 line by line on timelines of message blocks (DESIGN.md O-B)."""
    block_ids = _c(block_ids, np.int64)
    block_offsets = _c(block_offsets, np.int64)
    traj_ids = _c(traj_ids, np.int32)
    author = _c(author, np.uint8)
    tok_off = _c(tok_off, np.int64)
    tokens = _c(tokens, np.int32)
    logp = _c(logp, np.float32)
    tok_mask = _c(tok_mask, np.uint8)
    n = int(traj_ids.shape[0])
    B = int(block_ids.shape[0])
    N = int(tokens.shape[0])
    assert block_offsets.shape[0] == n + 1 and tok_off.shape[0] == B + 1 and author.shape[0] == B
    assert n == 0 or (int(block_offsets[-1]) == B and int(tok_off[-1]) == N)
    mt = np.zeros(max(N, 1), np.int32)
    mm = np.zeros(max(N, 1), np.uint8)
    ml = np.zeros(max(N, 1), np.float32) if logp is not None else None
    ms = np.zeros(max(N, 1), np.int32)
    mo = np.zeros(n + 1, np.int64)
    mbo = np.zeros(n + 1, np.int64)
    mbs = np.zeros(max(B, 1), np.int32)
    mba = np.zeros(max(B, 1), np.uint8)
    mbt = np.zeros(B + 1, np.int64)
    mor = np.zeros(max(n, 1), np.int32)
    mtr = np.zeros(max(n, 1), np.int32)
    ow = np.zeros(max(n, 1), np.int32)
    cnt = np.zeros(3, np.int64)
    rc = lib().ajt_oracle_merge_blocks(_p(block_ids), _p(block_offsets), _p(traj_ids), _p(author), _p(tok_off), _p(tokens),
                                       _p(logp), _p(tok_mask), C.c_int32(n), C.c_int32(match), _p(mt), _p(mm), _p(ml), _p(ms),
                                       _p(mo), _p(mbo), _p(mbs), _p(mba), _p(mbt), _p(mor), _p(mtr), _p(ow), _p(cnt))
    if rc != 0:
        raise ValueError(f"ajt_oracle_merge_blocks: invalid input (rc={rc})")
    M, Bo, No = int(cnt[0]), int(cnt[1]), int(cnt[2])
    return BlockMergeResult(mt[:No].copy(), mm[:No].copy(), None if ml is None else ml[:No].copy(), ms[:No].copy(),
                            mo[:M + 1].copy(), mbo[:M + 1].copy(), mbs[:Bo].copy(), mba[:Bo].copy(), mbt[:Bo + 1].copy(),
                            mor[:M].copy(), mtr[:M].copy(), ow[:n].copy(), M, Bo, No)


@dataclass
class LossResult:
    loss: float                  # sum over the given rows of w_t L_t (the whole loss when all rows are given)
    logp: np.ndarray             # float64 [R]
    w: np.ndarray                # float64 [R]
    g: np.ndarray                # float64 [R]
    Lt: np.ndarray               # float64 [R]
    dlogits: Optional[np.ndarray]  # float64 [R,V], before rounding
    stats: np.ndarray            # float64 [4]
    k3: Optional[np.ndarray] = None    # float64 [R]  low-variance KL estimator per token (extended form)
    ent: Optional[np.ndarray] = None   # float64 [R]  entropy of the row's softmax (extended form)
    ext: Optional[np.ndarray] = None   # float64 [2]  {sum w_t k3_t, sum w_t H_t}


def policy_loss(logits, targets, old_logp, adv, mask, seg_ids, S: int, eps_lo: float, eps_hi: float,
                seg_denom=None, inv_num_segs: float = 0.0, grad_scale: float = 1.0,
                row_ids=None, want_dlogits: bool = True, logits_is_bf16_bits: bool = False,
                ref_logp=None, kl_coef: float = 0.0, extended: bool = False, clip_c: float = 0.0) -> LossResult:
    """fp64 loss oracle (DESIGN.md O-L).  `logits` is float32 [R,V], or uint16 [R,V] holding bf16 bit
    patterns when logits_is_bf16_bits.  Per-token vectors have length T (all tokens of the call);
    `row_ids` (int64 [R]) says which tokens the given logits rows are (None => R == T)."""
    if logits_is_bf16_bits:
        logits = _c(logits, np.uint16)
        dt = DT_BF16
    else:
        logits = _c(logits, np.float32)
        dt = DT_F32
    R, V = int(logits.shape[0]), int(logits.shape[1])
    targets = _c(targets, np.int32)
    old_logp = _c(old_logp, np.float32)
    adv = _c(adv, np.float32)
    mask = _c(mask, np.uint8)
    seg_ids = _c(seg_ids, np.int32)
    T = int(targets.shape[0])
    row_ids = _c(row_ids, np.int64)
    if row_ids is None:
        assert R == T
    seg_denom = _c(seg_denom, np.float32)
    loss = np.zeros(1, np.float64)
    logp = np.zeros(max(R, 1), np.float64)
    w = np.zeros(max(R, 1), np.float64)
    g = np.zeros(max(R, 1), np.float64)
    Lt = np.zeros(max(R, 1), np.float64)
    dl = np.zeros((R, V), np.float64) if want_dlogits else None
    stats = np.zeros(4, np.float64)
    rc = lib().ajt_oracle_loss(_p(logits), C.c_int32(dt), C.c_int64(R), C.c_int32(V), C.c_int64(V), _p(row_ids),
                               _p(targets), _p(old_logp), _p(adv), _p(mask), _p(seg_ids), C.c_int64(T), C.c_int32(S),
                               C.c_double(eps_lo), C.c_double(eps_hi), _p(seg_denom), C.c_double(inv_num_segs),
                               C.c_double(grad_scale), _p(loss), _p(logp), _p(w), _p(g), _p(Lt), _p(dl), _p(stats))
    if rc != 0:
        raise ValueError(f"ajt_oracle_loss: invalid input (rc={rc})")
    if extended or ref_logp is not None or clip_c != 0.0:
        # steps 8-9 (KL against a reference policy, entropy): a second call of the extended entry point
        ref = _c(ref_logp, np.float32)
        k3 = np.zeros(max(R, 1), np.float64)
        ent = np.zeros(max(R, 1), np.float64)
        ext = np.zeros(2, np.float64)
        stats[:] = 0.0
        lib().ajt_oracle_loss_ex2.restype = C.c_int
        rc = lib().ajt_oracle_loss_ex2(_p(logits), C.c_int32(dt), C.c_int64(R), C.c_int32(V), C.c_int64(V), _p(row_ids),
                                      _p(targets), _p(old_logp), _p(adv), _p(mask), _p(seg_ids), C.c_int64(T), C.c_int32(S),
                                      C.c_double(eps_lo), C.c_double(eps_hi), _p(seg_denom), C.c_double(inv_num_segs),
                                      C.c_double(grad_scale), _p(loss), _p(logp), _p(w), _p(g), _p(Lt), _p(dl), _p(stats),
                                      _p(ref), C.c_double(kl_coef), _p(k3), _p(ent), _p(ext), C.c_double(clip_c))
        if rc != 0:
            raise ValueError(f"ajt_oracle_loss_ex2: invalid input (rc={rc})")
        return LossResult(float(loss[0]), logp[:R], w[:R], g[:R], Lt[:R], dl, stats, k3[:R], ent[:R], ext)
    return LossResult(float(loss[0]), logp[:R], w[:R], g[:R], Lt[:R], dl, stats)


def pack_loss_inputs(merged_tokens, merged_mask, merged_old_logp, merged_offsets, merged_origin, tl_seg, seg_adv=None):
    """Per-token loss inputs from merged sequences (reading L-12), sequence by sequence (ajt_oracle_pack in
    ajt_oracle.c): inside sequence m the row at position q predicts the token at q+1, so targets / mask / old_logp are those
    of q+1; the last position of every sequence has nothing to predict (0, 0, 0).  seg_ids = dense trajectory id of the
    surviving timeline; adv = that trajectory's advantage.
    Returns (targets int32, mask uint8, old_logp float32 | None, seg_ids int32, adv float32 | None)."""
    merged_offsets = _c(merged_offsets, np.int64)
    M = max(0, len(merged_offsets) - 1)
    N = int(merged_offsets[-1]) if len(merged_offsets) else 0
    targets = np.zeros(N, np.int32)
    mask = np.zeros(N, np.uint8)
    olp = None if merged_old_logp is None else np.zeros(N, np.float32)
    seg = np.zeros(N, np.int32)
    adv = None if seg_adv is None else np.zeros(N, np.float32)
    mt, mm = _c(merged_tokens, np.int32), _c(merged_mask, np.uint8)
    ml = None if merged_old_logp is None else _c(merged_old_logp, np.float32)
    mo, ts = _c(merged_origin, np.int32), _c(tl_seg, np.int32)
    sa = None if seg_adv is None else _c(seg_adv, np.float32)
    L = lib()
    L.ajt_oracle_pack.restype = C.c_int
    rc = L.ajt_oracle_pack(_p(mt), _p(mm), _p(ml), _p(merged_offsets), _p(mo), _p(ts), _p(sa), C.c_int64(M), _p(targets),
                           _p(mask), _p(olp), _p(seg), _p(adv))
    if rc != 0:
        raise ValueError("ajt_oracle_pack: invalid offsets")
    return targets, mask, olp, seg, adv


def pack_microbatches(lengths, budget: int):
    """Token-budget packing of consecutive merged sequences ("packed merged sequences", BASELINE.json north_star; DESIGN.md
    reading L-12): walk the sequences in order, open a new micro-batch whenever the next sequence would push the current one
    over `budget` rows (a sequence longer than the budget gets a micro-batch of its own).  Returns the list of
    (first_sequence, one_past_last_sequence)."""
    if budget < 1:
        raise ValueError("budget must be >= 1")
    out, a, used = [], 0, 0
    for k, L in enumerate(lengths):
        L = int(L)
        if used > 0 and used + L > budget:
            out.append((a, k))
            a, used = k, 0
        used += L
    if len(lengths) > a:
        out.append((a, len(lengths)))
    return out


def lm_head_logp(hidden_bits, weight_bits, targets, mask=None, round_logits_bf16: bool = False):
    """Log-prob and entropy of the target token under an LM head, without the method's tiling (the step before
    the loss in the actor update, forward half):
        z_t = W h_t  (fp64 from the exact bf16 inputs);  logp_t = z_{t,y_t} - logsumexp(z_t);  H_t = lse_t - sum_v p_tv z_tv
    hidden_bits uint16 [T,d], weight_bits uint16 [V,d] (bf16 bit patterns).  Rows with mask 0 give 0, 0."""
    def f64(bits):
        b = np.ascontiguousarray(bits, np.uint16).astype(np.uint32) << 16
        return b.view(np.float32).astype(np.float64)
    H, W = f64(hidden_bits), f64(weight_bits)
    T = H.shape[0]
    logp = np.zeros(T, np.float64)
    ent = np.zeros(T, np.float64)
    for a in range(0, T, 256):
        z = H[a:a + 256] @ W.T                      # library matmul as a step
        if round_logits_bf16:                       # the logits as a bf16-storing forward pass would hand them to the loss
            z = round_bf16(z)
        m = z.max(axis=1, keepdims=True)
        lse = m[:, 0] + np.log(np.exp(z - m).sum(axis=1))
        p = np.exp(z - lse[:, None])
        rows = np.arange(z.shape[0])
        logp[a:a + 256] = z[rows, np.asarray(targets[a:a + 256], np.int64)] - lse
        ent[a:a + 256] = lse - (p * z).sum(axis=1)
    if mask is not None:
        on = np.asarray(mask) != 0
        logp, ent = np.where(on, logp, 0.0), np.where(on, ent, 0.0)
    return logp, ent


def lm_head_loss_bwd(hidden_bits, weight_bits, targets, old_logp, adv, mask, seg_ids, S: int, eps_lo: float, eps_hi: float,
                     seg_denom=None, inv_num_segs: float = 0.0, grad_scale: float = 1.0, round_dz_bf16: bool = False):
    """The policy loss straight from the hidden states and its gradients w.r.t. both of them (SURVEY.md §8(f)
    f3, backward half; the actor update of PAPER.md:136).  The plain chain rule through z_t = W h_t:
        steps 1-6 of O-L on z (fp64 from the exact bf16 inputs; NOT rounded to bf16: reading H-1) give loss and, per row,
        dZ_tv = g_t (1[v = y_t] - p_tv);   dH = dZ W  ([T,V] x [V,d]);   dW = dZ^T H  ([V,T] x [T,d])
    round_dz_bf16: dZ is rounded to bf16 (RNE) before the two products, as a tensor-core path that feeds dZ as a bf16 operand
    does (reading H-4) -- the variant the kernel is compared with element by element; the unrounded one is the definition.
    Returns dict(loss, logp[T], lse[T], g[T], dH[T,d], dW[V,d]) in fp64.  CPU-sized inputs only (one [T,V] fp64 matrix)."""
    def f64(bits):
        b = np.ascontiguousarray(bits, np.uint16).astype(np.uint32) << 16
        return b.view(np.float32).astype(np.float64)
    H, W = f64(hidden_bits), f64(weight_bits)
    T, V = H.shape[0], W.shape[0]
    y = np.asarray(targets, np.int64)
    m = (np.asarray(mask) != 0).astype(np.float64)
    sg = np.asarray(seg_ids, np.int64)
    old, A = np.asarray(old_logp, np.float64), np.asarray(adv, np.float64)
    z = H @ W.T                                                   # library matmul as a step
    zmax = z.max(axis=1)
    lse = zmax + np.log(np.exp(z - zmax[:, None]).sum(axis=1))    # step 1
    logp = z[np.arange(T), y] - lse
    p = np.exp(z - lse[:, None])
    r = np.exp(logp - old)                                        # step 2
    rc = np.clip(r, 1.0 - eps_lo, 1.0 + eps_hi)
    L = -np.minimum(r * A, rc * A)                                # step 3
    Ns = np.zeros(S, np.float64)                                  # step 4
    np.add.at(Ns, sg, m)
    if seg_denom is not None:
        Ns = np.asarray(seg_denom, np.float64)
    inv = inv_num_segs if inv_num_segs != 0.0 else (1.0 / max(1, int((Ns > 0).sum())) if (Ns > 0).any() else 0.0)
    w = np.where(Ns[sg] > 0, m * inv / np.where(Ns[sg] > 0, Ns[sg], 1.0), 0.0)
    loss = float(np.sum(w * L))                                   # step 5
    hi = (A > 0) & (r > 1.0 + eps_hi)                             # step 6
    lo = (A < 0) & (r < 1.0 - eps_lo)
    g = np.where(hi | lo, 0.0, grad_scale * w * (-A * r))
    dZ = -g[:, None] * p
    dZ[np.arange(T), y] += g
    if round_dz_bf16:
        dZ = round_bf16(dZ)
    return dict(loss=loss, logp=logp * m, lse=lse * m, g=g, dH=dZ @ W, dW=dZ.T @ H, w=w, Lt=L)


def round_bf16(x: np.ndarray) -> np.ndarray:
    """fp64 -> nearest bf16 (ties to even), as fp64."""
    a = np.ascontiguousarray(x, np.float64)
    out = np.empty_like(a)
    lib().ajt_oracle_round_bf16_array(_p(a), _p(out), C.c_int64(a.size))
    return out
