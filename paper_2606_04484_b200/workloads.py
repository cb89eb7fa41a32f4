"""Seeded synthetic inputs shaped like the paper's agent workloads.

This module serves BOTH the CUDA path's tests/bench and the CPU oracle's tests.
It holds none of the method's arithmetic: no prefix matching, no merging, no
softmax, no ratio, no clipping.  It only draws random token streams with the
prefix structure of multi-turn agent episodes ("later turns reuse earlier turns
as prompt", §4.4.2), per-token loss-mask boundaries (mask = 1 only
on LLM-generated tokens, eq. (1)) and the per-token side inputs
of the loss (targets, advantages, segment ids).

Configs follow BASELINE.json `configs[0..4]`; where BASELINE.json is silent the
recipe of SURVEY.md §8(d) is used (restated in DESIGN.md "Input recipe").

Everything is a pure function of (config, seed): numpy Philox streams keyed by
(seed, config index, trajectory, field), so the GPU box and the CPU box
regenerate identical data without shipping files.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Tuple

import numpy as np

BASE_SEED = 20260604  # seed = 20260604 + config_index

# field ids for RNG stream keys
_F_STRUCT, _F_TOKENS, _F_LOGP, _F_REWARD, _F_MISC = 0, 1, 2, 3, 4


def rng_for(seed: int, *key: int) -> np.random.Generator:
    """Counter-based stream keyed by (seed, *key)."""
    ss = np.random.SeedSequence([int(seed) & 0xFFFFFFFF] + [int(k) & 0xFFFFFFFF for k in key])
    return np.random.Generator(np.random.Philox(ss))


# --------------------------------------------------------------------------- merge


@dataclass
class MergeSpec:
    name: str
    index: int                      # position in BASELINE.json configs
    n_traj: int
    turns: Tuple[int, int]          # inclusive range of K per trajectory
    prompt: int                     # P
    append: Tuple[int, int]         # inclusive range of a_k
    vocab: int
    p_break: float
    rewrite: str                    # "cut" (keep c tokens, redraw the tail at 25-100 % length) | "fresh" (10-30 % fresh context)
    cap: Optional[int] = None       # context cap (an append that would exceed it forces a fresh rewrite)
    token_law: str = "uniform"      # "uniform" | "zipf"
    order: str = "round_robin"      # emission order of timelines: "round_robin" by turn | "traj_major"


MERGE_SPECS: Dict[str, MergeSpec] = {
    # configs[0]  "tiny"
    "c1": MergeSpec("c1", 0, n_traj=32, turns=(6, 6), prompt=64, append=(32, 128), vocab=1024,
                    p_break=0.2, rewrite="cut"),
    # configs[1]  "single-model GRPO batch"
    "c2": MergeSpec("c2", 1, n_traj=64, turns=(8, 8), prompt=512, append=(256, 1024), vocab=151936,
                    p_break=0.1, rewrite="cut"),
    # configs[2]  "long-horizon agent"
    "c3": MergeSpec("c3", 2, n_traj=256, turns=(20, 40), prompt=2048, append=(512, 4096), vocab=151936,
                    p_break=0.3, rewrite="fresh", cap=32768, token_law="zipf"),
    # configs[3]  "heterogeneous multi-model team": built by merge_workload_c4 (two calls)
}


@dataclass
class MergeInputs:
    tokens: np.ndarray       # int32 [N_in]
    offsets: np.ndarray      # int64 [n+1]
    traj_ids: np.ndarray     # int32 [n]
    resp_start: np.ndarray   # int32 [n]
    old_logp: np.ndarray     # float32 [N_in]  (carried per-token log-probs)
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.traj_ids.shape[0])

    @property
    def n_tokens(self) -> int:
        return int(self.tokens.shape[0])


_ZIPF_CACHE: Dict[Tuple[int, float], np.ndarray] = {}


def _zipf_cdf(vocab: int, s: float) -> np.ndarray:
    key = (vocab, s)
    if key not in _ZIPF_CACHE:
        w = np.arange(1, vocab + 1, dtype=np.float64) ** (-s)
        c = np.cumsum(w)
        _ZIPF_CACHE[key] = c / c[-1]
    return _ZIPF_CACHE[key]


def draw_tokens(rng: np.random.Generator, count: int, vocab: int, law: str) -> np.ndarray:
    if count <= 0:
        return np.zeros(0, dtype=np.int32)
    if law == "uniform":
        return rng.integers(0, vocab, size=count, dtype=np.int64).astype(np.int32)
    if law == "zipf":   # rank r ∝ r^-1.1, truncated at vocab; token id = rank-1
        u = rng.random(count)
        return np.minimum(np.searchsorted(_zipf_cdf(vocab, 1.1), u, side="left"), vocab - 1).astype(np.int32)
    raise ValueError(law)


def _one_trajectory(spec: MergeSpec, seed: int, traj: int, stream: int = 0):
    """Returns a list of (context int32 array, resp_start) — one per turn (= per LLM call)."""
    rs = rng_for(seed, spec.index, stream, traj, _F_STRUCT)
    rt = rng_for(seed, spec.index, stream, traj, _F_TOKENS)
    K = int(rs.integers(spec.turns[0], spec.turns[1] + 1))
    ctx = draw_tokens(rt, spec.prompt, spec.vocab, spec.token_law)
    out = []
    for k in range(1, K + 1):
        a = int(rs.integers(spec.append[0], spec.append[1] + 1))
        f = float(rs.uniform(0.3, 0.7))
        brk = bool(rs.random() < spec.p_break) and k > 1
        frac = float(rs.uniform(0.1, 0.3))
        cutu = float(rs.random())
        shrink = float(rs.uniform(0.25, 1.0))
        L = ctx.shape[0]
        force_fresh = spec.cap is not None and L + a > spec.cap
        if force_fresh or (brk and spec.rewrite == "fresh"):
            # summarise: a fresh context of 10-30 % of the old length (new prefix)
            newL = max(1, int(round(frac * L)))
            ctx = draw_tokens(rt, newL, spec.vocab, spec.token_law)
        elif brk and spec.rewrite == "cut":
            # edit / compact the tail of the history: keep the first c tokens, redraw the rest at
            # 25-100 % of its old length (so the new chain can end shorter than the old one: the case
            # that separates the two owner rules)
            c = min(L - 1, int(cutu * L))
            tail = draw_tokens(rt, max(1, int(round(shrink * (L - c)))), spec.vocab, spec.token_law)
            # make sure the first redrawn token really differs so the prefix is broken at c
            tail[0] = (ctx[c] + 1 + (tail[0] % (spec.vocab - 1))) % spec.vocab
            ctx = np.concatenate([ctx[:c], tail])
        q = max(1, int(round(f * a)))
        app = draw_tokens(rt, a, spec.vocab, spec.token_law)
        ctx = np.concatenate([ctx, app])
        out.append((ctx, ctx.shape[0] - q))
    return out


def _assemble(per_traj: List[List[Tuple[np.ndarray, int]]], traj_keys: List[int], order: str,
              seed: int, cfg_index: int, stream: int = 0) -> MergeInputs:
    items = []  # (traj_key, ctx, resp_start)
    if order == "traj_major":
        for key, tl in zip(traj_keys, per_traj):
            for ctx, rs in tl:
                items.append((key, ctx, rs))
    elif order == "round_robin":
        kmax = max(len(tl) for tl in per_traj)
        for k in range(kmax):
            for key, tl in zip(traj_keys, per_traj):
                if k < len(tl):
                    items.append((key, tl[k][0], tl[k][1]))
    else:
        raise ValueError(order)
    n = len(items)
    lens = np.array([it[1].shape[0] for it in items], dtype=np.int64)
    offsets = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(lens, out=offsets[1:])
    tokens = np.concatenate([it[1] for it in items]).astype(np.int32) if n else np.zeros(0, np.int32)
    traj_ids = np.array([it[0] for it in items], dtype=np.int32)
    resp_start = np.array([it[2] for it in items], dtype=np.int32)
    rl = rng_for(seed, cfg_index, stream, 0x7FFF, _F_LOGP)
    old_logp = (-np.abs(rl.standard_normal(tokens.shape[0], dtype=np.float32)) - 0.05).astype(np.float32)
    return MergeInputs(tokens, offsets, traj_ids, resp_start, old_logp,
                       meta={"n_groups": len(traj_keys), "order": order})


def merge_workload(config: str, seed: Optional[int] = None, order: Optional[str] = None,
                   n_traj: Optional[int] = None) -> MergeInputs:
    """Merge-stage input of BASELINE.json configs[0..2] ("c1", "c2", "c3").

    `n_traj` shrinks the batch (same per-trajectory law) for CPU-sized tests.
    """
    spec = MERGE_SPECS[config]
    seed = BASE_SEED + spec.index if seed is None else seed
    nt = spec.n_traj if n_traj is None else n_traj
    per_traj = [_one_trajectory(spec, seed, t) for t in range(nt)]
    # traj ids are opaque keys: spread them out, not 0..n-1
    keys = [1000 + 7 * t for t in range(nt)]
    mi = _assemble(per_traj, keys, order or spec.order, seed, spec.index)
    mi.meta.update(config=config, seed=seed, vocab=spec.vocab)
    return mi


def merge_workload_c4(seed: Optional[int] = None, n_episodes: int = 128) -> Dict[str, MergeInputs]:
    """configs[3]: 128 episodes x 3 agents, interleaved timelines; agents 0,1 -> model A (V=151936),
    agent 2 -> model B (V=128256).  Group key = (episode, agent).  Returns {"A": ..., "B": ...}."""
    seed = BASE_SEED + 3 if seed is None else seed
    out = {}
    for model, agents, vocab in (("A", (0, 1), 151936), ("B", (2,), 128256)):
        spec = MergeSpec("c4" + model, 3, n_traj=n_episodes * len(agents), turns=(8, 16), prompt=512,
                         append=(256, 1024), vocab=vocab, p_break=0.15, rewrite="cut", cap=16384)
        per_traj, keys = [], []
        for ep in range(n_episodes):
            for ag in agents:
                per_traj.append(_one_trajectory(spec, seed, ep * 3 + ag, stream=1))
                keys.append(ep * 3 + ag)
        mi = _assemble(per_traj, keys, "round_robin", seed, 3, stream=1 + (model == "B"))
        mi.meta.update(config="c4" + model, seed=seed, vocab=vocab)
        out[model] = mi
    return out


def explicit_mask(mi: MergeInputs) -> np.ndarray:
    """uint8 [N_in] mask equivalent to resp_start: mask_j[p] = (p >= resp_start[j])."""
    m = np.zeros(mi.n_tokens, dtype=np.uint8)
    for j in range(mi.n):
        m[mi.offsets[j] + mi.resp_start[j]: mi.offsets[j + 1]] = 1
    return m


# --------------------------------------------------------------------------- loss side inputs


def advantages_pm1(seed: int, cfg_index: int, n_traj: int) -> np.ndarray:
    """c1: adv = +-1 per trajectory (Bernoulli 1/2)."""
    r = rng_for(seed, cfg_index, 0, 0, _F_REWARD)
    return np.where(r.random(n_traj) < 0.5, -1.0, 1.0).astype(np.float32)


def advantages_group_zscore(seed: int, cfg_index: int, n_traj: int, group: int = 8, p: float = 0.4) -> np.ndarray:
    """c2: rewards ~ Bernoulli(p); advantage = per-group z-score (r-mean)/(std+1e-6), 0 for constant
    groups (the zero-variance "dummy task" of PAPER.md:147, C3)."""
    r = rng_for(seed, cfg_index, 0, 0, _F_REWARD)
    rew = (r.random(n_traj) < p).astype(np.float64)
    adv = np.zeros(n_traj, dtype=np.float64)
    for g0 in range(0, n_traj, group):
        x = rew[g0:g0 + group]
        sd = x.std()
        adv[g0:g0 + group] = 0.0 if sd == 0 else (x - x.mean()) / (sd + 1e-6)
    return adv.astype(np.float32)


@dataclass
class LossVectors:
    targets: np.ndarray   # int32 [T]
    adv: np.ndarray       # float32 [T]
    mask: np.ndarray      # uint8 [T]
    seg_ids: np.ndarray   # int32 [T]
    S: int
    noise: np.ndarray     # float32 [T]: old_logp = (harness estimate of logp) + noise


def loss_sweep_vectors(T: int, V: int, S: int, rho: float, seed: Optional[int] = None,
                       cell: int = 0) -> LossVectors:
    """configs[4] cell: mask laid out as alternating env/response runs of geometric length (mean 256) with
    response density rho; S contiguous segments of near-equal length; adv ~ N(0,1) per segment; old_logp
    noise sigma 0.05 for 90 % of tokens and 0.3 for 10 % so both clip sides fire."""
    seed = BASE_SEED + 4 if seed is None else seed
    r = rng_for(seed, 4, cell, T & 0xFFFFFFFF, _F_MISC)
    targets = r.integers(0, V, size=T, dtype=np.int64).astype(np.int32)
    # alternating runs: response runs mean 256*rho/(0.5), env runs mean 256*(1-rho)/0.5 -> overall mean 256
    mask = np.zeros(T, dtype=np.uint8)
    pos, is_resp = 0, False
    mean_resp, mean_env = 512.0 * rho, 512.0 * (1.0 - rho)
    while pos < T:
        m = mean_resp if is_resp else mean_env
        ln = int(r.geometric(1.0 / max(m, 1.0)))
        if is_resp:
            mask[pos:pos + ln] = 1
        pos += ln
        is_resp = not is_resp
    S = max(1, min(S, T))
    bounds = (np.arange(S + 1, dtype=np.int64) * T) // S
    seg_ids = np.repeat(np.arange(S, dtype=np.int32), np.diff(bounds))
    adv_seg = r.standard_normal(S).astype(np.float32)
    adv = adv_seg[seg_ids]
    sig = np.where(r.random(T) < 0.9, 0.05, 0.3).astype(np.float32)
    noise = (r.standard_normal(T).astype(np.float32) * sig).astype(np.float32)
    return LossVectors(targets, adv, mask, seg_ids, S, noise)


def small_logits(T: int, V: int, sigma: float, seed: int, key: int = 0) -> np.ndarray:
    """float32 [T,V] ~ N(0, sigma) (sigma is a standard deviation).  CPU-sized only;
    large matrices are drawn on the GPU by the harness with a seeded torch.Generator."""
    r = rng_for(seed, 0xA0, key, T & 0xFFFFFFFF, V)
    return (r.standard_normal((T, V), dtype=np.float32) * np.float32(sigma)).astype(np.float32)


# --------------------------------------------------------------------------- block-level (text matching) inputs

AUTHOR_ENV, AUTHOR_USER, AUTHOR_LLM = 0, 1, 2   # author labels of eq. (1)


@dataclass
class BlockSpec:
    name: str
    index: int
    n_traj: int
    turns: Tuple[int, int]        # LLM calls per trajectory
    env_blocks: Tuple[int, int]   # env / user blocks appended before each call
    block_len: Tuple[int, int]    # tokens per block
    vocab: int
    p_break: float                # per turn: one earlier block is edited (new text), which breaks the prefix there
    p_drift: float                # per assistant block re-sent as prompt: re-tokenised differently, same text (Fig. 5)


BLOCK_SPECS: Dict[str, BlockSpec] = {
    # shapes follow configs[0] / configs[1] / configs[2] with their appends split into message blocks
    "b1": BlockSpec("b1", 10, n_traj=32, turns=(6, 6), env_blocks=(1, 2), block_len=(8, 64), vocab=1024, p_break=0.2, p_drift=0.3),
    "b2": BlockSpec("b2", 11, n_traj=64, turns=(8, 8), env_blocks=(1, 3), block_len=(64, 512), vocab=151936, p_break=0.1,
                    p_drift=0.2),
    "b3": BlockSpec("b3", 12, n_traj=256, turns=(20, 40), env_blocks=(1, 3), block_len=(128, 1024), vocab=151936, p_break=0.1,
                    p_drift=0.1),
}


@dataclass
class BlockInputs:
    block_ids: np.ndarray       # int64 [B]   text id of each block (equal ids <=> equal text)
    block_offsets: np.ndarray   # int64 [n+1] blocks of timeline i
    traj_ids: np.ndarray        # int32 [n]
    author: np.ndarray          # uint8 [B]
    tok_off: np.ndarray         # int64 [B+1] tokens of block b
    tokens: np.ndarray          # int32 [N]
    logp: np.ndarray            # float32 [N]  (log-probs of generated tokens; 0 on prompt blocks)
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.traj_ids.shape[0])


def _block_trajectory(spec: BlockSpec, seed: int, traj: int):
    """One trajectory: per LLM call a list of blocks (text id, author, tokens, logp).  Within a call the context blocks are
    the prompt (author env / user; assistant messages of earlier calls come back as env-labelled prompt blocks, possibly
    re-tokenised) and the last block is the generated answer (author llm)."""
    rs = rng_for(seed, spec.index, 0, traj, _F_STRUCT)
    rt = rng_for(seed, spec.index, 0, traj, _F_TOKENS)
    rl = rng_for(seed, spec.index, 0, traj, _F_LOGP)
    next_id = [(traj + 1) << 32]

    def new_block(author):
        L = int(rs.integers(spec.block_len[0], spec.block_len[1] + 1))
        next_id[0] += 1
        return dict(id=next_id[0] * 0x9E3779B97F4A7C15 % (1 << 63), author=author, tok=draw_tokens(rt, L, spec.vocab, "uniform"))

    K = int(rs.integers(spec.turns[0], spec.turns[1] + 1))
    ctx = [new_block(AUTHOR_USER)]      # the task prompt
    calls = []
    for k in range(1, K + 1):
        if k > 1 and rs.random() < spec.p_break:
            e = int(rs.integers(0, len(ctx)))          # the agent edits / compacts its history from block e on
            keep = int(rs.integers(1, 3))
            ctx = ctx[:e] + [new_block(AUTHOR_ENV) for _ in range(keep)]
        for _ in range(int(rs.integers(spec.env_blocks[0], spec.env_blocks[1] + 1))):
            ctx.append(new_block(AUTHOR_ENV))
        ans = new_block(AUTHOR_LLM)
        ans["logp"] = (-np.abs(rl.standard_normal(ans["tok"].shape[0], dtype=np.float32)) - 0.05).astype(np.float32)
        calls.append([dict(b) for b in ctx] + [ans])
        # the answer goes back into the context as a prompt block: same text, not generated any more; the chat template
        # may strip its thinking part, so the token ids differ although the text id is the same
        back = dict(id=ans["id"], author=AUTHOR_ENV, tok=ans["tok"])
        if rs.random() < spec.p_drift and ans["tok"].shape[0] > 4:
            cut = int(rs.integers(1, ans["tok"].shape[0] // 2 + 1))
            back["tok"] = ans["tok"][cut:]
        ctx.append(back)
    return calls


def block_workload(config: str, seed: Optional[int] = None, n_traj: Optional[int] = None, order: str = "round_robin") -> BlockInputs:
    """Timelines of message blocks for the text-level matching path."""
    spec = BLOCK_SPECS[config]
    seed = BASE_SEED + spec.index if seed is None else seed
    nt = spec.n_traj if n_traj is None else n_traj
    per_traj = [_block_trajectory(spec, seed, t) for t in range(nt)]
    keys = [2000 + 5 * t for t in range(nt)]
    items = []
    if order == "traj_major":
        for key, calls in zip(keys, per_traj):
            items += [(key, c) for c in calls]
    else:
        for k in range(max(len(c) for c in per_traj)):
            items += [(key, calls[k]) for key, calls in zip(keys, per_traj) if k < len(calls)]
    n = len(items)
    nb = np.array([len(c) for _, c in items], dtype=np.int64)
    block_offsets = np.zeros(n + 1, np.int64)
    np.cumsum(nb, out=block_offsets[1:])
    blocks = [b for _, c in items for b in c]
    lens = np.array([b["tok"].shape[0] for b in blocks], dtype=np.int64)
    tok_off = np.zeros(len(blocks) + 1, np.int64)
    np.cumsum(lens, out=tok_off[1:])
    tokens = np.concatenate([b["tok"] for b in blocks]).astype(np.int32)
    logp = np.concatenate([b.get("logp", np.zeros(b["tok"].shape[0], np.float32)) for b in blocks]).astype(np.float32)
    return BlockInputs(np.array([b["id"] for b in blocks], dtype=np.int64), block_offsets,
                       np.array([k for k, _ in items], dtype=np.int32), np.array([b["author"] for b in blocks], dtype=np.uint8),
                       tok_off, tokens, logp, meta=dict(config=config, seed=seed, vocab=spec.vocab, n_groups=nt))
