"""Pins for the block-level merge oracle (Algorithm 1 on message blocks).

P-B1 hand traces (tests/golden/block_hand_traces.json: Fig. 5's text-vs-token case, latest llm block wins, later-shorter
     absorbs first, episodes never mix)
P-B2 an independent formulation (Algorithm 1 on Python lists of dict blocks, absorbed SET, blocks mutated in place exactly as
     lines 12-14 say) agrees with the C oracle on random tiny inputs, both Match modes
P-B3 without tokenizer drift the flattened text-level result equals the (separately pinned) token-level oracle under the
     Algorithm-1 owner rule
P-B4 invariants on the seeded workloads; text-level merges at least as much as token-level
"""
import json
import os

import numpy as np
import pytest

import oracle
from paper_2606_04484_b200 import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))


def pack(timelines, traj):
    """timelines: list of lists of [id, author, tokens(, logp)]."""
    ids, auth, toks, lps, boff, toff = [], [], [], [], [0], [0]
    for tl in timelines:
        for b in tl:
            ids.append(b[0]); auth.append(b[1]); toks += list(b[2])
            lps += list(b[3]) if len(b) > 3 else [-(0.5 + 0.01 * len(lps) + 0.001 * k) for k in range(len(b[2]))]
            toff.append(len(toks))
        boff.append(len(ids))
    return dict(block_ids=np.array(ids, np.int64), block_offsets=np.array(boff, np.int64), traj_ids=np.array(traj, np.int32),
                author=np.array(auth, np.uint8), tok_off=np.array(toff, np.int64), tokens=np.array(toks, np.int32),
                logp=np.array(lps, np.float32))


CASES = json.load(open(os.path.join(HERE, "golden", "block_hand_traces.json")))["cases"]


@pytest.mark.parametrize("case", CASES, ids=[c["name"] for c in CASES])
def test_hand_traces(case):
    x = pack(case["timelines"], case["traj"])
    for mode, key in ((oracle.MATCH_TEXT, "text"), (oracle.MATCH_TOKEN, "token")):
        if key not in case:
            continue
        e = case[key]
        r = oracle.merge_blocks(**x, match=mode)
        assert r.M == e["M"]
        assert r.merged_origin.tolist() == e["origin"]
        assert r.owner.tolist() == e["owner"]
        assert r.merged_block_src.tolist() == e["block_src"]
        assert r.merged_block_author.tolist() == e["block_author"]
        assert r.merged_tokens.tolist() == e["tokens"]
        assert r.merged_mask.tolist() == e["mask"]
        assert r.merged_tok_src.tolist() == e["tok_src"]
        assert r.merged_offsets.tolist() == e["offsets"]
        assert r.merged_block_offsets.tolist() == e["block_offsets"]
        assert r.merged_block_tok_off.tolist() == e["block_tok_off"]
        # log-probs travel with the tokens (line 14): where the mask is 1 they are the supplying timeline's
        src_pos = []
        for m in range(r.M):
            s = int(r.merged_origin[m])
            for k in range(int(r.merged_block_offsets[m + 1] - r.merged_block_offsets[m])):
                sj = int(r.merged_block_src[r.merged_block_offsets[m] + k])
                sb = int(x["block_offsets"][sj]) + k
                src_pos += list(range(int(x["tok_off"][sb]), int(x["tok_off"][sb + 1])))
        want = np.where(r.merged_mask != 0, x["logp"][np.array(src_pos, np.int64)], 0.0).astype(np.float32)
        assert np.array_equal(r.merged_logp, want)


# ---- P-B2: Algorithm 1 written a second time, on Python objects

def algorithm1_python(timelines, traj, match):
    """timelines: list of lists of dict(id, author, tok, lp).  Mutates copies of the blocks exactly as lines 11-14 say."""
    T = [[dict(b, src=i) for b in tl] for i, tl in enumerate(timelines)]
    n = len(T)
    A = set()
    absorber = list(range(n))

    def same(a, b):
        return a["id"] == b["id"] if match == oracle.MATCH_TEXT else list(a["tok0"]) == list(b["tok0"])

    for i in range(n - 1, 0, -1):
        if i in A:
            continue
        for j in range(i - 1, -1, -1):
            if j in A or traj[j] != traj[i]:
                continue
            if len(T[i]) >= len(T[j]) and all(same(T[i][k], T[j][k]) for k in range(len(T[j]))):
                for k in range(len(T[j])):
                    if T[j][k]["author"] == 2 and T[i][k]["author"] != 2:
                        T[i][k]["author"] = 2
                        T[i][k]["tok"] = T[j][k]["tok"]
                        T[i][k]["lp"] = T[j][k]["lp"]
                        T[i][k]["src"] = T[j][k]["src"]
                A.add(j)
                absorber[j] = i
    surv = [i for i in range(n) if i not in A]
    return T, surv, absorber


def random_blocks(rng, n, n_groups):
    """Random tiny timelines with frequent shared prefixes, drift and edits."""
    pool = {}   # id -> canonical tokens
    tls, traj = [], []
    for i in range(n):
        g = int(rng.integers(0, n_groups))
        same = [t for t, tg in zip(tls, traj) if tg == g]
        if same and rng.random() < 0.75:
            base = same[int(rng.integers(0, len(same)))]
            keep = int(rng.integers(1, len(base) + 1))
            tl = []
            for b in base[:keep]:
                nb = dict(id=b["id"], author=0 if b["author"] == 2 else b["author"], tok=b["tok"], lp=[0.0] * len(b["tok"]))
                if b["author"] == 2 and rng.random() < 0.4 and len(b["tok"]) > 1:
                    nb["tok"] = b["tok"][1:]       # drift: same text, other tokens
                    nb["lp"] = [0.0] * len(nb["tok"])
                if rng.random() < 0.15:
                    nb["author"] = 2               # a block that is llm in both (a resampled call)
                    nb["lp"] = [-float(rng.random()) - 0.1 for _ in nb["tok"]]
                tl.append(nb)
        else:
            tl = []
        for _ in range(int(rng.integers(1, 4))):
            bid = int(rng.integers(1, 1 << 40))
            pool[bid] = [int(v) for v in rng.integers(0, 50, size=int(rng.integers(1, 5)))]
            au = int(rng.integers(0, 3))
            tl.append(dict(id=bid, author=au, tok=pool[bid], lp=[-float(rng.random()) - 0.1 if au == 2 else 0.0 for _ in pool[bid]]))
        for b in tl:
            b["tok0"] = b["tok"]
        tls.append(tl)
        traj.append(g)
    return tls, traj


@pytest.mark.parametrize("seed", range(40))
@pytest.mark.parametrize("mode", [oracle.MATCH_TEXT, oracle.MATCH_TOKEN])
def test_second_formulation(seed, mode):
    rng = np.random.default_rng(1000 + seed)
    tls, traj = random_blocks(rng, int(rng.integers(2, 14)), int(rng.integers(1, 4)))
    x = pack([[[b["id"], b["author"], b["tok"], b["lp"]] for b in tl] for tl in tls], traj)
    r = oracle.merge_blocks(**x, match=mode)
    T, surv, absorber = algorithm1_python(tls, traj, mode)
    assert r.merged_origin.tolist() == surv
    assert r.owner.tolist() == [surv.index(a) for a in absorber]
    toks = [t for s in surv for b in T[s] for t in b["tok"]]
    mask = [int(b["author"] == 2) for s in surv for b in T[s] for _ in b["tok"]]
    lps = [np.float32(lp) if b["author"] == 2 else np.float32(0) for s in surv for b in T[s] for lp in b["lp"]]
    assert r.merged_tokens.tolist() == toks and r.merged_mask.tolist() == mask
    assert np.array_equal(r.merged_logp, np.array(lps, np.float32))
    assert r.merged_block_src.tolist() == [b["src"] for s in surv for b in T[s]]
    assert r.merged_block_author.tolist() == [b["author"] for s in surv for b in T[s]]
    assert r.merged_block_offsets.tolist() == np.cumsum([0] + [len(T[s]) for s in surv]).tolist()


# ---- P-B3: no drift => the text-level result, flattened, is the token-level merge under Algorithm 1's owner rule

def test_no_drift_equals_token_level_oracle():
    spec = W.BLOCK_SPECS["b1"]
    W.BLOCK_SPECS["_nodrift"] = W.BlockSpec("_nodrift", 13, n_traj=24, turns=(5, 7), env_blocks=(1, 2), block_len=(4, 40), vocab=1024,
                                            p_break=spec.p_break, p_drift=0.0)
    bi = W.block_workload("_nodrift")
    r = oracle.merge_blocks(bi.block_ids, bi.block_offsets, bi.traj_ids, bi.author, bi.tok_off, bi.tokens, bi.logp)
    # the same timelines as flat token streams; mask = tokens of llm blocks
    offsets = bi.tok_off[bi.block_offsets]
    tmask = np.repeat((bi.author == W.AUTHOR_LLM).astype(np.uint8), np.diff(bi.tok_off))
    t = oracle.merge_timelines(bi.tokens, offsets, bi.traj_ids, None, tmask, bi.logp, owner_rule=oracle.OWNER_PAPER)
    assert (r.M, r.N_out) == (t.M, t.N_out) and r.M < bi.n
    assert np.array_equal(r.merged_tokens, t.merged_tokens) and np.array_equal(r.merged_mask, t.merged_mask)
    assert np.array_equal(r.merged_tok_src, t.merged_src) and np.array_equal(r.merged_logp, t.merged_old_logp)
    assert np.array_equal(r.merged_offsets, t.merged_offsets) and np.array_equal(r.merged_origin, t.merged_origin)
    assert np.array_equal(r.owner, t.owner) and np.array_equal(r.merged_traj, t.merged_traj)
    # and with no drift the two Match modes agree
    k = oracle.merge_blocks(bi.block_ids, bi.block_offsets, bi.traj_ids, bi.author, bi.tok_off, bi.tokens, bi.logp,
                            match=oracle.MATCH_TOKEN)
    assert np.array_equal(k.merged_tokens, r.merged_tokens) and np.array_equal(k.owner, r.owner)


# ---- P-B4: invariants on the seeded workloads

@pytest.mark.parametrize("config", ["b1", "b2"])
def test_invariants(config):
    bi = W.block_workload(config)
    r = oracle.merge_blocks(bi.block_ids, bi.block_offsets, bi.traj_ids, bi.author, bi.tok_off, bi.tokens, bi.logp)
    k = oracle.merge_blocks(bi.block_ids, bi.block_offsets, bi.traj_ids, bi.author, bi.tok_off, bi.tokens, bi.logp,
                            match=oracle.MATCH_TOKEN)
    assert r.M <= k.M < bi.n and r.N_out <= k.N_out    # "text ... yields more aggressive merging"
    assert r.M < k.M                                   # the drifted blocks make the difference (Fig. 5)
    assert r.B_out <= bi.block_ids.shape[0] and r.N_out == r.merged_tokens.shape[0]
    assert np.all(np.diff(r.merged_origin) > 0)        # original order (line 22)
    for j in range(bi.n):
        m = int(r.owner[j])
        s = int(r.merged_origin[m])
        assert bi.traj_ids[s] == bi.traj_ids[j] and s >= j
        Kj = int(bi.block_offsets[j + 1] - bi.block_offsets[j])
        mine = bi.block_ids[bi.block_offsets[j]:bi.block_offsets[j + 1]]
        assert np.array_equal(mine, bi.block_ids[bi.block_offsets[s]:bi.block_offsets[s] + Kj])      # recoverable prefix
        # "preserving which tokens were LLM-generated": every llm block of j is llm in its survivor
        llm = bi.author[bi.block_offsets[j]:bi.block_offsets[j + 1]] == W.AUTHOR_LLM
        got = r.merged_block_author[r.merged_block_offsets[m]:r.merged_block_offsets[m] + Kj]
        assert np.all(got[llm] == W.AUTHOR_LLM)
    # a block's tokens come from a member of the survivor's group that has the same text at that position
    for m in range(r.M):
        for k_ in range(int(r.merged_block_offsets[m + 1] - r.merged_block_offsets[m])):
            sj = int(r.merged_block_src[r.merged_block_offsets[m] + k_])
            assert int(r.owner[sj]) == m
            assert bi.block_ids[bi.block_offsets[sj] + k_] == bi.block_ids[bi.block_offsets[int(r.merged_origin[m])] + k_]


def test_rejects_bad_input():
    x = pack([[[1, 1, [1]]], []], [0, 0])     # the second timeline has no block: K_i >= 1 is required
    with pytest.raises(ValueError):
        oracle.merge_blocks(**x)


def test_explicit_token_mask_travels_with_the_tokens():
    """Reading B-2: when block k of the survivor takes tokens and log-probs from an absorbed timeline (lines 12-14), the per-token
    mask it carries is the supplier's; blocks the survivor keeps carry its own mask.  Hand example."""
    tls = [[[1, 1, [10, 11]], [2, 2, [20, 21, 22]]],                       # T_0: user, llm (generated here)
           [[1, 1, [10, 11]], [2, 0, [21, 22]], [3, 2, [30, 31]]]]         # T_1: the answer comes back re-tokenised, then a new answer
    x = pack(tls, [4, 4])
    #            T_0: u  u  l  l  l   T_1: u  u  e  e  l  l
    tok_mask = np.array([0, 1, 1, 0, 1,       1, 0, 1, 1, 0, 1], np.uint8)   # arbitrary per-token masks, not derived from authors
    r = oracle.merge_blocks(**x, tok_mask=tok_mask)
    assert r.M == 1 and r.merged_block_src.tolist() == [1, 0, 1]
    assert r.merged_tokens.tolist() == [10, 11, 20, 21, 22, 30, 31]
    assert r.merged_mask.tolist() == [1, 0, 1, 0, 1, 0, 1]               # T_1's own mask, T_0's for the replaced block, T_1's own
    assert r.merged_tok_src.tolist() == [1, -1, 0, -1, 0, -1, 1]
    want_lp = np.where(np.array(r.merged_mask) != 0, x["logp"][[5, 6, 2, 3, 4, 9, 10]], 0).astype(np.float32)
    assert np.array_equal(r.merged_logp, want_lp)
