"""Pins for the merge oracle (CPU only).  DESIGN.md pins P-M1..P-M5.

The oracle (oracle/ajt_oracle.c) is the definition by brute force; here it is checked against things
other than itself: hand traces of Algorithm 1 stored under tests/golden/, a literal transcription of
Algorithm 1's reverse double loop in pure Python, a pure-Python set definition, invariants and a closed form.
"""
import json
import os

import numpy as np
import pytest

import oracle
from paper_2606_04484_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def pack(timelines, traj, resp_start):
    lens = [len(t) for t in timelines]
    offsets = np.zeros(len(timelines) + 1, np.int64)
    offsets[1:] = np.cumsum(lens)
    tokens = np.array([x for t in timelines for x in t], dtype=np.int64).astype(np.int32)
    return tokens, offsets, np.array(traj, np.int32), np.array(resp_start, np.int32)


# ------------------------------------------------------------------ P-M1 hand traces of Algorithm 1

with open(os.path.join(GOLDEN, "merge_hand_traces.json")) as f:
    TRACES = json.load(f)["cases"]


@pytest.mark.parametrize("case", TRACES, ids=[c["name"] for c in TRACES])
@pytest.mark.parametrize("rule", ["paper", "longest"])
def test_hand_traces(case, rule):
    tokens, offsets, traj, rs = pack(case["timelines"], case["traj"], case["resp_start"])
    logp = -np.arange(1, tokens.shape[0] + 1, dtype=np.float32)  # distinct per (timeline, position)
    r = oracle.merge_timelines(tokens, offsets, traj, rs, None, logp,
                               oracle.OWNER_PAPER if rule == "paper" else oracle.OWNER_LONGEST)
    assert r.merged_origin.tolist() == case["survivors"]
    assert r.owner.tolist() == case["owner_" + rule]
    exp = case["merged_" + rule]
    assert r.M == len(exp)
    assert r.merged_traj.tolist() == [case["traj"][s] for s in case["survivors"]]
    for m, e in enumerate(exp):
        a, b = r.merged_offsets[m], r.merged_offsets[m + 1]
        assert r.merged_tokens[a:b].tolist() == e["tokens"]
        assert r.merged_mask[a:b].tolist() == e["mask"]
        assert r.merged_src[a:b].tolist() == e["src"]
        for p, s in enumerate(e["src"]):   # log-prob comes from the src timeline at the same position
            want = 0.0 if s < 0 else float(logp[offsets[s] + p])
            assert r.merged_old_logp[a + p] == want
    assert r.N_out == sum(len(e["tokens"]) for e in exp)


def test_explicit_mask_two_members_same_position():
    # reading M-7: two members with mask 1 at the same position -> OR; src/logp from the largest index
    tokens, offsets, traj, _ = pack([[5, 6], [5, 6]], [0, 0], [0, 0])
    mask_in = np.array([1, 1, 0, 1], np.uint8)
    logp = np.array([-1, -2, -3, -4], np.float32)
    for rule in (oracle.OWNER_PAPER, oracle.OWNER_LONGEST):
        r = oracle.merge_timelines(tokens, offsets, traj, None, mask_in, logp, rule)
        assert r.merged_origin.tolist() == [1]
        assert r.merged_mask.tolist() == [1, 1]
        assert r.merged_src.tolist() == [0, 1]
        assert r.merged_old_logp.tolist() == [-1.0, -4.0]


def test_invalid_inputs():
    tokens, offsets, traj, rs = pack([[1], [1, 2]], [0, 0], [0, 0])
    bad = offsets.copy()
    bad[1] = 0  # zero-length timeline (reading M-9)
    with pytest.raises(ValueError):
        oracle.merge_timelines(tokens, bad, traj, rs)
    with pytest.raises(ValueError):
        oracle.merge_timelines(tokens, offsets, traj, rs, owner_rule=7)


# ------------------------------------------------------------------ P-M2 two independent formulations


def algorithm1_literal(timelines, groups, masks, logps):
    """Algorithm 1 transcribed line by line, with the repairs of reading M-1 and the
    group test of M-4 inside the match.  Works on per-token (author==llm) flags.  Returns survivors (in
    original order), absorber[j], and the merged per-token (mask, src, logp) of every survivor."""
    n = len(timelines)
    tok = [list(t) for t in timelines]
    llm = [list(m) for m in masks]
    lp = [list(x) for x in logps]
    src = [[j if m else -1 for m in masks[j]] for j in range(n)]
    absorbed = set()                                           # 1: A <- {}
    absorber = {}
    for i in range(n - 1, 0, -1):                              # 2: for i = n downto 2
        if i in absorbed:                                      # 3-5
            continue
        for j in range(i - 1, -1, -1):                         # 6: for j = i-1 downto 1
            if j in absorbed:                                  # 7-8
                continue
            if groups[i] == groups[j] and len(tok[i]) >= len(tok[j]) and \
                    all(tok[i][k] == tok[j][k] for k in range(len(tok[j]))):   # 9
                for k in range(len(tok[j])):                   # 10
                    if llm[j][k] and not llm[i][k]:            # 11
                        llm[i][k] = 1                          # 12
                        tok[i][k] = tok[j][k]                  # 13
                        lp[i][k] = lp[j][k]                    # 14
                        src[i][k] = src[j][k]
                absorbed.add(j)                                # 18
                absorber[j] = i
    survivors = [i for i in range(n) if i not in absorbed]     # 22
    return survivors, absorber, {s: (tok[s], llm[s], src[s], lp[s]) for s in survivors}


def set_definition(timelines, groups, masks, rule):
    """DESIGN.md O-M steps 1-4 as sets, pure Python, independent of the C oracle."""
    n = len(timelines)

    def ext(i, j):
        return (groups[i] == groups[j] and i > j and len(timelines[i]) >= len(timelines[j])
                and timelines[i][:len(timelines[j])] == timelines[j])

    E = {j: [i for i in range(n) if ext(i, j)] for j in range(n)}
    surv = [j for j in range(n) if not E[j]]
    own = {}
    for j in range(n):
        if not E[j]:
            own[j] = j
        elif rule == "paper":
            own[j] = max(E[j])
        else:
            C = [i for i in E[j] if i in surv]
            own[j] = min(C, key=lambda i: (-len(timelines[i]), i))
    merged = {}
    for s in surv:
        G = [j for j in range(n) if own[j] == s]
        mask, src = [], []
        for p in range(len(timelines[s])):
            K = [j for j in G if p < len(timelines[j]) and masks[j][p]]
            mask.append(1 if K else 0)
            src.append(max(K) if K else -1)
        merged[s] = (mask, src)
    return surv, own, merged


def random_tiny(rng, allow_explicit_mask):
    n = int(rng.integers(1, 13))
    alpha = int(rng.integers(2, 4))
    ngroups = int(rng.integers(1, 4))
    timelines, groups = [], []
    for j in range(n):
        g = int(rng.integers(0, ngroups))
        same = [t for t, gg in zip(timelines, groups) if gg == g]
        if same and rng.random() < 0.7:     # extend / copy / truncate an earlier one so prefixes are frequent
            base = list(same[int(rng.integers(0, len(same)))])
            mode = rng.random()
            if mode < 0.6:
                base = base + [int(x) for x in rng.integers(0, alpha, size=int(rng.integers(0, 5)))]
            elif mode < 0.8:
                base = base[:max(1, int(rng.integers(1, len(base) + 1)))]
            t = base[:16]
        else:
            t = [int(x) for x in rng.integers(0, alpha, size=int(rng.integers(1, 9)))]
        timelines.append(t)
        groups.append(g)
    if allow_explicit_mask:
        masks = [[int(x) for x in rng.integers(0, 2, size=len(t))] for t in timelines]
        rs = None
    else:
        rs = [int(rng.integers(0, len(t) + 1)) for t in timelines]
        masks = [[1 if p >= rs[j] else 0 for p in range(len(t))] for j, t in enumerate(timelines)]
    return timelines, groups, masks, rs


@pytest.mark.parametrize("explicit", [False, True])
def test_two_formulations_agree_with_oracle(explicit):
    rng = np.random.default_rng(1234 + explicit)
    n_branch = 0
    for trial in range(400):
        timelines, groups, masks, rs = random_tiny(rng, explicit)
        n = len(timelines)
        tokens, offsets, traj, _ = pack(timelines, [g * 5 - 3 for g in groups], [0] * n)
        mask_flat = np.array([m for mm in masks for m in mm], np.uint8)
        logp_flat = -np.arange(1, tokens.shape[0] + 1, dtype=np.float32)
        logps = [logp_flat[offsets[j]:offsets[j + 1]].tolist() for j in range(n)]
        rs_arr = None if explicit else np.array(rs, np.int32)
        mi = mask_flat if explicit else None

        # (A) literal Algorithm 1  vs  oracle under AJT_OWNER_PAPER
        surv, absorber, merged = algorithm1_literal(timelines, groups, masks, logps)
        r = oracle.merge_timelines(tokens, offsets, traj, rs_arr, mi, logp_flat, oracle.OWNER_PAPER)
        assert r.merged_origin.tolist() == surv
        for j in range(n):
            assert r.merged_origin[r.owner[j]] == absorber.get(j, j)
        for m, s in enumerate(surv):
            a, b = r.merged_offsets[m], r.merged_offsets[m + 1]
            tk, ll, sr, lp = merged[s]
            assert r.merged_tokens[a:b].tolist() == tk
            assert r.merged_mask[a:b].tolist() == ll
            assert r.merged_src[a:b].tolist() == sr
            got = r.merged_old_logp[a:b].tolist()
            assert got == [lp[p] if ll[p] else 0.0 for p in range(len(tk))]

        # (B) set definition vs oracle under both rules; survivors identical under both rules (lemma)
        for rule, rc in (("paper", oracle.OWNER_PAPER), ("longest", oracle.OWNER_LONGEST)):
            surv2, own, mg = set_definition(timelines, groups, masks, rule)
            r2 = oracle.merge_timelines(tokens, offsets, traj, rs_arr, mi, logp_flat, rc)
            assert surv2 == surv and r2.merged_origin.tolist() == surv
            assert [int(r2.merged_origin[o]) for o in r2.owner] == [own[j] for j in range(n)]
            assert np.array_equal(r2.merged_tokens, r.merged_tokens)
            assert np.array_equal(r2.merged_offsets, r.merged_offsets)
            for m, s in enumerate(surv):
                a, b = r2.merged_offsets[m], r2.merged_offsets[m + 1]
                assert r2.merged_mask[a:b].tolist() == mg[s][0]
                assert r2.merged_src[a:b].tolist() == mg[s][1]
        rl = oracle.merge_timelines(tokens, offsets, traj, rs_arr, mi, logp_flat, oracle.OWNER_LONGEST)
        n_branch += int(not np.array_equal(rl.owner, r.owner))
    assert n_branch > 5     # the random cases do exercise branching, where the two rules differ


# ------------------------------------------------------------------ P-M3 invariants


def check_invariants(mi: W.MergeInputs, r: oracle.MergeResult, mask_in=None):
    n = mi.n
    L = np.diff(mi.offsets)
    assert r.N_out <= mi.n_tokens
    assert r.merged_offsets[0] == 0 and r.merged_offsets[-1] == r.N_out
    assert np.all(np.diff(r.merged_origin) > 0)                      # original order
    assert np.array_equal(np.diff(r.merged_offsets), L[r.merged_origin])   # survivors keep their own length
    assert np.array_equal(r.merged_traj, mi.traj_ids[r.merged_origin])
    for j in range(n):                                               # recoverability (reading M-12)
        m = r.owner[j]
        assert 0 <= m < r.M
        assert r.merged_traj[m] == mi.traj_ids[j]
        a = r.merged_offsets[m]
        assert r.merged_offsets[m + 1] - a >= L[j]
        x = mi.tokens[mi.offsets[j]:mi.offsets[j + 1]]
        assert np.array_equal(r.merged_tokens[a:a + L[j]], x)
        if mask_in is None:
            mj = np.arange(L[j]) >= mi.resp_start[j]
        else:
            mj = mask_in[mi.offsets[j]:mi.offsets[j + 1]] != 0
        assert np.all(r.merged_mask[a:a + L[j]][mj] == 1)
        assert np.all(r.merged_src[a:a + L[j]][mj] >= j)
    # src consistency: src >= 0 <=> mask; src's owner is this sequence; logp gathered from src
    seq_of = np.repeat(np.arange(r.M), np.diff(r.merged_offsets))
    pos = np.arange(r.N_out) - r.merged_offsets[seq_of]
    has = r.merged_src >= 0
    assert np.array_equal(has, r.merged_mask == 1)
    assert np.array_equal(r.owner[r.merged_src[has]], seq_of[has])
    if r.merged_old_logp is not None:
        assert np.array_equal(r.merged_old_logp[has], mi.old_logp[mi.offsets[r.merged_src[has]] + pos[has]])
        assert np.all(r.merged_old_logp[~has] == 0)


@pytest.mark.parametrize("cfg,order", [("c1", "round_robin"), ("c1", "traj_major"), ("c2", "round_robin")])
@pytest.mark.parametrize("rule", [oracle.OWNER_LONGEST, oracle.OWNER_PAPER])
def test_invariants_on_configs(cfg, order, rule):
    mi = W.merge_workload(cfg, order=order, n_traj=16 if cfg == "c2" else None)
    r = oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp, rule)
    check_invariants(mi, r)
    assert r.N_out < mi.n_tokens
    # explicit mask equivalent to resp_start
    r2 = oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, None, W.explicit_mask(mi), mi.old_logp, rule)
    for f in ("merged_tokens", "merged_mask", "merged_src", "merged_old_logp", "merged_offsets", "merged_origin",
              "merged_traj", "owner"):
        assert np.array_equal(getattr(r, f), getattr(r2, f)), f
    # idempotence: merging the merged output changes nothing
    r3 = oracle.merge_timelines(r.merged_tokens, r.merged_offsets, r.merged_traj, None, r.merged_mask,
                                r.merged_old_logp, rule)
    assert r3.M == r.M and r3.N_out == r.N_out
    assert np.array_equal(r3.merged_tokens, r.merged_tokens)
    assert np.array_equal(r3.merged_mask, r.merged_mask)
    assert np.array_equal(r3.owner, np.arange(r.M))


def test_rules_share_survivors_and_branching_exists_on_c1():
    mi = W.merge_workload("c1")
    a = oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp, oracle.OWNER_LONGEST)
    b = oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp, oracle.OWNER_PAPER)
    for f in ("merged_tokens", "merged_offsets", "merged_origin", "merged_traj"):
        assert np.array_equal(getattr(a, f), getattr(b, f))
    assert not np.array_equal(a.owner, b.owner)     # cut-point rewrites create branching (reading M-15)
    assert a.merged_mask.sum() == b.merged_mask.sum() == sum(
        int(mi.offsets[j + 1] - mi.offsets[j] - mi.resp_start[j]) for j in range(mi.n))


def test_no_shared_prefix_means_equality():
    rng = np.random.default_rng(7)
    timelines = [[int(x) for x in rng.integers(0, 1 << 30, size=int(rng.integers(3, 20)))] for _ in range(20)]
    tokens, offsets, traj, rs = pack(timelines, [0] * 20, [1] * 20)
    r = oracle.merge_timelines(tokens, offsets, traj, rs)
    assert r.N_out == tokens.shape[0] and r.M == 20
    assert np.array_equal(r.merged_tokens, tokens) and np.array_equal(r.owner, np.arange(20))
    # N_out == N_in  <=>  nobody has an extender: adding one extender breaks equality
    timelines.append(timelines[3] + [1])
    tokens, offsets, traj, rs = pack(timelines, [0] * 21, [1] * 21)
    r = oracle.merge_timelines(tokens, offsets, traj, rs)
    assert r.N_out == tokens.shape[0] - len(timelines[3]) and r.M == 20


# ------------------------------------------------------------------ P-M5 closed form for a break-free chain


def test_chain_closed_form():
    with open(os.path.join(GOLDEN, "chain_closed_form.json")) as f:
        gold = json.load(f)
    for c in gold["cases"]:
        P, K, a = c["P"], c["K"], c["a"]
        rng = np.random.default_rng(P + K + a)
        ctx = [int(x) for x in rng.integers(0, 1 << 20, size=P)]
        timelines = []
        for k in range(K):
            ctx = ctx + [int(x) for x in rng.integers(0, 1 << 20, size=a)]
            timelines.append(list(ctx))
        tokens, offsets, traj, rs = pack(timelines, [3] * K, [len(t) - 1 for t in timelines])
        assert tokens.shape[0] == c["N_in"] == K * P + a * K * (K + 1) // 2
        r = oracle.merge_timelines(tokens, offsets, traj, rs)
        assert r.N_out == c["N_out"] == P + K * a and r.M == 1
    lo, hi = gold["paper_consistency"]["range"]
    for calls in gold["paper_consistency"]["calls"]:
        assert lo <= (calls + 1) / 2 <= hi
    assert abs(2160 / 346 - gold["paper_consistency"]["reported"]) < 0.01
