"""GPU parity: ajt_merge_timelines (through the C ABI) vs the brute-force oracle, bit for bit in all nine
outputs (pin P-M6), under both owner rules, on every BASELINE.json config plus edge cases."""
import json
import os

import numpy as np
import pytest
import torch

import oracle
import paper_2606_04484_b200 as ajt
from paper_2606_04484_b200 import workloads as W
from helpers import assert_merge_equal, gpu_merge

pytestmark = pytest.mark.gpu

RULES = [ajt.OWNER_LONGEST, ajt.OWNER_PAPER]


def oracle_merge(mi, rule, mask_in=None, with_logp=True):
    return oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, None if mask_in is not None else mi.resp_start,
                                  mask_in, mi.old_logp if with_logp else None, rule)


def from_lists(timelines, traj, resp_start, seed=0):
    lens = [len(t) for t in timelines]
    offsets = np.zeros(len(timelines) + 1, np.int64)
    offsets[1:] = np.cumsum(lens)
    tokens = np.array([x for t in timelines for x in t], dtype=np.int64).astype(np.int32)
    lp = -np.arange(1, tokens.shape[0] + 1, dtype=np.float32)
    return W.MergeInputs(tokens, offsets, np.array(traj, np.int32), np.array(resp_start, np.int32), lp)


@pytest.mark.parametrize("rule", RULES)
@pytest.mark.parametrize("cfg,order", [("c1", "round_robin"), ("c1", "traj_major"), ("c2", "round_robin")])
def test_configs_small(cfg, order, rule):
    mi = W.merge_workload(cfg, order=order)
    g, status = gpu_merge(mi, rule)
    assert status == 0
    assert_merge_equal(g, oracle_merge(mi, rule))


@pytest.mark.parametrize("rule", RULES)
def test_config_c4_both_models(rule):
    for model, mi in W.merge_workload_c4().items():
        g, status = gpu_merge(mi, rule)
        assert status == 0, model
        assert_merge_equal(g, oracle_merge(mi, rule))


@pytest.mark.parametrize("rule", RULES)
def test_config_c3_full_size(rule):
    mi = W.merge_workload("c3")
    g, status = gpu_merge(mi, rule)
    assert status == 0
    assert_merge_equal(g, oracle_merge(mi, rule))


@pytest.mark.parametrize("rule", RULES)
def test_explicit_mask_and_no_logp(rule):
    mi = W.merge_workload("c1")
    rng = np.random.default_rng(3)
    mk = (rng.random(mi.n_tokens) < 0.4).astype(np.uint8)      # arbitrary masks: overlapping members (reading M-7)
    g, status = gpu_merge(mi, rule, use_explicit_mask=True, mask_in=mk)
    assert status == 0
    assert_merge_equal(g, oracle_merge(mi, rule, mask_in=mk))
    g, status = gpu_merge(mi, rule, with_logp=False)
    assert_merge_equal(g, oracle_merge(mi, rule, with_logp=False))


@pytest.mark.parametrize("pad", [1, 2, 3])
def test_unaligned_token_base(pad):
    mi = W.merge_workload("c1")
    g, status = gpu_merge(mi, ajt.OWNER_LONGEST, pad=pad)
    assert status == 0
    assert_merge_equal(g, oracle_merge(mi, ajt.OWNER_LONGEST))


@pytest.mark.parametrize("rule", RULES)
@pytest.mark.parametrize("cfg", ["c1", "c2"])
def test_weak_hash_exercises_exact_repair_path(cfg, rule):
    # a 4-bit hash makes hash-equal, token-different candidates common: results must still be exact (M5)
    mi = W.merge_workload(cfg)
    g, status = gpu_merge(mi, rule, flags=ajt.MERGE_WEAK_HASH)
    assert status & ajt.STATUS_HASH_COLLISION and not (status & ~ajt.STATUS_HASH_COLLISION)
    assert_merge_equal(g, oracle_merge(mi, rule))


def test_hand_traces_on_gpu():
    with open(os.path.join(os.path.dirname(__file__), "golden", "merge_hand_traces.json")) as f:
        cases = json.load(f)["cases"]
    for c in cases:
        mi = from_lists(c["timelines"], c["traj"], c["resp_start"])
        for rule in RULES:
            for flags in (0, ajt.MERGE_WEAK_HASH):
                g, status = gpu_merge(mi, rule, flags=flags)
                assert not (status & ~ajt.STATUS_HASH_COLLISION), c["name"]
                assert_merge_equal(g, oracle_merge(mi, rule))


def test_random_tiny_cases():
    rng = np.random.default_rng(77)
    for trial in range(120):
        n = int(rng.integers(1, 40))
        ng = int(rng.integers(1, 5))
        tls, groups = [], []
        for j in range(n):
            gsel = int(rng.integers(0, ng))
            same = [t for t, gg in zip(tls, groups) if gg == gsel]
            if same and rng.random() < 0.75:
                base = list(same[int(rng.integers(0, len(same)))])
                m = rng.random()
                if m < 0.6:
                    base = base + [int(x) for x in rng.integers(0, 3, size=int(rng.integers(0, 300)))]
                elif m < 0.8:
                    base = base[:max(1, int(rng.integers(1, len(base) + 1)))]
                t = base
            else:
                t = [int(x) for x in rng.integers(0, 3, size=int(rng.integers(1, 200)))]
            tls.append(t)
            groups.append(gsel)
        mi = from_lists(tls, [g * 11 - 20 for g in groups], [int(rng.integers(0, len(t) + 1)) for t in tls])
        for rule in RULES:
            g, status = gpu_merge(mi, rule, flags=ajt.MERGE_WEAK_HASH if trial % 3 == 0 else 0)
            assert not (status & ~ajt.STATUS_HASH_COLLISION)
            assert_merge_equal(g, oracle_merge(mi, rule))


def test_edge_cases():
    # n = 1; all singletons; one long timeline spanning many hash windows; duplicates; negative tokens
    rng = np.random.default_rng(5)
    mi = from_lists([[3, 4, 5]], [9], [1])
    g, st = gpu_merge(mi, ajt.OWNER_LONGEST)
    assert st == 0
    assert_merge_equal(g, oracle_merge(mi, ajt.OWNER_LONGEST))
    mi = from_lists([[int(x) for x in rng.integers(-5, 5, size=50)] for _ in range(30)], list(range(30)), [10] * 30)
    g, st = gpu_merge(mi, ajt.OWNER_PAPER)
    assert st == 0 and g.M == 30
    assert_merge_equal(g, oracle_merge(mi, ajt.OWNER_PAPER))
    long = [int(x) for x in rng.integers(-2**31, 2**31 - 1, size=70000)]
    mi = from_lists([long[:10], long[:2049], long[:2048], long[:40000], long, long, long[:69999]], [0] * 7,
                    [5, 100, 2048, 39000, 69000, 70000, 0])
    for rule in RULES:
        g, st = gpu_merge(mi, rule)
        assert st == 0
        assert_merge_equal(g, oracle_merge(mi, rule))


def test_one_giant_group_uses_global_sort_path():
    # k = 120 timelines in one group -> 7260 keys > 2048: the segmented sort goes through global memory
    rng = np.random.default_rng(8)
    base = [int(x) for x in rng.integers(0, 50, size=4000)]
    tls = []
    for j in range(120):
        L = int(rng.integers(1, 4000))
        t = base[:L]
        if rng.random() < 0.3:
            t = t[:-1] + [t[-1] + 1]
        tls.append(t)
    mi = from_lists(tls, [5] * 120, [int(rng.integers(0, len(t))) for t in tls])
    for rule in RULES:
        for flags in (0, ajt.MERGE_WEAK_HASH):
            g, st = gpu_merge(mi, rule, flags=flags)
            assert not (st & ~ajt.STATUS_HASH_COLLISION)
            assert_merge_equal(g, oracle_merge(mi, rule))


def test_many_timelines_uses_the_global_memory_group_kernel():
    # n > 7,936 timelines: grouping no longer fits one CTA's shared memory (merge_group_kernel<false>, arrays in the workspace)
    rng = np.random.default_rng(21)
    for n, ngroups in ((9000, 600), (20000, 4000)):
        gs = [int(rng.integers(0, ngroups)) for _ in range(n)]
        tls = [None] * n
        last = {}
        for j in range(n):
            g = gs[j]
            if g in last and rng.random() < 0.7:
                t = last[g] + [int(x) for x in rng.integers(0, 9, size=int(rng.integers(0, 12)))]
            else:
                t = [int(x) for x in rng.integers(0, 9, size=int(rng.integers(1, 30)))]
            tls[j] = t
            last[g] = t
        mi = from_lists(tls, [7 * g - 11 for g in gs], [int(rng.integers(0, len(t) + 1)) for t in tls])
        for rule in RULES:
            g, st = gpu_merge(mi, rule)
            assert st == 0, st
            assert_merge_equal(g, oracle_merge(mi, rule))
        assert g.M < n


def test_empty_and_invalid():
    dev = "cuda"
    z32 = torch.zeros(1, dtype=torch.int32, device=dev)
    out = ajt.merge_timelines(z32[:0], torch.zeros(1, dtype=torch.int64, device=dev), z32[:0], z32[:0])
    f = out.finalize()
    assert f.M == 0 and f.N_out == 0
    # zero-length timeline -> status bit
    tokens = torch.arange(6, dtype=torch.int32, device=dev)
    offs = torch.tensor([0, 3, 3, 6], dtype=torch.int64, device=dev)
    out = ajt.merge_timelines(tokens, offs, torch.zeros(3, dtype=torch.int32, device=dev),
                              torch.zeros(3, dtype=torch.int32, device=dev))
    assert ajt.last_status(out.workspace) & ajt.STATUS_ZERO_LEN
    offs = torch.tensor([0, 4, 3, 6], dtype=torch.int64, device=dev)
    out = ajt.merge_timelines(tokens, offs, torch.zeros(3, dtype=torch.int32, device=dev),
                              torch.zeros(3, dtype=torch.int32, device=dev))
    assert ajt.last_status(out.workspace) & ajt.STATUS_BAD_OFFSETS


def test_probe_capacity_status():
    # 200 timelines in one group need 20100 pairs; the default workspace holds 64*200+4096 = 16896: the status bit is set,
    # counts are {0, 0}, finalize() raises; a workspace sized from the group histogram works (no silent empty merge)
    tls = [[1] * (j + 1) for j in range(200)]
    mi = from_lists(tls, [0] * 200, [0] * 200)
    dev = "cuda"
    args = (torch.from_numpy(mi.tokens).to(dev), torch.from_numpy(mi.offsets).to(dev), torch.from_numpy(mi.traj_ids).to(dev),
            torch.from_numpy(mi.resp_start).to(dev), None, torch.from_numpy(mi.old_logp).to(dev))
    out = ajt.merge_timelines(*args)
    assert ajt.last_status(out.workspace) & ajt.STATUS_PROBE_CAPACITY
    assert out.counts.cpu().tolist() == [0, 0]
    with pytest.raises(ajt.AjtError):
        out.finalize()
    n_pairs = 200 * 201 // 2
    big = ajt.merge_workspace_bytes_for_pairs(mi.n, mi.n_tokens, n_pairs)
    assert big > ajt.merge_workspace_bytes(mi.n, mi.n_tokens)
    out = ajt.merge_timelines(*args, workspace_bytes=big)
    assert ajt.last_status(out.workspace) == 0
    assert_merge_equal(out.finalize(), oracle_merge(mi, ajt.OWNER_LONGEST))
    # the host-buffer call reports the same condition as an error code, and takes the pairs from a larger arena
    with pytest.raises(ajt.AjtError) as ei:
        ajt.merge_timelines_host(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp)
    assert ei.value.code == -3
    arena = torch.empty(ajt.merge_host_arena_bytes(mi.n, mi.n_tokens) + big, dtype=torch.uint8, device=dev)
    h = ajt.merge_timelines_host(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp, arena=arena)
    r = oracle_merge(mi, ajt.OWNER_LONGEST)
    assert h["status"] == 0 and h["M"] == r.M and np.array_equal(h["merged_tokens"][:r.N_out].numpy(), r.merged_tokens)


def test_long_trajectories_over_127_calls():
    # trajectories averaging more than ~127 LLM calls exceed the default pair capacity; sized from the histogram
    # they merge exactly.  4 trajectories x 160 calls, appended context, a few rewrites.
    rng = np.random.default_rng(31)
    tls, traj = [], []
    ctx = {g: [int(x) for x in rng.integers(0, 50, size=20)] for g in range(4)}
    for k in range(160):
        for g in range(4):
            if k and rng.random() < 0.05:
                c = int(rng.integers(0, len(ctx[g])))
                ctx[g] = ctx[g][:c] + [int(x) for x in rng.integers(50, 99, size=int(rng.integers(1, 30)))]
            ctx[g] = ctx[g] + [int(x) for x in rng.integers(0, 50, size=int(rng.integers(1, 12)))]
            tls.append(list(ctx[g]))
            traj.append(g)
    mi = from_lists(tls, traj, [max(0, len(t) - 3) for t in tls])
    n_pairs = 4 * (160 * 161 // 2)
    dev = "cuda"
    for rule in RULES:
        out = ajt.merge_timelines(torch.from_numpy(mi.tokens).to(dev), torch.from_numpy(mi.offsets).to(dev),
                                  torch.from_numpy(mi.traj_ids).to(dev), torch.from_numpy(mi.resp_start).to(dev), None,
                                  torch.from_numpy(mi.old_logp).to(dev), owner_rule=rule,
                                  workspace_bytes=ajt.merge_workspace_bytes_for_pairs(mi.n, mi.n_tokens, n_pairs))
        assert ajt.last_status(out.workspace) == 0
        assert_merge_equal(out.finalize(), oracle_merge(mi, rule))


def test_host_buffer_variant():
    mi = W.merge_workload("c1")
    h = ajt.merge_timelines_host(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp)
    r = oracle_merge(mi, ajt.OWNER_LONGEST)
    assert h["status"] == 0 and h["M"] == r.M and h["N_out"] == r.N_out
    assert np.array_equal(h["merged_tokens"][:r.N_out].numpy(), r.merged_tokens)
    assert np.array_equal(h["merged_mask"][:r.N_out].numpy(), r.merged_mask)
    assert np.array_equal(h["merged_src"][:r.N_out].numpy(), r.merged_src)
    assert np.array_equal(h["merged_old_logp"][:r.N_out].numpy(), r.merged_old_logp)
    assert np.array_equal(h["merged_offsets"][:r.M + 1].numpy(), r.merged_offsets)
    assert np.array_equal(h["owner"][:mi.n].numpy(), r.owner)
