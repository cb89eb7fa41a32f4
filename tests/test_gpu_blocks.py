"""GPU parity: ajt_merge_blocks (text-level matching; Alg. 1 lines 10-17) through the C ABI vs the
block-level oracle, bit-exact in every output.  Hand traces, random tiny inputs, the seeded block workloads (b1, b2 in full;
b3 at the size the oracle finishes in seconds), explicit token masks, weak hash (repair path), edge cases."""
import json
import os

import numpy as np
import pytest
import torch

import oracle
import paper_2606_04484_b200 as ajt
from paper_2606_04484_b200 import workloads as W

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))

FIELDS = ("merged_tokens", "merged_mask", "merged_logp", "merged_tok_src", "merged_offsets", "merged_block_offsets",
          "merged_block_src", "merged_block_author", "merged_block_tok_off", "merged_origin", "merged_traj", "owner")


def gpu_blocks(x, flags=0, tok_mask=None, with_logp=True):
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    out = ajt.merge_blocks(d(x["block_ids"]), d(x["block_offsets"]), d(x["traj_ids"]), d(x["author"]), d(x["tok_off"]),
                           d(x["tokens"]), d(x["logp"]) if with_logp else None, None if tok_mask is None else d(tok_mask),
                           flags=flags)
    status = ajt.last_status(out.workspace)
    return out.finalize(), status


def assert_equal(g, r):
    assert (g.M, g.B_out, g.N_out) == (r.M, r.B_out, r.N_out), ((g.M, g.B_out, g.N_out), (r.M, r.B_out, r.N_out))
    for f in FIELDS:
        b = getattr(r, f)
        a = getattr(g, f)
        if b is None:
            assert a is None
            continue
        a = a.cpu().numpy()
        if f == "merged_logp":
            a, b = a.view(np.uint32), b.view(np.uint32)
        if not np.array_equal(a, b):
            bad = np.nonzero(a != b)[0]
            raise AssertionError(f"{f}: {bad.size} mismatches, first at {bad[:5]}: gpu {a[bad[:5]]} oracle {b[bad[:5]]}")


def as_dict(bi):
    return dict(block_ids=bi.block_ids, block_offsets=bi.block_offsets, traj_ids=bi.traj_ids, author=bi.author,
                tok_off=bi.tok_off, tokens=bi.tokens, logp=bi.logp)


def run(x, flags=0, tok_mask=None, with_logp=True):
    g, status = gpu_blocks(x, flags, tok_mask, with_logp)
    assert status & ~ajt.STATUS_HASH_COLLISION == 0, status
    r = oracle.merge_blocks(x["block_ids"], x["block_offsets"], x["traj_ids"], x["author"], x["tok_off"], x["tokens"],
                            x["logp"] if with_logp else None, tok_mask)
    assert_equal(g, r)
    return g, r, status


def test_hand_traces():
    from test_oracle_blocks import CASES, pack
    for case in CASES:
        g, r, _ = run(pack(case["timelines"], case["traj"]))
        assert g.merged_tokens.cpu().tolist() == case["text"]["tokens"]
        assert g.merged_block_src.cpu().tolist() == case["text"]["block_src"]


@pytest.mark.parametrize("seed", range(12))
def test_random_tiny(seed):
    from test_oracle_blocks import pack, random_blocks
    rng = np.random.default_rng(5000 + seed)
    tls, traj = random_blocks(rng, int(rng.integers(2, 40)), int(rng.integers(1, 5)))
    run(pack([[[b["id"], b["author"], b["tok"], b["lp"]] for b in tl] for tl in tls], traj))


@pytest.mark.parametrize("config", ["b1", "b2"])
def test_seeded_workloads(config):
    bi = W.block_workload(config)
    g, r, _ = run(as_dict(bi))
    assert g.M < bi.n and g.N_out < bi.tokens.shape[0]
    if config == "b1":
        run(as_dict(W.block_workload(config, order="traj_major")))


def test_b3_reduced():
    bi = W.block_workload("b3", n_traj=48)     # several scan tiles (2048 merged blocks each), ~25 M tokens in
    g, r, _ = run(as_dict(bi))
    assert g.B_out > 2 * 2048


def test_explicit_token_mask_and_no_logp():
    bi = W.block_workload("b1")
    rng = np.random.default_rng(3)
    tm = (rng.random(bi.tokens.shape[0]) < 0.5).astype(np.uint8)
    run(as_dict(bi), tok_mask=tm)
    run(as_dict(bi), with_logp=False)


def test_weak_hash_takes_the_repair_path():
    bi = W.block_workload("b1")
    g, r, status = run(as_dict(bi), flags=ajt.MERGE_WEAK_HASH)


def test_empty_blocks_and_single_timeline():
    from test_oracle_blocks import pack
    x = pack([[[1, 1, [1, 2]], [2, 2, []], [3, 0, [4]]],
              [[1, 1, [1, 2]], [2, 0, []], [3, 0, [4]], [9, 2, [7, 7, 7]]]], [5, 5])
    run(x)
    run(pack([[[1, 2, [3]]]], [0]))


def test_probe_capacity_and_larger_workspace():
    # one group of 220 timelines: 24,310 (timeline, earlier length) pairs > the 64 n + 4096 the default workspace holds
    tls = [[[7, 1, [1]]] + [[100 + k, 2 if k == j else 0, [k]] for k in range(j + 1)] for j in range(220)]
    from test_oracle_blocks import pack
    x = pack(tls, [3] * 220)
    g, status = gpu_blocks(x)
    assert status & ajt.STATUS_PROBE_CAPACITY
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    out = ajt.merge_blocks(d(x["block_ids"]), d(x["block_offsets"]), d(x["traj_ids"]), d(x["author"]), d(x["tok_off"]), d(x["tokens"]),
                           d(x["logp"]), extra_workspace_bytes=32 * 24310)
    assert ajt.last_status(out.workspace) == 0
    r = oracle.merge_blocks(x["block_ids"], x["block_offsets"], x["traj_ids"], x["author"], x["tok_off"], x["tokens"], x["logp"])
    assert_equal(out.finalize(), r)
    assert r.M == 1


def test_bad_offsets_set_status():
    bi = W.block_workload("b1")
    x = as_dict(bi)
    x["block_offsets"] = x["block_offsets"].copy()
    x["block_offsets"][3] = x["block_offsets"][2]        # an empty timeline
    g, status = gpu_blocks(x)
    assert status & (ajt.STATUS_ZERO_LEN | ajt.STATUS_BAD_OFFSETS)
