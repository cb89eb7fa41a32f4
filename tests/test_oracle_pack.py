"""Pins for oracle.pack_loss_inputs (reading L-12: next-token alignment inside each merged sequence).

P-K1 hand example; P-K2 a second formulation (one global shift, then the sequence ends are cleared) on the seeded c1 merge;
P-K3 the property that makes it the right alignment: scoring the packed rows with a next-token model's own log-probs gives,
per sequence, exactly sum_{q>=1} mask[q] log p(x_q | x_<q) computed sequence by sequence."""
import numpy as np

import oracle
from helpers import seg_ids_from_merged, shift_for_next_token
from paper_2606_04484_b200 import workloads as W


def test_hand_example():
    # two sequences: [5 6 7] (mask 0 1 1, survivor timeline 3) and [8 9] (mask 0 1, survivor timeline 1)
    tok = np.array([5, 6, 7, 8, 9], np.int32)
    msk = np.array([0, 1, 1, 0, 1], np.uint8)
    lp = np.array([0, -.5, -.25, 0, -1.5], np.float32)
    off = np.array([0, 3, 5], np.int64)
    origin = np.array([3, 1], np.int32)
    tl_seg = np.array([9, 0, 9, 2], np.int32)
    adv = np.array([1.5, 0.0, -2.0], np.float32)
    t, m, o, s, a = oracle.pack_loss_inputs(tok, msk, lp, off, origin, tl_seg, adv)
    assert t.tolist() == [6, 7, 0, 9, 0]
    assert m.tolist() == [1, 1, 0, 1, 0]
    assert o.tolist() == [-.5, -.25, 0, -1.5, 0]
    assert s.tolist() == [2, 2, 2, 0, 0]
    assert a.tolist() == [-2.0, -2.0, -2.0, 1.5, 1.5]


def test_global_shift_formulation():
    mi = W.merge_workload("c1")
    r = oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp)
    uniq, tl_seg = np.unique(mi.traj_ids, return_inverse=True)
    t, m, o, s, _ = oracle.pack_loss_inputs(r.merged_tokens, r.merged_mask, r.merged_old_logp, r.merged_offsets, r.merged_origin,
                                            tl_seg.astype(np.int32))
    t2, m2, o2 = shift_for_next_token(r.merged_tokens, r.merged_mask, r.merged_old_logp, r.merged_offsets)
    s2, S, _ = seg_ids_from_merged(r.merged_offsets, r.merged_traj)
    assert np.array_equal(t, t2) and np.array_equal(m, m2) and np.array_equal(o, o2) and np.array_equal(s, s2)
    assert S == uniq.shape[0]


def test_alignment_scores_each_sequence():
    rng = np.random.default_rng(5)
    V = 11
    lens = [4, 1, 6, 2]
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    tok = rng.integers(0, V, size=off[-1]).astype(np.int32)
    msk = (rng.random(off[-1]) < 0.6).astype(np.uint8)
    table = rng.standard_normal((V, V))                      # a bigram "model": log p(next | current) = table[current, next]
    t, m, _, _, _ = oracle.pack_loss_inputs(tok, msk, None, off, np.arange(4, dtype=np.int32), np.zeros(4, np.int32))
    packed = sum(float(table[tok[q], t[q]]) for q in range(off[-1]) if m[q])
    direct = 0.0
    for k in range(4):
        x, mm = tok[off[k]:off[k + 1]], msk[off[k]:off[k + 1]]
        direct += sum(float(table[x[q - 1], x[q]]) for q in range(1, len(x)) if mm[q])
    assert abs(packed - direct) < 1e-12
    assert int(m.sum()) == sum(int(msk[off[k] + 1:off[k + 1]].sum()) for k in range(4))


def test_pack_microbatches_hand_and_properties():
    # P-K4 hand example (budget 10): 5+5 fits, the third 5 opens a batch, 20 is alone (longer than the budget), 1+1 close
    assert oracle.pack_microbatches([5, 5, 5, 20, 1, 1], 10) == [(0, 2), (2, 3), (3, 4), (4, 6)]
    assert oracle.pack_microbatches([], 10) == []
    assert oracle.pack_microbatches([3], 10) == [(0, 1)]
    # P-K5 what "greedy, in order" fixes on random inputs: the batches tile the sequences in order; a batch is within the
    # budget unless it is a single sequence; and it is maximal (the next sequence would not have fitted)
    rng = np.random.default_rng(5)
    for _ in range(200):
        L = [int(x) for x in rng.integers(1, 40, size=int(rng.integers(1, 60)))]
        B = int(rng.integers(1, 80))
        mb = oracle.pack_microbatches(L, B)
        assert mb[0][0] == 0 and mb[-1][1] == len(L) and all(mb[i][1] == mb[i + 1][0] for i in range(len(mb) - 1))
        for a, b in mb:
            assert b > a and (sum(L[a:b]) <= B or b - a == 1)
            if b < len(L):
                assert sum(L[a:b]) + L[b] > B
