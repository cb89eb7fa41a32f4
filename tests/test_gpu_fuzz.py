"""GPU fuzz against the oracle: seeded random inputs at small and medium sizes that mix the conditions the targeted tests take
one at a time (many members per survivor, duplicates, one-token differences, unaligned bases, explicit masks, both owner
rules, weak hash -> repair path, pair capacity; every loss kernel variant with ragged vocabularies, padded rows, in-place
backward, extreme mask densities; random LM-head shapes).  An earlier run of these generators found the only out-of-bounds
read this library had (block merge after a fatal status)."""
import numpy as np
import pytest
import torch
from types import SimpleNamespace

import oracle
import paper_2606_04484_b200 as ajt
from helpers import assert_merge_equal

pytestmark = pytest.mark.gpu


def rand_merge(rng):
    n = int(rng.integers(1, 120)); ng = int(rng.integers(1, 9)); alpha = int(rng.integers(2, 6))
    scale = int(rng.choice([4, 40, 400, 3000]))
    tls, gs = [], []
    for _ in range(n):
        g = int(rng.integers(0, ng))
        same = [t for t, gg in zip(tls, gs) if gg == g]
        if same and rng.random() < 0.8:
            base = same[int(rng.integers(0, len(same)))] if rng.random() < 0.5 else same[-1]
            m = rng.random()
            if m < 0.65:
                t = np.concatenate([base, rng.integers(0, alpha, size=int(rng.integers(0, scale)))])
            elif m < 0.8:
                t = base[:max(1, int(rng.integers(1, len(base) + 1)))]
            elif m < 0.9:
                t = base.copy(); k = int(rng.integers(0, len(t))); t[k] = (t[k] + 1) % alpha
            else:
                t = base.copy()
        else:
            t = rng.integers(0, alpha, size=int(rng.integers(1, scale + 1)))
        tls.append(t.astype(np.int32)); gs.append(g)
    offsets = np.zeros(n + 1, np.int64)
    np.cumsum([len(t) for t in tls], out=offsets[1:])
    tokens = np.concatenate(tls).astype(np.int32)
    return SimpleNamespace(tokens=tokens, offsets=offsets, traj_ids=(np.array(gs, np.int32) * 977 - 5000).astype(np.int32),
                           resp_start=np.array([int(rng.integers(0, len(t) + 1)) for t in tls], np.int32),
                           old_logp=(-rng.random(tokens.shape[0])).astype(np.float32), n_tokens=int(tokens.shape[0]), n=n)


@pytest.mark.parametrize("chunk", range(4))
def test_merge_fuzz(chunk):
    for c in range(60):
        rng = np.random.default_rng(31000 + 60 * chunk + c)
        mi = rand_merge(rng)
        rule, flags, explicit, pad = int(rng.integers(0, 2)), int(rng.integers(0, 2)), bool(rng.integers(0, 2)), int(rng.integers(0, 4))
        d = lambda a: torch.from_numpy(a).cuda()
        tf = torch.zeros(mi.n_tokens + pad, dtype=torch.int32, device="cuda")
        tf[pad:] = d(mi.tokens)
        mk_np = None
        if explicit:
            mk_np = np.concatenate([(np.arange(mi.offsets[j + 1] - mi.offsets[j]) >= mi.resp_start[j]) for j in range(mi.n)])
            mk_np = np.where(rng.random(mk_np.shape[0]) < 0.1, ~mk_np, mk_np).astype(np.uint8)
        out = ajt.merge_timelines(tf[pad:], d(mi.offsets), d(mi.traj_ids), None if explicit else d(mi.resp_start),
                                  d(mk_np) if explicit else None, d(mi.old_logp), owner_rule=rule, flags=flags)
        st = ajt.last_status(out.workspace)
        if st & ajt.STATUS_PROBE_CAPACITY:
            assert out.counts.cpu().tolist() == [0, 0]
            continue
        assert st & ~ajt.STATUS_HASH_COLLISION == 0, (c, st)
        r = oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, None if explicit else mi.resp_start, mk_np, mi.old_logp, rule)
        assert_merge_equal(out.finalize(), r)


@pytest.mark.parametrize("chunk", range(3))
def test_blocks_fuzz(chunk):
    from test_gpu_blocks import assert_equal, gpu_blocks
    from test_oracle_blocks import pack, random_blocks
    for c in range(70):
        rng = np.random.default_rng(32000 + 70 * chunk + c)
        tls, traj = random_blocks(rng, int(rng.integers(2, 200)), int(rng.integers(1, 7)))
        x = pack([[[b["id"], b["author"], b["tok"], b["lp"]] for b in tl] for tl in tls], traj)
        g, st = gpu_blocks(x, flags=int(rng.integers(0, 2)))
        if st & ajt.STATUS_PROBE_CAPACITY:
            assert (g.M, g.B_out, g.N_out) == (0, 0, 0)
            continue
        assert st & ~ajt.STATUS_HASH_COLLISION == 0, (c, st)
        assert_equal(g, oracle.merge_blocks(x["block_ids"], x["block_offsets"], x["traj_ids"], x["author"], x["tok_off"], x["tokens"],
                                            x["logp"]))


VS = [8, 24, 1000, 1001, 4864, 4872, 9728, 38912, 38920, 77824, 77832, 100000, 128256, 151936, 155640, 155648, 160000]


@pytest.mark.parametrize("chunk", range(3))
def test_loss_fuzz(chunk):
    from test_gpu_loss import run_and_check
    from test_gpu_loss_ext import run_ext
    for c in range(16):
        seed = 33000 + 16 * chunk + c
        rng = np.random.default_rng(seed)
        V = int(rng.choice(VS)); T = int(rng.integers(1, 200 if V > 50000 else 700)); S = int(rng.integers(1, 40))
        rho = float(rng.choice([0.0, 0.05, 0.3, 0.7, 1.0])); dt = torch.bfloat16 if rng.random() < 0.8 else torch.float32
        pad = int(rng.choice([0, 0, 8, 64, 3])); eps = (float(rng.choice([0.1, 0.2])), float(rng.choice([0.2, 0.28])))
        gs = float(rng.choice([1.0, 1.0, 0.37, 3.0]))
        if rng.random() < 0.5:
            run_and_check(T, V, S, rho, dt, sigma=float(rng.choice([1.0, 3.0])), eps=eps, grad_scale=gs, seed=seed, ld=V + pad if pad else None,
                          inplace=(dt == torch.bfloat16 and pad == 0 and rng.random() < 0.3))
        else:
            run_ext(T, V, S, rho, dt, kl_coef=float(rng.choice([0.0, 2e-3, 0.5])), sigma=float(rng.choice([1.0, 3.0])), eps=eps, seed=seed,
                    with_ref=bool(rng.random() < 0.8), grad_scale=gs)


def test_lm_head_fuzz():
    from test_gpu_lmhead import run
    for c in range(120):
        rng = np.random.default_rng(34000 + c)
        T = int(rng.integers(1, 700)); d = 64 * int(rng.integers(1, 9))
        V = int(rng.choice([8, 100, 255, 256, 257, 1023, 1024, 1025, 5000, 20011]))
        run(T, d, V, seed=34000 + c, mask_frac=(None if rng.random() < 0.5 else 0.5), wscale=float(rng.choice([0.05, 0.3])))
