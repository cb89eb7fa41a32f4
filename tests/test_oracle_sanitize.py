"""the oracle built with -fsanitize=address,undefined, run over the hand traces, random tiny merges, block
merges, the loss (plain and extended) and the pack routine in a child process.  Any out-of-bounds access, use of
uninitialised stack, signed overflow or misaligned access in oracle/ajt_oracle.c aborts the child."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CHILD = r'''
import json, os, sys
import numpy as np
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))
import oracle
oracle.build()
cases = json.load(open(os.path.join(ROOT, "tests", "golden", "merge_hand_traces.json")))["cases"]
for c in cases:
    lens = [len(t) for t in c["timelines"]]
    off = np.zeros(len(lens) + 1, np.int64); off[1:] = np.cumsum(lens)
    tok = np.array([x for t in c["timelines"] for x in t], np.int64).astype(np.int32)
    lp = -np.arange(1, tok.shape[0] + 1, dtype=np.float32)
    for rule in (0, 1):
        oracle.merge_timelines(tok, off, np.array(c["traj"], np.int32), np.array(c["resp_start"], np.int32), None, lp, rule)
rng = np.random.default_rng(0)
for _ in range(60):
    n = int(rng.integers(1, 14)); tls = []
    for j in range(n):
        if tls and rng.random() < 0.7:
            b = list(tls[int(rng.integers(0, len(tls)))]); tls.append(b + [int(x) for x in rng.integers(0, 3, size=int(rng.integers(0, 9)))])
        else:
            tls.append([int(x) for x in rng.integers(0, 3, size=int(rng.integers(1, 12)))])
    lens = [len(t) for t in tls]; off = np.zeros(n + 1, np.int64); off[1:] = np.cumsum(lens)
    tok = np.array([x for t in tls for x in t], np.int32)
    mk = (rng.random(tok.shape[0]) < 0.5).astype(np.uint8)
    r = oracle.merge_timelines(tok, off, rng.integers(0, 3, size=n).astype(np.int32), None, mk, np.zeros(tok.shape[0], np.float32), int(rng.integers(0, 2)))
    tl_seg = rng.integers(0, 4, size=n).astype(np.int32)
    oracle.pack_loss_inputs(r.merged_tokens, r.merged_mask, r.merged_old_logp, r.merged_offsets, r.merged_origin, tl_seg, np.ones(4, np.float32))
from paper_2606_04484_b200 import workloads as W
bi = W.block_workload("b1")
oracle.merge_blocks(bi.block_ids, bi.block_offsets, bi.traj_ids, bi.author, bi.tok_off, bi.tokens, bi.logp)
T, V, S = 37, 53, 5
z = rng.standard_normal((T, V)).astype(np.float32)
y = rng.integers(0, V, size=T).astype(np.int32); m = (rng.random(T) < 0.6).astype(np.uint8); sg = rng.integers(0, S, size=T).astype(np.int32)
old = rng.standard_normal(T).astype(np.float32) * 0.1 - 4; adv = rng.standard_normal(T).astype(np.float32)
oracle.policy_loss(z, y, old, adv, m, sg, S, 0.2, 0.28)
oracle.policy_loss(z, y, old, adv, m, sg, S, 0.2, 0.28, ref_logp=old + 0.01, kl_coef=2e-3)
print("SANITIZED-OK")
'''


def test_oracle_under_asan_ubsan():
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    ubsan = subprocess.run(["gcc", "-print-file-name=libubsan.so"], capture_output=True, text=True).stdout.strip()
    if not (os.path.isabs(asan) and os.path.exists(asan)):
        pytest.skip("libasan is not installed with this gcc")
    env = dict(os.environ, AJT_ORACLE_SANITIZE="1", LD_PRELOAD=asan + (":" + ubsan if os.path.exists(ubsan) else ""),
               ASAN_OPTIONS="detect_leaks=0:halt_on_error=1", UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1", OMP_NUM_THREADS="2")
    r = subprocess.run([sys.executable, "-c", "ROOT = %r\n" % ROOT + CHILD], env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and "SANITIZED-OK" in r.stdout, (r.stdout[-2000:], r.stderr[-4000:])
