#!/usr/bin/env python
"""bench.py — one "step" = one pass of the whole hot path (SURVEY.md §8(a) rows M1-M7 + L0-L4) over one
synthetic batch of BASELINE.json configs[1] ("single-model GRPO batch"):

    ajt_merge_timelines      over the batch's 512 timelines (N_in ~ 1.76 M tokens)
    ajt_policy_loss_fwd_bwd  over one 40,960-row micro-batch of the merged tokens, bf16 logits [40960,151936]

`value` = algorithmic bytes of the step / device time (GB/s), inputs resident in HBM.  `e2e` = the same metric
through the *_host C-ABI calls with pinned HOST buffers (H2D and D2H inside the timed region).
`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload.

Launch: `python bench.py --gpus N --steps K --warmup W`; for N>1 under torch.distributed.run (one rank per GPU,
weak scaling: every rank runs its own seeded batch, no data-path collective — merging never crosses trajectories
and loss rows are independent given the per-trajectory normalisers).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "merge Gtokens/s and policy-loss fwd+bwd logits GB/s (fraction of B200 HBM peak)"
MB_ROWS = 40960          # loss micro-batch rows (BASELINE.json configs[1]: "~40k merged tokens")
V = 151936
EPS = (0.2, 0.28)

from paper_2606_04484_b200.harness import (NOMINAL_HBM_GBS, loss_bytes as _loss_bytes, measured_peak, merge_bytes)  # noqa: E402


def loss_bytes(T: int, Vv: int, n_unmasked: int, b_in: int = 2) -> int:
    return _loss_bytes(T, Vv, n_unmasked, b_in)


# ----------------------------------------------------------------------------------------- clocks sampler


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML every 20 ms on a thread (nvidia-smi -lms block-buffers
    its output when piped, so the same counters are read in-process)."""
    BAD = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.stop_flag = threading.Event()
        self.th = None
        self.max_mhz = None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            idx = self.index
            if vis:
                try:
                    idx = int(vis.split(",")[self.index])
                except Exception:
                    idx = self.index
            h = pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
        except Exception:
            return

        def rd():
            while not self.stop_flag.is_set():
                try:
                    mhz = float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM))
                    try:
                        rs = int(pynvml.nvmlDeviceGetCurrentClocksEventReasons(h))
                    except Exception:
                        rs = int(pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(h))
                    try:
                        pw = pynvml.nvmlDeviceGetPowerUsage(h) / 1000.0
                    except Exception:
                        pw = None
                    self.rows.append((time.time(), mhz, rs, pw))
                except Exception:
                    pass
                time.sleep(0.02)
        self.th = threading.Thread(target=rd, daemon=True)
        self.th.start()

    def stop(self):
        self.stop_flag.set()
        if self.th is not None:
            self.th.join(timeout=2)

    def summary(self, t0: float, t1: float) -> dict:
        sel = [r for r in self.rows if t0 <= r[0] <= t1] or [r for r in self.rows if t0 - 0.05 <= r[0] <= t1 + 0.05]
        reasons = set()
        for r in sel:
            for bit, nm in self.BAD.items():
                if r[2] & bit:
                    reasons.add(nm)
        pw = [r[3] for r in sel if r[3] is not None]
        return {"sm_mhz": float(np.median([r[1] for r in sel])) if sel else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(reasons), "samples": len(sel), "power_w_max": max(pw) if pw else None}


# ----------------------------------------------------------------------------------------- workload (harness)


def harness_old_logp(torch, logits_t, targets_t, noise):
    from paper_2606_04484_b200.harness import harness_old_logp as f
    return f(logits_t, targets_t, noise)


def fill_logits(torch, buf, seed: int, sigma: float = 3.0, slab: int = 2048):
    from paper_2606_04484_b200.harness import fill_logits as f
    f(buf, seed, sigma, slab)


def loss_side_inputs(W, merged_tokens, merged_mask, merged_old_logp, merged_offsets, merged_traj, seed: int):
    """Index plumbing from the merge output to the loss call (reading L-12) plus the batch-wide
    per-trajectory normalisers the caller owns when it streams micro-batches (reading L-4)."""
    targets, mask, _ = W.shift_for_next_token(merged_tokens, merged_mask, merged_old_logp, merged_offsets)
    seg, S, _ = W.seg_ids_from_merged(merged_offsets, merged_traj)
    adv = W.advantages_group_zscore(seed, 1, S)[seg]
    Ns = np.bincount(seg, weights=mask.astype(np.float64), minlength=S).astype(np.float32)
    inv = 1.0 / max(1, int((Ns > 0).sum()))
    return targets, mask, seg, S, adv.astype(np.float32), Ns, float(np.float32(inv))


def oracle_step_time(oracle, mi, logits_bits, targets, old_logp, adv, mask, seg, S, Ns, inv, rows: int):
    """Times the oracle, as it stands, on (full merge) + (the first `rows` rows of the loss micro-batch).
    Returns (t_merge, t_loss_rows, n_unmasked_in_rows)."""
    t0 = time.perf_counter()
    oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp, oracle.OWNER_LONGEST)
    t1 = time.perf_counter()
    rid = np.arange(rows, dtype=np.int64)
    oracle.policy_loss(logits_bits[:rows], targets, old_logp, adv, mask, seg, S, float(np.float32(EPS[0])),
                       float(np.float32(EPS[1])), seg_denom=Ns, inv_num_segs=inv, row_ids=rid, want_dlogits=True,
                       logits_is_bf16_bits=True)
    t2 = time.perf_counter()
    return t1 - t0, t2 - t1, int(mask[:rows].sum())


def extrapolated_gbs(n, N_in, N_out, T, n_unmasked_full, t_merge, t_loss_rows, rows, n_unmasked_rows):
    """Loss rows are independent: the micro-batch's loss time is extrapolated from the sample at the sample's
    algorithmic byte rate; the merge is timed in full."""
    rate = loss_bytes(rows, V, n_unmasked_rows) / max(t_loss_rows, 1e-9)
    t_step = t_merge + loss_bytes(T, V, n_unmasked_full) / rate
    return (merge_bytes(n, N_in, N_out) + loss_bytes(T, V, n_unmasked_full)) / t_step / 1e9, t_step


# ----------------------------------------------------------------------------------------- reference arm (oracle)


def run_reference(args, rank: int):
    """`--impl reference`: the CPU oracle as it stands, on the box's host cores, same config / metric / unit.
    Each step = the full merge of the batch + a bounded sample of loss rows (the rest extrapolated; rows are
    independent).  Under torchrun only rank 0 works."""
    if rank != 0:
        return
    import torch

    import oracle
    from paper_2606_04484_b200 import workloads as W

    oracle.build()
    seed = W.BASE_SEED + 1
    mi = W.merge_workload("c2", seed=seed)
    r = oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp, oracle.OWNER_LONGEST)
    targets, mask, seg, S, adv, Ns, inv = loss_side_inputs(W, r.merged_tokens, r.merged_mask, r.merged_old_logp,
                                                           r.merged_offsets, r.merged_traj, seed)
    T = min(args.loss_rows, r.N_out)
    targets, mask, seg, adv = targets[:T], mask[:T], seg[:T], adv[:T]
    rows_max = 1024
    g = torch.Generator().manual_seed(seed)
    logits = (torch.randn((rows_max, V), generator=g) * 3.0).to(torch.bfloat16)
    noise = (W.rng_for(seed, 1, 99).standard_normal(T) * 0.05).astype(np.float32)
    old = np.zeros(T, np.float32)
    old[:rows_max] = harness_old_logp(torch, logits, torch.from_numpy(targets[:rows_max]), noise[:rows_max]).numpy()
    bits = logits.view(torch.int16).numpy().view(np.uint16)
    # calibrate: size the per-step sample so that warmup + steps stay within ~2 minutes
    tm, tl, nu = oracle_step_time(oracle, mi, bits, targets, old, adv, mask, seg, S, Ns, inv, 64)
    budget = 120.0 / max(1, args.steps + args.warmup)
    rows = int(min(rows_max, max(64, 64 * max(0.0, budget - tm) / max(tl, 1e-6))))
    for _ in range(args.warmup):
        oracle_step_time(oracle, mi, bits, targets, old, adv, mask, seg, S, Ns, inv, rows)
    t_m = t_l = 0.0
    t0 = time.perf_counter()
    for _ in range(args.steps):
        a, b, nu = oracle_step_time(oracle, mi, bits, targets, old, adv, mask, seg, S, Ns, inv, rows)
        t_m += a
        t_l += b
    wall = time.perf_counter() - t0
    K = max(1, args.steps)
    val, t_step = extrapolated_gbs(mi.n, mi.n_tokens, r.N_out, T, int(mask.sum()), t_m / K, t_l / K, rows, nu)
    cores = oracle.num_threads()
    sample = (f"per step: full merge of the batch ({mi.n} timelines, {mi.n_tokens} tokens) + first {rows} of {T} loss rows "
              f"({nu} unmasked) x V={V}; micro-batch time extrapolated at the sample's byte rate (rows are independent)")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "GB/s", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t_step * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64 (oracle)", "data": "synthetic",
            "config": workload_config(mi.n, mi.n_tokens, r.N_out, T, float(mask.mean())),
            "cpu_baseline": {"value": val, "unit": "GB/s", "cores": cores, "kind": "oracle", "sample": sample,
                             "measured_wall_s": wall},
            "e2e": {"value": val, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def workload_config(n, N_in, N_out, T, rho):
    return {"workload": "BASELINE.json configs[1] single-model GRPO batch: merge of 64 trajectories x 8 turns "
                        f"({n} timelines, N_in={N_in}, N_out={N_out}) + policy-loss fwd+bwd over one micro-batch "
                        f"[{T},{V}] bf16 of the merged tokens (mask density {rho:.3f}), eps 0.2/0.28, group z-score adv",
            "owner_rule": "longest", "loss_rows": T, "vocab": V, "merge_timelines": n, "N_in": N_in, "N_out": N_out,
            "l2": "inputs larger than L2: every step streams the 12.4 GB logits micro-batch (two buffers alternate), "
                  "which also evicts the 7 MB merge input between merge calls"}


# ----------------------------------------------------------------------------------------- our arm (CUDA)


def run_ours(args, rank: int, world: int, local_rank: int):
    import torch
    import torch.distributed as dist

    import paper_2606_04484_b200 as ajt
    from paper_2606_04484_b200 import workloads as W

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    ajt.lib()  # fail loudly if libajt.so is missing

    # ---- inputs (seeded, synthetic; weak scaling: every rank owns its own batch)
    seed = W.BASE_SEED + 1 + 1000 * rank
    mi = W.merge_workload("c2", seed=seed)
    d = lambda a: torch.from_numpy(a).to(dev)
    tokens, offsets, traj, rs, lp = d(mi.tokens), d(mi.offsets), d(mi.traj_ids), d(mi.resp_start), d(mi.old_logp)
    stream = torch.cuda.Stream(dev)
    with torch.cuda.stream(stream):
        mout = ajt.merge_timelines(tokens, offsets, traj, rs, None, lp, owner_rule=ajt.OWNER_LONGEST)
        stream.synchronize()
        assert ajt.last_status(mout.workspace) == 0
        fin = mout.finalize()
    n, N_in, N_out, M = mi.n, mi.n_tokens, fin.N_out, fin.M
    cpu = lambda t: t.cpu().numpy()
    targets, mask, seg, S, adv, Ns, inv = loss_side_inputs(W, cpu(fin.merged_tokens), cpu(fin.merged_mask),
                                                           cpu(fin.merged_old_logp), cpu(fin.merged_offsets),
                                                           cpu(fin.merged_traj), seed)
    T = min(args.loss_rows, N_out)
    n_mb = 2 if N_out >= 2 * T else 1
    Ns_d = d(Ns)
    mbs = []
    for k in range(n_mb):
        sl = slice(k * T, (k + 1) * T)
        logits = torch.empty((T, V), dtype=torch.bfloat16, device=dev)
        fill_logits(torch, logits, seed * 7 + k)
        tg = d(targets[sl].copy())
        noise = (W.rng_for(seed, 1, 99 + k).standard_normal(T) * 0.05).astype(np.float32)
        old = harness_old_logp(torch, logits, tg, noise)
        mbs.append(dict(logits=logits, targets=tg, old=old, adv=d(adv[sl].copy()), mask=d(mask[sl].copy()),
                        seg=d(seg[sl].copy()), n_unmasked=int(mask[sl].sum())))
    dlogits = torch.empty((T, V), dtype=torch.bfloat16, device=dev)
    lout = None
    # The stages are chained on the device: the merge's outputs feed ajt_pack_loss_inputs (next-token alignment, segment ids,
    # advantages: reading L-12), ajt_segment_counts gives the batch-wide N_s (reading L-4), and the loss call reads the
    # micro-batch's rows of those arrays.  Nothing goes through the host inside a step.  (`old` was synthesised in the set-up
    # from the same targets: input synthesis, BASELINE.json configs.)
    uniq, tl_seg = np.unique(mi.traj_ids, return_inverse=True)
    assert int(uniq.shape[0]) == S
    tl_seg_d = d(tl_seg.astype(np.int32))
    seg_adv_d = d(W.advantages_group_zscore(seed, 1, S).astype(np.float32))
    with torch.cuda.stream(stream):
        pk = ajt.pack_loss_inputs(mout, tl_seg_d, S, seg_adv_d, stream=stream)
        stream.synchronize()
    for k in range(n_mb):       # the device chain reproduces the set-up's host arrays bit for bit
        sl = slice(k * T, (k + 1) * T)
        assert torch.equal(pk.targets[sl], mbs[k]["targets"]) and torch.equal(pk.mask[sl], mbs[k]["mask"])
        assert torch.equal(pk.seg_ids[sl], mbs[k]["seg"]) and torch.equal(pk.adv[sl], mbs[k]["adv"])
        mbs[k].update(targets=pk.targets[sl], mask=pk.mask[sl], seg=pk.seg_ids[sl], adv=pk.adv[sl])
    pk_mask_all, pk_seg_all = pk.mask[:N_out], pk.seg_ids[:N_out]

    def step(k: int, ev=None):
        nonlocal lout
        mb = mbs[k % n_mb]
        if ev:
            ev[0].record(stream)
        ajt.merge_timelines(tokens, offsets, traj, rs, None, lp, owner_rule=ajt.OWNER_LONGEST, out=mout, stream=stream)
        if ev:
            ev[1].record(stream)
        ajt.pack_loss_inputs(mout, tl_seg_d, S, seg_adv_d, out=pk, stream=stream)
        ajt.segment_counts(pk_mask_all, pk_seg_all, S, out=Ns_d, stream=stream)
        if ev:
            ev[3].record(stream)
        lout = ajt.policy_loss_fwd_bwd(mb["logits"], mb["targets"], mb["old"], mb["adv"], mb["mask"], mb["seg"], S, EPS[0],
                                       EPS[1], seg_denom=Ns_d, inv_num_segs=inv, dlogits=dlogits, out=lout, stream=stream)
        if ev:
            ev[2].record(stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    def max_over_ranks(x: float) -> float:
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t[0])

    def sum_over_ranks(x: float) -> float:
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return float(t[0])

    K, Wm = args.steps, args.warmup
    with torch.cuda.stream(stream):
        for k in range(Wm):
            step(k)
        barrier()
        sampler = ClockSampler(local_rank)
        sampler.start()
        time.sleep(0.3)
        evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(K)]
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        tw0 = time.time()
        e0.record(stream)
        for k in range(K):
            step(k, evs[k])
        e1.record(stream)
        barrier()
        tw1 = time.time()
    total_ms = max_over_ranks(e0.elapsed_time(e1))
    merge_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in evs]))
    bridge_ms = float(np.mean([e[1].elapsed_time(e[3]) for e in evs]))
    loss_ms = float(np.mean([e[3].elapsed_time(e[2]) for e in evs]))
    assert ajt.last_status(mout.workspace) == 0 and ajt.last_status(lout.workspace) == 0
    clocks = sampler.summary(tw0, tw1)

    b_merge = merge_bytes(n, N_in, N_out)
    b_loss = [loss_bytes(T, V, mb["n_unmasked"]) for mb in mbs]
    step_bytes = float(np.mean([b_merge + b_loss[k % n_mb] for k in range(K)]))
    loss_b = float(np.mean([b_loss[k % n_mb] for k in range(K)]))
    ms_per_step = total_ms / K
    value = sum_over_ranks(step_bytes) / (ms_per_step * 1e-3) / 1e9
    peak, peak_src = measured_peak()

    # ---- HBM ceilings of this box, measured now with the library's probe kernels; dlogits is scratch here
    ceilings = None
    if rank == 0:
        nb = (int(dlogits.numel()) * 2) & ~15
        sink = torch.zeros(4, dtype=torch.int32, device=dev)

        def probe(mode, dst, src, moved):
            best = 1e30
            with torch.cuda.stream(stream):
                for _ in range(4):
                    a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a0.record(stream)
                    ajt.hbm_probe(dst, src, nb, mode, stream=stream)
                    a1.record(stream)
                    stream.synchronize()
                    best = min(best, a0.elapsed_time(a1))
            return moved / (best * 1e-3) / 1e9

        ceilings = {"read_gb_per_s": probe(0, sink, mbs[0]["logits"], nb), "write_gb_per_s": probe(1, dlogits, None, nb),
                    "memset_gb_per_s": probe(3, dlogits, None, nb), "copy_gb_per_s": probe(2, dlogits, mbs[0]["logits"], 2 * nb),
                    "bytes": nb, "how": "ajt_hbm_probe (16-byte loads / stores over the 12.4 GB logits / dlogits buffers, best of 4)"}

    # ---- e2e: the *_host C-ABI calls, pinned HOST buffers, H2D + D2H inside the timed region
    e2e = None
    if not args.no_e2e:
        e2e = run_e2e(torch, ajt, mi, mbs[0], S, Ns, inv, T, dev, stream, K, Wm, b_merge + b_loss[0], barrier,
                      max_over_ranks, sum_over_ranks)
    sampler.stop()

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu:
        cpu_baseline = run_cpu_baseline(torch, mi, mbs[0], targets[:T], mask[:T], seg[:T], adv[:T], S, Ns, inv, T, n, N_in,
                                        N_out)

    if rank == 0:
        traffic = None
        tp = os.path.join(ROOT, "profiles", "traffic.json")
        if os.path.exists(tp):
            try:
                with open(tp) as f:
                    traffic = json.load(f).get("loss_rows_kernel_dram_bytes_per_launch")
            except Exception:
                traffic = None
        ach = loss_b / (loss_ms * 1e-3) / 1e9
        mg = b_merge / (merge_ms * 1e-3) / 1e9
        line = {
            "metric": METRIC, "value": value, "unit": "GB/s", "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32 (bf16 logits/dlogits in HBM, fp64 scalar; merge int32/u64)", "data": "synthetic",
            "config": workload_config(n, N_in, N_out, T, float(np.mean([mb["n_unmasked"] for mb in mbs]) / T)),
            "merge": {"ms": merge_ms, "merged_gtokens_per_s": N_out / (merge_ms * 1e-3) / 1e9,
                      "input_gtokens_per_s": N_in / (merge_ms * 1e-3) / 1e9, "gb_per_s": mg, "frac_of_measured": mg / peak,
                      "frac_of_nominal_8tbs": mg / NOMINAL_HBM_GBS, "token_reduction_factor": N_in / N_out, "M": M,
                      "algorithmic_bytes": b_merge},
            "bridge": {"ms": bridge_ms, "what": "ajt_pack_loss_inputs over the N_out merged tokens + ajt_segment_counts "
                       "(device-resident chain between the stages; its bytes are not counted in `value`)"},
            "loss": {"ms": loss_ms, "logits_gb_per_s": ach, "frac_of_measured": ach / peak,
                     "frac_of_nominal_8tbs": ach / NOMINAL_HBM_GBS, "algorithmic_bytes": loss_b,
                     "dense_2TV_gb_per_s": 4.0 * T * V / (loss_ms * 1e-3) / 1e9},
            "roofline": {"bound": "hbm", "kernel": "loss_rows_kernel (timed as the ajt_policy_loss_fwd_bwd call: prep + rows + "
                         "final launches; rows is >99% of it, profiles/)", "achieved": ach, "peak": peak, "unit": "GB/s",
                         "frac": ach / peak, "traffic": traffic, "peak_source": peak_src},
            "hbm_ceilings": ceilings, "clocks": clocks, "gpu_launches": K * (6 + 1 + 1 + 3),   # merge 6, pack 1, segment counts 1, loss 3 (prep, rows, final)
            "e2e": e2e, "cpu_baseline": cpu_baseline,
            "paper_context": "paper reports only end-to-end actor-update 2160 s -> 346 s (6.25x) with merging on AppWorld, "
                             "8-GPU node at most, GPU model and precision not stated (PAPER.md:373,395); not comparable",
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def run_e2e(torch, ajt, mi, mb, S, Ns, inv, T, dev, stream, K, Wm, step_bytes, barrier, max_over_ranks, sum_over_ranks):
    """Same step through ajt_merge_timelines_host + ajt_policy_loss_fwd_bwd_host: every input starts in pinned HOST
    memory and every output ends there; the copies run inside the timed region."""
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_tok, h_off, h_traj, h_rs, h_lp = pin(mi.tokens), pin(mi.offsets), pin(mi.traj_ids), pin(mi.resp_start), pin(mi.old_logp)
    h_logits = torch.empty((T, V), dtype=torch.bfloat16, pin_memory=True)
    h_logits.copy_(mb["logits"])
    h_dlogits = torch.empty((T, V), dtype=torch.bfloat16, pin_memory=True)
    h_vec = {k: mb[k].cpu().pin_memory() for k in ("targets", "old", "adv", "mask", "seg")}
    h_Ns = pin(Ns)
    m_arena = torch.empty(ajt.merge_host_arena_bytes(mi.n, mi.n_tokens), dtype=torch.uint8, device=dev)
    l_arena = torch.empty(ajt.loss_host_arena_bytes(T, V, S, V, ajt.DT_BF16), dtype=torch.uint8, device=dev)
    m_out = None
    res = {}

    def step():
        nonlocal m_out
        r = ajt.merge_timelines_host(h_tok, h_off, h_traj, h_rs, None, h_lp, owner_rule=ajt.OWNER_LONGEST, arena=m_arena,
                                     out=m_out, stream=stream)
        m_out = {k: r[k] for k in ("merged_tokens", "merged_mask", "merged_src", "merged_old_logp", "merged_offsets",
                                   "merged_origin", "merged_traj", "owner")}
        res["merge"] = r
        res["loss"] = ajt.policy_loss_fwd_bwd_host(h_logits, h_vec["targets"], h_vec["old"], h_vec["adv"], h_vec["mask"],
                                                   h_vec["seg"], S, EPS[0], EPS[1], ajt.DT_BF16, seg_denom=h_Ns,
                                                   inv_num_segs=inv, dlogits=h_dlogits, arena=l_arena, stream=stream)

    Ke = max(1, min(K, args_e2e_steps(K)))
    with torch.cuda.stream(stream):
        for _ in range(min(Wm, 2)):
            step()
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(Ke):
            step()
        e1.record(stream)
        barrier()
    ms = max_over_ranks(e0.elapsed_time(e1)) / Ke
    assert res["merge"]["status"] == 0 and res["loss"]["status"] == 0
    No, M, n, N = res["merge"]["N_out"], res["merge"]["M"], mi.n, mi.n_tokens
    n_up = int(mb["n_unmasked"])   # the host call uploads only the rows the kernel reads (mask != 0)
    h2d = 4 * N + 8 * (n + 1) + 4 * n + 4 * n + 4 * N + n_up * V * 2 + 17 * T + 4 * S
    d2h = No * (4 + 1 + 4 + 4) + 8 * (M + 1) + 4 * M + 4 * M + 4 * n + 16 + 4 + T * V * 2 + 4 + 4
    return {"value": sum_over_ranks(float(step_bytes)) / (ms * 1e-3) / 1e9, "unit": "GB/s", "h2d_bytes_per_step": int(h2d),
            "d2h_bytes_per_step": int(d2h), "ms_per_step": ms, "steps": Ke,
            "api": "ajt_merge_timelines_host + ajt_policy_loss_fwd_bwd_host (pinned host buffers)",
            "pcie_gb_per_s": (h2d + d2h) / (ms * 1e-3) / 1e9, "loss": res["loss"]["loss"]}


def args_e2e_steps(K: int) -> int:
    return max(1, min(K, 5))   # each e2e step moves ~25 GB over PCIe (~0.5-1 s)


def run_cpu_baseline(torch, mi, mb, targets, mask, seg, adv, S, Ns, inv, T, n, N_in, N_out):
    """The oracle as it stands on the GPU box's host cores, on a bounded sample (~10-30 s of CPU work): the full
    merge of the batch + loss rows in slabs of 2048 until ~20 s are spent (the whole micro-batch if it gets there)."""
    import oracle

    oracle.build()
    slab = 2048
    old = mb["old"].cpu().numpy().astype(np.float32)
    t0 = time.perf_counter()
    oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp, oracle.OWNER_LONGEST)
    tm = time.perf_counter() - t0
    tl, rows, nu = 0.0, 0, 0
    while rows < T and tl < 20.0:
        b = min(T, rows + slab)
        bits = mb["logits"][rows:b].contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
        rid = np.arange(rows, b, dtype=np.int64)
        t0 = time.perf_counter()
        oracle.policy_loss(bits, targets, old, adv, mask, seg, S, float(np.float32(EPS[0])), float(np.float32(EPS[1])),
                           seg_denom=Ns, inv_num_segs=inv, row_ids=rid, want_dlogits=True, logits_is_bf16_bits=True)
        tl += time.perf_counter() - t0
        nu += int(mask[rows:b].sum())
        rows = b
    val, t_step = extrapolated_gbs(n, N_in, N_out, T, int(mask.sum()), tm, tl, rows, nu)
    how = "no extrapolation" if rows == T else "rest of the micro-batch extrapolated at the sample's byte rate"
    return {"value": val, "unit": "GB/s", "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"full merge of the batch ({n} timelines, {N_in} tokens: {tm * 1e3:.1f} ms) + first {rows} of {T} loss rows "
                      f"({nu} unmasked) x V={V} in {tl:.2f} s, fp64 dlogits included; {how}",
            "est_ms_per_step": t_step * 1e3, "merge_ms": tm * 1e3}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--loss-rows", type=int, default=MB_ROWS, help="rows of the loss micro-batch (profiling runs only; "
                    "the default is the workload BASELINE.json names)")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg")
    ap.add_argument("--no-cpu", action="store_true", help="skip the oracle cpu_baseline leg")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if world != args.gpus and rank == 0:
        print(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}; launch with torch.distributed.run for N>1", file=sys.stderr)
    run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
