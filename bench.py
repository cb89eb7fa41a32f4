#!/usr/bin/env python
"""bench.py — one "step" = one pass of the whole hot path (SURVEY.md §8(a) rows M1-M7 + L0-L4) over one synthetic batch
of BASELINE.json configs[2] ("long-horizon agent", the largest single-GPU configuration):

    ajt_merge_timelines      over the batch's ~7.9k timelines (N_in ~ 69 M tokens, 277 MB)
    ajt_pack_loss_inputs + ajt_segment_counts   the device-resident bridge (next-token alignment, batch-wide N_s)
    ajt_policy_loss_fwd_bwd  over one 65,536-row chunk of the merged tokens, bf16 logits [65536,151936] (19.9 GB in,
                             19.9 GB out), with the chunk's real targets / mask / segments from the merge output

`value` = algorithmic bytes of the step / device time (GB/s), inputs resident in HBM.  `e2e` = the same metric through the
*_host C-ABI calls with pinned HOST buffers (H2D and D2H inside the timed region).  `configs` = one compact record per
BASELINE.json config (c1, c2, c3, c4 A/B, three c5 cells): merged tokens/s, merge GB/s, logits GB/s, token-reduction
factor, each as a fraction of the measured and of the nominal HBM rate, and the oracle's merge time on the host cores
(one thread and all).  `--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload.

Launch: `python bench.py --gpus N --steps K --warmup W`; for N>1 under torch.distributed.run (one rank per GPU): ONE batch
is split N ways — trajectory groups go to ranks (paper_2606_04484_b200.shard), every rank merges its share, the batch-wide
per-trajectory token counts N_s are all-reduced (NCCL) inside the step, every rank runs the loss over one chunk of its own
merged tokens, and the scalar is all-reduced.
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
CHUNK_ROWS = 65536       # BASELINE.json configs[2]: "64k-token chunks of bf16 logits [65536,151936]"
V = 151936
EPS = (0.2, 0.28)
HEADLINE = "c3"

from paper_2606_04484_b200.harness import (NOMINAL_HBM_GBS, L2Flusher, fill_logits, harness_old_logp, loss_bytes,  # noqa: E402
                                           measured_peak, merge_bytes, time_calls)


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




# ----------------------------------------------------------------------------------------- workload plumbing (no method arithmetic)

CFG_INDEX = {"c1": 0, "c2": 1, "c3": 2, "c4A": 3, "c4B": 3}
CFG_EPS = {"c1": (0.2, 0.2), "c2": (0.2, 0.28), "c3": (0.2, 0.28), "c4A": (0.2, 0.2), "c4B": (0.2, 0.2)}
CFG_WHAT = {
    "c1": "configs[0] tiny: 32 trajectories x 6 turns, vocab 1024, fp32 logits over all merged tokens",
    "c2": "configs[1] single-model GRPO batch: 64 trajectories x 8 turns, one 40,960-row micro-batch [40960,151936] bf16",
    "c3": "configs[2] long-horizon agent: 256 trajectories x 20-40 turns, contexts to 32k, one chunk [65536,151936] bf16",
    "c4A": "configs[3] team, model A (agents 0,1; vocab 151936): one chunk [65536,151936] bf16",
    "c4B": "configs[3] team, model B (agent 2; vocab 128256): one chunk [65536,128256] bf16",
}


def merge_inputs(W, name: str, seed=None):
    if name in ("c4A", "c4B"):
        return W.merge_workload_c4(seed=seed)[name[-1]]
    return W.merge_workload(name, seed=seed)


def seg_advantages(W, name: str, seed: int, S: int) -> np.ndarray:
    if name == "c1":
        return W.advantages_pm1(seed, 0, S).astype(np.float32)
    return W.advantages_group_zscore(seed, CFG_INDEX[name], S).astype(np.float32)


def loss_traffic(T: int, Vv: int):
    """DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) of ONE loss rows-kernel launch at shape [T, Vv], from the
    committed ncu --set full captures (profiles/r02_traffic.csv; the commands are in profiles/r02_README.md), or None."""
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "r02_traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["kernel"].startswith("loss_rows") and row["shape"] == f"{T}x{Vv}":
                    return float(row["dram_bytes_per_launch"]), row["note"]
    except Exception:
        pass
    return None, None


def fracs(gbs: float, peak: float) -> dict:
    return {"gb_per_s": gbs, "frac_of_measured": gbs / peak, "frac_of_nominal_8tbs": gbs / NOMINAL_HBM_GBS}


class Batch:
    """One batch resident on the device: merge inputs, merge outputs, and the packed per-token loss inputs the bridge
    derives from them (ajt_pack_loss_inputs + ajt_segment_counts).  All of it through the library's calls."""

    def __init__(self, torch, ajt, W, name, mi, seed, dev, stream, tl_seg=None, S=None):
        self.torch, self.ajt, self.name, self.mi, self.stream = torch, ajt, name, mi, stream
        d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
        self.tokens, self.offsets, self.traj, self.rs, self.lp = d(mi.tokens), d(mi.offsets), d(mi.traj_ids), d(mi.resp_start), d(mi.old_logp)
        if tl_seg is None:
            uniq, tl_seg = np.unique(mi.traj_ids, return_inverse=True)
            S = int(uniq.shape[0])
        self.S = S
        self.tl_seg_h = tl_seg.astype(np.int32)
        self.seg_adv_h = seg_advantages(W, name, seed, S)
        self.tl_seg, self.seg_adv = d(self.tl_seg_h), d(self.seg_adv_h)
        self.Ns = torch.zeros(S, dtype=torch.float32, device=dev)
        with torch.cuda.stream(stream):
            self.mout = ajt.merge_timelines(self.tokens, self.offsets, self.traj, self.rs, None, self.lp,
                                            owner_rule=ajt.OWNER_LONGEST, stream=stream)
            self.pk = ajt.pack_loss_inputs(self.mout, self.tl_seg, S, self.seg_adv, stream=stream)
            stream.synchronize()
        st = ajt.last_status(self.mout.workspace, stream)
        assert st == 0, f"{name}: merge status {st}"
        self.fin = self.mout.finalize()
        self.n, self.N_in, self.N_out, self.M = mi.n, mi.n_tokens, self.fin.N_out, self.fin.M
        self.mask_all, self.seg_all = self.pk.mask[:self.N_out], self.pk.seg_ids[:self.N_out]
        with torch.cuda.stream(stream):
            ajt.segment_counts(self.mask_all, self.seg_all, S, out=self.Ns, stream=stream)
            stream.synchronize()

    def merge(self):
        self.ajt.merge_timelines(self.tokens, self.offsets, self.traj, self.rs, None, self.lp, owner_rule=self.ajt.OWNER_LONGEST,
                                 out=self.mout, stream=self.stream)

    def bridge(self, accumulate_into=None):
        self.ajt.pack_loss_inputs(self.mout, self.tl_seg, self.S, self.seg_adv, out=self.pk, stream=self.stream)
        self.ajt.segment_counts(self.mask_all, self.seg_all, self.S, out=self.Ns, stream=self.stream)

    def rows(self, a: int, b: int) -> dict:
        pk = self.pk
        return dict(targets=pk.targets[a:b], mask=pk.mask[a:b], seg=pk.seg_ids[a:b], adv=pk.adv[a:b],
                    n_unmasked=int(pk.mask[a:b].sum().item()), T=b - a)

    def check_pack_against_oracle(self, oracle, n_seq: int = 24):
        """The device bridge against oracle.pack_loss_inputs on the first merged sequences (reading L-12)."""
        f, cpu = self.fin, (lambda t: t.cpu().numpy())
        m = min(n_seq, f.M)
        off = cpu(f.merged_offsets[:m + 1])
        No = int(off[-1])
        t, mk, lp, sg, av = oracle.pack_loss_inputs(cpu(f.merged_tokens[:No]), cpu(f.merged_mask[:No]), cpu(f.merged_old_logp[:No]),
                                                    off, cpu(f.merged_origin[:m]), self.tl_seg_h, self.seg_adv_h)
        pk = self.pk
        assert np.array_equal(cpu(pk.targets[:No]), t) and np.array_equal(cpu(pk.mask[:No]), mk)
        assert np.array_equal(cpu(pk.seg_ids[:No]), sg) and np.array_equal(cpu(pk.adv[:No]), av)
        assert np.array_equal(cpu(pk.old_logp[:No]), lp)


def noise_for(W, seed: int, key: int, T: int, sigma: float = 0.05) -> np.ndarray:
    return (W.rng_for(seed, CFG_INDEX.get("c2", 1), 99 + key).standard_normal(T) * sigma).astype(np.float32)


def oracle_merge_times(oracle, mi) -> dict:
    """The brute-force merge oracle on the host cores: one thread, then all of them."""
    allc = oracle.num_threads()
    out = {}
    for nm, nt in (("one_thread", 1), ("all_cores", allc)):
        oracle.set_threads(nt)
        t0 = time.perf_counter()
        oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp, oracle.OWNER_LONGEST)
        out[nm + "_ms"] = (time.perf_counter() - t0) * 1e3
    oracle.set_threads(allc)
    out["cores"] = allc
    return out


# ----------------------------------------------------------------------------------------- our arm (CUDA)


def run_ours(args, rank: int, world: int, local_rank: int):
    import torch
    import torch.distributed as dist

    import paper_2606_04484_b200 as ajt
    from paper_2606_04484_b200 import shard as SH
    from paper_2606_04484_b200 import workloads as W

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    ajt.lib()  # fail loudly if libajt.so is missing
    peak, peak_src = measured_peak()
    stream = torch.cuda.Stream(dev)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)

    # ---- the batch (seeded, synthetic).  N > 1: ONE batch split by trajectory groups, every rank keeps its share
    seed = W.BASE_SEED + CFG_INDEX[HEADLINE]
    mi_full = merge_inputs(W, HEADLINE, seed)
    uniq, tl_seg_full = np.unique(mi_full.traj_ids, return_inverse=True)
    S = int(uniq.shape[0])
    if world > 1:
        sh = SH.shard_merge_inputs(mi_full.tokens, mi_full.offsets, mi_full.traj_ids, mi_full.resp_start, None, mi_full.old_logp,
                                   rank=rank, world=world)
        mi = W.MergeInputs(sh.tokens, sh.offsets, sh.traj_ids, sh.resp_start, sh.old_logp)
        tl_seg = tl_seg_full[sh.index]
    else:
        mi, tl_seg = mi_full, tl_seg_full
    B = Batch(torch, ajt, W, HEADLINE, mi, seed, dev, stream, tl_seg=tl_seg, S=S)
    T = min(args.loss_rows, B.N_out)
    n_ch = 2 if B.N_out >= 2 * T else 1
    big_rows = 131072 if (world == 1 and not args.no_configs) else T   # the largest configs[4] cell shares the buffers
    logits_big = torch.empty((big_rows, V), dtype=torch.bfloat16, device=dev)
    dlogits_big = torch.empty((big_rows, V), dtype=torch.bfloat16, device=dev)
    fill_logits(logits_big, seed * 7 + rank)
    logits, dlogits = logits_big[:T], dlogits_big[:T]
    chunks = []
    for k in range(n_ch):
        r = B.rows(k * T, (k + 1) * T)
        r["old"] = harness_old_logp(logits, r["targets"], noise_for(W, seed, k, T))   # input synthesis: new logp + N(0, 0.05)
        chunks.append(r)
    Ns_loc = B.Ns                                      # this rank's per-trajectory counts; all-reduced inside the step
    Ns_glob = torch.zeros_like(Ns_loc)
    loss_acc = torch.zeros(1, dtype=torch.float64, device=dev)
    lout = None

    def step(k: int, ev=None):
        nonlocal lout
        ch = chunks[k % n_ch]
        if ev:
            ev[0].record(stream)
        B.merge()
        if ev:
            ev[1].record(stream)
        B.bridge()
        Ns_glob.copy_(Ns_loc)
        if world > 1:
            dist.all_reduce(Ns_glob)                   # N_s over the whole batch (kilobytes)
        if ev:
            ev[2].record(stream)
        lout = ajt.policy_loss_fwd_bwd(logits, ch["targets"], ch["old"], ch["adv"], ch["mask"], ch["seg"], S, EPS[0], EPS[1],
                                       seg_denom=Ns_glob, inv_num_segs=0.0, dlogits=dlogits, out=lout, stream=stream)
        if ev:
            ev[3].record(stream)
        if world > 1:
            loss_acc.copy_(lout.loss.double())
            dist.all_reduce(loss_acc)                  # the scalar (one double)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    def reduce_ranks(x: float, op) -> float:
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=op)
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
        l0 = ajt.launch_count()
        tw0 = time.time()
        e0.record(stream)
        for k in range(K):
            step(k, evs[k])
        e1.record(stream)
        barrier()
        tw1 = time.time()
        launches = ajt.launch_count() - l0
    total_ms = reduce_ranks(e0.elapsed_time(e1), dist.ReduceOp.MAX if world > 1 else None)
    merge_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in evs]))
    bridge_ms = float(np.mean([e[1].elapsed_time(e[2]) for e in evs]))
    loss_ms = float(np.mean([e[2].elapsed_time(e[3]) for e in evs]))
    assert ajt.last_status(B.mout.workspace) == 0 and ajt.last_status(lout.workspace) == 0
    clocks = sampler.summary(tw0, tw1)

    b_merge = merge_bytes(B.n, B.N_in, B.N_out)
    b_loss = [loss_bytes(T, V, ch["n_unmasked"]) for ch in chunks]
    step_bytes = float(np.mean([b_merge + b_loss[k % n_ch] for k in range(K)]))
    loss_b = float(np.mean([b_loss[k % n_ch] for k in range(K)]))
    ms_per_step = total_ms / K
    value = reduce_ranks(step_bytes, dist.ReduceOp.SUM if world > 1 else None) / (ms_per_step * 1e-3) / 1e9
    rho = float(np.mean([ch["n_unmasked"] for ch in chunks]) / T)

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

        ceilings = {"read_gb_per_s": probe(0, sink, logits, nb), "write_gb_per_s": probe(1, dlogits, None, nb),
                    "memset_gb_per_s": probe(3, dlogits, None, nb), "copy_gb_per_s": probe(2, dlogits, logits, 2 * nb),
                    "bytes": nb, "how": "ajt_hbm_probe (16-byte loads / stores over the logits / dlogits chunk buffers, best of 4)"}

    # ---- e2e: the *_host C-ABI calls, pinned HOST buffers, H2D + D2H inside the timed region
    e2e = None
    if not args.no_e2e:
        e2e = run_e2e(torch, ajt, mi, B, chunks[0], logits, dlogits, S, T, dev, stream, K, Wm, b_merge, barrier, reduce_ranks,
                      dist, world)
    sampler.stop()

    cpu_baseline, cfg_records = None, None
    if rank == 0 and not args.no_cpu:
        cpu_baseline = run_cpu_baseline(torch, B, chunks[0], logits, S, T)
    if rank == 0 and world == 1 and not args.no_configs:
        cfg_records = run_config_records(torch, ajt, W, B, chunks[0], logits_big, dlogits_big, dev, stream, peak,
                                         dict(merge_ms=merge_ms, loss_ms=loss_ms, T=T, rho=rho), with_oracle=not args.no_cpu)

    if rank == 0:
        shape_key = f"loss_rows_kernel[{T}x{V},rho={rho:.2f}]"
        traffic, traffic_note = loss_traffic(T, V)
        ach = loss_b / (loss_ms * 1e-3) / 1e9
        mg = b_merge / (merge_ms * 1e-3) / 1e9
        line = {
            "metric": METRIC, "value": value, "unit": "GB/s", "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None,
            "dtype": "f32 (bf16 logits/dlogits in HBM, fp64 scalar; merge int32/u64)", "data": "synthetic",
            "config": workload_config(mi_full.n, mi_full.n_tokens, B, T, rho, world),
            "merge_c3": {"ms": merge_ms, "merged_gtokens_per_s": B.N_out / (merge_ms * 1e-3) / 1e9,
                         "input_gtokens_per_s": B.N_in / (merge_ms * 1e-3) / 1e9, **fracs(mg, peak),
                         "token_reduction_factor": B.N_in / B.N_out, "M": B.M, "n": B.n, "N_in": B.N_in, "N_out": B.N_out,
                         "algorithmic_bytes": b_merge, "target": "north_star: >= 0.40 of the nominal 8 TB/s"},
            "bridge": {"ms": bridge_ms, "what": "ajt_pack_loss_inputs over the N_out merged tokens + ajt_segment_counts "
                       "(device-resident chain between the stages" + (", then the NCCL all-reduce of N_s" if world > 1 else "") +
                       "; its bytes are not counted in `value`)"},
            "loss": {"ms": loss_ms, "logits_gb_per_s": ach, "frac_of_measured": ach / peak,
                     "frac_of_nominal_8tbs": ach / NOMINAL_HBM_GBS, "algorithmic_bytes": loss_b,
                     "dense_2TV_gb_per_s": 4.0 * T * V / (loss_ms * 1e-3) / 1e9, "mask_density": rho,
                     "chunks_in_batch": int((B.N_out + T - 1) // T),
                     "batch_loss_s_extrapolated": float((B.N_out + T - 1) // T) * loss_ms * 1e-3,
                     "extrapolation": "the batch's merged tokens in chunks of loss_rows x this call's time (chunks are "
                                      "independent given the batch-wide N_s; SURVEY.md 8(d) configs[2])"},
            "roofline": {"bound": "hbm", "kernel": shape_key + " (timed as the ajt_policy_loss_fwd_bwd call: prep + rows + final "
                         "launches; rows is >99% of it, profiles/)", "achieved": ach, "peak": peak, "unit": "GB/s",
                         "frac": ach / peak, "traffic": traffic, "traffic_note": traffic_note, "peak_source": peak_src},
            "hbm_ceilings": ceilings, "clocks": clocks, "gpu_launches": int(launches),
            "gpu_launches_how": "counted by the library (ajt_launch_count before / after the timed region): merge 7, pack 1, "
                                "segment counts 1, loss 3 per step",
            "e2e": e2e, "cpu_baseline": cpu_baseline, "configs": cfg_records,
            "paper_context": "paper reports only end-to-end actor-update 2160 s -> 346 s (6.25x) with merging on AppWorld, "
                             "8-GPU node at most, GPU model and precision not stated (PAPER.md:373,395); not comparable",
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def workload_config(n, N_in, B, T, rho, world):
    return {"workload": "BASELINE.json configs[2] long-horizon agent (the largest single-GPU configuration): merge of 256 "
                        f"trajectories x 20-40 turns ({n} timelines, N_in={N_in}, contexts to 32k tokens, Zipf(1.1) tokens) + "
                        f"policy-loss fwd+bwd over one chunk [{T},{V}] bf16 of the merged tokens with the merge's own targets / "
                        f"mask / segments (mask density {rho:.3f}), eps 0.2/0.28, group z-score advantages"
                        + (f"; the batch is split over {world} ranks by trajectory group, this record describes rank 0's share "
                           f"(n={B.n}, N_in={B.N_in})" if world > 1 else ""),
            "owner_rule": "longest", "loss_rows": T, "vocab": V, "merge_timelines": n, "N_in": N_in, "N_out": B.N_out,
            "parallelism": "single GPU" if world == 1 else f"dp{world}: groups -> ranks, all-reduce of N_s and of the scalar",
            "l2": "inputs larger than L2: every step streams the 277 MB token array and a 19.9 GB logits chunk (126 MB L2)"}


def mem_available_gb() -> float:
    try:
        with open("/proc/meminfo") as f:
            for ln in f:
                if ln.startswith("MemAvailable:"):
                    return float(ln.split()[1]) / 1e6
    except Exception:
        pass
    return 0.0


def run_e2e(torch, ajt, mi, B, ch, logits, dlogits, S, T, dev, stream, K, Wm, b_merge, barrier, reduce_ranks, dist, world):
    """Same step through ajt_merge_timelines_host + ajt_policy_loss_fwd_bwd_host2: every input starts in pinned HOST memory;
    the merge's outputs and the loss / status come back to the host; the gradient stays on the device (where the backward
    pass continues).  The copies run inside the timed region.  The logits chunk needs T x V x 2 bytes of pinned host memory:
    on a box without that much the leg uses as many rows as fit and says so."""
    Te = T
    need_gb = T * V * 2 / 1e9 + 4.0
    if mem_available_gb() < need_gb + 8.0:
        Te = max(1024, min(T, int((mem_available_gb() - 12.0) * 1e9 / (V * 2)) // 1024 * 1024))
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_tok, h_off, h_traj, h_rs, h_lp = pin(mi.tokens), pin(mi.offsets), pin(mi.traj_ids), pin(mi.resp_start), pin(mi.old_logp)
    h_logits = torch.empty((Te, V), dtype=torch.bfloat16, pin_memory=True)
    h_logits.copy_(logits[:Te])
    h_vec = {k: ch[k][:Te].cpu().pin_memory() for k in ("targets", "old", "adv", "mask", "seg")}
    Ns = B.Ns.clone()
    if world > 1:
        dist.all_reduce(Ns)
    h_Ns = Ns.cpu().pin_memory()
    m_arena = torch.empty(ajt.merge_host_arena_bytes(mi.n, mi.n_tokens), dtype=torch.uint8, device=dev)
    l_arena = torch.empty(ajt.loss_host_arena_bytes(Te, V, S, V, ajt.DT_BF16), dtype=torch.uint8, device=dev)
    ctx = ajt.HostCtx()
    m_out = None
    res = {}

    def step():
        nonlocal m_out
        r = ajt.merge_timelines_host(h_tok, h_off, h_traj, h_rs, None, h_lp, owner_rule=ajt.OWNER_LONGEST, arena=m_arena,
                                     out=m_out, stream=stream)
        m_out = {k: r[k] for k in ("merged_tokens", "merged_mask", "merged_src", "merged_old_logp", "merged_offsets",
                                   "merged_origin", "merged_traj", "owner")}
        res["merge"] = r
        res["loss"] = ajt.policy_loss_fwd_bwd_host2(h_logits, h_vec["targets"], h_vec["old"], h_vec["adv"], h_vec["mask"],
                                                    h_vec["seg"], S, EPS[0], EPS[1], ajt.DT_BF16, dlogits[:Te], seg_denom=h_Ns,
                                                    inv_num_segs=0.0, want_logp=True, ctx=ctx, arena=l_arena, stream=stream)

    Ke = max(1, min(K, 5))   # each e2e step moves ~10 GB over PCIe
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
    ms = reduce_ranks(e0.elapsed_time(e1), dist.ReduceOp.MAX if world > 1 else None) / Ke
    ctx.close()
    assert res["merge"]["status"] == 0 and res["loss"]["status"] == 0
    No, M, n, N = res["merge"]["N_out"], res["merge"]["M"], mi.n, mi.n_tokens
    n_up = int(h_vec["mask"].sum().item())   # the host call uploads only the rows the kernel reads (mask != 0)
    step_bytes = b_merge + loss_bytes(Te, V, n_up)
    h2d = 4 * N + 8 * (n + 1) + 4 * n + 4 * n + 4 * N + n_up * V * 2 + 17 * Te + 4 * S
    d2h = No * (4 + 1 + 4 + 4) + 8 * (M + 1) + 4 * M + 4 * M + 4 * n + 16 + 4 + 4 + 4 * Te + 4
    return {"value": reduce_ranks(float(step_bytes), dist.ReduceOp.SUM if world > 1 else None) / (ms * 1e-3) / 1e9, "unit": "GB/s",
            "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h), "ms_per_step": ms, "steps": Ke, "loss_rows": Te,
            "api": "ajt_merge_timelines_host + ajt_policy_loss_fwd_bwd_host2 (pinned host buffers; merged sequences, loss, "
                   "log-probs and status return to the host, dlogits stay on the device for the backward pass)",
            "note": None if Te == T else f"host memory holds {Te} of the chunk's {T} logits rows pinned; the loss leg ran on those",
            "pcie_gb_per_s": (h2d + d2h) / (ms * 1e-3) / 1e9, "loss": res["loss"]["loss"]}


def run_cpu_baseline(torch, B, ch, logits, S, T):
    """The oracle as it stands on the GPU box's host cores, on a bounded sample (~10-30 s of CPU work): the full merge of
    the batch + loss rows of the chunk in slabs of 1024 until ~15 s are spent; the rest of the chunk is extrapolated at the
    sample's byte rate (rows are independent)."""
    import oracle

    oracle.build()
    mi = B.mi
    t0 = time.perf_counter()
    oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp, oracle.OWNER_LONGEST)
    tm = time.perf_counter() - t0
    B.check_pack_against_oracle(oracle)
    cpu = lambda t: t.cpu().numpy()
    targets, mask, seg, adv, old = cpu(ch["targets"]), cpu(ch["mask"]), cpu(ch["seg"]), cpu(ch["adv"]), cpu(ch["old"])
    Ns = cpu(B.Ns)
    inv = float(np.float32(1.0 / max(1, int((Ns > 0).sum()))))
    slab, tl, rows, nu = 1024, 0.0, 0, 0
    while rows < T and tl < 15.0:
        b = min(T, rows + slab)
        bits = logits[rows:b].contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
        rid = np.arange(rows, b, dtype=np.int64)
        t0 = time.perf_counter()
        oracle.policy_loss(bits, targets, old, adv, mask, seg, S, float(np.float32(EPS[0])), float(np.float32(EPS[1])),
                           seg_denom=Ns, inv_num_segs=inv, row_ids=rid, want_dlogits=True, logits_is_bf16_bits=True)
        tl += time.perf_counter() - t0
        nu += int(mask[rows:b].sum())
        rows = b
    rate = loss_bytes(rows, V, nu) / max(tl, 1e-9)
    b_all = loss_bytes(T, V, int(mask.sum()))
    t_step = tm + b_all / rate
    val = (merge_bytes(B.n, B.N_in, B.N_out) + b_all) / t_step / 1e9
    how = "no extrapolation" if rows == T else "rest of the chunk extrapolated at the sample's byte rate"
    return {"value": val, "unit": "GB/s", "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"full merge of the batch ({B.n} timelines, {B.N_in} tokens: {tm * 1e3:.0f} ms) + first {rows} of {T} loss rows "
                      f"({nu} unmasked) x V={V} in {tl:.2f} s, fp64 dlogits included; {how}",
            "est_ms_per_step": t_step * 1e3, "merge_ms": tm * 1e3}


def run_config_records(torch, ajt, W, B3, ch3, logits_big, dlogits_big, dev, stream, peak, head, with_oracle=True):
    """One compact record per BASELINE.json config (north_star "Report throughput ..."; SURVEY.md §8(d) "Reported per
    config"): merge ms / merged tokens per s / GB/s / token-reduction factor, loss ms / logits GB/s, fractions of the measured
    and nominal HBM rate, and the merge oracle's time on the host cores with one thread and with all of them.  Calls whose
    inputs fit in the 126 MB L2 are timed cold (a 256 MB write before every repetition)."""
    oracle = None
    if with_oracle:
        import oracle as _o
        _o.build()
        oracle = _o
    flush = L2Flusher(dev)
    L2 = 126 << 20
    recs = {}

    def time_med(fn, cold):
        ms = time_calls(fn, stream, reps=5, warmup=2, flush=flush if cold else None)
        return float(np.median(ms))

    def loss_rec(lg, dl, targets, old, adv, mask, seg, S, Vv, eps, seg_denom=None):
        T = int(lg.shape[0])
        b_in = 2 if lg.dtype == torch.bfloat16 else 4
        nu = int(mask.sum().item())
        lo = None

        def call():
            nonlocal lo
            lo = ajt.policy_loss_fwd_bwd(lg, targets, old, adv, mask, seg, S, eps[0], eps[1], seg_denom=seg_denom, inv_num_segs=0.0,
                                         V=Vv, dlogits=dl, out=lo, stream=stream)
        cold = T * Vv * b_in < L2
        ms = time_med(call, cold)
        assert ajt.last_status(lo.workspace, stream) == 0
        b = loss_bytes(T, Vv, nu, b_in)
        return {"T": T, "V": Vv, "dtype": "bf16" if b_in == 2 else "f32", "mask_density": nu / max(1, T), "ms": ms,
                "algorithmic_bytes": b, **{("logits_" + k if k == "gb_per_s" else k): v for k, v in fracs(b / ms / 1e6, peak).items()},
                "l2": "cold" if cold else "larger than L2", "traffic": loss_traffic(T, Vv)[0]}

    def merge_rec(Bx, ms=None):
        cold = 4 * Bx.N_in * 2 < L2
        if ms is None:
            ms = time_med(Bx.merge, cold)
        b = merge_bytes(Bx.n, Bx.N_in, Bx.N_out)
        r = {"n": Bx.n, "N_in": Bx.N_in, "N_out": Bx.N_out, "M": Bx.M, "token_reduction_factor": Bx.N_in / max(1, Bx.N_out),
             "ms": ms, "merged_gtokens_per_s": Bx.N_out / ms / 1e6, "input_gtokens_per_s": Bx.N_in / ms / 1e6, "algorithmic_bytes": b,
             **fracs(b / ms / 1e6, peak), "l2": "cold" if cold else "larger than L2"}
        if oracle is not None:
            r["oracle_merge"] = oracle_merge_times(oracle, Bx.mi)
        return r

    # c3: the headline step's own measurements
    recs["c3"] = {"what": CFG_WHAT["c3"], "merge": merge_rec(B3, head["merge_ms"]),
                  "loss": {"T": head["T"], "V": V, "dtype": "bf16", "mask_density": head["rho"], "ms": head["loss_ms"],
                           "algorithmic_bytes": loss_bytes(head["T"], V, ch3["n_unmasked"]),
                           **{("logits_" + k if k == "gb_per_s" else k): v
                              for k, v in fracs(loss_bytes(head["T"], V, ch3["n_unmasked"]) / head["loss_ms"] / 1e6, peak).items()},
                           "l2": "larger than L2", "traffic": loss_traffic(head["T"], V)[0]}}
    for name in ("c1", "c2", "c4A", "c4B"):
        seed = W.BASE_SEED + CFG_INDEX[name]
        Bx = Batch(torch, ajt, W, name, merge_inputs(W, name, seed), seed, dev, stream)
        rec = {"what": CFG_WHAT[name], "merge": merge_rec(Bx)}
        if name == "c1":
            T = Bx.N_out
            lg = torch.empty((T, 1024), dtype=torch.float32, device=dev)
            g = torch.Generator(device=dev).manual_seed(seed)
            lg.copy_(torch.randn((T, 1024), generator=g, device=dev) * 2.0)
            dl, Vv = torch.empty((T, 1024), dtype=torch.bfloat16, device=dev), 1024
        else:
            T = min({"c2": 40960}.get(name, CHUNK_ROWS), Bx.N_out)
            Vv = 128256 if name == "c4B" else V
            lg, dl = logits_big[:T], dlogits_big[:T]
        r = Bx.rows(0, T)
        old = harness_old_logp(lg[:, :Vv] if lg.shape[1] != Vv else lg, r["targets"], noise_for(W, seed, 0, T))
        rec["loss"] = loss_rec(lg, dl, r["targets"], old, r["adv"], r["mask"], r["seg"], Bx.S, Vv, CFG_EPS[name], seg_denom=Bx.Ns)
        recs[name] = rec
        del Bx
    # c5: three cells of the loss sweep (smallest; V = 32,000 at mask density 0.7; largest)
    for cell, (T, Vv, rho, S) in enumerate(((4096, 32000, 0.3, 8), (16384, 32000, 0.7, 64), (131072, V, 0.7, 512))):
        if T > logits_big.shape[0]:
            continue
        lv = W.loss_sweep_vectors(T, Vv, S, rho, cell=cell)
        dd = lambda a: torch.from_numpy(a).to(dev)
        lg, dl = logits_big[:T], dlogits_big[:T]
        tg = dd(lv.targets)
        old = harness_old_logp(lg[:, :Vv] if Vv != V else lg, tg, lv.noise)
        rec = loss_rec(lg, dl, tg, old, dd(lv.adv), dd(lv.mask), dd(lv.seg_ids), S, Vv, (0.2, 0.28))
        rec["S"] = S
        recs[f"c5[{T}x{Vv},rho={rho}]"] = {"what": "configs[4] loss sweep cell", "loss": rec}
    # f3: log-probs and the loss with its gradients straight from hidden states, the one tensor-core stage
    try:
        recs["lm_head[40960x4096x151936]"] = lm_head_record(torch, ajt, W, dev, stream)
    except Exception as e:   # measurement extra: never takes the bench line down
        recs["lm_head[40960x4096x151936]"] = {"error": repr(e)[:200]}
    return recs


def lm_head_record(torch, ajt, W, dev, stream):
    """ajt_lm_head_logp (forward) and ajt_lm_head_loss_bwd (loss + dH + dW) at 40,960 x 4,096 x 151,936 with the mask of a
    configs[4] cell (density ~0.35): TFLOP/s over the unmasked rows (2 T d V forward; 8 T d V for the whole backward call,
    which recomputes the logits tiles), against the measured cuBLAS bf16 rates of MEASURED_PEAKS.json."""
    T, d, Vv, S = 40960, 4096, V, 64
    g = torch.Generator(device=dev).manual_seed(6)
    Hh = torch.randn((T, d), generator=g, device=dev).to(torch.bfloat16)
    Ww = (torch.randn((Vv, d), generator=g, device=dev) * 0.02).to(torch.bfloat16)
    lv = W.loss_sweep_vectors(T, Vv, S, 0.35, cell=9)
    dd = lambda a: torch.from_numpy(a).to(dev)
    y, adv, mask, seg = dd(lv.targets), dd(lv.adv), dd(lv.mask), dd(lv.seg_ids)
    with torch.cuda.stream(stream):
        lp, _ = ajt.lm_head_logp(Hh, Ww, y, mask, stream=stream)
        stream.synchronize()
    old = (lp + dd(lv.noise)).contiguous()
    dW = torch.zeros((Vv, d), dtype=torch.float32, device=dev)
    st = {"ws": None}

    def bwd():
        o = ajt.lm_head_loss_bwd(Hh, Ww, y, old, adv, mask, seg, S, EPS[0], EPS[1], dW=dW, accumulate_dw=False, workspace=st["ws"],
                                 stream=stream)
        st["ws"] = o["workspace"]

    def fwd():
        ajt.lm_head_logp(Hh, Ww, y, mask, stream=stream)

    ms_b = float(np.median(time_calls(bwd, stream, reps=3, warmup=1)))
    ms_f = float(np.median(time_calls(fwd, stream, reps=3, warmup=1)))
    Tu = int(lv.mask.sum())
    burst = sust = None
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            mp = json.load(f)
        burst, sust = float(mp["bf16_tflops"]), float(mp["bf16_tflops_sustained"])
    except Exception:
        pass
    tf_f, tf_b = 2.0 * Tu * d * Vv / ms_f / 1e9, 8.0 * Tu * d * Vv / ms_b / 1e9
    return {"what": "SURVEY.md §8(f) f3: LM head fused with the loss, forward and backward (tcgen05 / TMEM / TMA); bound: tensor",
            "rows": T, "unmasked_rows": Tu, "d": d, "V": Vv,
            "forward": {"ms": ms_f, "tflops": tf_f, "frac_of_bf16_burst": tf_f / burst if burst else None,
                        "frac_of_bf16_sustained": tf_f / sust if sust else None},
            "loss_fwd_bwd": {"ms": ms_b, "tflops": tf_b, "frac_of_bf16_burst": tf_b / burst if burst else None,
                             "frac_of_bf16_sustained": tf_b / sust if sust else None,
                             "flops": "8 T d V: logits tiles twice (forward, recomputed for dZ), dH = dZ W, dW = dZ^T H"}}


# ----------------------------------------------------------------------------------------- reference arm (oracle)


def run_reference(args, rank: int):
    """`--impl reference`: the CPU oracle as it stands, on the box's host cores, same config / metric / unit.  Each step =
    the full merge of the batch + a bounded sample of the chunk's loss rows (the rest extrapolated: rows are independent).
    Under torchrun only rank 0 works."""
    if rank != 0:
        return
    import torch

    import oracle
    from paper_2606_04484_b200 import workloads as W

    oracle.build()
    seed = W.BASE_SEED + CFG_INDEX[HEADLINE]
    mi = merge_inputs(W, HEADLINE, seed)
    r = oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp, oracle.OWNER_LONGEST)
    uniq, tl_seg = np.unique(mi.traj_ids, return_inverse=True)
    S = int(uniq.shape[0])
    seg_adv = seg_advantages(W, HEADLINE, seed, S)
    targets, mask, _, seg, adv = oracle.pack_loss_inputs(r.merged_tokens, r.merged_mask, r.merged_old_logp, r.merged_offsets,
                                                         r.merged_origin, tl_seg.astype(np.int32), seg_adv)
    Ns = np.bincount(seg, weights=mask.astype(np.float64), minlength=S).astype(np.float32)   # the oracle's step 4 input
    inv = float(np.float32(1.0 / max(1, int((Ns > 0).sum()))))
    T = min(args.loss_rows, r.N_out)
    n_unm = int(mask[:T].sum())
    rows_max = min(2048, T)
    g = torch.Generator().manual_seed(seed)
    logits = (torch.randn((rows_max, V), generator=g) * 3.0).to(torch.bfloat16)
    # the sample is every (T / rows_max)-th row of the chunk, so it carries the chunk's own mix of prompt (masked) and
    # response rows; a leading slab would hold prompt rows only
    rid_all = np.unique(np.linspace(0, T - 1, rows_max).astype(np.int64))
    rows_max = int(rid_all.shape[0])
    old = np.zeros(T, np.float32)
    old[rid_all] = harness_old_logp(logits[:rows_max], torch.from_numpy(targets[rid_all]), noise_for(W, seed, 0, rows_max)).numpy()
    bits = logits.view(torch.int16).numpy().view(np.uint16)

    def one_step(rows):
        pick = np.unique(np.linspace(0, rows_max - 1, rows).astype(np.int64))   # evenly spaced among the sampled rows
        rid, bt = rid_all[pick], np.ascontiguousarray(bits[pick])
        t0 = time.perf_counter()
        oracle.merge_timelines(mi.tokens, mi.offsets, mi.traj_ids, mi.resp_start, None, mi.old_logp, oracle.OWNER_LONGEST)
        t1 = time.perf_counter()
        oracle.policy_loss(bt, targets[:T], old, adv[:T], mask[:T], seg[:T], S, float(np.float32(EPS[0])),
                           float(np.float32(EPS[1])), seg_denom=Ns, inv_num_segs=inv, row_ids=rid,
                           want_dlogits=True, logits_is_bf16_bits=True)
        return t1 - t0, time.perf_counter() - t1, int(mask[rid].sum())

    tm, tl, nu = one_step(min(256, rows_max))
    budget = 120.0 / max(1, args.steps + args.warmup)   # warm-up + steps stay within ~2 minutes
    rows = int(min(rows_max, max(32, 256 * max(0.0, budget - tm) / max(tl, 1e-6))))
    for _ in range(args.warmup):
        one_step(rows)
    t_m = t_l = 0.0
    t0 = time.perf_counter()
    for _ in range(args.steps):
        a, b, nu = one_step(rows)
        t_m += a
        t_l += b
    wall = time.perf_counter() - t0
    K = max(1, args.steps)
    rate = loss_bytes(rows, V, nu) / max(t_l / K, 1e-9)
    b_all = loss_bytes(T, V, n_unm)
    t_step = t_m / K + b_all / rate
    val = (merge_bytes(mi.n, mi.n_tokens, r.N_out) + b_all) / t_step / 1e9
    cores = oracle.num_threads()
    sample = (f"per step: full merge of the batch ({mi.n} timelines, {mi.n_tokens} tokens) + {rows} of the chunk's {T} loss rows, evenly "
              f"spaced ({nu} unmasked) x V={V}; the chunk's time is extrapolated at the sample's byte rate (rows are independent)")

    class _B:   # what workload_config reads
        n, N_in, N_out = mi.n, mi.n_tokens, r.N_out
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "GB/s", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t_step * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64 (oracle)", "data": "synthetic",
            "config": workload_config(mi.n, mi.n_tokens, _B, T, n_unm / T, 1),
            "cpu_baseline": {"value": val, "unit": "GB/s", "cores": cores, "kind": "oracle", "sample": sample,
                             "measured_wall_s": wall},
            "e2e": {"value": val, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--loss-rows", type=int, default=CHUNK_ROWS, help="rows of the loss chunk (profiling runs only; the default "
                    "is the workload BASELINE.json names)")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg")
    ap.add_argument("--no-cpu", action="store_true", help="skip the oracle legs (cpu_baseline, oracle merge times)")
    ap.add_argument("--no-configs", action="store_true", help="skip the per-config records")
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
