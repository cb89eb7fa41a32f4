"""Per-config measurement of the CUDA path on one GPU: `python -m paper_2606_04484_b200.sweep [--configs c1,c2,c3,c4,c5]`.

One JSON line per (config, stage): merge time / merged tokens/s / GB/s / token-reduction factor, loss time / logits GB/s,
each as a fraction of the measured HBM peak (MEASURED_PEAKS.json) and of the nominal 8 TB/s.
Inputs are the seeded synthetic workloads of DESIGN.md "Input recipe".  Calls whose inputs fit in L2 are timed cold
(a 256 MB write between repetitions) and the line says so.  bench.py is the driver's contract; this is the wider table
behind profiles/*_sweep.md.  The oracle is not used here (parity at these sizes is tests/test_gpu_fullsize.py).
"""
from __future__ import annotations

import argparse
import json
import sys
import time

import numpy as np
import torch

import paper_2606_04484_b200 as ajt
from paper_2606_04484_b200 import harness as H
from paper_2606_04484_b200 import workloads as W

L2_BYTES = 126 << 20


def _stats(ms):
    a = np.asarray(ms, dtype=np.float64)
    return float(np.median(a)), float(a.min())


def _emit(out, **kw):
    line = json.dumps(kw)
    print(line, flush=True)
    if out:
        out.write(line + "\n")
        out.flush()


def measure_merge(name: str, mi, dev, stream, reps: int, out, rules=(("longest", ajt.OWNER_LONGEST),)):
    d = lambda a: torch.from_numpy(a).to(dev)
    tokens, offsets, traj, rs, lp = d(mi.tokens), d(mi.offsets), d(mi.traj_ids), d(mi.resp_start), d(mi.old_logp)
    peak, _ = H.measured_peak()
    fin = None
    for rname, rule in rules:
        with torch.cuda.stream(stream):
            mo = ajt.merge_timelines(tokens, offsets, traj, rs, None, lp, owner_rule=rule, stream=stream)
            stream.synchronize()
        status = ajt.last_status(mo.workspace, stream)
        assert status == 0, status
        fin = mo.finalize()
        cold = 4 * mi.n_tokens * 2 < L2_BYTES
        flush = H.L2Flusher(dev) if cold else None
        call = lambda: ajt.merge_timelines(tokens, offsets, traj, rs, None, lp, owner_rule=rule, out=mo, stream=stream)
        med, best = _stats(H.time_calls(call, stream, reps=reps, flush=flush))
        b = H.merge_bytes(mi.n, mi.n_tokens, fin.N_out)
        gbs = b / (med * 1e-3) / 1e9
        _emit(out, stage="merge", config=name, owner_rule=rname, n=mi.n, N_in=mi.n_tokens, N_out=fin.N_out, M=fin.M,
              token_reduction_factor=mi.n_tokens / max(1, fin.N_out), ms_median=med, ms_best=best,
              merged_gtokens_per_s=fin.N_out / (med * 1e-3) / 1e9, input_gtokens_per_s=mi.n_tokens / (med * 1e-3) / 1e9,
              algorithmic_bytes=b, gb_per_s=gbs, frac_of_measured=gbs / peak, frac_of_nominal_8tbs=gbs / H.NOMINAL_HBM_GBS,
              l2="cold (256 MB flush between calls)" if cold else "input larger than L2", reps=reps)
    return fin


def measure_blocks(name: str, bi, dev, stream, reps: int, out):
    """ajt_merge_blocks (text-level matching) on a seeded block workload."""
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    ids, boff, traj, au, toff, tok, lp = (d(bi.block_ids), d(bi.block_offsets), d(bi.traj_ids), d(bi.author), d(bi.tok_off),
                                          d(bi.tokens), d(bi.logp))
    peak, _ = H.measured_peak()
    with torch.cuda.stream(stream):
        mo = ajt.merge_blocks(ids, boff, traj, au, toff, tok, lp, stream=stream)
        stream.synchronize()
    status = ajt.last_status(mo.workspace, stream)
    assert status == 0, status
    fin = mo.finalize()
    B, N = int(bi.block_ids.shape[0]), int(bi.tokens.shape[0])
    cold = 4 * N < L2_BYTES
    flush = H.L2Flusher(dev) if cold else None
    call = lambda: ajt.merge_blocks(ids, boff, traj, au, toff, tok, lp, out=mo, stream=stream)
    med, best = _stats(H.time_calls(call, stream, reps=reps, flush=flush))
    # algorithmic bytes: 9 B per input block (id, author) + 8 B of tok_off per block read; per OUTPUT token 4 (token) + 4 (logp)
    # read and 4 + 4 + 4 + 1 written; absorbed timelines' tokens are never touched
    b = 17 * B + 21 * fin.N_out + 25 * fin.B_out + 20 * bi.n
    gbs = b / (med * 1e-3) / 1e9
    _emit(out, stage="merge_blocks", config=name, n=bi.n, B_in=B, N_in=N, M=fin.M, B_out=fin.B_out, N_out=fin.N_out,
          token_reduction_factor=N / max(1, fin.N_out), ms_median=med, ms_best=best,
          merged_gtokens_per_s=fin.N_out / (med * 1e-3) / 1e9, algorithmic_bytes=b, gb_per_s=gbs, frac_of_measured=gbs / peak,
          frac_of_nominal_8tbs=gbs / H.NOMINAL_HBM_GBS, l2="cold (256 MB flush between calls)" if cold else "output larger than L2",
          reps=reps)
    return fin


def measure_loss(name: str, logits, targets, old, adv, mask, seg, S, eps, dev, stream, reps, out, seg_denom=None, inv=0.0,
                 dlogits=None, extra=None, ext=False):
    T, V = logits.shape
    b_in = 2 if logits.dtype == torch.bfloat16 else 4
    if dlogits is None:
        dlogits = torch.empty((T, V), dtype=torch.bfloat16, device=dev)
    lo = None

    ref = old + 0.01 if ext else None   # extended form (steps 8-9): KL against a reference policy + row entropy, same read

    def call():
        nonlocal lo
        if ext:
            lo = ajt.policy_loss_fwd_bwd_ext(logits, targets, old, adv, mask, seg, S, eps[0], eps[1], ref_logp=ref, kl_coef=2e-3,
                                             seg_denom=seg_denom, inv_num_segs=inv, dlogits=dlogits, out=lo, stream=stream)
        else:
            lo = ajt.policy_loss_fwd_bwd(logits, targets, old, adv, mask, seg, S, eps[0], eps[1], seg_denom=seg_denom,
                                         inv_num_segs=inv, dlogits=dlogits, out=lo, stream=stream)

    cold = T * V * b_in < L2_BYTES
    flush = H.L2Flusher(dev) if cold else None
    med, best = _stats(H.time_calls(call, stream, reps=reps, flush=flush))
    status = ajt.last_status(lo.workspace, stream)
    assert status == 0, status
    nu = int(mask.sum().item())
    b = H.loss_bytes(T, V, nu, b_in)
    gbs = b / (med * 1e-3) / 1e9
    peak, _ = H.measured_peak()
    kw = dict(stage="loss_ext" if ext else "loss", config=name, T=T, V=V, S=S, dtype="bf16" if b_in == 2 else "f32", mask_density=nu / max(1, T),
              ms_median=med, ms_best=best, algorithmic_bytes=b, logits_gb_per_s=gbs, frac_of_measured=gbs / peak,
              frac_of_nominal_8tbs=gbs / H.NOMINAL_HBM_GBS, dense_2TV_gb_per_s=2.0 * T * V * 2 / (med * 1e-3) / 1e9,
              loss=float(lo.loss.item()), l2="cold (256 MB flush between calls)" if cold else "input larger than L2", reps=reps)
    if extra:
        kw.update(extra)
    _emit(out, **kw)
    return dlogits


def loss_inputs_from_merge(fin, seed, cfg_index, adv_kind, dev):
    cpu = lambda t: t.cpu().numpy()
    targets, mask, _ = W.shift_for_next_token(cpu(fin.merged_tokens), cpu(fin.merged_mask), cpu(fin.merged_old_logp),
                                              cpu(fin.merged_offsets))
    seg, S, _ = W.seg_ids_from_merged(cpu(fin.merged_offsets), cpu(fin.merged_traj))
    if adv_kind == "pm1":
        adv = W.advantages_pm1(seed, cfg_index, S)[seg]
    else:
        adv = W.advantages_group_zscore(seed, cfg_index, S)[seg]
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    return d(targets), d(mask), d(seg), S, d(adv.astype(np.float32))


def chunked_loss(name, fin, V, eps, seed, cfg_index, adv_kind, rows, n_chunks, dev, stream, reps, out, dtype=torch.bfloat16,
                 sigma=3.0):
    targets, mask, seg, S, adv = loss_inputs_from_merge(fin, seed, cfg_index, adv_kind, dev)
    if V < 151936:   # model B of configs[3]: token ids are already < its vocabulary
        assert int(targets.max().item()) < V
    Ns = ajt.segment_counts(mask, seg, S)
    T_all = int(targets.numel())
    rows = min(rows, T_all)
    logits = torch.empty((rows, V), dtype=dtype, device=dev)
    dlogits = torch.empty((rows, V), dtype=torch.bfloat16, device=dev)
    n_avail = max(1, T_all // rows)
    for c in range(min(n_chunks, n_avail)):
        k = (c * max(1, n_avail // max(1, n_chunks))) % n_avail     # spread the timed chunks over the batch
        sl = slice(k * rows, (k + 1) * rows)
        H.fill_logits(logits, seed * 13 + c, sigma)
        noise = (W.rng_for(seed, cfg_index, 99 + c).standard_normal(rows) * 0.05).astype(np.float32)
        tg = targets[sl].contiguous()
        old = H.harness_old_logp(logits, tg, noise)
        measure_loss(name, logits, tg, old, adv[sl].contiguous(), mask[sl].contiguous(), seg[sl].contiguous(), S, eps, dev, stream,
                     reps, out, seg_denom=Ns, inv=0.0, dlogits=dlogits,
                     extra=dict(chunk=k, chunks_in_batch=-(-T_all // rows), batch_rows=T_all))
    del logits, dlogits
    torch.cuda.empty_cache()


def run_c5(dev, stream, reps, out, quick=False):
    Ts = (4096, 16384, 65536, 131072)
    Vs = (32000, 128256, 151936)
    if quick:
        Ts, Vs = (4096, 65536), (32000, 151936)
    cell = 0
    for V in Vs:
        for T in Ts:
            logits = torch.empty((T, V), dtype=torch.bfloat16, device=dev)
            dlogits = torch.empty((T, V), dtype=torch.bfloat16, device=dev)
            H.fill_logits(logits, 5000 + cell)
            for rho in (0.3, 0.7):
                Ss = (64,) if not (T == 65536 and V == 151936 and rho == 0.7) else (8, 64, 512)
                for S in Ss:
                    lv = W.loss_sweep_vectors(T, V, S, rho, cell=cell)
                    d = lambda a: torch.from_numpy(a).to(dev)
                    tg = d(lv.targets)
                    old = H.harness_old_logp(logits, tg, lv.noise)
                    r = reps if T * V < (1 << 32) else max(5, reps // 2)
                    measure_loss("c5", logits, tg, old, d(lv.adv), d(lv.mask), d(lv.seg_ids), lv.S, (0.2, 0.28), dev, stream, r, out,
                                 dlogits=dlogits, extra=dict(rho=rho))
                    if S == 64 and T == 65536:   # the extended form beside the plain call on the 64k-row cells
                        measure_loss("c5", logits, tg, old, d(lv.adv), d(lv.mask), d(lv.seg_ids), lv.S, (0.2, 0.28), dev, stream,
                                     r, out, dlogits=dlogits, extra=dict(rho=rho), ext=True)
                cell += 1
            del logits, dlogits
            torch.cuda.empty_cache()


def measure_lm_head(name: str, T: int, d: int, V: int, dev, stream, reps: int, out, rho: float = 1.0):
    """ajt_lm_head_logp (forward half): dense contraction on the tensor cores, reported in TFLOP/s against
    the measured bf16 matmul throughput of MEASURED_PEAKS.json (burst figure: the kernel is timed alone)."""
    g = torch.Generator(device=dev).manual_seed(17)
    Hh = torch.randn((T, d), generator=g, device=dev).to(torch.bfloat16)
    Ww = (torch.randn((V, d), generator=g, device=dev) * 0.02).to(torch.bfloat16)
    y = torch.randint(0, V, (T,), generator=g, device=dev, dtype=torch.int32)
    ws = torch.empty(int(ajt.lib().ajt_lm_head_workspace_bytes(T, d, V)) + 256, dtype=torch.uint8, device=dev)
    mask = None
    if rho < 1.0:   # response / env runs as in the loss sweep: only the unmasked rows are worth a log-prob
        mask = torch.from_numpy(W.loss_sweep_vectors(T, V, 64, rho, cell=7).mask).to(dev)
    call = lambda: ajt.lm_head_logp(Hh, Ww, y, mask, workspace=ws, stream=stream)
    med, best = _stats(H.time_calls(call, stream, reps=reps, flush=None))
    n_rows = T if mask is None else int(mask.sum().item())
    flops = 2.0 * n_rows * d * V
    tf = flops / (med * 1e-3) / 1e12
    peak = None
    try:
        import json as _j, os as _o
        with open(_o.path.join(H.ROOT, "MEASURED_PEAKS.json")) as f:
            peak = float(_j.load(f)["bf16_tflops"])
    except Exception:
        peak = 2250.0 * 0.7   # B200_PROFILING.md fallback: nominal dense bf16 x typical cuBLAS fraction
    _emit(out, stage="lm_head_logp", config=name, T=T, d=d, V=V, ms_median=med, ms_best=best, flops=flops, tflop_per_s=tf,
          rows_unmasked=n_rows, mask_density=n_rows / T, peak_tflops=peak, frac_of_measured=tf / peak, frac_of_nominal_2250=tf / 2250.0,
          logits_bytes_not_written=2.0 * T * V, reps=reps)


def stock_bandwidth(dev, out):
    """Context for the rooflines: what stock library kernels (torch fill_ / copy_, cudaMemset) reach on this box when they move
    the bytes of the loss step (12.9 GB arrays; the bench micro-batch reads 27 % of the rows and writes all of them)."""
    n = 6 * (1 << 30)
    a = torch.empty(n, dtype=torch.bfloat16, device=dev)
    b = torch.empty(n, dtype=torch.bfloat16, device=dev)
    k = int(n * 0.27)

    def run(f, name, nbytes):
        ts = []
        for _ in range(6):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); f(); e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        t = float(np.min(ts))
        _emit(out, stage="stock_bandwidth", what=name, ms_best=t, bytes=nbytes, gb_per_s=nbytes / t / 1e6)

    sink = torch.zeros(4, dtype=torch.int32, device=dev)
    run(lambda: ajt.hbm_probe(sink, a, 2 * n, 0), "ajt_hbm_probe read 12.9 GB (ld.global.v4)", 2 * n)
    run(lambda: ajt.hbm_probe(a, None, 2 * n, 1), "ajt_hbm_probe write 12.9 GB (st.global.v4)", 2 * n)
    run(lambda: ajt.hbm_probe(a, None, 2 * n, 3), "cudaMemsetAsync 12.9 GB", 2 * n)
    run(lambda: ajt.hbm_probe(b, a, 2 * n, 2), "ajt_hbm_probe copy 12.9 GB -> 12.9 GB", 4 * n)
    run(lambda: a.zero_(), "zero_ 12.9 GB (write only)", 2 * n)
    run(lambda: a.fill_(1.0), "fill_ 12.9 GB (write only)", 2 * n)
    run(lambda: b.copy_(a), "copy_ 12.9 GB -> 12.9 GB (read + write)", 4 * n)
    run(lambda: (b[:k].copy_(a[:k]), b[k:].fill_(0.0)), "27 % copied + 73 % filled: the bench step's read / write mix, 2 kernels",
        4 * k + 2 * (n - k))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="c1,c2,c3,c4,c5")
    ap.add_argument("--reps", type=int, default=20)
    ap.add_argument("--out", default=None, help="also append the JSON lines to this file")
    ap.add_argument("--merge-only", action="store_true")
    ap.add_argument("--quick", action="store_true", help="c5: 2x2 cells instead of 4x3")
    ap.add_argument("--both-rules", action="store_true")
    ap.add_argument("--stock-bandwidth", action="store_true", help="time torch fill_ / copy_ on 12.9 GB arrays and exit")
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("sweep: no CUDA device; the hot path has no CPU fallback")
    ajt.lib()
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    stream = torch.cuda.Stream(dev)
    out = open(args.out, "a") if args.out else None
    if args.stock_bandwidth:
        stock_bandwidth(dev, out)
        return
    rules = (("longest", ajt.OWNER_LONGEST), ("paper", ajt.OWNER_PAPER)) if args.both_rules else (("longest", ajt.OWNER_LONGEST),)
    cfgs = [c.strip() for c in args.configs.split(",") if c.strip()]
    t0 = time.time()
    for c in cfgs:
        if c == "c1":
            mi = W.merge_workload("c1")
            fin = measure_merge("c1", mi, dev, stream, args.reps, out, rules)
            if not args.merge_only:   # all merged tokens in one call, fp32 logits, V = 1024
                chunked_loss("c1", fin, 1024, (0.2, 0.2), W.BASE_SEED, 0, "pm1", fin.N_out, 1, dev, stream, args.reps, out,
                             dtype=torch.float32, sigma=2.0)
        elif c == "c2":
            mi = W.merge_workload("c2", seed=W.BASE_SEED + 1)
            fin = measure_merge("c2", mi, dev, stream, args.reps, out, rules)
            if not args.merge_only:
                chunked_loss("c2", fin, 151936, (0.2, 0.28), W.BASE_SEED + 1, 1, "zscore", 40960, 3, dev, stream, args.reps, out)
        elif c == "c3":
            mi = W.merge_workload("c3")
            fin = measure_merge("c3", mi, dev, stream, args.reps, out, rules)
            if not args.merge_only:
                chunked_loss("c3", fin, 151936, (0.2, 0.2), W.BASE_SEED + 2, 2, "zscore", 65536, 8, dev, stream,
                             max(5, args.reps // 2), out)
        elif c == "c4":
            for model, mi in W.merge_workload_c4().items():
                fin = measure_merge("c4" + model, mi, dev, stream, args.reps, out, rules)
                if not args.merge_only:
                    chunked_loss("c4" + model, fin, mi.meta["vocab"], (0.2, 0.2), W.BASE_SEED + 3, 3, "zscore", 65536, 4, dev, stream,
                                 max(5, args.reps // 2), out)
        elif c in W.BLOCK_SPECS:
            measure_blocks(c, W.block_workload(c), dev, stream, args.reps, out)
        elif c == "h1":   # Qwen3-8B-like head (d = 4096, V = 151936) over the bench micro-batch's rows
            measure_lm_head("h1", 40960, 4096, 151936, dev, stream, max(3, args.reps // 4), out)
            measure_lm_head("h1", 40960, 4096, 151936, dev, stream, max(3, args.reps // 4), out, rho=0.3)
        elif c == "h0":
            measure_lm_head("h0", 8192, 2048, 32000, dev, stream, args.reps, out)
        elif c == "c5":
            if not args.merge_only:
                run_c5(dev, stream, args.reps, out, quick=args.quick)
        else:
            raise SystemExit(f"unknown config {c}")
    print(f"# sweep done in {time.time() - t0:.1f} s", file=sys.stderr)


if __name__ == "__main__":
    main()
