"""Measurement harness used by bench.py and the full-size tests: algorithmic byte counts, input synthesis on the device, CUDA-event
timing with an L2 flush.  None of the method's steps is computed here (the one softmax below only SYNTHESISES the
`old_logp` input as "new logp + noise", BASELINE.json configs), and nothing here touches the oracle."""
from __future__ import annotations

import json
import os
from typing import Callable, List, Optional

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
FALLBACK_HBM_GBS = 6650.0   # /opt/skills/guides/B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
NOMINAL_HBM_GBS = 8000.0    # BASELINE.json north_star "~8 TB/s"


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            with open(p) as f:
                return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def merge_bytes(n: int, N_in: int, N_out: int, with_logp: bool = True) -> int:
    """read every input token once, write every output once."""
    return 4 * N_in + 9 * N_out + (4 * N_out if with_logp else 0) + 20 * n


def loss_bytes(T: int, V: int, n_unmasked: int, b_in: int = 2) -> int:
    """read each UNMASKED row once, write EVERY row once, 17 B/token of side inputs."""
    return n_unmasked * V * b_in + T * V * 2 + 17 * T


def fill_logits(buf: torch.Tensor, seed: int, sigma: float = 3.0, slab: int = 2048) -> None:
    g = torch.Generator(device=buf.device).manual_seed(seed)
    for a in range(0, buf.shape[0], slab):
        b = min(buf.shape[0], a + slab)
        buf[a:b] = (torch.randn((b - a, buf.shape[1]), generator=g, device=buf.device, dtype=torch.float32) * sigma).to(buf.dtype)


def harness_old_logp(logits_t: torch.Tensor, targets_t: torch.Tensor, noise: np.ndarray) -> torch.Tensor:
    """INPUT synthesis, not the method: old_logp = (library log-softmax of the row at its target) + noise
    (BASELINE.json configs: "old_logp = new logp + N(0,0.05)")."""
    T = logits_t.shape[0]
    out = torch.empty(T, dtype=torch.float32, device=logits_t.device)
    step = max(1, (1 << 27) // max(1, logits_t.shape[1]))
    for a in range(0, T, step):
        z = logits_t[a:a + step].float()
        lse = torch.logsumexp(z, dim=-1)
        out[a:a + step] = z.gather(1, targets_t[a:a + step].long()[:, None])[:, 0] - lse
    return out + torch.from_numpy(noise).to(out.device)


class L2Flusher:
    """Writes a buffer larger than the 126 MB L2 so that the next call starts cold."""

    def __init__(self, device, mbytes: int = 256):
        self.buf = torch.empty(mbytes << 20, dtype=torch.uint8, device=device)
        self.k = 0

    def __call__(self):
        self.k = (self.k + 1) & 0x7F
        self.buf.fill_(self.k)


def time_calls(fn: Callable[[], None], stream: torch.cuda.Stream, reps: int = 20, warmup: int = 3,
               flush: Optional[L2Flusher] = None) -> List[float]:
    """Per-call device times in ms: CUDA events recorded on `stream` right around each call (the optional L2 flush
    runs on the same stream before the start event)."""
    with torch.cuda.stream(stream):
        for _ in range(warmup):
            if flush:
                flush()
            fn()
        stream.synchronize()
        evs = []
        for _ in range(reps):
            if flush:
                flush()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            fn()
            e1.record(stream)
            evs.append((e0, e1))
        stream.synchronize()
    return [a.elapsed_time(b) for a, b in evs]
