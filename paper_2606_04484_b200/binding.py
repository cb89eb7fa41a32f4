"""ctypes binding of libajt.so: argument marshalling only (include/ajt.h is the contract).

torch is used for device memory and streams; numpy / pinned torch tensors for the *_host variants.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libajt.so")

OWNER_LONGEST, OWNER_PAPER = 0, 1
DT_BF16, DT_F32 = 0, 1
MERGE_WEAK_HASH = 1
STATUS_BAD_TARGET, STATUS_BAD_SEG, STATUS_BAD_OFFSETS, STATUS_ZERO_LEN = 1, 2, 4, 8
STATUS_PROBE_CAPACITY, STATUS_HASH_COLLISION, STATUS_INTERNAL = 16, 32, 64

_EXPORTS = [
    "ajt_version", "ajt_strerror", "ajt_last_status",
    "ajt_merge_workspace_bytes", "ajt_merge_workspace_bytes_for_pairs", "ajt_merge_timelines", "ajt_merge_host_arena_bytes", "ajt_merge_timelines_host",
    "ajt_loss_workspace_bytes", "ajt_policy_loss_fwd_bwd", "ajt_loss_host_arena_bytes", "ajt_policy_loss_fwd_bwd_host",
    "ajt_segment_counts", "ajt_policy_loss_fwd_bwd_ext", "ajt_merge_blocks_workspace_bytes", "ajt_merge_blocks",
    "ajt_pack_loss_inputs", "ajt_pack_microbatches", "ajt_lm_head_workspace_bytes", "ajt_lm_head_bwd_workspace_bytes",
    "ajt_lm_head_loss_bwd", "ajt_lm_head_logp",
    "ajt_hbm_probe", "ajt_launch_count", "ajt_host_ctx_create", "ajt_host_ctx_destroy", "ajt_policy_loss_fwd_bwd_host2",
    "ajt_loss_static_scratch_bytes", "ajt_policy_loss_fwd_bwd_static",
]

_lib = None


class AjtError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {strerror(code)} (code {code})")


def library_path() -> str:
    return _LIB_PATH


def exported_symbols():
    return list(_EXPORTS)


def lib():
    """Loads libajt.so.  Fails loudly when it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise RuntimeError(f"{_LIB_PATH} is missing: build it with `python -m paper_2606_04484_b200.build` "
                               "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(_LIB_PATH)
        L.ajt_version.restype = C.c_int
        L.ajt_strerror.restype = C.c_char_p
        L.ajt_strerror.argtypes = [C.c_int]
        L.ajt_last_status.restype = C.c_int
        for f in ("ajt_merge_workspace_bytes", "ajt_merge_host_arena_bytes"):
            getattr(L, f).restype = C.c_size_t
            getattr(L, f).argtypes = [C.c_int32, C.c_int64]
        L.ajt_merge_workspace_bytes_for_pairs.restype = C.c_size_t
        L.ajt_merge_workspace_bytes_for_pairs.argtypes = [C.c_int32, C.c_int64, C.c_int64]
        L.ajt_lm_head_workspace_bytes.restype = C.c_size_t
        L.ajt_lm_head_workspace_bytes.argtypes = [C.c_int64, C.c_int32, C.c_int32]
        L.ajt_lm_head_bwd_workspace_bytes.restype = C.c_size_t
        L.ajt_lm_head_bwd_workspace_bytes.argtypes = [C.c_int64, C.c_int32, C.c_int32, C.c_int32]
        L.ajt_lm_head_loss_bwd.restype = C.c_int
        L.ajt_merge_blocks_workspace_bytes.restype = C.c_size_t
        L.ajt_merge_blocks_workspace_bytes.argtypes = [C.c_int32, C.c_int64]
        L.ajt_loss_workspace_bytes.restype = C.c_size_t
        L.ajt_loss_workspace_bytes.argtypes = [C.c_int64, C.c_int32, C.c_int32]
        L.ajt_loss_host_arena_bytes.restype = C.c_size_t
        L.ajt_loss_host_arena_bytes.argtypes = [C.c_int64, C.c_int32, C.c_int32, C.c_int64, C.c_int32]
        for f in ("ajt_merge_timelines", "ajt_merge_timelines_host", "ajt_policy_loss_fwd_bwd",
                  "ajt_policy_loss_fwd_bwd_host", "ajt_segment_counts", "ajt_policy_loss_fwd_bwd_ext", "ajt_merge_blocks",
                  "ajt_pack_loss_inputs", "ajt_pack_microbatches", "ajt_lm_head_logp", "ajt_hbm_probe", "ajt_host_ctx_create",
                  "ajt_policy_loss_fwd_bwd_host2"):
            getattr(L, f).restype = C.c_int
        L.ajt_launch_count.restype = C.c_uint64
        L.ajt_host_ctx_destroy.restype = None
        L.ajt_host_ctx_destroy.argtypes = [C.c_void_p]
        _lib = L
    return _lib


def version() -> int:
    return int(lib().ajt_version())


def strerror(code: int) -> str:
    return lib().ajt_strerror(int(code)).decode()


def merge_workspace_bytes(n: int, n_tokens: int) -> int:
    return int(lib().ajt_merge_workspace_bytes(n, n_tokens))


def merge_workspace_bytes_for_pairs(n: int, n_tokens: int, n_pairs: int) -> int:
    return int(lib().ajt_merge_workspace_bytes_for_pairs(n, n_tokens, n_pairs))


def launch_count() -> int:
    """Kernels launched by the library in this process so far (include/ajt_test.h)."""
    return int(lib().ajt_launch_count())


def merge_host_arena_bytes(n: int, n_tokens: int) -> int:
    return int(lib().ajt_merge_host_arena_bytes(n, n_tokens))


def loss_workspace_bytes(T: int, V: int, S: int) -> int:
    return int(lib().ajt_loss_workspace_bytes(T, V, S))


def loss_host_arena_bytes(T: int, V: int, S: int, ld: int, dtype: int) -> int:
    return int(lib().ajt_loss_host_arena_bytes(T, V, S, ld, dtype))


def _dp(t: Optional[torch.Tensor]):
    return None if t is None else C.c_void_p(t.data_ptr())


def _hp(a):
    if a is None:
        return None
    if isinstance(a, torch.Tensor):
        return C.c_void_p(a.data_ptr())
    return a.ctypes.data_as(C.c_void_p)


def _stream(stream: Optional[torch.cuda.Stream] = None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _check_dev(t: Optional[torch.Tensor], dtype, name: str):
    if t is None:
        return
    if not t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous CUDA tensor of {dtype}, got {t.dtype} on {t.device}")


def _require_cuda():
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2606_04484_b200: no CUDA device; the hot path has no CPU fallback")


def last_status(workspace: torch.Tensor, stream=None) -> int:
    bits = C.c_uint32(0)
    rc = lib().ajt_last_status(_dp(workspace), _stream(stream), C.byref(bits))
    if rc != 0:
        raise AjtError(rc, "ajt_last_status")
    return int(bits.value)


# ------------------------------------------------------------------------------------------- merge


@dataclass
class MergeOutput:
    """Device tensors at worst-case capacity; only the first N_out / M entries are defined.  `finalize()`
    synchronises, reads `counts` and returns views of the right length."""
    merged_tokens: torch.Tensor
    merged_mask: torch.Tensor
    merged_src: torch.Tensor
    merged_old_logp: Optional[torch.Tensor]
    merged_offsets: torch.Tensor
    merged_origin: torch.Tensor
    merged_traj: torch.Tensor
    owner: torch.Tensor
    counts: torch.Tensor
    workspace: torch.Tensor
    M: int = -1
    N_out: int = -1

    def finalize(self) -> "MergeOutput":
        """Synchronises; raises AjtError when the call ended on a fatal status (the outputs are then empty)."""
        c = self.counts.cpu()
        M, No = int(c[0]), int(c[1])
        st = int(self.workspace[:4].view(torch.int32).cpu()[0]) & 0xFFFFFFFF
        if st & STATUS_PROBE_CAPACITY:
            raise AjtError(-3, "ajt_merge_timelines (AJT_STATUS_PROBE_CAPACITY: size the workspace with "
                               "merge_workspace_bytes_for_pairs)")
        if st & (STATUS_BAD_OFFSETS | STATUS_ZERO_LEN):
            raise AjtError(-1, "ajt_merge_timelines (bad offsets or a zero-length timeline)")
        return MergeOutput(self.merged_tokens[:No], self.merged_mask[:No], self.merged_src[:No],
                           None if self.merged_old_logp is None else self.merged_old_logp[:No],
                           self.merged_offsets[:M + 1], self.merged_origin[:M], self.merged_traj[:M], self.owner,
                           self.counts, self.workspace, M, No)


def merge_timelines(tokens: torch.Tensor, offsets: torch.Tensor, traj_ids: torch.Tensor,
                    resp_start: Optional[torch.Tensor] = None, mask_in: Optional[torch.Tensor] = None,
                    old_logp_in: Optional[torch.Tensor] = None, owner_rule: int = OWNER_LONGEST, flags: int = 0,
                    out: Optional[MergeOutput] = None, workspace_bytes: Optional[int] = None,
                    stream=None) -> MergeOutput:
    """ajt_merge_timelines (include/ajt.h).  All tensors live on the current CUDA device."""
    _require_cuda()
    _check_dev(tokens, torch.int32, "tokens")
    _check_dev(offsets, torch.int64, "offsets")
    _check_dev(traj_ids, torch.int32, "traj_ids")
    _check_dev(resp_start, torch.int32, "resp_start")
    _check_dev(mask_in, torch.uint8, "mask_in")
    _check_dev(old_logp_in, torch.float32, "old_logp_in")
    n, N = int(traj_ids.numel()), int(tokens.numel())
    dev = tokens.device
    if out is None:
        wsb = merge_workspace_bytes(n, N) if workspace_bytes is None else int(workspace_bytes)
        out = MergeOutput(
            torch.empty(max(N, 1), dtype=torch.int32, device=dev), torch.empty(max(N, 1), dtype=torch.uint8, device=dev),
            torch.empty(max(N, 1), dtype=torch.int32, device=dev),
            None if old_logp_in is None else torch.empty(max(N, 1), dtype=torch.float32, device=dev),
            torch.empty(n + 1, dtype=torch.int64, device=dev), torch.empty(max(n, 1), dtype=torch.int32, device=dev),
            torch.empty(max(n, 1), dtype=torch.int32, device=dev), torch.empty(max(n, 1), dtype=torch.int32, device=dev),
            torch.empty(2, dtype=torch.int64, device=dev), torch.empty(wsb, dtype=torch.uint8, device=dev))
    rc = lib().ajt_merge_timelines(
        _dp(tokens), _dp(offsets), _dp(traj_ids), _dp(resp_start), _dp(mask_in), _dp(old_logp_in),
        C.c_int32(n), C.c_int64(N), C.c_int32(owner_rule), C.c_uint32(flags),
        _dp(out.merged_tokens), _dp(out.merged_mask), _dp(out.merged_src), _dp(out.merged_old_logp),
        _dp(out.merged_offsets), _dp(out.merged_origin), _dp(out.merged_traj), _dp(out.owner), _dp(out.counts),
        _dp(out.workspace), C.c_size_t(out.workspace.numel()), _stream(stream))
    if rc != 0:
        raise AjtError(rc, "ajt_merge_timelines")
    return out


AUTHOR_ENV, AUTHOR_USER, AUTHOR_LLM = 0, 1, 2


def merge_blocks_workspace_bytes(n: int, n_blocks: int) -> int:
    return int(lib().ajt_merge_blocks_workspace_bytes(C.c_int32(n), C.c_int64(n_blocks)))


@dataclass
class BlockMergeOutput:
    """Device tensors at worst-case capacity; `finalize()` synchronises, reads `counts` and returns views of the right length."""
    merged_tokens: torch.Tensor
    merged_mask: torch.Tensor
    merged_logp: Optional[torch.Tensor]
    merged_tok_src: torch.Tensor
    merged_offsets: torch.Tensor
    merged_block_offsets: torch.Tensor
    merged_block_src: torch.Tensor
    merged_block_author: torch.Tensor
    merged_block_tok_off: torch.Tensor
    merged_origin: torch.Tensor
    merged_traj: torch.Tensor
    owner: torch.Tensor
    counts: torch.Tensor
    workspace: torch.Tensor
    M: int = -1
    B_out: int = -1
    N_out: int = -1

    def finalize(self) -> "BlockMergeOutput":
        c = self.counts.cpu()
        M, Bo, No = int(c[0]), int(c[1]), int(c[2])
        return BlockMergeOutput(self.merged_tokens[:No], self.merged_mask[:No],
                                None if self.merged_logp is None else self.merged_logp[:No], self.merged_tok_src[:No],
                                self.merged_offsets[:M + 1], self.merged_block_offsets[:M + 1], self.merged_block_src[:Bo],
                                self.merged_block_author[:Bo], self.merged_block_tok_off[:Bo + 1], self.merged_origin[:M],
                                self.merged_traj[:M], self.owner, self.counts, self.workspace, M, Bo, No)


def merge_blocks(block_ids: torch.Tensor, block_offsets: torch.Tensor, traj_ids: torch.Tensor, author: torch.Tensor,
                 tok_off: torch.Tensor, tokens: torch.Tensor, logp: Optional[torch.Tensor] = None,
                 tok_mask: Optional[torch.Tensor] = None, flags: int = 0, out: Optional[BlockMergeOutput] = None,
                 stream=None, extra_workspace_bytes: int = 0) -> BlockMergeOutput:
    """ajt_merge_blocks (include/ajt.h): Algorithm 1 with text-level matching on timelines of message blocks."""
    _require_cuda()
    _check_dev(block_ids, torch.int64, "block_ids")
    _check_dev(block_offsets, torch.int64, "block_offsets")
    _check_dev(traj_ids, torch.int32, "traj_ids")
    _check_dev(author, torch.uint8, "author")
    _check_dev(tok_off, torch.int64, "tok_off")
    _check_dev(tokens, torch.int32, "tokens")
    _check_dev(logp, torch.float32, "logp")
    _check_dev(tok_mask, torch.uint8, "tok_mask")
    n, B, N = int(traj_ids.numel()), int(block_ids.numel()), int(tokens.numel())
    dev = block_ids.device
    if out is None:
        e = lambda k, dt: torch.empty(max(k, 1), dtype=dt, device=dev)
        out = BlockMergeOutput(e(N, torch.int32), e(N, torch.uint8), None if logp is None else e(N, torch.float32),
                               e(N, torch.int32), e(n + 1, torch.int64), e(n + 1, torch.int64), e(B, torch.int32),
                               e(B, torch.uint8), e(B + 1, torch.int64), e(n, torch.int32), e(n, torch.int32), e(n, torch.int32),
                               e(3, torch.int64), e(merge_blocks_workspace_bytes(n, B) + int(extra_workspace_bytes), torch.uint8))
    rc = lib().ajt_merge_blocks(
        _dp(block_ids), _dp(block_offsets), _dp(traj_ids), _dp(author), _dp(tok_off), _dp(tokens), _dp(logp), _dp(tok_mask),
        C.c_int32(n), C.c_int64(B), C.c_int64(N), C.c_uint32(flags),
        _dp(out.merged_tokens), _dp(out.merged_mask), _dp(out.merged_logp), _dp(out.merged_tok_src), _dp(out.merged_offsets),
        _dp(out.merged_block_offsets), _dp(out.merged_block_src), _dp(out.merged_block_author), _dp(out.merged_block_tok_off),
        _dp(out.merged_origin), _dp(out.merged_traj), _dp(out.owner), _dp(out.counts), _dp(out.workspace),
        C.c_size_t(out.workspace.numel()), _stream(stream))
    if rc != 0:
        raise AjtError(rc, "ajt_merge_blocks")
    return out


@dataclass
class PackedLossInputs:
    """Device tensors at the capacity of the merge outputs; the first N_out entries are defined."""
    targets: torch.Tensor
    mask: torch.Tensor
    old_logp: Optional[torch.Tensor]
    seg_ids: torch.Tensor
    adv: Optional[torch.Tensor]
    status: torch.Tensor


def pack_loss_inputs(mo, tl_seg: torch.Tensor, S: int, seg_adv: Optional[torch.Tensor] = None,
                     out: Optional[PackedLossInputs] = None, stream=None) -> PackedLossInputs:
    """ajt_pack_loss_inputs (include/ajt.h).  `mo`: an un-finalized MergeOutput / BlockMergeOutput (capacity-sized tensors and
    the device `counts`); nothing is read back to the host."""
    _require_cuda()
    _check_dev(tl_seg, torch.int32, "tl_seg")
    _check_dev(seg_adv, torch.float32, "seg_adv")
    logp = getattr(mo, "merged_old_logp", None) if hasattr(mo, "merged_old_logp") else getattr(mo, "merged_logp", None)
    counts = mo.counts
    if counts.numel() == 3:       # block-level merge: {M, B_out, N_out}
        counts = torch.stack((counts[0], counts[2]))
    cap = int(mo.merged_tokens.numel())
    dev = mo.merged_tokens.device
    if out is None:
        out = PackedLossInputs(torch.empty(cap, dtype=torch.int32, device=dev), torch.empty(cap, dtype=torch.uint8, device=dev),
                               None if logp is None else torch.empty(cap, dtype=torch.float32, device=dev),
                               torch.empty(cap, dtype=torch.int32, device=dev),
                               None if seg_adv is None else torch.empty(cap, dtype=torch.float32, device=dev),
                               torch.empty(1, dtype=torch.int32, device=dev))
    rc = lib().ajt_pack_loss_inputs(_dp(mo.merged_tokens), _dp(mo.merged_mask), _dp(logp), _dp(mo.merged_offsets),
                                    _dp(mo.merged_origin), _dp(tl_seg), _dp(seg_adv), _dp(counts), C.c_int64(cap), C.c_int32(S),
                                    _dp(out.targets), _dp(out.mask), _dp(out.old_logp), _dp(out.seg_ids), _dp(out.adv),
                                    _dp(out.status), _stream(stream))
    if rc != 0:
        raise AjtError(rc, "ajt_pack_loss_inputs")
    return out


def pack_microbatches(mo, budget: int, stream=None):
    """ajt_pack_microbatches (include/ajt.h): token-budget packing of the merged sequences.  Returns device tensors
    (mb_seq int32 [n+2], mb_row int64 [n+2], n_mb int32 [1]); entries 0 .. n_mb are defined."""
    _require_cuda()
    counts = mo.counts
    if counts.numel() == 3:
        counts = torch.stack((counts[0], counts[2]))
    cap = int(mo.merged_offsets.numel()) + 1
    dev = mo.merged_offsets.device
    mb_seq = torch.empty(cap, dtype=torch.int32, device=dev)
    mb_row = torch.empty(cap, dtype=torch.int64, device=dev)
    n_mb = torch.zeros(1, dtype=torch.int32, device=dev)
    rc = lib().ajt_pack_microbatches(_dp(mo.merged_offsets), _dp(counts), C.c_int64(int(budget)), C.c_int32(cap), _dp(mb_seq),
                                     _dp(mb_row), _dp(n_mb), _stream(stream))
    if rc != 0:
        raise AjtError(rc, "ajt_pack_microbatches")
    return mb_seq, mb_row, n_mb


def merge_timelines_host(tokens, offsets, traj_ids, resp_start=None, mask_in=None, old_logp_in=None,
                         owner_rule: int = OWNER_LONGEST, flags: int = 0, arena: Optional[torch.Tensor] = None,
                         out: Optional[dict] = None, stream=None) -> dict:
    """ajt_merge_timelines_host: HOST buffers (numpy arrays or CPU torch tensors, pinned for speed).  Raises AjtError
    on a fatal status (pair capacity: pass a larger `arena`; bad offsets; zero-length timeline)."""
    _require_cuda()
    n, N = int(len(traj_ids)), int(len(tokens))
    if arena is None:
        arena = torch.empty(merge_host_arena_bytes(n, N), dtype=torch.uint8, device="cuda")
    if out is None:
        pin = dict(pin_memory=True)
        out = dict(merged_tokens=torch.empty(max(N, 1), dtype=torch.int32, **pin),
                   merged_mask=torch.empty(max(N, 1), dtype=torch.uint8, **pin),
                   merged_src=torch.empty(max(N, 1), dtype=torch.int32, **pin),
                   merged_old_logp=None if old_logp_in is None else torch.empty(max(N, 1), dtype=torch.float32, **pin),
                   merged_offsets=torch.empty(n + 1, dtype=torch.int64, **pin),
                   merged_origin=torch.empty(max(n, 1), dtype=torch.int32, **pin),
                   merged_traj=torch.empty(max(n, 1), dtype=torch.int32, **pin),
                   owner=torch.empty(max(n, 1), dtype=torch.int32, **pin))
    counts = np.zeros(2, np.int64)
    status = C.c_uint32(0)
    rc = lib().ajt_merge_timelines_host(
        _hp(tokens), _hp(offsets), _hp(traj_ids), _hp(resp_start), _hp(mask_in), _hp(old_logp_in),
        C.c_int32(n), C.c_int64(N), C.c_int32(owner_rule), C.c_uint32(flags),
        _hp(out["merged_tokens"]), _hp(out["merged_mask"]), _hp(out["merged_src"]), _hp(out["merged_old_logp"]),
        _hp(out["merged_offsets"]), _hp(out["merged_origin"]), _hp(out["merged_traj"]), _hp(out["owner"]),
        _hp(counts), C.byref(status), _dp(arena), C.c_size_t(arena.numel()), _stream(stream))
    if rc != 0:
        raise AjtError(rc, "ajt_merge_timelines_host")
    out = dict(out)
    out["M"], out["N_out"], out["status"] = int(counts[0]), int(counts[1]), int(status.value)
    return out


# ------------------------------------------------------------------------------------------- loss


@dataclass
class LossOutput:
    dlogits: torch.Tensor            # bf16 [T, ld]
    loss: torch.Tensor               # f32 [1] (device)
    logp: Optional[torch.Tensor]     # f32 [T]
    stats: Optional[torch.Tensor]    # f32 [4]
    workspace: torch.Tensor
    k3: Optional[torch.Tensor] = None    # f32 [T]  extended form: low-variance KL estimator per token
    ent: Optional[torch.Tensor] = None   # f32 [T]  extended form: entropy of each unmasked row
    ext: Optional[torch.Tensor] = None   # f32 [2]  extended form: {sum w_t k3_t, sum w_t H_t}


def policy_loss_fwd_bwd(logits: torch.Tensor, targets: torch.Tensor, old_logp: torch.Tensor, adv: torch.Tensor,
                        mask: torch.Tensor, seg_ids: torch.Tensor, S: int, eps_lo: float, eps_hi: float,
                        seg_denom: Optional[torch.Tensor] = None, inv_num_segs: float = 0.0, grad_scale: float = 1.0,
                        V: Optional[int] = None, dlogits: Optional[torch.Tensor] = None, want_logp: bool = False,
                        want_stats: bool = False, out: Optional[LossOutput] = None, stream=None) -> LossOutput:
    """ajt_policy_loss_fwd_bwd (include/ajt.h).  logits: CUDA [T, ld] bf16 or f32; V defaults to ld.
    Pass dlogits=logits (bf16) for the in-place backward."""
    _require_cuda()
    if logits.dim() != 2 or not logits.is_cuda or logits.stride(1) != 1:
        raise TypeError("logits: expected a 2-D CUDA tensor with unit column stride")
    if logits.dtype == torch.bfloat16:
        dt = DT_BF16
    elif logits.dtype == torch.float32:
        dt = DT_F32
    else:
        raise TypeError("logits: bf16 or f32 only")
    T, ld = int(logits.shape[0]), int(logits.stride(0)) if logits.shape[0] > 1 else int(logits.shape[1])
    V = int(logits.shape[1]) if V is None else int(V)
    _check_dev(targets, torch.int32, "targets")
    _check_dev(old_logp, torch.float32, "old_logp")
    _check_dev(adv, torch.float32, "adv")
    _check_dev(mask, torch.uint8, "mask")
    _check_dev(seg_ids, torch.int32, "seg_ids")
    _check_dev(seg_denom, torch.float32, "seg_denom")
    dev = logits.device
    if out is None:
        if dlogits is None:
            dlogits = torch.empty((T, ld), dtype=torch.bfloat16, device=dev)
        out = LossOutput(dlogits, torch.empty(1, dtype=torch.float32, device=dev),
                         torch.empty(max(T, 1), dtype=torch.float32, device=dev) if want_logp else None,
                         torch.empty(4, dtype=torch.float32, device=dev) if want_stats else None,
                         torch.empty(loss_workspace_bytes(T, V, S), dtype=torch.uint8, device=dev))
    if out.dlogits.dtype != torch.bfloat16 or not out.dlogits.is_cuda:
        raise TypeError("dlogits: expected a CUDA bf16 tensor")
    rc = lib().ajt_policy_loss_fwd_bwd(
        _dp(logits), _dp(targets), _dp(old_logp), _dp(adv), _dp(mask), _dp(seg_ids),
        C.c_float(eps_lo), C.c_float(eps_hi), C.c_int64(T), C.c_int32(V), C.c_int32(S), C.c_int64(ld), C.c_int32(dt),
        _dp(seg_denom), C.c_float(inv_num_segs), C.c_float(grad_scale), _dp(out.dlogits), _dp(out.loss), _dp(out.logp),
        _dp(out.stats), _dp(out.workspace), C.c_size_t(out.workspace.numel()), _stream(stream))
    if rc != 0:
        raise AjtError(rc, "ajt_policy_loss_fwd_bwd")
    return out


def loss_static_scratch_bytes() -> int:
    L = lib()
    L.ajt_loss_static_scratch_bytes.restype = C.c_size_t
    return int(L.ajt_loss_static_scratch_bytes())


def policy_loss_fwd_bwd_static(logits: torch.Tensor, targets: torch.Tensor, old_logp: torch.Tensor, adv: torch.Tensor,
                               mask: torch.Tensor, seg_ids: torch.Tensor, S: int, eps_lo: float, eps_hi: float,
                               dlogits: torch.Tensor, loss: torch.Tensor, logp: Optional[torch.Tensor] = None,
                               stats: Optional[torch.Tensor] = None, status: Optional[torch.Tensor] = None,
                               seg_denom: Optional[torch.Tensor] = None, inv_num_segs: float = 0.0, grad_scale: float = 1.0,
                               V: Optional[int] = None, stream=None) -> None:
    """ajt_policy_loss_fwd_bwd_static (include/ajt.h): the loss call with its scratch in the library's static device array.
    Allocates nothing: every output tensor is the caller's."""
    _require_cuda()
    if logits.dim() != 2 or not logits.is_cuda or logits.stride(1) != 1:
        raise TypeError("logits: expected a 2-D CUDA tensor with unit column stride")
    if logits.dtype == torch.bfloat16:
        dt = DT_BF16
    elif logits.dtype == torch.float32:
        dt = DT_F32
    else:
        raise TypeError("logits: bf16 or f32 only")
    T, ld = int(logits.shape[0]), int(logits.stride(0)) if logits.shape[0] > 1 else int(logits.shape[1])
    V = int(logits.shape[1]) if V is None else int(V)
    _check_dev(targets, torch.int32, "targets")
    _check_dev(old_logp, torch.float32, "old_logp")
    _check_dev(adv, torch.float32, "adv")
    _check_dev(mask, torch.uint8, "mask")
    _check_dev(seg_ids, torch.int32, "seg_ids")
    _check_dev(seg_denom, torch.float32, "seg_denom")
    _check_dev(loss, torch.float32, "loss")
    _check_dev(logp, torch.float32, "logp")
    _check_dev(stats, torch.float32, "stats")
    _check_dev(status, torch.int32, "status")
    if dlogits.dtype != torch.bfloat16 or not dlogits.is_cuda:
        raise TypeError("dlogits: expected a CUDA bf16 tensor")
    rc = lib().ajt_policy_loss_fwd_bwd_static(
        _dp(logits), _dp(targets), _dp(old_logp), _dp(adv), _dp(mask), _dp(seg_ids),
        C.c_float(eps_lo), C.c_float(eps_hi), C.c_int64(T), C.c_int32(V), C.c_int32(S), C.c_int64(ld), C.c_int32(dt),
        _dp(seg_denom), C.c_float(inv_num_segs), C.c_float(grad_scale), _dp(dlogits), _dp(loss), _dp(logp), _dp(stats),
        _dp(status), _stream(stream))
    if rc != 0:
        raise AjtError(rc, "ajt_policy_loss_fwd_bwd_static")


def policy_loss_fwd_bwd_ext(logits: torch.Tensor, targets: torch.Tensor, old_logp: torch.Tensor, adv: torch.Tensor,
                            mask: torch.Tensor, seg_ids: torch.Tensor, S: int, eps_lo: float, eps_hi: float,
                            ref_logp: Optional[torch.Tensor] = None, kl_coef: float = 0.0,
                            seg_denom: Optional[torch.Tensor] = None, inv_num_segs: float = 0.0, grad_scale: float = 1.0,
                            V: Optional[int] = None, dlogits: Optional[torch.Tensor] = None, want_logp: bool = False,
                            want_stats: bool = False, want_rows: bool = True, out: Optional[LossOutput] = None,
                            stream=None, clip_c: float = 0.0) -> LossOutput:
    """ajt_policy_loss_fwd_bwd_ext (include/ajt.h): the loss call plus the KL term against `ref_logp` (low_var_kl), the
    per-row entropy and the optional dual-clip bound `clip_c`, from the same single read of each row."""
    _require_cuda()
    if logits.dim() != 2 or not logits.is_cuda or logits.stride(1) != 1:
        raise TypeError("logits: expected a 2-D CUDA tensor with unit column stride")
    if logits.dtype == torch.bfloat16:
        dt = DT_BF16
    elif logits.dtype == torch.float32:
        dt = DT_F32
    else:
        raise TypeError("logits: bf16 or f32 only")
    T, ld = int(logits.shape[0]), int(logits.stride(0)) if logits.shape[0] > 1 else int(logits.shape[1])
    V = int(logits.shape[1]) if V is None else int(V)
    _check_dev(targets, torch.int32, "targets")
    _check_dev(old_logp, torch.float32, "old_logp")
    _check_dev(adv, torch.float32, "adv")
    _check_dev(mask, torch.uint8, "mask")
    _check_dev(seg_ids, torch.int32, "seg_ids")
    _check_dev(seg_denom, torch.float32, "seg_denom")
    _check_dev(ref_logp, torch.float32, "ref_logp")
    dev = logits.device
    if out is None:
        if dlogits is None:
            dlogits = torch.empty((T, ld), dtype=torch.bfloat16, device=dev)
        f32 = lambda n: torch.empty(n, dtype=torch.float32, device=dev)
        out = LossOutput(dlogits, f32(1), f32(max(T, 1)) if want_logp else None, f32(4) if want_stats else None,
                         torch.empty(loss_workspace_bytes(T, V, S), dtype=torch.uint8, device=dev),
                         f32(max(T, 1)) if want_rows else None, f32(max(T, 1)) if want_rows else None, f32(2))
    if out.dlogits.dtype != torch.bfloat16 or not out.dlogits.is_cuda:
        raise TypeError("dlogits: expected a CUDA bf16 tensor")
    if out.ext is None:
        raise TypeError("out.ext: the extended call needs a [2] f32 CUDA tensor")
    rc = lib().ajt_policy_loss_fwd_bwd_ext(
        _dp(logits), _dp(targets), _dp(old_logp), _dp(adv), _dp(mask), _dp(seg_ids),
        C.c_float(eps_lo), C.c_float(eps_hi), C.c_int64(T), C.c_int32(V), C.c_int32(S), C.c_int64(ld), C.c_int32(dt),
        _dp(seg_denom), C.c_float(inv_num_segs), C.c_float(grad_scale), _dp(ref_logp), C.c_float(kl_coef), C.c_float(clip_c),
        _dp(out.dlogits), _dp(out.loss), _dp(out.logp), _dp(out.stats), _dp(out.k3), _dp(out.ent), _dp(out.ext),
        _dp(out.workspace), C.c_size_t(out.workspace.numel()), _stream(stream))
    if rc != 0:
        raise AjtError(rc, "ajt_policy_loss_fwd_bwd_ext")
    return out


def lm_head_logp(hidden: torch.Tensor, weight: torch.Tensor, targets: torch.Tensor, mask: Optional[torch.Tensor] = None,
                 want_entropy: bool = True, workspace: Optional[torch.Tensor] = None, stream=None, want_lse: bool = False,
                 round_logits_bf16: bool = False):
    """ajt_lm_head_logp (include/ajt.h): (logp f32 [T], entropy f32 [T] | None) from hidden [T, d] and weight [V, d] (bf16);
    with want_lse also the row log-sum-exps as a third element."""
    _require_cuda()
    _check_dev(hidden, torch.bfloat16, "hidden")
    _check_dev(weight, torch.bfloat16, "weight")
    _check_dev(targets, torch.int32, "targets")
    _check_dev(mask, torch.uint8, "mask")
    if hidden.dim() != 2 or weight.dim() != 2 or hidden.stride(1) != 1 or weight.stride(1) != 1 or hidden.shape[1] != weight.shape[1]:
        raise TypeError("hidden [T, d] and weight [V, d] with unit column stride")
    T, d, V = int(hidden.shape[0]), int(hidden.shape[1]), int(weight.shape[0])
    dev = hidden.device
    logp = torch.empty(max(T, 1), dtype=torch.float32, device=dev)
    ent = torch.empty(max(T, 1), dtype=torch.float32, device=dev) if want_entropy else None
    lse = torch.empty(max(T, 1), dtype=torch.float32, device=dev) if want_lse else None
    if workspace is None:
        workspace = torch.empty(int(lib().ajt_lm_head_workspace_bytes(C.c_int64(T), C.c_int32(d), C.c_int32(V))) + 256, dtype=torch.uint8,
                                device=dev)
    rc = lib().ajt_lm_head_logp(_dp(hidden), _dp(weight), _dp(targets), _dp(mask), C.c_int64(T), C.c_int32(d), C.c_int32(V),
                                C.c_int64(int(hidden.stride(0)) if T > 1 else d), C.c_int64(int(weight.stride(0)) if V > 1 else d),
                                _dp(logp), _dp(ent), _dp(lse), C.c_uint32(1 if round_logits_bf16 else 0), _dp(workspace),
                                C.c_size_t(workspace.numel()), _stream(stream))
    if rc != 0:
        raise AjtError(rc, "ajt_lm_head_logp")
    if want_lse:
        return logp[:T], (None if ent is None else ent[:T]), lse[:T]
    return logp[:T], (None if ent is None else ent[:T])


def lm_head_loss_bwd(hidden: torch.Tensor, weight: torch.Tensor, targets: torch.Tensor, old_logp: torch.Tensor, adv: torch.Tensor,
                     mask: Optional[torch.Tensor], seg_ids: torch.Tensor, S: int, eps_lo: float, eps_hi: float,
                     seg_denom: Optional[torch.Tensor] = None, inv_num_segs: float = 0.0, grad_scale: float = 1.0,
                     dW: Optional[torch.Tensor] = None, accumulate_dw: bool = False, round_logits_bf16: bool = False,
                     workspace: Optional[torch.Tensor] = None, stream=None) -> dict:
    """ajt_lm_head_loss_bwd (include/ajt.h): loss, dH (bf16 [T, d]) and dW (fp32 [V, d]) from hidden states and head weights."""
    _require_cuda()
    _check_dev(hidden, torch.bfloat16, "hidden")
    _check_dev(weight, torch.bfloat16, "weight")
    _check_dev(targets, torch.int32, "targets")
    _check_dev(old_logp, torch.float32, "old_logp")
    _check_dev(adv, torch.float32, "adv")
    _check_dev(mask, torch.uint8, "mask")
    _check_dev(seg_ids, torch.int32, "seg_ids")
    _check_dev(seg_denom, torch.float32, "seg_denom")
    T, d = int(hidden.shape[0]), int(hidden.shape[1])
    V = int(weight.shape[0])
    dev = hidden.device
    dH = torch.empty((T, d), dtype=torch.bfloat16, device=dev)
    if dW is None:
        dW = torch.empty((V, d), dtype=torch.float32, device=dev)
        accumulate_dw = False
    _check_dev(dW, torch.float32, "dW")
    loss = torch.empty(1, dtype=torch.float32, device=dev)
    logp = torch.empty(max(T, 1), dtype=torch.float32, device=dev)
    if workspace is None:
        workspace = torch.empty(int(lib().ajt_lm_head_bwd_workspace_bytes(T, d, V, S)) + 256, dtype=torch.uint8, device=dev)
    rc = lib().ajt_lm_head_loss_bwd(_dp(hidden), _dp(weight), _dp(targets), _dp(old_logp), _dp(adv), _dp(mask), _dp(seg_ids),
                                    C.c_float(eps_lo), C.c_float(eps_hi), C.c_int64(T), C.c_int32(d), C.c_int32(V), C.c_int32(S),
                                    C.c_int64(d), C.c_int64(d), _dp(seg_denom), C.c_float(inv_num_segs), C.c_float(grad_scale),
                                    _dp(dH), C.c_int64(d), _dp(dW), C.c_int64(d), C.c_int32(1 if accumulate_dw else 0), _dp(loss),
                                    _dp(logp), C.c_uint32(1 if round_logits_bf16 else 0), _dp(workspace),
                                    C.c_size_t(workspace.numel()), _stream(stream))
    if rc != 0:
        raise AjtError(rc, "ajt_lm_head_loss_bwd")
    return dict(loss=loss, dH=dH, dW=dW, logp=logp[:T], workspace=workspace)


def hbm_probe(dst: Optional[torch.Tensor], src: Optional[torch.Tensor], nbytes: int, mode: int, stream=None) -> None:
    """ajt_hbm_probe (include/ajt.h): 0 read src, 1 write dst, 2 copy src -> dst, 3 cudaMemsetAsync(dst)."""
    _require_cuda()
    rc = lib().ajt_hbm_probe(_dp(dst), _dp(src), C.c_size_t(nbytes), C.c_int32(mode), _stream(stream))
    if rc != 0:
        raise AjtError(rc, "ajt_hbm_probe")


def segment_counts(mask: torch.Tensor, seg_ids: torch.Tensor, S: int, out: Optional[torch.Tensor] = None,
                   accumulate: bool = False, status: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """ajt_segment_counts (include/ajt.h): seg_denom[s] (+)= number of masked-in tokens of trajectory s."""
    _require_cuda()
    _check_dev(mask, torch.uint8, "mask")
    _check_dev(seg_ids, torch.int32, "seg_ids")
    if out is None:
        out = torch.empty(S, dtype=torch.float32, device=mask.device)
        accumulate = False
    _check_dev(out, torch.float32, "seg_denom")
    _check_dev(status, torch.int32, "status")
    rc = lib().ajt_segment_counts(_dp(mask), _dp(seg_ids), C.c_int64(int(mask.numel())), C.c_int32(S),
                                  C.c_int32(1 if accumulate else 0), _dp(out), _dp(status), _stream(stream))
    if rc != 0:
        raise AjtError(rc, "ajt_segment_counts")
    return out


def policy_loss_fwd_bwd_host(logits, targets, old_logp, adv, mask, seg_ids, S: int, eps_lo: float, eps_hi: float,
                             dtype: int, V: Optional[int] = None, seg_denom=None, inv_num_segs: float = 0.0,
                             grad_scale: float = 1.0, dlogits=None, want_logp: bool = False, want_stats: bool = False,
                             arena: Optional[torch.Tensor] = None, stream=None) -> dict:
    """ajt_policy_loss_fwd_bwd_host: HOST buffers.  logits: [T, ld] CPU tensor (bf16 / f32) or numpy
    (uint16 bit patterns for bf16 / float32)."""
    _require_cuda()
    T, ld = int(logits.shape[0]), int(logits.shape[1])
    V = ld if V is None else int(V)
    if arena is None:
        arena = torch.empty(loss_host_arena_bytes(T, V, S, ld, dtype), dtype=torch.uint8, device="cuda")
    if dlogits is None:
        dlogits = torch.empty((T, ld), dtype=torch.bfloat16, pin_memory=True)
    loss = np.zeros(1, np.float32)
    logp = np.zeros(max(T, 1), np.float32) if want_logp else None
    stats = np.zeros(4, np.float32) if want_stats else None
    status = C.c_uint32(0)
    rc = lib().ajt_policy_loss_fwd_bwd_host(
        _hp(logits), _hp(targets), _hp(old_logp), _hp(adv), _hp(mask), _hp(seg_ids), C.c_float(eps_lo), C.c_float(eps_hi),
        C.c_int64(T), C.c_int32(V), C.c_int32(S), C.c_int64(ld), C.c_int32(dtype), _hp(seg_denom), C.c_float(inv_num_segs),
        C.c_float(grad_scale), _hp(dlogits), _hp(loss), _hp(logp), _hp(stats), C.byref(status), _dp(arena),
        C.c_size_t(arena.numel()), _stream(stream))
    if rc != 0:
        raise AjtError(rc, "ajt_policy_loss_fwd_bwd_host")
    return dict(dlogits=dlogits, loss=float(loss[0]), logp=logp, stats=stats, status=int(status.value))


class HostCtx:
    """ajt_host_ctx: the helper streams / events of the host slab pipeline, created once."""

    def __init__(self):
        _require_cuda()
        self.h = C.c_void_p(None)
        rc = lib().ajt_host_ctx_create(C.byref(self.h))
        if rc != 0:
            raise AjtError(rc, "ajt_host_ctx_create")

    def close(self):
        if self.h:
            lib().ajt_host_ctx_destroy(self.h)
            self.h = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def policy_loss_fwd_bwd_host2(logits, targets, old_logp, adv, mask, seg_ids, S: int, eps_lo: float, eps_hi: float,
                              dtype: int, dlogits_device: torch.Tensor, V: Optional[int] = None, seg_denom=None,
                              inv_num_segs: float = 0.0, grad_scale: float = 1.0, want_logp: bool = False,
                              want_stats: bool = False, ctx: Optional[HostCtx] = None, arena: Optional[torch.Tensor] = None,
                              stream=None) -> dict:
    """ajt_policy_loss_fwd_bwd_host2 with the gradient left on the device: HOST inputs, `dlogits_device` a CUDA bf16 [T, ld]
    tensor; only loss / logp / stats / status come back."""
    _require_cuda()
    T, ld = int(logits.shape[0]), int(logits.shape[1])
    V = ld if V is None else int(V)
    _check_dev(dlogits_device, torch.bfloat16, "dlogits_device")
    if arena is None:
        arena = torch.empty(loss_host_arena_bytes(T, V, S, ld, dtype), dtype=torch.uint8, device="cuda")
    loss = np.zeros(1, np.float32)
    logp = np.zeros(max(T, 1), np.float32) if want_logp else None
    stats = np.zeros(4, np.float32) if want_stats else None
    status = C.c_uint32(0)
    rc = lib().ajt_policy_loss_fwd_bwd_host2(
        _hp(logits), _hp(targets), _hp(old_logp), _hp(adv), _hp(mask), _hp(seg_ids), C.c_float(eps_lo), C.c_float(eps_hi),
        C.c_int64(T), C.c_int32(V), C.c_int32(S), C.c_int64(ld), C.c_int32(dtype), _hp(seg_denom), C.c_float(inv_num_segs),
        C.c_float(grad_scale), _dp(dlogits_device), C.c_int32(1), _hp(loss), _hp(logp), _hp(stats), C.byref(status),
        None if ctx is None else ctx.h, _dp(arena), C.c_size_t(arena.numel()), _stream(stream))
    if rc != 0:
        raise AjtError(rc, "ajt_policy_loss_fwd_bwd_host2")
    return dict(dlogits=dlogits_device, loss=float(loss[0]), logp=logp, stats=stats, status=int(status.value))
