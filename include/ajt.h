/*
 * ajt.h — C ABI of libajt.so: B200-native (sm_100a) timeline merging and policy-loss fwd+bwd.
 *
 * The two hot-path calls follow the paper's statement of the problem (arxiv/paper_2606_04484,
 * "AgentJet"; line numbers are /root/reference/PAPER.md):
 *
 *   ajt_merge_timelines      Timeline merging, Algorithm 1 (§4.4.2) on flat token
 *                            streams with token-level Match: every timeline whose token
 *                            context is a prefix of a LATER timeline of the same episode is absorbed;
 *                            the survivors carry the OR of the LLM loss masks (eq. (1))
 *                            and an index map back to the original timelines.
 *   ajt_policy_loss_fwd_bwd  "policy gradient ... loss terms are computed" (§4.2 step 4),
 *                            "GRPO-style policy-gradient updates", clip_ratio 0.2
 *                            (PAPER.md:531).  The formula is BASELINE.json north_star's: fused online
 *                            log-softmax over V, target gather, importance ratio vs old log-probs,
 *                            PPO/GRPO clip, masked per-trajectory mean; forward value and gradient
 *                            w.r.t. the logits, written in bf16 (DESIGN.md "O-L" steps 1-7).
 *
 * Conventions (all calls)
 *   - Plain pointers and sizes; no C++ or framework types.  Pointers marked DEVICE are CUDA device
 *     memory owned by the caller; the library allocates nothing and frees nothing.
 *   - Calls enqueue work on `stream` and return WITHOUT synchronising.  The return value reports
 *     host-detectable errors only (AJT_ERR_*).  Data-dependent faults set bits in a device status
 *     word inside the workspace (AJT_STATUS_*), read back with ajt_last_status(); outputs are then
 *     unspecified.  No exceptions, no abort(); thread-safe for distinct workspaces.  The only state kept between
 *     calls is a per-device table of launch facts (SM count, one-time shared-memory opt-in of the kernels), written
 *     once per device with idempotent values.
 *   - There is no CPU fallback: without a CUDA device every compute call returns AJT_ERR_CUDA.
 *   - The *_host variants take HOST buffers, stage them through a caller-provided device arena with
 *     cudaMemcpyAsync on `stream`, run the same kernels and copy the results back; they synchronise
 *     the stream before returning.
 */
#ifndef AJT_H_
#define AJT_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct CUstream_st* ajt_stream_t; /* cudaStream_t */

enum {
    AJT_OK = 0,
    AJT_ERR_INVALID_ARG = -1,
    AJT_ERR_WORKSPACE_TOO_SMALL = -2,
    AJT_ERR_CAPACITY = -3,
    AJT_ERR_CUDA = -4,
    AJT_ERR_UNSUPPORTED = -5
};

/* Owner rule (reading M-3). */
enum {
    AJT_OWNER_LONGEST = 0, /* BASELINE.json north_star: longest surviving extender, then lowest index */
    AJT_OWNER_PAPER = 1    /* Algorithm 1 literally: the latest extender */
};

enum { AJT_DT_BF16 = 0, AJT_DT_F32 = 1 };

/* ajt_merge_timelines `flags`: 0 (include/ajt_test.h defines a test hook). */

/* Device status bits (ajt_last_status). */
enum {
    AJT_STATUS_BAD_TARGET = 1,       /* targets[t] outside [0,V) on a masked-in row */
    AJT_STATUS_BAD_SEG = 2,          /* seg_ids[t] outside [0,S) on a masked-in row */
    AJT_STATUS_BAD_OFFSETS = 4,      /* offsets[0] != 0, decreasing, or offsets[n] != n_tokens */
    AJT_STATUS_ZERO_LEN = 8,         /* a timeline of length 0 (L_j >= 1 required) */
    AJT_STATUS_PROBE_CAPACITY = 16,  /* more candidate (timeline, earlier-length) pairs than the workspace holds */
    AJT_STATUS_HASH_COLLISION = 32,  /* informational: a hash-equal candidate failed the exact token comparison and was
                                        skipped (the outputs are exact either way) */
    AJT_STATUS_INTERNAL = 64
};

int ajt_version(void);                /* major*10000 + minor*100 + patch */
const char* ajt_strerror(int code);   /* static string for an AJT_ERR_* code */

/* Synchronises `stream`, copies the status word of `workspace` (DEVICE) to *bits.  Returns AJT_OK or AJT_ERR_CUDA. */
int ajt_last_status(const void* workspace, ajt_stream_t stream, uint32_t* bits);

/* ------------------------------------------------------------------------------------------------
 * Stage (a): timeline merging.  Algorithm 1; definition restated in DESIGN.md "O-M".
 *
 *   i extends j  <=>  traj_ids[i]==traj_ids[j], i>j, L_i>=L_j, tokens_i[0:L_j]==tokens_j
 *   j survives   <=>  no i extends j; survivors are numbered m=0..M-1 in ascending original index
 *   owner_tl(j)  =    j if it survives; else per `owner_rule` among the (surviving) extenders of j
 *   merged seq m =    the survivor's tokens; mask = OR of member masks; src / old_logp from the largest
 *                     member index whose mask is 1 at that position (Alg. 1 lines 10-17)
 *
 * Workspace: ajt_merge_workspace_bytes(n, n_tokens) bytes of DEVICE memory, 256-byte aligned.  It sizes
 * room for 64*n + 4096 candidate pairs.  The call needs one pair per (timeline, earlier-or-same timeline of its group):
 * n_pairs = sum over groups of k_g (k_g + 1) / 2, which the caller can count from traj_ids alone.  A batch that needs
 * more (groups of more than ~127 timelines on average) sets AJT_STATUS_PROBE_CAPACITY; size the workspace with
 * ajt_merge_workspace_bytes_for_pairs(n, n_tokens, n_pairs) instead (every extra 32 bytes hold one more pair; the
 * capacity always follows from `workspace_bytes`).
 *
 * All integer; outputs are bit-exact with the definition, whatever the prefix hash does: a candidate is accepted only
 * through exactly compared links or after an exact token comparison (AJT_STATUS_HASH_COLLISION is informational: a
 * hash-equal candidate was rejected by that comparison).  Only the first N_out / M entries of the outputs are written.
 * `counts` is DEVICE memory: synchronise the stream before reading it.  After a fatal status (bad offsets, zero-length
 * timeline, pair capacity) the outputs are unspecified except counts = {0, 0} and merged_offsets[0] = 0, so that a chained
 * call (ajt_pack_loss_inputs) does nothing.  The call is five plain kernel launches on `stream` (no cooperative launch, no
 * host read-back): it can be captured in a CUDA graph.
 */
size_t ajt_merge_workspace_bytes(int32_t n, int64_t n_tokens);
size_t ajt_merge_workspace_bytes_for_pairs(int32_t n, int64_t n_tokens, int64_t n_pairs);

int ajt_merge_timelines(
    /* inputs, DEVICE, read-only */
    const int32_t* tokens,      /* [n_tokens] packed token ids (opaque 32-bit patterns, compared bitwise) */
    const int64_t* offsets,     /* [n+1] offsets[0]=0, strictly increasing, offsets[n]=n_tokens */
    const int32_t* traj_ids,    /* [n] opaque group keys; need not be contiguous or sorted */
    const int32_t* resp_start,  /* [n] mask_j[p] = (p >= resp_start[j]); may be NULL if mask_in is given */
    const uint8_t* mask_in,     /* [n_tokens] explicit per-token 0/1 mask, or NULL -> use resp_start */
    const float* old_logp_in,   /* [n_tokens] per-token log-probs carried on the timelines, or NULL */
    int32_t n, int64_t n_tokens, int32_t owner_rule, uint32_t flags,
    /* outputs, DEVICE, caller-allocated with worst-case capacity (n_tokens tokens, n sequences) */
    int32_t* merged_tokens,     /* [N_out] */
    uint8_t* merged_mask,       /* [N_out] */
    int32_t* merged_src,        /* [N_out] original timeline index supplying mask/logp here, -1 if mask 0 */
    float* merged_old_logp,     /* [N_out], or NULL (must be NULL iff old_logp_in is NULL) */
    int64_t* merged_offsets,    /* [M+1] */
    int32_t* merged_origin,     /* [M] original index of the surviving timeline */
    int32_t* merged_traj,       /* [M] its traj_id */
    int32_t* owner,             /* [n] merged-sequence index m whose first L_j tokens are timeline j */
    int64_t* counts,            /* [2] {M, N_out} */
    void* workspace, size_t workspace_bytes, ajt_stream_t stream);

/* ------------------------------------------------------------------------------------------------
 * Stage (a'), text-level matching: Algorithm 1 on timelines of MESSAGE BLOCKS (eq. (1)) with
 * Match = text, the paper's default strategy.
 *
 * Timeline i = blocks block_offsets[i] .. block_offsets[i+1].  Block b = (text, author, tokens, log-probs, mask): the text
 * is represented by a caller-supplied 64-bit id with equal ids <=> equal texts (reading B-1); author is AJT_AUTHOR_*;
 * tokens / logp / tok_mask of block b are elements tok_off[b] .. tok_off[b+1] of the packed arrays.
 *   i extends j  <=>  traj_ids equal, i > j, K_i >= K_j and block_ids_i[k] == block_ids_j[k] for k < K_j
 *   j is absorbed by its LATEST extender (the reverse double loop); survivors keep their order (line 22)
 *   block k of a survivor s: if some member has an llm block at k and s has not, the block takes author llm, tokens and
 *   log-probs (and mask) from the latest such member (lines 10-17); otherwise it stays s's own
 * tok_mask NULL -> mu = 1 exactly on the tokens of llm blocks.  Token-level matching of the same data is
 * ajt_merge_timelines on the flat token streams.
 *
 * Outputs (DEVICE, caller-allocated at worst-case capacity: n_tokens tokens, n_blocks blocks, n sequences):
 *   merged_tokens / merged_mask / merged_logp / merged_tok_src [N_out] (tok_src = supplying timeline where the mask is 1,
 *   else -1; logp 0 where the mask is 0), merged_offsets [M+1] (tokens), merged_block_offsets [M+1] (blocks),
 *   merged_block_src [B_out] (timeline whose block k stands at block k of the survivor), merged_block_author [B_out],
 *   merged_block_tok_off [B_out+1], merged_origin / merged_traj [M], owner [n], counts [3] = {M, B_out, N_out}.
 * All integer / byte work: bit-exact with the definition.  Workspace: ajt_merge_blocks_workspace_bytes(n, n_blocks) bytes
 * of DEVICE memory, 256-byte aligned (0 is returned for n_blocks >= 2^30); like ajt_merge_timelines it holds 64*n + 4096
 * candidate pairs and every extra 32 bytes the caller provides hold one more.  Status bits as for ajt_merge_timelines
 * (AJT_STATUS_BAD_OFFSETS also for a decreasing tok_off); `flags` as there.  Enqueues on `stream`, does not synchronise.
 */
enum { AJT_AUTHOR_ENV = 0, AJT_AUTHOR_USER = 1, AJT_AUTHOR_LLM = 2 };

size_t ajt_merge_blocks_workspace_bytes(int32_t n, int64_t n_blocks);

int ajt_merge_blocks(
    const int64_t* block_ids,      /* DEVICE [n_blocks] text ids */
    const int64_t* block_offsets,  /* DEVICE [n+1] block_offsets[0]=0, strictly increasing, block_offsets[n]=n_blocks */
    const int32_t* traj_ids,       /* DEVICE [n] */
    const uint8_t* author,         /* DEVICE [n_blocks] AJT_AUTHOR_* */
    const int64_t* tok_off,        /* DEVICE [n_blocks+1] tok_off[0]=0, non-decreasing, tok_off[n_blocks]=n_tokens */
    const int32_t* tokens,         /* DEVICE [n_tokens] */
    const float* logp,             /* DEVICE [n_tokens] or NULL */
    const uint8_t* tok_mask,       /* DEVICE [n_tokens] or NULL */
    int32_t n, int64_t n_blocks, int64_t n_tokens, uint32_t flags,
    int32_t* merged_tokens, uint8_t* merged_mask, float* merged_logp /* NULL iff logp is NULL */, int32_t* merged_tok_src,
    int64_t* merged_offsets, int64_t* merged_block_offsets, int32_t* merged_block_src, uint8_t* merged_block_author,
    int64_t* merged_block_tok_off, int32_t* merged_origin, int32_t* merged_traj, int32_t* owner, int64_t* counts,
    void* workspace, size_t workspace_bytes, ajt_stream_t stream);

/* HOST-buffer variant: same arguments but every array pointer is HOST memory (pinned for speed).
 * `arena` is DEVICE scratch of at least ajt_merge_host_arena_bytes(n, n_tokens) bytes; whatever it holds beyond that goes
 * to the candidate pairs (ajt_merge_workspace_bytes_for_pairs(n, n_tokens, n_pairs) - ajt_merge_workspace_bytes(n, n_tokens)
 * more bytes hold n_pairs).  Synchronises.  A fatal status is an error of this call: AJT_ERR_CAPACITY for
 * AJT_STATUS_PROBE_CAPACITY, AJT_ERR_INVALID_ARG for bad offsets / zero-length timelines (status_bits is still filled). */
size_t ajt_merge_host_arena_bytes(int32_t n, int64_t n_tokens);

int ajt_merge_timelines_host(
    const int32_t* tokens, const int64_t* offsets, const int32_t* traj_ids, const int32_t* resp_start,
    const uint8_t* mask_in, const float* old_logp_in, int32_t n, int64_t n_tokens, int32_t owner_rule,
    uint32_t flags, int32_t* merged_tokens, uint8_t* merged_mask, int32_t* merged_src, float* merged_old_logp,
    int64_t* merged_offsets, int32_t* merged_origin, int32_t* merged_traj, int32_t* owner,
    int64_t* counts /* HOST [2] */, uint32_t* status_bits /* HOST [1] or NULL */,
    void* arena /* DEVICE */, size_t arena_bytes, ajt_stream_t stream);

/* ------------------------------------------------------------------------------------------------
 * Bridge (a) -> (b): per-token loss inputs from the merge outputs, on the device ("the packed merged sequences",
 * BASELINE.json north_star; reading L-12).  For position q of merged sequence m:
 *   targets[q] = merged_tokens[q+1], mask[q] = merged_mask[q+1], old_logp[q] = merged_old_logp[q+1]
 *   (next-token alignment inside the sequence); at the LAST position of every sequence all three are 0
 *   seg_ids[q] = tl_seg[merged_origin[m]];   adv[q] = seg_adv[seg_ids[q]]
 * tl_seg [n]: caller's dense trajectory id in [0,S) of every ORIGINAL timeline (the traj_ids renumbered on the host);
 * seg_adv [S]: one advantage per trajectory (GRPO).  counts = the merge call's {M, N_out} (DEVICE): nothing is
 * read back to the host between the merge, this call and the loss.  Only the first N_out entries of the outputs are
 * written; a micro-batch is then any row range of them (rows are independent given ajt_segment_counts, reading L-4).
 * merged_old_logp / old_logp and seg_adv / adv may be NULL in pairs.  status_bits DEVICE [1] or NULL: AJT_STATUS_BAD_SEG
 * when a tl_seg value is outside [0,S) (segment 0 is used).  All pointers DEVICE; enqueues on `stream`. */
int ajt_pack_loss_inputs(
    const int32_t* merged_tokens, const uint8_t* merged_mask, const float* merged_old_logp, const int64_t* merged_offsets,
    const int32_t* merged_origin, const int32_t* tl_seg, const float* seg_adv, const int64_t* counts,
    int64_t capacity_tokens /* size of the token arrays (>= N_out) */, int32_t S,
    int32_t* targets, uint8_t* mask, float* old_logp, int32_t* seg_ids, float* adv,
    uint32_t* status_bits, ajt_stream_t stream);

/* Token-budget packing of the merged sequences into micro-batches, on the device ("the packed merged sequences",
 * BASELINE.json north_star): consecutive sequences are taken in order while the rows of the
 * micro-batch stay <= budget (a sequence longer than the budget gets a micro-batch of its own).  Micro-batch b is
 * sequences mb_seq[b] .. mb_seq[b+1] = rows mb_row[b] .. mb_row[b+1] of the arrays ajt_pack_loss_inputs writes, so a loss
 * call per micro-batch is a row range of them.  merged_offsets / counts: the merge call's (DEVICE).  mb_seq / mb_row:
 * DEVICE [capacity], n_mb DEVICE [1]; entries up to n_mb (inclusive: the closing entry {M, N_out}) are written when
 * n_mb < capacity (size them M + 1).  Enqueues on `stream`. */
int ajt_pack_microbatches(const int64_t* merged_offsets, const int64_t* counts, int64_t budget, int32_t capacity,
                          int32_t* mb_seq, int64_t* mb_row, int32_t* n_mb, ajt_stream_t stream);

/* ------------------------------------------------------------------------------------------------
 * Stage (b): token-level clipped policy-gradient loss, forward and backward w.r.t. the logits.
 * Definition, for t in [0,T):
 *   lse_t = log sum_v exp(z_tv);  logp_t = z_{t,y_t} - lse_t;  r_t = exp(logp_t - old_logp_t)
 *   L_t   = -min(r_t A_t, clip(r_t, 1-eps_lo, 1+eps_hi) A_t)
 *   N_s   = sum_{t: seg_t = s} mask_t  (or seg_denom[s]);  S' = #{s: N_s > 0}  (or 1/inv_num_segs)
 *   w_t   = mask_t / (N_{seg_t} S');   loss = sum_t w_t L_t
 *   g_t   = grad_scale w_t (-A_t r_t) [not (A_t>0 and r_t>1+eps_hi)] [not (A_t<0 and r_t<1-eps_lo)]
 *   dlogits_tv = g_t (1[v = y_t] - exp(z_tv - lse_t))      stored as bf16, round-to-nearest-even
 * Rows with mask_t = 0 are not read; their dlogits rows are written as zeros.
 *
 * Arithmetic: fp32 on chip, the scalar loss accumulated in fp64 in a fixed order (bitwise reproducible).
 * Fast path (one HBM read of each unmasked row, one write of every row): bf16 logits, V % 8 == 0,
 * ld_logits % 8 == 0, 16-byte aligned base pointers, V <= 155648.  Everything else (fp32 logits, odd V,
 * larger V) takes a slower generic kernel with the same results.
 *
 * `dlogits` may alias `logits` when logits_dtype is AJT_DT_BF16 (in-place backward).
 * Workspace: ajt_loss_workspace_bytes(T, V, S) bytes of DEVICE memory, 256-byte aligned.
 */
size_t ajt_loss_workspace_bytes(int64_t T, int32_t V, int32_t S);

int ajt_policy_loss_fwd_bwd(
    const void* logits,         /* DEVICE [T, ld_logits] row-major, logits_dtype; columns [0,V) are used */
    const int32_t* targets,     /* DEVICE [T] in [0,V) */
    const float* old_logp,      /* DEVICE [T] */
    const float* adv,           /* DEVICE [T] per-token advantage */
    const uint8_t* mask,        /* DEVICE [T] 0/1 */
    const int32_t* seg_ids,     /* DEVICE [T] in [0,S): trajectory of each token */
    float eps_lo, float eps_hi,
    int64_t T, int32_t V, int32_t S, int64_t ld_logits, int32_t logits_dtype,
    const float* seg_denom,     /* DEVICE [S] or NULL: override N_s (chunked streaming, reading L-4) */
    float inv_num_segs,         /* 0 -> compute 1/S' from this call's tokens; else used as given */
    float grad_scale,           /* upstream dLoss, normally 1.0f */
    void* dlogits,              /* DEVICE [T, ld_logits] bf16 */
    float* loss_out,            /* DEVICE [1]: this call's sum_t w_t L_t (the caller sums chunks) */
    float* logp_out,            /* DEVICE [T] or NULL: logp_t where mask_t = 1, 0 elsewhere */
    float* stats_out,           /* DEVICE [4] or NULL: {n_masked, n_clipped_hi, n_clipped_lo, sum_t w_t (-log r_t)} */
    void* workspace, size_t workspace_bytes, ajt_stream_t stream);

/* Extended form: the same call with the protocol's "other loss terms" fused into the same single
 * read of each row (DESIGN.md "O-L" steps 8-9, readings L-16, L-17):
 *   step 8  KL penalty against a reference policy with the low-variance estimator the protocol names
 *           (`kl_loss_coef = 2e-3`, `low_var_kl`):
 *             d_t = ref_logp_t - logp_t;   k3_t = min(exp(d_t) - d_t - 1, 10)
 *             loss = sum_t w_t (L_t + kl_coef k3_t);   g_t += grad_scale w_t kl_coef (1 - exp(d_t)) [k3_t < 10]
 *           switched off by ref_logp = NULL or kl_coef = 0 (then k3_t = 0).
 *   step 9  entropy of each unmasked row's softmax (the policy entropy the paper monitors),
 *             H_t = lse_t - sum_v p_tv z_tv,   reported only (no gradient).
 *   step 3b the optional three-parameter "dual-clip" bound (reading L-18): clip_c > 1 caps the surrogate
 *           of negative-advantage tokens, L_t = min(L_t, -A_t clip_c), with zero gradient where the cap is active
 *           (r_t > clip_c); clip_c = 0 switches it off.  (stats_out does not count capped tokens.)
 * Extra arguments: ref_logp DEVICE [T] or NULL; kl_coef >= 0; clip_c >= 0; k3_out, ent_out DEVICE [T] or NULL (k3_t, H_t where
 * mask_t = 1, 0 elsewhere); ext_out DEVICE [2], required: {sum_t w_t k3_t, sum_t w_t H_t} of this call.
 * Everything else (arguments, workspace, layouts, error behaviour, paths) is as for ajt_policy_loss_fwd_bwd; with
 * ref_logp = NULL the loss, dlogits, logp_out and stats_out are bit-identical to that call's. */
int ajt_policy_loss_fwd_bwd_ext(
    const void* logits, const int32_t* targets, const float* old_logp, const float* adv, const uint8_t* mask,
    const int32_t* seg_ids, float eps_lo, float eps_hi, int64_t T, int32_t V, int32_t S, int64_t ld_logits,
    int32_t logits_dtype, const float* seg_denom, float inv_num_segs, float grad_scale,
    const float* ref_logp, float kl_coef, float clip_c,
    void* dlogits, float* loss_out, float* logp_out, float* stats_out,
    float* k3_out, float* ent_out, float* ext_out,
    void* workspace, size_t workspace_bytes, ajt_stream_t stream);

/* ------------------------------------------------------------------------------------------------
 * Log-prob and entropy of the target token straight from the hidden states (the forward half of fusing the LM head
 * with the loss; the pass that yields the old / reference log-probs the loss consumes, PAPER.md:136,
 * 172-176):
 *   z_t = W h_t;   lse_t = logsumexp_v z_tv;   logp_out[t] = z_{t,y_t} - lse_t;   ent_out[t] = lse_t - sum_v softmax(z_t)_v z_tv;
 *   lse_out[t] = lse_t (what a later backward pass needs to recompute softmax tiles)
 * hidden DEVICE [T, ld_hidden] bf16 (columns [0,d)), weight DEVICE [V, ld_weight] bf16, targets DEVICE [T] in [0,V),
 * mask DEVICE [T] or NULL (rows with mask 0 give 0, 0, 0).  The [T, V] logits are never written: tiles of 128 x 256 are
 * produced by tcgen05.mma (bf16 x bf16 -> fp32 in tensor memory) and reduced on the fly.  Arithmetic: fp32.
 * Requires d % 64 == 0, ld % 8 == 0 and 16-byte aligned bases (AJT_ERR_UNSUPPORTED otherwise).
 * With a mask the unmasked rows are compacted first (their hidden rows gathered into the workspace), so masked rows cost
 * no flops.  Workspace: ajt_lm_head_workspace_bytes(T, d, V) bytes of DEVICE memory, 256-byte aligned; its first word is the
 * call's status word (ajt_last_status): AJT_STATUS_BAD_TARGET when an unmasked row's target is outside [0, V) (that row
 * returns 0, 0, 0). */
enum {
    AJT_LM_ROUND_LOGITS_BF16 = 1 /* round every logit to bf16 (RNE) before the softmax: the log-probs then agree with what
                                    ajt_policy_loss_fwd_bwd computes from the same logits STORED in bf16 (to fp32 rounding of
                                    the reductions), so that old / new log-prob ratios start at 1 (the train / inference
                                    consistency the paper is concerned with) */
};

size_t ajt_lm_head_workspace_bytes(int64_t T, int32_t d, int32_t V);

int ajt_lm_head_logp(const void* hidden, const void* weight, const int32_t* targets, const uint8_t* mask, int64_t T, int32_t d,
                     int32_t V, int64_t ld_hidden, int64_t ld_weight, float* logp_out, float* ent_out /* or NULL */,
                     float* lse_out /* or NULL */, uint32_t flags /* AJT_LM_* */, void* workspace, size_t workspace_bytes,
                     ajt_stream_t stream);

/* ajt_policy_loss_fwd_bwd for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same computation, the same kernels and the same results as ajt_policy_loss_fwd_bwd
 * (BASELINE.json north_star; DESIGN.md "O-L" steps 1-7), but the call's scratch lives in a file-scope
 * device array of the library instead of a caller-provided workspace.  The call allocates nothing (no cudaMalloc / cudaFree,
 * no allocating library routine).  Inputs and outputs are the caller's, exactly as for ajt_policy_loss_fwd_bwd.
 *   Limit: the scratch is ajt_loss_static_scratch_bytes() = 4 MiB per GPU (held by every GPU that loads the library until
 *   the process exits); a call needs ajt_loss_workspace_bytes(T, V, S) bytes of it (69 bytes per row + 4 S + ~1 KB: e.g.
 *   T = 40,960 rows with S = 4,096).  Larger calls return AJT_ERR_CAPACITY and launch nothing: use the workspace call.
 *   Sharing: every call on a device uses the same array, which keeps the previous call's contents; the call clears what must
 *   start at zero on `stream`.  Two such calls that overlap on one GPU (different streams, no dependency) RACE: order them.
 *   status_out: DEVICE [1] or NULL: the call's AJT_STATUS_* word, copied on `stream` (there is no workspace to pass to
 *   ajt_last_status).  Enqueues on `stream`, does not synchronise. */
size_t ajt_loss_static_scratch_bytes(void);

int ajt_policy_loss_fwd_bwd_static(const void* logits, const int32_t* targets, const float* old_logp, const float* adv,
                                   const uint8_t* mask, const int32_t* seg_ids, float eps_lo, float eps_hi, int64_t T, int32_t V,
                                   int32_t S, int64_t ld_logits, int32_t logits_dtype, const float* seg_denom, float inv_num_segs,
                                   float grad_scale, void* dlogits, float* loss_out, float* logp_out /* or NULL */,
                                   float* stats_out /* or NULL */, uint32_t* status_out /* or NULL */, ajt_stream_t stream);

/* The policy loss straight from the hidden states, forward AND backward ("policy gradient ... loss terms
 * are computed"): with z_t = W h_t and steps 1-6 of ajt_policy_loss_fwd_bwd on z,
 *   loss = sum_t w_t L_t;   dZ_tv = g_t (1[v = y_t] - exp(z_tv - lse_t));   dH = dZ W  [T, d] bf16;   dW (+)= dZ^T H  [V, d] fp32
 * The [T, V] logits are never written: tiles of 256 x 256 are recomputed by tcgen05.mma and turned into dZ in the epilogue;
 * dZ is staged in bf16 (round to nearest even: the operand precision of the two follow-on tensor-core products, reading
 * H-4) 4,096 unmasked rows at a time in the workspace, and dH / dW come out of the same TMA / tcgen05 mainloop.  Masked
 * rows (mask NULL: none) cost no flops; their dH rows are zero.  seg_denom DEVICE [S] or NULL (then N_s is counted from
 * this call's tokens), inv_num_segs as for ajt_policy_loss_fwd_bwd.  accumulate_dw != 0 adds to dW instead of overwriting.
 * loss_out DEVICE [1]; logp_out DEVICE [T] or NULL.  flags: AJT_LM_*.  Requires d % 64 == 0, ld_hidden / ld_weight / ld_dh
 * % 8 == 0, ld_dw % 4 == 0, 16-byte aligned bases.  Workspace: ajt_lm_head_bwd_workspace_bytes(T, d, V, S) bytes (its first
 * word is the status word: AJT_STATUS_BAD_TARGET, AJT_STATUS_BAD_SEG).  Enqueues on `stream`. */
size_t ajt_lm_head_bwd_workspace_bytes(int64_t T, int32_t d, int32_t V, int32_t S);

int ajt_lm_head_loss_bwd(const void* hidden, const void* weight, const int32_t* targets, const float* old_logp, const float* adv,
                         const uint8_t* mask, const int32_t* seg_ids, float eps_lo, float eps_hi, int64_t T, int32_t d, int32_t V,
                         int32_t S, int64_t ld_hidden, int64_t ld_weight, const float* seg_denom, float inv_num_segs,
                         float grad_scale, void* dH, int64_t ld_dh, float* dW, int64_t ld_dw, int32_t accumulate_dw,
                         float* loss_out, float* logp_out, uint32_t flags, void* workspace, size_t workspace_bytes,
                         ajt_stream_t stream);

/* Batch-wide per-trajectory normalisers for callers that stream the batch through several loss calls
 * (micro-batches, 64k-row chunks, or rows of one trajectory spread over several GPUs; reading L-4;
 * "masked per-trajectory mean", BASELINE.json north_star):
 *   seg_denom[s] (+)= #{t in [0,T) : seg_ids[t] = s and mask[t] != 0}
 * `accumulate` = 0 clears seg_denom (and *status_bits) first; != 0 adds to what is there, so a batch can be
 * counted chunk by chunk.  Counts are integers held in fp32: exact below 2^24 masked tokens per trajectory.
 * Pass the result as `seg_denom` to every ajt_policy_loss_fwd_bwd call of the batch with inv_num_segs = 0
 * (1/S' is then taken from seg_denom) — or all-reduce it across ranks first.
 * seg_denom: DEVICE [S].  status_bits: DEVICE [1] or NULL (AJT_STATUS_BAD_SEG when a masked-in token has
 * seg_ids[t] outside [0,S); that token is not counted).  Enqueues on `stream`, does not synchronise. */
int ajt_segment_counts(const uint8_t* mask /* DEVICE [T] */, const int32_t* seg_ids /* DEVICE [T] */, int64_t T, int32_t S,
                       int32_t accumulate, float* seg_denom, uint32_t* status_bits, ajt_stream_t stream);

/* HOST-buffer variant.  `arena` is DEVICE scratch of at least ajt_loss_host_arena_bytes(T, V, S, ld, dtype) bytes.
 * The per-token vectors go up first and the batch-wide normalisers are counted on the device; the matrix is cut into up
 * to 16 row slabs whose H2D copy, loss call and D2H copy overlap with their neighbours' (both PCIe directions busy at
 * once); rows with mask 0 are not copied up, since the kernel never reads them.  For that the call creates two helper streams and their events and destroys them before it returns: the only
 * resources the library ever creates (ajt_policy_loss_fwd_bwd_host2 takes them from a caller-owned context instead).  dlogits / logp rows are those of the device call; loss and stats[3] are the fp64
 * sums of the slabs' fp32 partials.  Pinned host buffers are needed for the overlap.  Synchronises. */
size_t ajt_loss_host_arena_bytes(int64_t T, int32_t V, int32_t S, int64_t ld_logits, int32_t logits_dtype);

/* Helper streams and events of the slab pipeline, created once and reused across calls (ajt_policy_loss_fwd_bwd_host2);
 * the only resources the library ever creates.  One context serves one call at a time. */
typedef struct ajt_host_ctx* ajt_host_ctx_t;
int ajt_host_ctx_create(ajt_host_ctx_t* ctx);
void ajt_host_ctx_destroy(ajt_host_ctx_t ctx);

/* ajt_policy_loss_fwd_bwd_host with two more choices: `dlogits_on_device` != 0 makes `dlogits` a DEVICE buffer
 * [T, ld_logits] bf16 (16-byte aligned) that receives the gradient, so that nothing but loss / logp / stats / status comes
 * back over PCIe (what a trainer wants: the backward pass continues on the device); `ctx` (or NULL: created and destroyed
 * inside the call) carries the helper streams.  Everything else as for ajt_policy_loss_fwd_bwd_host. */
int ajt_policy_loss_fwd_bwd_host2(
    const void* logits, const int32_t* targets, const float* old_logp, const float* adv, const uint8_t* mask,
    const int32_t* seg_ids, float eps_lo, float eps_hi, int64_t T, int32_t V, int32_t S, int64_t ld_logits,
    int32_t logits_dtype, const float* seg_denom, float inv_num_segs, float grad_scale,
    void* dlogits, int32_t dlogits_on_device, float* loss_out /* HOST [1] */, float* logp_out /* HOST [T] or NULL */,
    float* stats_out /* HOST [4] or NULL */, uint32_t* status_bits /* HOST [1] or NULL */,
    ajt_host_ctx_t ctx, void* arena /* DEVICE */, size_t arena_bytes, ajt_stream_t stream);

int ajt_policy_loss_fwd_bwd_host(
    const void* logits, const int32_t* targets, const float* old_logp, const float* adv, const uint8_t* mask,
    const int32_t* seg_ids, float eps_lo, float eps_hi, int64_t T, int32_t V, int32_t S, int64_t ld_logits,
    int32_t logits_dtype, const float* seg_denom, float inv_num_segs, float grad_scale,
    void* dlogits /* HOST bf16 */, float* loss_out /* HOST [1] */, float* logp_out /* HOST [T] or NULL */,
    float* stats_out /* HOST [4] or NULL */, uint32_t* status_bits /* HOST [1] or NULL */,
    void* arena /* DEVICE */, size_t arena_bytes, ajt_stream_t stream);

#ifdef __cplusplus
}
#endif
#endif /* AJT_H_ */
