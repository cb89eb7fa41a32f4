// Library-level entry points of libajt.so: version, error strings, status read-back and the HOST-buffer
// variants of the two hot-path calls (stage through a caller-provided device arena; no allocation here).
#include "ajt_common.cuh"

namespace {
inline size_t a256(size_t x) { return (x + 255) & ~(size_t)255; }
}  // namespace

extern "C" int ajt_version(void) { return AJT_VERSION_NUM; }

extern "C" const char* ajt_strerror(int code) {
    switch (code) {
        case AJT_OK: return "ok";
        case AJT_ERR_INVALID_ARG: return "invalid argument";
        case AJT_ERR_WORKSPACE_TOO_SMALL: return "workspace too small";
        case AJT_ERR_CAPACITY: return "capacity exceeded";
        case AJT_ERR_CUDA: return "CUDA error (no device, launch failure or runtime error)";
        case AJT_ERR_UNSUPPORTED: return "unsupported configuration";
        default: return "unknown error code";
    }
}

extern "C" int ajt_last_status(const void* workspace, ajt_stream_t stream, uint32_t* bits) {
    if (!workspace || !bits) return AJT_ERR_INVALID_ARG;
    cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
    if (cudaMemcpyAsync(bits, workspace, sizeof(uint32_t), cudaMemcpyDeviceToHost, s) != cudaSuccess) return AJT_ERR_CUDA;
    if (cudaStreamSynchronize(s) != cudaSuccess) return AJT_ERR_CUDA;
    return AJT_OK;
}

// ------------------------------------------------------------------------------------------------ loss, host buffers

namespace {
struct LossArena {
    size_t logits, targets, old_logp, adv, mask, seg, denom, loss, logp, stats, ws, total;
};
LossArena loss_arena(int64_t T, int32_t V, int32_t S, int64_t ld, int32_t dtype) {
    LossArena a;
    size_t o = 0;
    const size_t esz = dtype == AJT_DT_F32 ? 4 : 2;
    a.logits = o; o += a256((size_t)T * ld * esz);   // bf16: dlogits is written in place; f32: bf16 dlogits reuse the front
    a.targets = o; o += a256((size_t)T * 4);
    a.old_logp = o; o += a256((size_t)T * 4);
    a.adv = o; o += a256((size_t)T * 4);
    a.mask = o; o += a256((size_t)T);
    a.seg = o; o += a256((size_t)T * 4);
    a.denom = o; o += a256((size_t)S * 4);
    a.loss = o; o += 256;
    a.logp = o; o += a256((size_t)T * 4);
    a.stats = o; o += 256;
    a.ws = o; o += ajt_loss_workspace_bytes(T, V, S);
    a.total = o;
    // f32 logits cannot be overwritten in place by bf16 rows of the same stride without clobbering unread
    // rows, so they get a separate dlogits buffer
    if (dtype == AJT_DT_F32) a.total += a256((size_t)T * ld * 2);
    return a;
}
}  // namespace

extern "C" size_t ajt_loss_host_arena_bytes(int64_t T, int32_t V, int32_t S, int64_t ld, int32_t dtype) {
    if (T < 0 || V <= 0 || S <= 0 || ld < V) return 0;
    return loss_arena(T, V, S, ld, dtype).total;
}

extern "C" int ajt_policy_loss_fwd_bwd_host(const void* logits, const int32_t* targets, const float* old_logp, const float* adv,
                                            const uint8_t* mask, const int32_t* seg_ids, float eps_lo, float eps_hi, int64_t T,
                                            int32_t V, int32_t S, int64_t ld, int32_t dtype, const float* seg_denom,
                                            float inv_num_segs, float grad_scale, void* dlogits, float* loss_out,
                                            float* logp_out, float* stats_out, uint32_t* status_bits, void* arena,
                                            size_t arena_bytes, ajt_stream_t stream_) {
    cudaStream_t s = reinterpret_cast<cudaStream_t>(stream_);
    if (T < 0 || V <= 0 || S <= 0 || ld < V || !arena || !loss_out) return AJT_ERR_INVALID_ARG;
    if (dtype != AJT_DT_BF16 && dtype != AJT_DT_F32) return AJT_ERR_INVALID_ARG;
    if ((uintptr_t)arena & 255) return AJT_ERR_INVALID_ARG;
    const LossArena a = loss_arena(T, V, S, ld, dtype);
    if (arena_bytes < a.total) return AJT_ERR_WORKSPACE_TOO_SMALL;
    uint8_t* d = reinterpret_cast<uint8_t*>(arena);
    const size_t esz = dtype == AJT_DT_F32 ? 4 : 2;
    void* d_dlogits = dtype == AJT_DT_F32 ? (void*)(d + a.ws + ajt_loss_workspace_bytes(T, V, S)) : (void*)(d + a.logits);
#define AJT_CP(dst, src, bytes, kind) \
    if ((bytes) > 0 && cudaMemcpyAsync((dst), (src), (bytes), (kind), s) != cudaSuccess) return AJT_ERR_CUDA
    AJT_CP(d + a.logits, logits, (size_t)T * ld * esz, cudaMemcpyHostToDevice);
    AJT_CP(d + a.targets, targets, (size_t)T * 4, cudaMemcpyHostToDevice);
    AJT_CP(d + a.old_logp, old_logp, (size_t)T * 4, cudaMemcpyHostToDevice);
    AJT_CP(d + a.adv, adv, (size_t)T * 4, cudaMemcpyHostToDevice);
    AJT_CP(d + a.mask, mask, (size_t)T, cudaMemcpyHostToDevice);
    AJT_CP(d + a.seg, seg_ids, (size_t)T * 4, cudaMemcpyHostToDevice);
    if (seg_denom) AJT_CP(d + a.denom, seg_denom, (size_t)S * 4, cudaMemcpyHostToDevice);
    const int rc = ajt_policy_loss_fwd_bwd(d + a.logits, (const int32_t*)(d + a.targets), (const float*)(d + a.old_logp),
                                           (const float*)(d + a.adv), d + a.mask, (const int32_t*)(d + a.seg), eps_lo, eps_hi, T,
                                           V, S, ld, dtype, seg_denom ? (const float*)(d + a.denom) : nullptr, inv_num_segs,
                                           grad_scale, d_dlogits, (float*)(d + a.loss), logp_out ? (float*)(d + a.logp) : nullptr,
                                           stats_out ? (float*)(d + a.stats) : nullptr, d + a.ws,
                                           ajt_loss_workspace_bytes(T, V, S), stream_);
    if (rc != AJT_OK) return rc;
    AJT_CP(dlogits, d_dlogits, (size_t)T * ld * 2, cudaMemcpyDeviceToHost);
    AJT_CP(loss_out, d + a.loss, 4, cudaMemcpyDeviceToHost);
    if (logp_out) AJT_CP(logp_out, d + a.logp, (size_t)T * 4, cudaMemcpyDeviceToHost);
    if (stats_out) AJT_CP(stats_out, d + a.stats, 16, cudaMemcpyDeviceToHost);
    if (status_bits) AJT_CP(status_bits, d + a.ws, 4, cudaMemcpyDeviceToHost);
#undef AJT_CP
    return cudaStreamSynchronize(s) == cudaSuccess ? AJT_OK : AJT_ERR_CUDA;
}

// ------------------------------------------------------------------------------------------------ merge, host buffers

namespace {
struct MergeArena {
    size_t tokens, offsets, traj, resp, mask, logp, m_tokens, m_mask, m_src, m_logp, m_off, m_origin, m_traj, owner, counts, ws,
        ws_bytes, total;
};
MergeArena merge_arena(int32_t n, int64_t N) {
    MergeArena a;
    size_t o = 0;
    const size_t n4 = a256(((size_t)n + 1) * 4), n8 = a256(((size_t)n + 1) * 8), N4 = a256((size_t)N * 4), N1 = a256((size_t)N);
    a.tokens = o; o += N4; a.offsets = o; o += n8; a.traj = o; o += n4; a.resp = o; o += n4; a.mask = o; o += N1;
    a.logp = o; o += N4;
    a.m_tokens = o; o += N4; a.m_mask = o; o += N1; a.m_src = o; o += N4; a.m_logp = o; o += N4;
    a.m_off = o; o += n8; a.m_origin = o; o += n4; a.m_traj = o; o += n4; a.owner = o; o += n4; a.counts = o; o += 256;
    a.ws = o; a.ws_bytes = ajt_merge_workspace_bytes(n, N); o += a256(a.ws_bytes);
    a.total = o;
    return a;
}
}  // namespace

extern "C" size_t ajt_merge_host_arena_bytes(int32_t n, int64_t n_tokens) {
    if (n < 0 || n_tokens < 0) return 0;
    return merge_arena(n, n_tokens).total;
}

extern "C" int ajt_merge_timelines_host(const int32_t* tokens, const int64_t* offsets, const int32_t* traj_ids,
                                        const int32_t* resp_start, const uint8_t* mask_in, const float* old_logp_in, int32_t n,
                                        int64_t N, int32_t owner_rule, uint32_t flags, int32_t* merged_tokens,
                                        uint8_t* merged_mask, int32_t* merged_src, float* merged_old_logp,
                                        int64_t* merged_offsets, int32_t* merged_origin, int32_t* merged_traj, int32_t* owner,
                                        int64_t* counts, uint32_t* status_bits, void* arena, size_t arena_bytes,
                                        ajt_stream_t stream_) {
    cudaStream_t s = reinterpret_cast<cudaStream_t>(stream_);
    if (n < 0 || N < 0 || !arena || !counts || !offsets) return AJT_ERR_INVALID_ARG;
    if ((uintptr_t)arena & 255) return AJT_ERR_INVALID_ARG;
    if ((old_logp_in == nullptr) != (merged_old_logp == nullptr)) return AJT_ERR_INVALID_ARG;
    const MergeArena a = merge_arena(n, N);
    if (arena_bytes < a.total) return AJT_ERR_WORKSPACE_TOO_SMALL;
    uint8_t* d = reinterpret_cast<uint8_t*>(arena);
#define AJT_CP(dst, src, bytes, kind) \
    if ((bytes) > 0 && cudaMemcpyAsync((dst), (src), (bytes), (kind), s) != cudaSuccess) return AJT_ERR_CUDA
    AJT_CP(d + a.tokens, tokens, (size_t)N * 4, cudaMemcpyHostToDevice);
    AJT_CP(d + a.offsets, offsets, ((size_t)n + 1) * 8, cudaMemcpyHostToDevice);
    AJT_CP(d + a.traj, traj_ids, (size_t)n * 4, cudaMemcpyHostToDevice);
    if (resp_start) AJT_CP(d + a.resp, resp_start, (size_t)n * 4, cudaMemcpyHostToDevice);
    if (mask_in) AJT_CP(d + a.mask, mask_in, (size_t)N, cudaMemcpyHostToDevice);
    if (old_logp_in) AJT_CP(d + a.logp, old_logp_in, (size_t)N * 4, cudaMemcpyHostToDevice);
    const int rc = ajt_merge_timelines(
        (const int32_t*)(d + a.tokens), (const int64_t*)(d + a.offsets), (const int32_t*)(d + a.traj),
        resp_start ? (const int32_t*)(d + a.resp) : nullptr, mask_in ? d + a.mask : nullptr,
        old_logp_in ? (const float*)(d + a.logp) : nullptr, n, N, owner_rule, flags, (int32_t*)(d + a.m_tokens), d + a.m_mask,
        (int32_t*)(d + a.m_src), old_logp_in ? (float*)(d + a.m_logp) : nullptr, (int64_t*)(d + a.m_off),
        (int32_t*)(d + a.m_origin), (int32_t*)(d + a.m_traj), (int32_t*)(d + a.owner), (int64_t*)(d + a.counts), d + a.ws,
        a.ws_bytes, stream_);
    if (rc != AJT_OK) return rc;
    // the merged sizes are only known on the device: fetch {M, N_out}, then copy exactly that much back
    AJT_CP(counts, d + a.counts, 16, cudaMemcpyDeviceToHost);
    if (status_bits) AJT_CP(status_bits, d + a.ws, 4, cudaMemcpyDeviceToHost);
    if (cudaStreamSynchronize(s) != cudaSuccess) return AJT_ERR_CUDA;
    const size_t M = (size_t)counts[0], No = (size_t)counts[1];
    if (M > (size_t)n || No > (size_t)N) return AJT_ERR_CUDA;
    AJT_CP(merged_tokens, d + a.m_tokens, No * 4, cudaMemcpyDeviceToHost);
    AJT_CP(merged_mask, d + a.m_mask, No, cudaMemcpyDeviceToHost);
    AJT_CP(merged_src, d + a.m_src, No * 4, cudaMemcpyDeviceToHost);
    if (merged_old_logp) AJT_CP(merged_old_logp, d + a.m_logp, No * 4, cudaMemcpyDeviceToHost);
    AJT_CP(merged_offsets, d + a.m_off, (M + 1) * 8, cudaMemcpyDeviceToHost);
    AJT_CP(merged_origin, d + a.m_origin, M * 4, cudaMemcpyDeviceToHost);
    AJT_CP(merged_traj, d + a.m_traj, M * 4, cudaMemcpyDeviceToHost);
    AJT_CP(owner, d + a.owner, (size_t)n * 4, cudaMemcpyDeviceToHost);
#undef AJT_CP
    return cudaStreamSynchronize(s) == cudaSuccess ? AJT_OK : AJT_ERR_CUDA;
}
