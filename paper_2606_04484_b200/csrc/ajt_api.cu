// Library-level entry points of libajt.so: version, error strings, status read-back and the HOST-buffer
// variants of the two hot-path calls (stage through a caller-provided device arena; no allocation here).
#include <atomic>

#include "ajt_common.cuh"
#include "../../include/ajt_test.h"

namespace {
inline size_t a256(size_t x) { return (x + 255) & ~(size_t)255; }
std::atomic<unsigned long long> g_launches{0};
}  // namespace

void ajt::note_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }
extern "C" uint64_t ajt_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

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

// ------------------------------------------------------------------------------------------------ HBM ceilings (measurement)

namespace {
__global__ void __launch_bounds__(256) probe_read_kernel(const uint4* __restrict__ src, size_t n16, uint32_t* sink) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    uint32_t acc = 0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += stride) {
        uint4 v;
        asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(src + i));
        acc ^= v.x ^ v.y ^ v.z ^ v.w;
    }
    if (acc == 0x9E3779B9u) *sink = acc;   // keeps the loads alive; practically never taken
}
__global__ void __launch_bounds__(256) probe_write_kernel(uint4* __restrict__ dst, size_t n16) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += stride) ajt::stg128_stream(dst + i, make_uint4(0, 0, 0, 0));
}
__global__ void __launch_bounds__(256) probe_copy_kernel(uint4* __restrict__ dst, const uint4* __restrict__ src, size_t n16) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += stride) {
        uint4 v;
        asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(src + i));
        ajt::stg128_stream(dst + i, v);
    }
}
}  // namespace

extern "C" int ajt_hbm_probe(void* dst, const void* src, size_t bytes, int32_t mode, ajt_stream_t stream_) {
    cudaStream_t s = reinterpret_cast<cudaStream_t>(stream_);
    if (mode < 0 || mode > 3 || (bytes & 15) || ((mode != 0) && (!dst || ((uintptr_t)dst & 15))) ||
        ((mode == 0 || mode == 2) && (!src || ((uintptr_t)src & 15))))
        return AJT_ERR_INVALID_ARG;
    int dev = 0, num_sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return AJT_ERR_CUDA;
    if (cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || num_sms < 1) return AJT_ERR_CUDA;
    const size_t n16 = bytes / 16;
    const int grid = num_sms * 32;
    if (mode == 0) AJT_LAUNCH(probe_read_kernel<<<grid, 256, 0, s>>>(reinterpret_cast<const uint4*>(src), n16, reinterpret_cast<uint32_t*>(dst)));
    else if (mode == 1) AJT_LAUNCH(probe_write_kernel<<<grid, 256, 0, s>>>(reinterpret_cast<uint4*>(dst), n16));
    else if (mode == 2) AJT_LAUNCH(probe_copy_kernel<<<grid, 256, 0, s>>>(reinterpret_cast<uint4*>(dst), reinterpret_cast<const uint4*>(src), n16));
    else if (cudaMemsetAsync(dst, 0, bytes, s) != cudaSuccess) return AJT_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? AJT_OK : AJT_ERR_CUDA;
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

namespace {
// Per-slab partials -> running totals kept on the device in fp64 (no host read between slabs).
__global__ void host_acc_kernel(double* acc /* [5]: loss, stats[4] */, uint32_t* status_acc, const float* loss, const float* stats,
                                const uint32_t* ws_status) {
    acc[0] += (double)loss[0];
    if (stats)
        for (int k = 0; k < 4; ++k) acc[1 + k] += (double)stats[k];
    *status_acc |= *ws_status;
}
__global__ void host_fin_kernel(const double* acc, float* loss, float* stats) {
    loss[0] = (float)acc[0];
    for (int k = 0; k < 4; ++k) stats[k] = (float)acc[1 + k];
}
constexpr int kHostMaxSlabs = 16;
}  // namespace

// Slab pipeline: the per-token vectors go up first and the batch-wide normalisers are counted on the device (reading L-4);
// the [T, ld] matrix is cut into up to 16 row slabs, and slab i's H2D copy (helper stream 1), its loss call (the caller's
// stream) and its D2H copy (helper stream 2) overlap with the neighbours', so both PCIe directions stay busy at once.
struct ajt_host_ctx {
    cudaStream_t s_up, s_dn;
    cudaEvent_t ev_up[kHostMaxSlabs], ev_k[kHostMaxSlabs], ev0, ev_end;
};

extern "C" int ajt_host_ctx_create(ajt_host_ctx_t* out) {
    if (!out) return AJT_ERR_INVALID_ARG;
    ajt_host_ctx* c = new (std::nothrow) ajt_host_ctx();
    if (!c) return AJT_ERR_CAPACITY;
    bool ok = cudaStreamCreateWithFlags(&c->s_up, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&c->s_dn, cudaStreamNonBlocking) == cudaSuccess &&
              cudaEventCreateWithFlags(&c->ev0, cudaEventDisableTiming) == cudaSuccess &&
              cudaEventCreateWithFlags(&c->ev_end, cudaEventDisableTiming) == cudaSuccess;
    for (int i = 0; i < kHostMaxSlabs && ok; ++i)
        ok = cudaEventCreateWithFlags(&c->ev_up[i], cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&c->ev_k[i], cudaEventDisableTiming) == cudaSuccess;
    if (!ok) {
        ajt_host_ctx_destroy(c);
        return AJT_ERR_CUDA;
    }
    *out = c;
    return AJT_OK;
}

extern "C" void ajt_host_ctx_destroy(ajt_host_ctx_t c) {
    if (!c) return;
    for (int i = 0; i < kHostMaxSlabs; ++i) {
        if (c->ev_up[i]) cudaEventDestroy(c->ev_up[i]);
        if (c->ev_k[i]) cudaEventDestroy(c->ev_k[i]);
    }
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev_end) cudaEventDestroy(c->ev_end);
    if (c->s_up) cudaStreamDestroy(c->s_up);
    if (c->s_dn) cudaStreamDestroy(c->s_dn);
    delete c;
}

extern "C" int ajt_policy_loss_fwd_bwd_host(const void* logits, const int32_t* targets, const float* old_logp, const float* adv,
                                            const uint8_t* mask, const int32_t* seg_ids, float eps_lo, float eps_hi, int64_t T,
                                            int32_t V, int32_t S, int64_t ld, int32_t dtype, const float* seg_denom,
                                            float inv_num_segs, float grad_scale, void* dlogits, float* loss_out,
                                            float* logp_out, float* stats_out, uint32_t* status_bits, void* arena,
                                            size_t arena_bytes, ajt_stream_t stream_) {
    return ajt_policy_loss_fwd_bwd_host2(logits, targets, old_logp, adv, mask, seg_ids, eps_lo, eps_hi, T, V, S, ld, dtype,
                                         seg_denom, inv_num_segs, grad_scale, dlogits, 0, loss_out, logp_out, stats_out,
                                         status_bits, nullptr, arena, arena_bytes, stream_);
}

extern "C" int ajt_policy_loss_fwd_bwd_host2(const void* logits, const int32_t* targets, const float* old_logp, const float* adv,
                                             const uint8_t* mask, const int32_t* seg_ids, float eps_lo, float eps_hi, int64_t T,
                                             int32_t V, int32_t S, int64_t ld, int32_t dtype, const float* seg_denom,
                                             float inv_num_segs, float grad_scale, void* dlogits, int32_t dlogits_on_device,
                                             float* loss_out, float* logp_out, float* stats_out, uint32_t* status_bits,
                                             ajt_host_ctx_t ctx, void* arena, size_t arena_bytes, ajt_stream_t stream_) {
    cudaStream_t s = reinterpret_cast<cudaStream_t>(stream_);
    if (T < 0 || V <= 0 || S <= 0 || ld < V || !arena || !loss_out) return AJT_ERR_INVALID_ARG;
    if (dlogits_on_device && ((uintptr_t)dlogits & 15)) return AJT_ERR_INVALID_ARG;
    if (dtype != AJT_DT_BF16 && dtype != AJT_DT_F32) return AJT_ERR_INVALID_ARG;
    if (T > 0 && (!logits || !targets || !old_logp || !adv || !mask || !seg_ids || !dlogits)) return AJT_ERR_INVALID_ARG;
    if ((uintptr_t)arena & 255) return AJT_ERR_INVALID_ARG;
    const LossArena a = loss_arena(T, V, S, ld, dtype);
    if (arena_bytes < a.total) return AJT_ERR_WORKSPACE_TOO_SMALL;
    uint8_t* d = reinterpret_cast<uint8_t*>(arena);
    const size_t esz = dtype == AJT_DT_F32 ? 4 : 2;
    const size_t ws_bytes = ajt_loss_workspace_bytes(T, V, S);
    // where the kernel writes the gradient: the caller's device buffer, or the arena (bf16: in place over the uploaded rows)
    uint8_t* d_dl = dlogits_on_device ? reinterpret_cast<uint8_t*>(dlogits) : (dtype == AJT_DT_F32 ? d + a.ws + ws_bytes : d + a.logits);
    // accumulators live in the tail of the stats slot: [loss f32 | ... ] at a.loss, [stats 4 x f32 | acc 5 x f64 | status u32] at a.stats
    float* d_loss = reinterpret_cast<float*>(d + a.loss);
    float* d_stats = reinterpret_cast<float*>(d + a.stats);
    double* d_acc = reinterpret_cast<double*>(d + a.stats + 64);
    uint32_t* d_status = reinterpret_cast<uint32_t*>(d + a.stats + 128);
    float* d_denom = reinterpret_cast<float*>(d + a.denom);

    int rc = AJT_OK;
    ajt_host_ctx_t own = nullptr;   // helper streams / events: the caller's context, or one made for this call
    if (!ctx) {
        rc = ajt_host_ctx_create(&own);
        if (rc != AJT_OK) return rc;
        ctx = own;
    }
    cudaStream_t s_up = ctx->s_up, s_dn = ctx->s_dn;
    cudaEvent_t *ev_up = ctx->ev_up, *ev_k = ctx->ev_k, ev0 = ctx->ev0, ev_end = ctx->ev_end;
    const int nslab = (int)(T <= 0 ? 0 : (T < 256 * kHostMaxSlabs ? (T + 255) / 256 : kHostMaxSlabs));
    const int64_t rows_per = nslab ? (T + nslab - 1) / nslab : 0;
#define AJT_TRY(x) \
    do { \
        if (rc == AJT_OK && (x) != cudaSuccess) rc = AJT_ERR_CUDA; \
    } while (0)
#define AJT_CP(dst, src, bytes, kind, st) \
    do { \
        if ((bytes) > 0) AJT_TRY(cudaMemcpyAsync((dst), (src), (bytes), (kind), (st))); \
    } while (0)
    // ---- per-token vectors, normalisers, accumulators (caller's stream)
    AJT_CP(d + a.targets, targets, (size_t)T * 4, cudaMemcpyHostToDevice, s);
    AJT_CP(d + a.old_logp, old_logp, (size_t)T * 4, cudaMemcpyHostToDevice, s);
    AJT_CP(d + a.adv, adv, (size_t)T * 4, cudaMemcpyHostToDevice, s);
    AJT_CP(d + a.mask, mask, (size_t)T, cudaMemcpyHostToDevice, s);
    AJT_CP(d + a.seg, seg_ids, (size_t)T * 4, cudaMemcpyHostToDevice, s);
    AJT_TRY(cudaMemsetAsync(d + a.stats, 0, 256, s));
    AJT_TRY(cudaMemsetAsync(d + a.loss, 0, 256, s));
    if (rc == AJT_OK) {
        if (seg_denom) AJT_CP(d_denom, seg_denom, (size_t)S * 4, cudaMemcpyHostToDevice, s);
        else rc = ajt_segment_counts(d + a.mask, (const int32_t*)(d + a.seg), T, S, 0, d_denom, d_status, stream_);
    }
    AJT_TRY(cudaEventRecord(ev0, s));
    AJT_TRY(cudaStreamWaitEvent(s_up, ev0, 0));   // the uploads start after whatever the caller had queued on its stream
    // ---- slabs
    for (int i = 0; i < nslab && rc == AJT_OK; ++i) {
        const int64_t r0 = i * rows_per, r1 = (r0 + rows_per < T) ? r0 + rows_per : T;
        if (r1 <= r0) break;
        const int64_t R = r1 - r0;
        // only the rows the kernel reads go up: runs of consecutive rows with mask != 0 (the mask is host memory here)
        for (int64_t r = r0; r < r1;) {
            while (r < r1 && mask[r] == 0) ++r;
            int64_t e = r;
            while (e < r1 && mask[e] != 0) ++e;
            if (e > r)
                AJT_CP(d + a.logits + (size_t)r * ld * esz, (const uint8_t*)logits + (size_t)r * ld * esz, (size_t)(e - r) * ld * esz,
                       cudaMemcpyHostToDevice, s_up);
            r = e;
        }
        AJT_TRY(cudaEventRecord(ev_up[i], s_up));
        AJT_TRY(cudaStreamWaitEvent(s, ev_up[i], 0));
        if (rc != AJT_OK) break;
        rc = ajt_policy_loss_fwd_bwd(d + a.logits + (size_t)r0 * ld * esz, (const int32_t*)(d + a.targets) + r0,
                                     (const float*)(d + a.old_logp) + r0, (const float*)(d + a.adv) + r0, d + a.mask + r0,
                                     (const int32_t*)(d + a.seg) + r0, eps_lo, eps_hi, R, V, S, ld, dtype, d_denom, inv_num_segs,
                                     grad_scale, d_dl + (size_t)r0 * ld * 2, d_loss, logp_out ? (float*)(d + a.logp) + r0 : nullptr,
                                     stats_out ? d_stats : nullptr, d + a.ws, ws_bytes, stream_);
        if (rc != AJT_OK) break;
        AJT_LAUNCH(host_acc_kernel<<<1, 1, 0, s>>>(d_acc, d_status, d_loss, stats_out ? d_stats : nullptr, (const uint32_t*)(d + a.ws)));
        AJT_TRY(cudaEventRecord(ev_k[i], s));
        AJT_TRY(cudaStreamWaitEvent(s_dn, ev_k[i], 0));
        if (!dlogits_on_device)
            AJT_CP((uint8_t*)dlogits + (size_t)r0 * ld * 2, d_dl + (size_t)r0 * ld * 2, (size_t)R * ld * 2, cudaMemcpyDeviceToHost, s_dn);
    }
    if (rc == AJT_OK) {
        AJT_LAUNCH(host_fin_kernel<<<1, 1, 0, s>>>(d_acc, d_loss, d_stats));
        AJT_CP(loss_out, d_loss, 4, cudaMemcpyDeviceToHost, s);
        if (logp_out) AJT_CP(logp_out, d + a.logp, (size_t)T * 4, cudaMemcpyDeviceToHost, s);
        if (stats_out) AJT_CP(stats_out, d_stats, 16, cudaMemcpyDeviceToHost, s);
        if (status_bits) AJT_CP(status_bits, d_status, 4, cudaMemcpyDeviceToHost, s);
    }
    // ---- join and clean up (also on the error paths: nothing may still be running on the helper streams)
    if (s_dn && ev_end && cudaEventRecord(ev_end, s_dn) == cudaSuccess) cudaStreamWaitEvent(s, ev_end, 0);
    if (s_up) cudaStreamSynchronize(s_up);
    if (s_dn) cudaStreamSynchronize(s_dn);
    if (cudaStreamSynchronize(s) != cudaSuccess && rc == AJT_OK) rc = AJT_ERR_CUDA;
    if (own) ajt_host_ctx_destroy(own);
#undef AJT_CP
#undef AJT_TRY
    return rc;
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
    MergeArena a = merge_arena(n, N);
    if (arena_bytes < a.total) return AJT_ERR_WORKSPACE_TOO_SMALL;
    a.ws_bytes += (arena_bytes - a.total) & ~(size_t)255;   // the workspace comes last: a larger arena holds more candidate pairs
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
    uint32_t st = 0;
    if (cudaMemcpyAsync(&st, d + a.ws, 4, cudaMemcpyDeviceToHost, s) != cudaSuccess) return AJT_ERR_CUDA;
    if (cudaStreamSynchronize(s) != cudaSuccess) return AJT_ERR_CUDA;
    // a fatal data-dependent status is an error of this call: the merged outputs would be empty / unspecified
    if (st & AJT_STATUS_PROBE_CAPACITY) return AJT_ERR_CAPACITY;
    if (st & (AJT_STATUS_BAD_OFFSETS | AJT_STATUS_ZERO_LEN)) return AJT_ERR_INVALID_ARG;
    if (st & AJT_STATUS_INTERNAL) return AJT_ERR_CUDA;
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
