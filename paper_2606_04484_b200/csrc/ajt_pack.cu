// Bridge between the two stages: turns the merge outputs into the per-token inputs of the loss call without leaving the
// device (reading L-12; "the packed merged sequences", BASELINE.json north_star).
//
// For position q of merged sequence m (next-token alignment inside each sequence, never across a boundary):
//   targets[q] = tokens[q+1], mask[q] = mask[q+1], old_logp[q] = old_logp[q+1];   the last position of m: 0, 0, 0
//   seg_ids[q] = tl_seg[merged_origin[m]]   (dense trajectory id of the surviving timeline)
//   adv[q]     = seg_adv[seg_ids[q]]        (GRPO: one advantage per trajectory)
// One pass, 9 B read and 17 B written per token.  A warp takes 512 consecutive tokens, finds the sequence of the first one
// with one warp-uniform binary search and walks forward from there.
#include "ajt_common.cuh"

namespace {

constexpr int kPackTile = 512;

struct PackParams {
    const int32_t* merged_tokens;
    const uint8_t* merged_mask;
    const float* merged_old_logp;
    const int64_t* merged_offsets;
    const int32_t* merged_origin;
    const int32_t* tl_seg;
    const float* seg_adv;
    const int64_t* counts;
    int64_t cap;
    int32_t S;
    int32_t* targets;
    uint8_t* mask;
    float* old_logp;
    int32_t* seg_ids;
    float* adv;
    uint32_t* status;
};

__device__ __forceinline__ int64_t last_le(const int64_t* __restrict__ a, int64_t n, int64_t x) {
    int64_t lo = 0, hi = n - 1;
    while (lo < hi) {
        const int64_t mid = (lo + hi + 1) >> 1;
        if (__ldg(a + mid) <= x) lo = mid;
        else hi = mid - 1;
    }
    return lo;
}

__global__ void __launch_bounds__(256) pack_loss_inputs_kernel(const PackParams p) {
    const int64_t M = p.counts[0], N = p.counts[1];
    if (M <= 0 || N <= 0 || N > p.cap) return;   // nothing merged, or counts that cannot belong to these arrays
    const int lane = threadIdx.x & 31;
    const int64_t wglobal = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    const int64_t ntiles = (N + kPackTile - 1) / kPackTile;
    const bool vec_ok = ((((uintptr_t)p.targets | (uintptr_t)p.seg_ids | (uintptr_t)p.old_logp | (uintptr_t)p.adv) & 15) == 0) &&
                        (((uintptr_t)p.mask & 3) == 0);
    for (int64_t tile = wglobal; tile < ntiles; tile += nwarps) {
        const int64_t t0 = tile * kPackTile;
        int64_t m = last_le(p.merged_offsets, M, t0);
        int64_t mend = __ldg(p.merged_offsets + m + 1);
        int32_t sg = __ldg(p.tl_seg + __ldg(p.merged_origin + m));
        auto seg_checked = [&](int32_t s) {
            if ((unsigned)s >= (unsigned)p.S) {
                if (p.status) atomicOr(p.status, (uint32_t)AJT_STATUS_BAD_SEG);
                return 0;
            }
            return s;
        };
        sg = seg_checked(sg);
        float av = p.seg_adv ? __ldg(p.seg_adv + sg) : 0.f;
#pragma unroll 2
        for (int u = 0; u < kPackTile / 128; ++u) {
            const int64_t q0 = t0 + 128 * u + 4 * lane;
            if (q0 >= N) break;
            int32_t tg[4], sgs[4];
            float lp[4], ad[4];
            uint32_t mk = 0;
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int64_t q = q0 + e;
                tg[e] = 0; sgs[e] = 0; lp[e] = 0.f; ad[e] = 0.f;
                if (q < N) {
                    while (q >= mend) {   // next sequence (every sequence has at least one token)
                        ++m;
                        mend = __ldg(p.merged_offsets + m + 1);
                        sg = seg_checked(__ldg(p.tl_seg + __ldg(p.merged_origin + m)));
                        av = p.seg_adv ? __ldg(p.seg_adv + sg) : 0.f;
                    }
                    sgs[e] = sg;
                    ad[e] = av;
                    if (q + 1 < mend) {   // not the last position of its sequence
                        tg[e] = __ldg(p.merged_tokens + q + 1);
                        if (__ldg(p.merged_mask + q + 1) != 0) mk |= 1u << (8 * e);
                        if (p.merged_old_logp) lp[e] = __ldg(p.merged_old_logp + q + 1);
                    }
                }
            }
            if (vec_ok && q0 + 3 < N) {
                *reinterpret_cast<int4*>(p.targets + q0) = make_int4(tg[0], tg[1], tg[2], tg[3]);
                *reinterpret_cast<int4*>(p.seg_ids + q0) = make_int4(sgs[0], sgs[1], sgs[2], sgs[3]);
                *reinterpret_cast<uint32_t*>(p.mask + q0) = mk;
                if (p.old_logp) *reinterpret_cast<float4*>(p.old_logp + q0) = make_float4(lp[0], lp[1], lp[2], lp[3]);
                if (p.adv) *reinterpret_cast<float4*>(p.adv + q0) = make_float4(ad[0], ad[1], ad[2], ad[3]);
            } else {
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    if (q0 + e < N) {
                        p.targets[q0 + e] = tg[e];
                        p.seg_ids[q0 + e] = sgs[e];
                        p.mask[q0 + e] = (uint8_t)((mk >> (8 * e)) & 1u);
                        if (p.old_logp) p.old_logp[q0 + e] = lp[e];
                        if (p.adv) p.adv[q0 + e] = ad[e];
                    }
                }
            }
            const int64_t qn = q0 + 128;
            while (qn < N && qn >= mend) {
                ++m;
                mend = __ldg(p.merged_offsets + m + 1);
                sg = seg_checked(__ldg(p.tl_seg + __ldg(p.merged_origin + m)));
                av = p.seg_adv ? __ldg(p.seg_adv + sg) : 0.f;
            }
        }
    }
}

// Token-budget packing (north_star "packed merged sequences"): consecutive merged sequences go into
// micro-batches of at most `budget` rows, greedily and in order (a sequence longer than the budget gets a micro-batch of
// its own).  The recurrence is sequential in the sequences, so one CTA stages the offsets in shared memory (coalesced) and
// one thread walks them; M is a few thousand at most in the configs (micro-seconds).
constexpr int kMbStage = 4096;
__global__ void __launch_bounds__(1024) pack_microbatches_kernel(const int64_t* __restrict__ merged_offsets, const int64_t* __restrict__ counts,
                                                                 int64_t budget, int32_t cap, int32_t* __restrict__ mb_seq,
                                                                 int64_t* __restrict__ mb_row, int32_t* __restrict__ n_mb) {
    __shared__ int64_t s_off[kMbStage + 1];
    __shared__ int64_t s_used;
    __shared__ int s_nmb;
    const int64_t M = counts[0];
    if (threadIdx.x == 0) { s_used = 0; s_nmb = 0; }
    __syncthreads();
    for (int64_t m0 = 0; m0 < M; m0 += kMbStage) {
        const int cn = (int)min((int64_t)kMbStage, M - m0);
        for (int x = threadIdx.x; x <= cn; x += blockDim.x) s_off[x] = merged_offsets[m0 + x];
        __syncthreads();
        if (threadIdx.x == 0) {
            int64_t used = s_used;
            int nmb = s_nmb;
            for (int x = 0; x < cn; ++x) {
                const int64_t L = s_off[x + 1] - s_off[x];
                if (nmb == 0 || (used > 0 && used + L > budget)) {   // sequence m0 + x opens a micro-batch
                    if (nmb < cap) { mb_seq[nmb] = (int32_t)(m0 + x); mb_row[nmb] = s_off[x]; }
                    ++nmb;
                    used = 0;
                }
                used += L;
            }
            s_used = used;
            s_nmb = nmb;
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const int nmb = s_nmb;
        if (nmb < cap) { mb_seq[nmb] = (int32_t)M; mb_row[nmb] = counts[1]; }   // the closing entry
        *n_mb = nmb;
    }
}

}  // namespace

extern "C" int ajt_pack_microbatches(const int64_t* merged_offsets, const int64_t* counts, int64_t budget, int32_t capacity,
                                     int32_t* mb_seq, int64_t* mb_row, int32_t* n_mb, ajt_stream_t stream_) {
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    if (!merged_offsets || !counts || !mb_seq || !mb_row || !n_mb || budget < 1 || capacity < 1) return AJT_ERR_INVALID_ARG;
    AJT_LAUNCH(pack_microbatches_kernel<<<1, 1024, 0, stream>>>(merged_offsets, counts, budget, capacity, mb_seq, mb_row, n_mb));
    return cudaGetLastError() == cudaSuccess ? AJT_OK : AJT_ERR_CUDA;
}

extern "C" int ajt_pack_loss_inputs(const int32_t* merged_tokens, const uint8_t* merged_mask, const float* merged_old_logp,
                                    const int64_t* merged_offsets, const int32_t* merged_origin, const int32_t* tl_seg,
                                    const float* seg_adv, const int64_t* counts, int64_t capacity_tokens, int32_t S,
                                    int32_t* targets, uint8_t* mask, float* old_logp, int32_t* seg_ids, float* adv,
                                    uint32_t* status_bits, ajt_stream_t stream_) {
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    if (capacity_tokens < 0 || S <= 0) return AJT_ERR_INVALID_ARG;
    if (!merged_offsets || !merged_origin || !tl_seg || !counts) return AJT_ERR_INVALID_ARG;
    if (capacity_tokens > 0 && (!merged_tokens || !merged_mask || !targets || !mask || !seg_ids)) return AJT_ERR_INVALID_ARG;
    if ((merged_old_logp == nullptr) != (old_logp == nullptr)) return AJT_ERR_INVALID_ARG;
    if ((seg_adv == nullptr) != (adv == nullptr)) return AJT_ERR_INVALID_ARG;
    int dev = 0, num_sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return AJT_ERR_CUDA;
    if (cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || num_sms < 1) return AJT_ERR_CUDA;
    if (status_bits && cudaMemsetAsync(status_bits, 0, sizeof(uint32_t), stream) != cudaSuccess) return AJT_ERR_CUDA;
    if (capacity_tokens == 0) return AJT_OK;
    PackParams p;
    p.merged_tokens = merged_tokens; p.merged_mask = merged_mask; p.merged_old_logp = merged_old_logp;
    p.merged_offsets = merged_offsets; p.merged_origin = merged_origin; p.tl_seg = tl_seg; p.seg_adv = seg_adv; p.counts = counts;
    p.cap = capacity_tokens; p.S = S; p.targets = targets; p.mask = mask; p.old_logp = old_logp; p.seg_ids = seg_ids; p.adv = adv; p.status = status_bits;
    const int64_t want = (capacity_tokens + 8 * kPackTile - 1) / (8 * kPackTile);
    const int grid = (int)(want < (int64_t)num_sms * 8 ? (want < 1 ? 1 : want) : (int64_t)num_sms * 8);
    AJT_LAUNCH(pack_loss_inputs_kernel<<<grid, 256, 0, stream>>>(p));
    return cudaGetLastError() == cudaSuccess ? AJT_OK : AJT_ERR_CUDA;
}
