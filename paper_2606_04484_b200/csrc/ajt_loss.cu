// Stage (b): token-level clipped policy-gradient loss, forward + backward w.r.t. logits (sm_100a).
//
// What is computed: DESIGN.md "O-L" steps 1-7 (BASELINE.json north_star).
// Kernels:
//   K6  loss_prep_kernel   per-segment mask counts N_s, 1/S', and the compacted lists of rows to read
//                          (mask=1) and rows to zero-fill (mask=0)                          [L0]
//   K7  loss_rows_kernel   the HBM-bound row kernel: each unmasked [V] row is pulled ONCE from HBM by
//                          1-D TMA bulk copies into a shared-memory ring, parked in registers as packed
//                          bf16, reduced (max, sum-exp), turned into dlogits and stored ONCE.  A row of
//                          V=151936 bf16 (304 KB) does not fit one SM, so a 2-CTA cluster holds half a
//                          row each and exchanges the 16+16 warp partials over DSMEM (st.async +
//                          mbarrier complete_tx).  Masked rows are zero-filled by the producer warp with
//                          bulk stores from a zeroed shared buffer, overlapping the math.      [L1-L3]
//       loss_rows_generic  fallback for fp32 logits / odd V / unaligned / huge V (3 reads via L1/L2).
//   K8  loss_final_kernel  fixed-order fp64 reduction of the per-row terms -> loss, stats      [L4]
#include <math.h>

#include <mutex>

#include "ajt_common.cuh"
#include "ajt_token.cuh"

namespace {

using namespace ajt;

// 19 consumer warps + 1 producer warp = 20 warps: registers are allocated per 4 warps, so 20 warps x 96
// registers fill the 64K register file exactly; 64 of the 96 hold the row slice (16 x uint4).
constexpr int kConsWarps = 19;
constexpr int kConsumers = kConsWarps * 32;      // 608 consumer threads
constexpr int kThreads = kConsumers + 32;        // + 1 producer warp = 640
constexpr int kChunkElems = kConsumers * 8;      // 4864 bf16 per chunk: one 16-byte vector per consumer thread
constexpr int kChunkBytes = kChunkElems * 2;     // 9728 B
constexpr int kSlots = 20;                       // 190 KB ring
constexpr int kMaxCluster = 2;
constexpr float kLog2e = 1.4426950408889634f;
constexpr uint32_t kNegInf2 = 0xFF80FF80u;       // packed bf16 (-inf, -inf)

constexpr int kScalRing = 32;                    // per-row scalar records in flight (> kSlots: the producer is at most kSlots rows ahead)
struct __align__(16) RowScal {                   // written by the producer, read (broadcast) by every consumer
    int64_t row;
    int32_t y;
    int32_t ybad;
    float old, A, w, zy;
    float ref, pad0, pad1, pad2;                 // extended form only: reference-policy log-prob of the target
};
static_assert(sizeof(RowScal) == 48, "RowScal is three 16-byte vectors");

constexpr size_t kRowsSmemBytes = (size_t)kSlots * kChunkBytes + kChunkBytes /* zero buffer */ +
                                  (2 * kSlots + 2) * sizeof(uint64_t) + 2 * kConsWarps * kMaxCluster * sizeof(float2) +
                                  kScalRing * sizeof(RowScal) + 2 * kConsWarps * kMaxCluster * sizeof(float);

struct LossParams {
    const void* logits;
    const int32_t* targets;
    const float* old_logp;
    const float* adv;
    const uint8_t* mask;
    const int32_t* seg_ids;
    float eps_lo, eps_hi;
    int64_t T;
    int32_t V, S;
    int64_t ld;
    int32_t dtype;
    const float* seg_denom;
    float inv_num_segs, grad_scale;
    void* dlogits;
    float* loss_out;
    float* logp_out;
    float* stats_out;
    const float* ref_logp;  // extended form (steps 8-9): reference-policy log-probs [T] or NULL
    float kl_coef;
    float clip_c;           // extended form, step 3b: dual-clip bound for negative advantages (0: off)
    float* ext_out;         // [2] {sum w_t k3_t, sum w_t H_t} or NULL
    float* k3_out;          // [T] or NULL
    float* ent_out;         // [T] or NULL
    int32_t ext;            // 1: extended kernels (KL term and / or entropy requested)
    int32_t zero_rows;      // 1: the prep kernel zeroes logp_out / k3_out / ent_out of every row
    // workspace
    AjtCtrl* ctrl;
    uint64_t* tile_state;  // [ntiles] prep scan: bit 63 valid, bits 32..62 active rows of the tile, bits 0..31 masked rows
    int32_t* seg_cnt;      // [S]
    int4* rec_i;           // [T] compact records of the rows with mask = 1, ascending: {row, target, segment, 0}
    float2* rec_f;         // [T]   "  : {old_logp, adv}
    float* rec_r;          // [T]   "  : ref_logp (extended form)
    int32_t* list_zero;    // [T] rows with mask = 0, ascending
    double* row_val;       // [T] w_t L_t by compact index
    double* row_kl;        // [T] w_t (-log r_t) by compact index
    uint8_t* row_clip;     // [T] bit0 clipped high, bit1 clipped low
    double* row_k3;        // [T] w_t k3_t by compact index (extended form)
    double* row_ent;       // [T] w_t H_t   "
};

struct LossWs {
    size_t ctrl, tile_state, seg_cnt, zero_bytes, rec_i, rec_f, rec_r, list_zero, row_val, row_kl, row_clip, row_k3, row_ent, total;
};
constexpr int kPrepTile = 1024;

__host__ inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

__host__ LossWs loss_ws_layout(int64_t T, int32_t S) {
    LossWs w;
    size_t o = 0;
    w.ctrl = o; o += align256(sizeof(AjtCtrl));
    w.tile_state = o; o += align256((size_t)((T + kPrepTile - 1) / kPrepTile) * 8);
    w.seg_cnt = o; o += align256((size_t)S * 4);
    w.zero_bytes = o;  // [ctrl, tile_state, seg_cnt] are cleared by one memset per call
    w.rec_i = o; o += align256((size_t)T * 16);
    w.rec_f = o; o += align256((size_t)T * 8);
    w.rec_r = o; o += align256((size_t)T * 4);
    w.list_zero = o; o += align256((size_t)T * 4);
    w.row_val = o; o += align256((size_t)T * 8);
    w.row_kl = o; o += align256((size_t)T * 8);
    w.row_clip = o; o += align256((size_t)T);
    w.row_k3 = o; o += align256((size_t)T * 8);
    w.row_ent = o; o += align256((size_t)T * 8);
    w.total = o;
    return w;
}

// ------------------------------------------------------------------------------------------------ K6

constexpr uint64_t kTileValid = 1ull << 63;

// Grid-wide stable compaction in one pass.  Tiles of 1024 rows are handed out by an atomic ticket (so every predecessor of
// a tile has started: no deadlock whatever the grid); a tile publishes its (active, masked) counts, then sums the counts of
// all its predecessors (1024 at a time, spinning on the valid bit) to get its bases.  The last CTA to finish counts S'.
__global__ void __launch_bounds__(1024) loss_prep_kernel(const LossParams p, int ntiles) {
    __shared__ int s_cnt[2][32];
    __shared__ int s_red[2][32];
    __shared__ int s_tile, s_last;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (;;) {
        if (tid == 0) s_tile = atomicAdd(&p.ctrl->tile_counter, 1);
        __syncthreads();
        const int tile = s_tile;
        if (tile >= ntiles) break;
        const int64_t t = (int64_t)tile * kPrepTile + tid;
        const bool in = t < p.T;
        if (in && p.zero_rows) {   // per-row outputs: masked rows read 0; the rows kernel then writes the unmasked ones
            if (p.logp_out) p.logp_out[t] = 0.f;
            if (p.k3_out) p.k3_out[t] = 0.f;
            if (p.ent_out) p.ent_out[t] = 0.f;
        }
        bool act = in && p.mask[t] != 0;
        int sg = act ? p.seg_ids[t] : 0;
        if (act && (unsigned)sg >= (unsigned)p.S) {
            atomicOr(&p.ctrl->status, (uint32_t)AJT_STATUS_BAD_SEG);
            act = false;  // treated as a masked-out row
        }
        // N_s: warp-aggregated atomics (segments are contiguous runs, so lanes mostly share one id)
        const int key = act ? sg : -1 - lane;
        const unsigned peers = __match_any_sync(0xffffffffu, key);
        if (act && lane == __ffs(peers) - 1) atomicAdd(&p.seg_cnt[sg], __popc(peers));
        const unsigned ba = __ballot_sync(0xffffffffu, act);
        const unsigned bz = __ballot_sync(0xffffffffu, in && !act);
        if (lane == 0) {
            s_cnt[0][warp] = __popc(ba);
            s_cnt[1][warp] = __popc(bz);
        }
        __syncthreads();
        int pa = 0, pz = 0, ta = 0, tz = 0;
#pragma unroll
        for (int w = 0; w < 32; ++w) {
            const int ca = s_cnt[0][w], cz = s_cnt[1][w];
            if (w < warp) { pa += ca; pz += cz; }
            ta += ca; tz += cz;
        }
        if (tid == 0)
            atomicExch(reinterpret_cast<unsigned long long*>(&p.tile_state[tile]),
                       (unsigned long long)(kTileValid | ((uint64_t)ta << 32) | (uint64_t)tz));
        int sa = 0, sz = 0;
        for (int i = tid; i < tile; i += 1024) {
            uint64_t v;
            do {
                v = *reinterpret_cast<volatile uint64_t*>(&p.tile_state[i]);
            } while (!(v & kTileValid));
            sa += (int)((v >> 32) & 0x7fffffffu);
            sz += (int)(v & 0xffffffffu);
        }
#pragma unroll
        for (int o = 16; o; o >>= 1) {
            sa += __shfl_xor_sync(0xffffffffu, sa, o);
            sz += __shfl_xor_sync(0xffffffffu, sz, o);
        }
        if (lane == 0) { s_red[0][warp] = sa; s_red[1][warp] = sz; }
        __syncthreads();
        int base_a = 0, base_z = 0;
#pragma unroll
        for (int w = 0; w < 32; ++w) { base_a += s_red[0][w]; base_z += s_red[1][w]; }
        const unsigned lt = (1u << lane) - 1u;
        if (act) {
            const int idx = base_a + pa + __popc(ba & lt);
            p.rec_i[idx] = make_int4((int)t, p.targets[t], sg, 0);
            p.rec_f[idx] = make_float2(p.old_logp[t], p.adv[t]);
            if (p.ref_logp) p.rec_r[idx] = p.ref_logp[t];
        } else if (in) {
            p.list_zero[base_z + pz + __popc(bz & lt)] = (int32_t)t;
        }
        if (tile == ntiles - 1 && tid == 0) {
            p.ctrl->n_active = base_a + ta;
            p.ctrl->n_zero = base_z + tz;
        }
        __syncthreads();
    }
    // the last CTA to get here sees every N_s: S' = #{s : N_s > 0}
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = atomicAdd(&p.ctrl->done_counter, 1) == (int)gridDim.x - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    int live = 0;
    for (int s = tid; s < p.S; s += 1024) {
        const float d = p.seg_denom ? p.seg_denom[s] : (float)__ldcg(&p.seg_cnt[s]);
        live += d > 0.f;
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) live += __shfl_xor_sync(0xffffffffu, live, o);
    if (lane == 0) s_red[0][warp] = live;
    __syncthreads();
    if (tid == 0) {
        int tot = 0;
        for (int w = 0; w < 32; ++w) tot += s_red[0][w];
        p.ctrl->n_live_segs = tot;
        p.ctrl->inv_num_segs = p.inv_num_segs != 0.f ? p.inv_num_segs : (tot > 0 ? 1.0f / (float)tot : 0.f);
    }
}

// ------------------------------------------------------------------------------------------------ L2

// ------------------------------------------------------------------------------------------------ K7 (fast)

__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ float exp_diff(float m, float M) {  // exp(m - M), 0 when m = -inf
    return m == -INFINITY ? 0.f : ex2((m - M) * kLog2e);
}

// t = z - m, e = exp(t): s += e, u += e t.  (The extended kernels never feed padding here; a -inf logit makes the entropy
// NaN, as it does in the definition: the domain is finite logits, reading L-7.)
__device__ __forceinline__ void acc_exp(float x, float ms, float& s, float& u, bool ext) {
    const float t = x - ms;
    const float e = ex2(t * kLog2e);
    s += e;
    if (ext) u = fmaf(e, t, u);
}
// The same with the subtraction folded into one FFMA (k = -m log2(e)); u then collects e z, and the caller takes m s off.
__device__ __forceinline__ void acc_exp_fma(float x, float k, float& s, float& u, bool ext) {
    const float e = ex2(fmaf(x, kLog2e, k));
    s += e;
    if (ext) u = fmaf(e, x, u);
}
// re-base a partial (m, s, u = sum e^{z-m} (z-m)) onto the maximum M: returns the factor, updates s and u
__device__ __forceinline__ void rebase(float m, float M, float& s, float& u) {
    const float f = exp_diff(m, M);
    const float dm = m == -INFINITY ? 0.f : m - M;
    u = f * fmaf(dm, s, u);
    s = f * s;
}

// EXT: the extended form (steps 8-9): reference-policy log-prob per row, and u = sum_v e^{z-M} (z-M) beside the sum-exp so
// that the row entropy H = log S - u / S comes out of the same single read.
template <int NCH, int CSIZE, bool EXT>
__global__ void __launch_bounds__(kThreads, 1) loss_rows_kernel(const LossParams p) {
    extern __shared__ __align__(1024) uint8_t smem[];
    pdl_wait();
    uint8_t* ring = smem;
    uint8_t* zbuf = smem + (size_t)kSlots * kChunkBytes;
    uint64_t* full = reinterpret_cast<uint64_t*>(zbuf + kChunkBytes);
    uint64_t* empty = full + kSlots;
    uint64_t* pbar = empty + kSlots;
    float2* part = reinterpret_cast<float2*>(pbar + 2);  // [2][kConsWarps * kMaxCluster]
    RowScal* scal = reinterpret_cast<RowScal*>(part + 2 * kConsWarps * kMaxCluster);
    float* partu = reinterpret_cast<float*>(scal + kScalRing);  // [2][kConsWarps * kMaxCluster], extended form
    constexpr int kParts = kConsWarps * CSIZE;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t rank = CSIZE > 1 ? cluster_ctarank() : 0u;
    const int cid = blockIdx.x / CSIZE, NC = gridDim.x / CSIZE;

    // the slice of the vocabulary this CTA owns: 8-element (16-byte) granularity
    const int V = p.V;
    const int h = CSIZE == 1 ? V : (((V + CSIZE - 1) / CSIZE + 7) & ~7);
    const int sl_begin = (int)rank * h;
    const int sl_len = max(0, min(h, V - sl_begin));
    const int nch = (sl_len + kChunkElems - 1) / kChunkElems;

    if (tid == 0) {
        for (int i = 0; i < kSlots; ++i) {
            mbar_init(&full[i], 1);
            mbar_init(&empty[i], kConsWarps);
        }
        mbar_init(&pbar[0], kConsWarps);
        mbar_init(&pbar[1], kConsWarps);
        fence_mbar_init();
    }
    for (int i = tid; i < kChunkBytes / 16; i += kThreads) reinterpret_cast<uint4*>(zbuf)[i] = make_uint4(0, 0, 0, 0);
    fence_proxy_async_smem();
    if (CSIZE > 1) cluster_sync_all(); else __syncthreads();

    const int n_active = p.ctrl->n_active, n_zero = p.ctrl->n_zero;
    const int nrows = n_active > cid ? (n_active - cid + NC - 1) / NC : 0;
    const __nv_bfloat16* logits = reinterpret_cast<const __nv_bfloat16*>(p.logits);
    __nv_bfloat16* dlogits = reinterpret_cast<__nv_bfloat16*>(p.dlogits);

    if (warp == kConsWarps) {
        // ===== producer warp: TMA loads of unmasked rows + bulk zero-fill of masked rows =====
        if (lane == 0) {
            const int nzero = n_zero > cid ? (n_zero - cid + NC - 1) / NC : 0;
            int zdone = 0;
            auto zero_rows_until = [&](int target) {
                for (; zdone < target; ++zdone) {
                    const int64_t row = p.list_zero[cid + (int64_t)zdone * NC];
                    __nv_bfloat16* dst = dlogits + row * p.ld + sl_begin;
                    for (int ch = 0; ch < nch; ++ch) {
                        const uint32_t bytes = (uint32_t)min(kChunkElems, sl_len - ch * kChunkElems) * 2u;
                        bulk_store(dst + (size_t)ch * kChunkElems, zbuf, bytes);
                    }
                    bulk_commit();
                }
            };
            // Per-row scalars are gathered two rows ahead so that their dependent loads (record -> logits[row, y],
            // N_s) never sit on anybody's critical path: stage B holds row k+1's record with its two loads in
            // flight, stage C holds row k complete.  Published through shared memory before the row's first
            // full-barrier arrive (release) and read by the consumers after their wait (acquire).
            const float inv_S = p.ctrl->inv_num_segs;
            struct Stage { int4 ri; float2 rf; float zy, den, ref; };
            auto load_rec = [&](int k, Stage& st) {
                if (k < nrows) {
                    const int64_t idx = cid + (int64_t)k * NC;
                    st.ri = p.rec_i[idx];
                    st.rf = p.rec_f[idx];
                    if (EXT) st.ref = p.ref_logp ? p.rec_r[idx] : 0.f;
                }
            };
            auto load_dep = [&](int k, Stage& st) {
                if (k < nrows) {
                    const bool ybad = (unsigned)st.ri.y >= (unsigned)V;
                    st.zy = ybad ? 0.f : __bfloat162float(logits[(int64_t)st.ri.x * p.ld + st.ri.y]);
                    st.den = p.seg_denom ? p.seg_denom[st.ri.z] : (float)p.seg_cnt[st.ri.z];
                }
            };
            Stage A = {}, B = {}, C = {};
            load_rec(0, C);
            load_rec(1, B);
            load_dep(0, C);
            load_dep(1, B);
            int slot = 0;
            uint32_t ph = 0;
            for (int k = 0; k < nrows; ++k) {
                load_rec(k + 2, A);
                {
                    const bool ybad = (unsigned)C.ri.y >= (unsigned)V;
                    RowScal rs;
                    rs.row = C.ri.x;
                    rs.y = C.ri.y;
                    rs.ybad = ybad;
                    rs.old = C.rf.x;
                    rs.A = C.rf.y;
                    rs.w = (C.den > 0.f && !ybad) ? inv_S / C.den : 0.f;
                    rs.zy = C.zy;
                    rs.ref = C.ref;
                    rs.pad0 = rs.pad1 = rs.pad2 = 0.f;
                    scal[k & (kScalRing - 1)] = rs;
                }
                const int64_t row = C.ri.x;
                const __nv_bfloat16* src = logits + row * p.ld + sl_begin;
                for (int ch = 0; ch < nch; ++ch) {
                    mbar_wait(&empty[slot], ph ^ 1u);
                    const uint32_t bytes = (uint32_t)min(kChunkElems, sl_len - ch * kChunkElems) * 2u;
                    mbar_arrive_expect_tx(&full[slot], bytes);
                    bulk_load(ring + (size_t)slot * kChunkBytes, src + (size_t)ch * kChunkElems, bytes, &full[slot]);
                    if (++slot == kSlots) { slot = 0; ph ^= 1u; }
                }
                zero_rows_until((int)(((int64_t)(k + 1) * nzero) / nrows));
                C = B;
                B = A;
                load_dep(k + 2, B);
            }
            zero_rows_until(nzero);
            bulk_wait<0>();
        }
    } else {
        // ===== consumer warps =====
        int slot = 0;
        uint32_t ph = 0;
        for (int k = 0; k < nrows; ++k) {
            const int kidx = cid + k * NC;
            // ---- pass 1a: ring -> registers (packed bf16), packed running max
            uint4 r[NCH];
            uint32_t mx = kNegInf2;
            int64_t row = 0;
            int y = 0;
            bool ybad = false;
            float old = 0.f, A = 0.f, w = 0.f, zy = 0.f, ref = 0.f;
#pragma unroll
            for (int ch = 0; ch < NCH; ++ch) {
                r[ch] = make_uint4(kNegInf2, kNegInf2, kNegInf2, kNegInf2);
                if (ch < nch) {
                    mbar_wait(&full[slot], ph);
                    if (ch == 0) {  // the producer published this row's scalars before arming the first chunk
                        const uint4 s0 = lds128(&scal[k & (kScalRing - 1)]), s1 = lds128(&scal[k & (kScalRing - 1)].old);
                        row = (int64_t)(((uint64_t)s0.y << 32) | s0.x);
                        y = (int)s0.z;
                        ybad = s0.w != 0;
                        old = __uint_as_float(s1.x);
                        A = __uint_as_float(s1.y);
                        w = __uint_as_float(s1.z);
                        zy = __uint_as_float(s1.w);
                        if (EXT) ref = scal[k & (kScalRing - 1)].ref;
                    }
                    if (ch * kChunkElems + tid * 8 < sl_len) r[ch] = lds128(ring + (size_t)slot * kChunkBytes + tid * 16);
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&empty[slot]);
                    if (++slot == kSlots) { slot = 0; ph ^= 1u; }
                    mx = max_bf16x2(mx, max_bf16x2(max_bf16x2(r[ch].x, r[ch].y), max_bf16x2(r[ch].z, r[ch].w)));
                }
            }
            // ---- pass 1b: thread-local sum of exp(x - m_thread) from registers: one MUFU per element
            const float m = fmaxf(bf16lo(mx), bf16hi(mx));
            const float ms = m == -INFINITY ? 0.f : m;
            float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f, u0 = 0.f, u1 = 0.f;
            const float kms = -ms * kLog2e;
#pragma unroll
            for (int ch = 0; ch < NCH; ++ch) {
                if (ch < nch && (!EXT || ch * kChunkElems + tid * 8 < sl_len)) {   // EXT: no -inf padding in e * t
                    acc_exp_fma(bf16lo(r[ch].x), kms, s0, u0, EXT);
                    acc_exp_fma(bf16hi(r[ch].x), kms, s1, u1, EXT);
                    acc_exp_fma(bf16lo(r[ch].y), kms, s2, u0, EXT);
                    acc_exp_fma(bf16hi(r[ch].y), kms, s3, u1, EXT);
                    acc_exp_fma(bf16lo(r[ch].z), kms, s0, u0, EXT);
                    acc_exp_fma(bf16hi(r[ch].z), kms, s1, u1, EXT);
                    acc_exp_fma(bf16lo(r[ch].w), kms, s2, u0, EXT);
                    acc_exp_fma(bf16hi(r[ch].w), kms, s3, u1, EXT);
                }
            }
            float s = (s0 + s1) + (s2 + s3);
            // ---- warp partial, published to every CTA of the cluster
            const float mw = warp_max(m);
            float sw, uw = 0.f;
            if (EXT) {
                float u = fmaf(-ms, s, u0 + u1);   // sum e (z - m)
                rebase(m, mw, s, u);
                sw = warp_sum(s);
                uw = warp_sum(u);
            } else {
                sw = warp_sum(s * exp_diff(m, mw));
            }
            const int par = k & 1;
            float2* mypart = part + par * kParts;
            float* mypartu = partu + par * kParts;
            if (lane == 0) {
                mypart[rank * kConsWarps + warp] = make_float2(mw, sw);
                if (EXT) mypartu[rank * kConsWarps + warp] = uw;
                if (CSIZE > 1) {
                    const uint64_t v = ((uint64_t)__float_as_uint(sw) << 32) | (uint64_t)__float_as_uint(mw);
                    const uint32_t a = smem_u32(&mypart[rank * kConsWarps + warp]), b = smem_u32(&pbar[par]);
                    const uint32_t au = smem_u32(&mypartu[rank * kConsWarps + warp]);
#pragma unroll
                    for (uint32_t q = 0; q < (uint32_t)CSIZE; ++q)
                        if (q != rank) {
                            st_async_b64(mapa(a, q), v, mapa(b, q));
                            if (EXT) st_async_b32(mapa(au, q), __float_as_uint(uw), mapa(b, q));
                        }
                    if (warp == 0) mbar_arrive_expect_tx(&pbar[par], (uint32_t)((CSIZE - 1) * kConsWarps * (EXT ? 12 : 8)));
                    else mbar_arrive(&pbar[par]);
                } else {
                    mbar_arrive(&pbar[par]);
                }
            }
            mbar_wait(&pbar[par], (uint32_t)(k >> 1) & 1u);
            // ---- combine the 16*CSIZE partials (every warp redundantly; 1 MUFU + 10 shuffles)
            float2 pv = lane < kParts ? mypart[lane] : make_float2(-INFINITY, 0.f);
            float2 pw = (kParts > 32 && lane + 32 < kParts) ? mypart[lane + 32] : make_float2(-INFINITY, 0.f);
            const float M = warp_max(fmaxf(pv.x, pw.x));
            float S, U = 0.f;
            if (EXT) {
                float uv = lane < kParts ? mypartu[lane] : 0.f;
                float ux = (kParts > 32 && lane + 32 < kParts) ? mypartu[lane + 32] : 0.f;
                rebase(pv.x, M, pv.y, uv);
                rebase(pw.x, M, pw.y, ux);
                S = warp_sum(pv.y + pw.y);
                U = warp_sum(uv + ux);
            } else {
                S = warp_sum(pv.y * exp_diff(pv.x, M) + pw.y * exp_diff(pw.x, M));
            }
            const TokScalars ts = token_scalars(M, S, zy, old, A, w, p.eps_lo, p.eps_hi, p.grad_scale,
                                                EXT && p.ref_logp != nullptr && p.kl_coef != 0.f, ref, p.kl_coef, EXT ? p.clip_c : 0.f);
            if (tid == 0 && rank == 0) {
                p.row_val[kidx] = ts.wl;
                p.row_kl[kidx] = ts.wkl;
                p.row_clip[kidx] = (uint8_t)(w > 0.f ? ts.clip : 0);
                if (p.logp_out) p.logp_out[row] = ybad ? 0.f : ts.logp;
                if (ybad) atomicOr(&p.ctrl->status, (uint32_t)AJT_STATUS_BAD_TARGET);
                if (EXT) {
                    const float H = ybad ? 0.f : ts.logS - U / S;   // step 9: H = lse - sum p z = log S - sum e^{z-M}(z-M) / S
                    p.row_k3[kidx] = ts.wk3;
                    p.row_ent[kidx] = (double)w * (double)H;
                    if (p.k3_out) p.k3_out[row] = ybad ? 0.f : ts.k3;
                    if (p.ent_out) p.ent_out[row] = H;
                }
            }
            // ---- pass 2: dlogits = g (1[v=y] - exp(z - lse)), bf16 RNE, one 16-byte store per vector
            __nv_bfloat16* drow = dlogits + row * p.ld + sl_begin;
            const float g = ts.g;
            if (g != 0.f) {
                const float coef = -g, k2 = -ts.lse * kLog2e;
#pragma unroll
                for (int ch = 0; ch < NCH; ++ch) {
                    if (ch < nch && ch * kChunkElems + tid * 8 < sl_len) {
                        uint4 o;
                        o.x = pack_bf16x2(coef * ex2(fmaf(bf16lo(r[ch].x), kLog2e, k2)), coef * ex2(fmaf(bf16hi(r[ch].x), kLog2e, k2)));
                        o.y = pack_bf16x2(coef * ex2(fmaf(bf16lo(r[ch].y), kLog2e, k2)), coef * ex2(fmaf(bf16hi(r[ch].y), kLog2e, k2)));
                        o.z = pack_bf16x2(coef * ex2(fmaf(bf16lo(r[ch].z), kLog2e, k2)), coef * ex2(fmaf(bf16hi(r[ch].z), kLog2e, k2)));
                        o.w = pack_bf16x2(coef * ex2(fmaf(bf16lo(r[ch].w), kLog2e, k2)), coef * ex2(fmaf(bf16hi(r[ch].w), kLog2e, k2)));
                        stg128_stream(drow + (size_t)ch * kChunkElems + tid * 8, o);
                    }
                }
                // the target column: g (1 - p_y); same thread that stored the vector holding it, so ordered
                const int yl = y - sl_begin;
                if ((unsigned)yl < (unsigned)sl_len && ((yl % kChunkElems) >> 3) == tid) {
                    const float py = ex2(fmaf(zy, kLog2e, k2));
                    drow[yl] = __float2bfloat16_rn(fmaf(coef, py, g));
                }
            } else {
                const uint4 z4 = make_uint4(0, 0, 0, 0);
#pragma unroll
                for (int ch = 0; ch < NCH; ++ch)
                    if (ch < nch && ch * kChunkElems + tid * 8 < sl_len) stg128_stream(drow + (size_t)ch * kChunkElems + tid * 8, z4);
            }
        }
    }
    if (CSIZE > 1) cluster_sync_all();  // peers may still be writing into this CTA's shared memory
}

// ------------------------------------------------------------------------------------------------ K7 (generic)

template <typename TIn>
__device__ __forceinline__ float ld_logit(const TIn* p, int64_t i);
template <>
__device__ __forceinline__ float ld_logit<float>(const float* p, int64_t i) { return p[i]; }
template <>
__device__ __forceinline__ float ld_logit<__nv_bfloat16>(const __nv_bfloat16* p, int64_t i) { return __bfloat162float(p[i]); }

// One group of G threads per row (G = 32 or 256).  Three sweeps over the row (max, sum-exp, write); the
// second and third hit L1/L2.  Used for fp32 logits (config c1), V % 8 != 0, unaligned pointers, V > 155648.
template <typename TIn, int G>
__global__ void __launch_bounds__(256) loss_rows_generic(const LossParams p) {
    pdl_wait();
    constexpr int kGroups = 256 / G;
    __shared__ float s_red[3][kGroups][8];
    const int tid = threadIdx.x, gl = tid % G, gi = tid / G, lane = tid & 31, wig = gl >> 5;
    const TIn* logits = reinterpret_cast<const TIn*>(p.logits);
    __nv_bfloat16* dlogits = reinterpret_cast<__nv_bfloat16*>(p.dlogits);
    const float inv_S = p.ctrl->inv_num_segs;
    const int V = p.V;
    const int64_t nrow_groups = (p.T + kGroups - 1) / kGroups;
    for (int64_t rg = blockIdx.x; rg < nrow_groups; rg += gridDim.x) {
        const int64_t row = rg * kGroups + gi;
        const bool inrange = row < p.T;
        const bool act = inrange && p.mask[row] != 0;
        int y = 0, sg = 0;
        float old = 0.f, A = 0.f, w = 0.f, zy = 0.f, ref = 0.f;
        bool ybad = false;
        if (act) {
            if (p.ext && p.ref_logp) ref = p.ref_logp[row];
            y = p.targets[row];
            sg = p.seg_ids[row];
            old = p.old_logp[row];
            A = p.adv[row];
            ybad = (unsigned)y >= (unsigned)V;
            const bool sbad = (unsigned)sg >= (unsigned)p.S;
            const float denom = sbad ? 0.f : (p.seg_denom ? p.seg_denom[sg] : (float)p.seg_cnt[sg]);
            w = (denom > 0.f && !ybad) ? inv_S / denom : 0.f;
            zy = ybad ? 0.f : ld_logit<TIn>(logits, row * p.ld + y);
        }
        const TIn* zrow = logits + row * p.ld;
        float m = -INFINITY;
        if (act)
            for (int v = gl; v < V; v += G) m = fmaxf(m, ld_logit<TIn>(zrow, v));
        m = warp_max(m);
        if (G > 32) {
            if (lane == 0) s_red[0][gi][wig] = m;
            __syncthreads();
            m = s_red[0][gi][0];
#pragma unroll
            for (int i = 1; i < G / 32; ++i) m = fmaxf(m, s_red[0][gi][i]);
        }
        float s = 0.f, u = 0.f;   // u = sum e^{z-m} (z-m): entropy of the row (extended form)
        if (act)
            for (int v = gl; v < V; v += G) acc_exp(ld_logit<TIn>(zrow, v), m, s, u, true);
        s = warp_sum(s);
        u = warp_sum(u);
        if (G > 32) {
            if (lane == 0) {
                s_red[1][gi][wig] = s;
                s_red[2][gi][wig] = u;
            }
            __syncthreads();
            s = 0.f;
            u = 0.f;
#pragma unroll
            for (int i = 0; i < G / 32; ++i) {
                s += s_red[1][gi][i];
                u += s_red[2][gi][i];
            }
        }
        if (inrange) {
            __nv_bfloat16* drow = dlogits + row * p.ld;
            float g = 0.f, lse = 0.f;
            if (act) {
                const TokScalars ts = token_scalars(m, s, zy, old, A, w, p.eps_lo, p.eps_hi, p.grad_scale,
                                                    p.ext && p.ref_logp != nullptr && p.kl_coef != 0.f, ref, p.kl_coef, p.ext ? p.clip_c : 0.f);
                g = ts.g;
                lse = ts.lse;
                if (gl == 0) {
                    p.row_val[row] = ts.wl;
                    p.row_kl[row] = ts.wkl;
                    p.row_clip[row] = (uint8_t)(w > 0.f ? ts.clip : 0);
                    if (p.logp_out) p.logp_out[row] = ybad ? 0.f : ts.logp;
                    if (ybad) atomicOr(&p.ctrl->status, (uint32_t)AJT_STATUS_BAD_TARGET);
                    if (p.ext) {
                        const float H = ybad ? 0.f : ts.logS - u / s;
                        p.row_k3[row] = ts.wk3;
                        p.row_ent[row] = (double)w * (double)H;
                        if (p.k3_out) p.k3_out[row] = ybad ? 0.f : ts.k3;
                        if (p.ent_out) p.ent_out[row] = H;
                    }
                }
            } else if (gl == 0) {
                p.row_val[row] = 0.0;
                p.row_kl[row] = 0.0;
                p.row_clip[row] = 0;
                if (p.logp_out) p.logp_out[row] = 0.f;
                if (p.ext) {
                    p.row_k3[row] = 0.0;
                    p.row_ent[row] = 0.0;
                    if (p.k3_out) p.k3_out[row] = 0.f;
                    if (p.ent_out) p.ent_out[row] = 0.f;
                }
            }
            if (g != 0.f) {
                const float coef = -g, k2 = -lse * kLog2e;
                for (int v = gl; v < V; v += G) {
                    const float pv = ex2(fmaf(ld_logit<TIn>(zrow, v), kLog2e, k2));
                    drow[v] = __float2bfloat16_rn(v == y ? fmaf(coef, pv, g) : coef * pv);
                }
            } else {
                for (int v = gl; v < V; v += G) drow[v] = __float2bfloat16_rn(0.f);
            }
        }
        if (G > 32) __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------------ K8

// fp32 logits with V <= 2048 (configs[0]): ONE read of every unmasked row.  A warp per row; lane l keeps vectors l + 32 j
// (j < NV = ceil(V / 128)) of the row in registers as float4, so the maximum, the sum of exponentials (kept in place of the
// logits) and the gradient all come from the same 16-byte loads, and dlogits leave as 8-byte stores (256 contiguous bytes per
// instruction).  Same per-row outputs as loss_rows_generic (by_row layout for the final kernel).
template <int NV>
__global__ void __launch_bounds__(256) loss_rows_f32_regs(const LossParams p) {
    pdl_wait();
    const int lane = threadIdx.x & 31;
    const int64_t wglobal = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    const float* logits = reinterpret_cast<const float*>(p.logits);
    __nv_bfloat16* dlogits = reinterpret_cast<__nv_bfloat16*>(p.dlogits);
    const float inv_S = p.ctrl->inv_num_segs;
    const int V = p.V, nvec = V >> 2;
    for (int64_t row = wglobal; row < p.T; row += nwarps) {
        const bool act = p.mask[row] != 0;
        uint2* const drow = reinterpret_cast<uint2*>(dlogits + row * p.ld);
        if (!act) {
#pragma unroll
            for (int j = 0; j < NV; ++j)
                if (lane + 32 * j < nvec) drow[lane + 32 * j] = make_uint2(0u, 0u);
            if (lane == 0) {
                p.row_val[row] = 0.0;
                p.row_kl[row] = 0.0;
                p.row_clip[row] = 0;
                if (p.logp_out) p.logp_out[row] = 0.f;
                if (p.ext) {
                    p.row_k3[row] = 0.0;
                    p.row_ent[row] = 0.0;
                    if (p.k3_out) p.k3_out[row] = 0.f;
                    if (p.ent_out) p.ent_out[row] = 0.f;
                }
            }
            continue;
        }
        const float4* const zrow = reinterpret_cast<const float4*>(logits + row * p.ld);
        float4 x[NV];
#pragma unroll
        for (int j = 0; j < NV; ++j)
            x[j] = lane + 32 * j < nvec ? __ldg(zrow + lane + 32 * j) : make_float4(-INFINITY, -INFINITY, -INFINITY, -INFINITY);
        const float ref = p.ext && p.ref_logp ? p.ref_logp[row] : 0.f;
        const int y = p.targets[row], sg = p.seg_ids[row];
        const float old = p.old_logp[row], A = p.adv[row];
        const bool ybad = (unsigned)y >= (unsigned)V, sbad = (unsigned)sg >= (unsigned)p.S;
        const float denom = sbad ? 0.f : (p.seg_denom ? p.seg_denom[sg] : (float)p.seg_cnt[sg]);
        const float w = (denom > 0.f && !ybad) ? inv_S / denom : 0.f;
        float m = -INFINITY;
#pragma unroll
        for (int j = 0; j < NV; ++j) m = fmaxf(m, fmaxf(fmaxf(x[j].x, x[j].y), fmaxf(x[j].z, x[j].w)));
        m = warp_max(m);
        // the target's logit sits in exactly one lane's registers
        float zy = 0.f;
#pragma unroll
        for (int j = 0; j < NV; ++j) {
            const int v0 = 4 * (lane + 32 * j);
            if (!ybad && y >= v0 && y < v0 + 4) zy = y == v0 ? x[j].x : y == v0 + 1 ? x[j].y : y == v0 + 2 ? x[j].z : x[j].w;
        }
        zy = warp_sum(zy);
        float s = 0.f, u = 0.f;   // x becomes e^{z - m}; u = sum e^{z-m} (z-m): entropy of the row (extended form)
#pragma unroll
        for (int j = 0; j < NV; ++j) {
            float* f = reinterpret_cast<float*>(&x[j]);
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const float t = f[i] - m;
                const float e = ex2(t * kLog2e);   // padding lanes: e^{-inf} = 0
                s += e;
                if (p.ext && e > 0.f) u = fmaf(e, t, u);
                f[i] = e;
            }
        }
        s = warp_sum(s);
        u = warp_sum(u);
        const TokScalars ts = token_scalars(m, s, zy, old, A, w, p.eps_lo, p.eps_hi, p.grad_scale,
                                            p.ext && p.ref_logp != nullptr && p.kl_coef != 0.f, ref, p.kl_coef, p.ext ? p.clip_c : 0.f);
        if (lane == 0) {
            p.row_val[row] = ts.wl;
            p.row_kl[row] = ts.wkl;
            p.row_clip[row] = (uint8_t)(w > 0.f ? ts.clip : 0);
            if (p.logp_out) p.logp_out[row] = ybad ? 0.f : ts.logp;
            if (ybad) atomicOr(&p.ctrl->status, (uint32_t)AJT_STATUS_BAD_TARGET);
            if (p.ext) {
                const float H = ybad ? 0.f : ts.logS - u / s;
                p.row_k3[row] = ts.wk3;
                p.row_ent[row] = (double)w * (double)H;
                if (p.k3_out) p.k3_out[row] = ybad ? 0.f : ts.k3;
                if (p.ent_out) p.ent_out[row] = H;
            }
        }
        const float g = ts.g;
        if (g != 0.f) {
            const float coef = -g * ex2((m - ts.lse) * kLog2e);   // p_v = e^{z_v - m} e^{m - lse}
#pragma unroll
            for (int j = 0; j < NV; ++j) {
                if (lane + 32 * j >= nvec) continue;
                const int v0 = 4 * (lane + 32 * j);
                float d0 = coef * x[j].x, d1 = coef * x[j].y, d2 = coef * x[j].z, d3 = coef * x[j].w;
                if (y == v0) d0 += g;
                if (y == v0 + 1) d1 += g;
                if (y == v0 + 2) d2 += g;
                if (y == v0 + 3) d3 += g;
                drow[lane + 32 * j] = make_uint2(pack_bf16x2(d0, d1), pack_bf16x2(d2, d3));
            }
        } else {
#pragma unroll
            for (int j = 0; j < NV; ++j)
                if (lane + 32 * j < nvec) drow[lane + 32 * j] = make_uint2(0u, 0u);
        }
    }
}

// Fixed-order fp64 reduction: thread i sums elements i, i+1024, ...; then a shared-memory tree.
__global__ void __launch_bounds__(1024) loss_final_kernel(const LossParams p, int by_row) {
    pdl_wait();
    __shared__ double s_a[1024], s_b[1024];
    __shared__ int s_c[2][1024];
    const int tid = threadIdx.x;
    const int64_t n = by_row ? p.T : (int64_t)p.ctrl->n_active;
    double a = 0.0, b = 0.0;
    int c1 = 0, c2 = 0;
    for (int64_t i = tid; i < n; i += 1024) {
        a += p.row_val[i];
        b += p.row_kl[i];
        const int c = p.row_clip[i];
        c1 += c & 1;
        c2 += (c >> 1) & 1;
    }
    s_a[tid] = a; s_b[tid] = b; s_c[0][tid] = c1; s_c[1][tid] = c2;
    __syncthreads();
    for (int o = 512; o; o >>= 1) {
        if (tid < o) {
            s_a[tid] += s_a[tid + o];
            s_b[tid] += s_b[tid + o];
            s_c[0][tid] += s_c[0][tid + o];
            s_c[1][tid] += s_c[1][tid + o];
        }
        __syncthreads();
    }
    double pg = s_a[0];
    if (p.ext) {   // steps 8-9: second fixed-order pass over the KL and entropy terms, same tree
        __syncthreads();
        a = 0.0;
        b = 0.0;
        for (int64_t i = tid; i < n; i += 1024) {
            a += p.row_k3[i];
            b += p.row_ent[i];
        }
        const double hold = s_b[0];
        __syncthreads();
        s_a[tid] = a; s_b[tid] = b;
        __syncthreads();
        for (int o = 512; o; o >>= 1) {
            if (tid < o) {
                s_a[tid] += s_a[tid + o];
                s_b[tid] += s_b[tid + o];
            }
            __syncthreads();
        }
        if (tid == 0) {
            pg += (double)p.kl_coef * s_a[0];
            if (p.ext_out) {
                p.ext_out[0] = (float)s_a[0];
                p.ext_out[1] = (float)s_b[0];
            }
            s_b[0] = hold;
        }
    }
    if (tid == 0) {
        p.loss_out[0] = (float)pg;
        if (p.stats_out) {
            p.stats_out[0] = (float)p.ctrl->n_active;
            p.stats_out[1] = (float)s_c[0][0];
            p.stats_out[2] = (float)s_c[1][0];
            p.stats_out[3] = (float)s_b[0];
        }
    }
}

// ------------------------------------------------------------------------------------------------ segment counts

// N_s += #{t in this call : seg_t = s, mask_t = 1}.  Counts are integers held in fp32 (exact below 2^24), so the
// float atomics commute and the result does not depend on the order of arrival.
__global__ void __launch_bounds__(256) segment_counts_kernel(const uint8_t* __restrict__ mask, const int32_t* __restrict__ seg_ids,
                                                             int64_t T, int32_t S, float* __restrict__ denom,
                                                             uint32_t* __restrict__ status) {
    const int lane = threadIdx.x & 31;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t gtid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    // Vector body: 4 positions per thread and iteration (one 4-byte mask load, one 16-byte segment-id load), whenever both
    // arrays reach their alignment at the same position h; segments are long runs, so a warp's 128 positions almost always
    // carry one id and cost one atomic.  Counts are integers below 2^24, so the float adds are exact in any order.
    int64_t h = (4 - (int64_t)(reinterpret_cast<uintptr_t>(mask) & 3)) & 3;
    const bool vec = ((reinterpret_cast<uintptr_t>(seg_ids) >> 2) + (uintptr_t)h) % 4 == 0;
    if (!vec) h = T;
    if (h > T) h = T;
    const int64_t nq = vec ? (T - h) / 4 : 0;
    const int64_t nq_pad = (nq + 31) & ~(int64_t)31;
    for (int64_t q = gtid; q < nq_pad; q += stride) {
        int sg = -1, cnt = 0;
        if (q < nq) {
            const uint32_t m4 = *reinterpret_cast<const uint32_t*>(mask + h + 4 * q);
            if (m4) {
                const int4 s4 = *reinterpret_cast<const int4*>(seg_ids + h + 4 * q);
                const int sv[4] = {s4.x, s4.y, s4.z, s4.w};
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    if (!((m4 >> (8 * i)) & 0xffu)) continue;
                    if ((unsigned)sv[i] >= (unsigned)S) {
                        if (status) atomicOr(status, (uint32_t)AJT_STATUS_BAD_SEG);
                        continue;
                    }
                    if (sg < 0) sg = sv[i];
                    if (sv[i] == sg) ++cnt;
                    else atomicAdd(&denom[sv[i]], 1.0f);
                }
            }
        }
        const unsigned have = __ballot_sync(0xffffffffu, cnt > 0);
        if (!have) continue;
        const int s0 = __shfl_sync(0xffffffffu, sg, __ffs(have) - 1);
        if (__all_sync(0xffffffffu, cnt == 0 || sg == s0)) {
            const int tot = __reduce_add_sync(0xffffffffu, cnt);
            if (lane == 0) atomicAdd(&denom[s0], (float)tot);
        } else if (cnt > 0) {
            atomicAdd(&denom[sg], (float)cnt);
        }
    }
    // scalar head / tail (and the whole range when the two alignments never meet)
    const int64_t t_tail = vec ? h + 4 * nq : 0;
    const int64_t n_sc = vec ? h + (T - t_tail) : T;
    for (int64_t i = gtid; i < n_sc; i += stride) {
        const int64_t t = (vec && i >= h) ? t_tail + (i - h) : i;
        if (mask[t] == 0) continue;
        const int sg = seg_ids[t];
        if ((unsigned)sg >= (unsigned)S) {
            if (status) atomicOr(status, (uint32_t)AJT_STATUS_BAD_SEG);
            continue;
        }
        atomicAdd(&denom[sg], 1.0f);
    }
}

template <int NCH, int CSIZE, bool EXT>
cudaError_t launch_rows_t(const LossParams& p, int num_sms, cudaStream_t stream) {
    auto kern = loss_rows_kernel<NCH, CSIZE, EXT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRowsSmemBytes);
    if (e != cudaSuccess) return e;
    return launch_dependent(kern, (num_sms / CSIZE) * CSIZE, kThreads, kRowsSmemBytes, stream, CSIZE, p);
}

template <int NCH, int CSIZE>
cudaError_t launch_rows(const LossParams& p, int num_sms, cudaStream_t stream) {
    return p.ext ? launch_rows_t<NCH, CSIZE, true>(p, num_sms, stream) : launch_rows_t<NCH, CSIZE, false>(p, num_sms, stream);
}

}  // namespace

extern "C" size_t ajt_loss_workspace_bytes(int64_t T, int32_t V, int32_t S) {
    (void)V;
    if (T < 0 || S < 0) return 0;
    return loss_ws_layout(T, S).total;
}

namespace {
struct LossExt {   // steps 8-9 (ajt_policy_loss_fwd_bwd_ext)
    int32_t on;
    const float* ref_logp;
    float kl_coef;
    float *k3_out, *ent_out, *ext_out;
    float clip_c;
};

int loss_call(const void* logits, const int32_t* targets, const float* old_logp, const float* adv, const uint8_t* mask,
              const int32_t* seg_ids, float eps_lo, float eps_hi, int64_t T, int32_t V, int32_t S, int64_t ld_logits,
              int32_t logits_dtype, const float* seg_denom, float inv_num_segs, float grad_scale, void* dlogits, float* loss_out,
              float* logp_out, float* stats_out, const LossExt& x, void* workspace, size_t workspace_bytes,
              ajt_stream_t stream_) {
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    if (x.on && (!x.ext_out || !(x.kl_coef >= 0.f) || !(x.clip_c >= 0.f))) return AJT_ERR_INVALID_ARG;
    if (T < 0 || V <= 0 || S <= 0 || ld_logits < V || T >= ((int64_t)1 << 31)) return AJT_ERR_INVALID_ARG;
    if (!(eps_lo >= 0.f) || !(eps_hi >= 0.f) || inv_num_segs < 0.f) return AJT_ERR_INVALID_ARG;
    if (logits_dtype != AJT_DT_BF16 && logits_dtype != AJT_DT_F32) return AJT_ERR_INVALID_ARG;
    if (!loss_out || !workspace) return AJT_ERR_INVALID_ARG;
    if (T > 0 && (!logits || !targets || !old_logp || !adv || !mask || !seg_ids || !dlogits)) return AJT_ERR_INVALID_ARG;
    if ((uintptr_t)workspace & 255) return AJT_ERR_INVALID_ARG;
    const LossWs ws = loss_ws_layout(T, S);
    if (workspace_bytes < ws.total) return AJT_ERR_WORKSPACE_TOO_SMALL;

    int dev = 0, num_sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return AJT_ERR_CUDA;
    if (cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || num_sms < 2) return AJT_ERR_CUDA;

    uint8_t* wsb = reinterpret_cast<uint8_t*>(workspace);
    LossParams p;
    p.logits = logits; p.targets = targets; p.old_logp = old_logp; p.adv = adv; p.mask = mask; p.seg_ids = seg_ids;
    p.eps_lo = eps_lo; p.eps_hi = eps_hi; p.T = T; p.V = V; p.S = S; p.ld = ld_logits; p.dtype = logits_dtype;
    p.seg_denom = seg_denom; p.inv_num_segs = inv_num_segs; p.grad_scale = grad_scale;
    p.dlogits = dlogits; p.loss_out = loss_out; p.logp_out = logp_out; p.stats_out = stats_out;
    p.ctrl = reinterpret_cast<AjtCtrl*>(wsb + ws.ctrl);
    p.tile_state = reinterpret_cast<uint64_t*>(wsb + ws.tile_state);
    p.seg_cnt = reinterpret_cast<int32_t*>(wsb + ws.seg_cnt);
    p.rec_i = reinterpret_cast<int4*>(wsb + ws.rec_i);
    p.rec_f = reinterpret_cast<float2*>(wsb + ws.rec_f);
    p.list_zero = reinterpret_cast<int32_t*>(wsb + ws.list_zero);
    p.row_val = reinterpret_cast<double*>(wsb + ws.row_val);
    p.row_kl = reinterpret_cast<double*>(wsb + ws.row_kl);
    p.row_clip = wsb + ws.row_clip;
    p.ext = x.on; p.ref_logp = x.ref_logp; p.kl_coef = x.kl_coef; p.clip_c = x.clip_c; p.k3_out = x.k3_out; p.ent_out = x.ent_out; p.ext_out = x.ext_out;
    p.rec_r = reinterpret_cast<float*>(wsb + ws.rec_r);
    p.row_k3 = reinterpret_cast<double*>(wsb + ws.row_k3);
    p.row_ent = reinterpret_cast<double*>(wsb + ws.row_ent);

    const bool aligned = (((uintptr_t)logits | (uintptr_t)dlogits) & 15) == 0 && (ld_logits % 8) == 0 && (V % 8) == 0;
    const bool fast = logits_dtype == AJT_DT_BF16 && aligned && T > 0 && V <= 2 * 16 * kChunkElems - 16;
    p.zero_rows = fast ? 1 : 0;   // the fast kernels write the per-row outputs of unmasked rows only
    if (cudaMemsetAsync(p.ctrl, 0, ws.zero_bytes, stream) != cudaSuccess) return AJT_ERR_CUDA;
    const int ntiles = (int)((T + kPrepTile - 1) / kPrepTile);
    AJT_LAUNCH(loss_prep_kernel<<<max(1, min(ntiles, num_sms)), 1024, 0, stream>>>(p, ntiles));

    cudaError_t e = cudaSuccess;
    int by_row = 0;
    if (fast && V <= 8 * kChunkElems) e = launch_rows<8, 1>(p, num_sms, stream);
    else if (fast && V <= 16 * kChunkElems) e = launch_rows<16, 1>(p, num_sms, stream);
    else if (fast) e = launch_rows<16, 2>(p, num_sms, stream);
    else if (T > 0) {
        by_row = 1;
        const int grid = num_sms * 8;
        const bool f32_regs = logits_dtype == AJT_DT_F32 && V <= 2048 && (V % 4) == 0 && (ld_logits % 4) == 0 &&
                              ((uintptr_t)logits & 15) == 0 && ((uintptr_t)dlogits & 7) == 0;
        if (f32_regs) {
            e = V <= 1024 ? launch_dependent(loss_rows_f32_regs<8>, grid, 256, 0, stream, 1, p)
                          : launch_dependent(loss_rows_f32_regs<16>, grid, 256, 0, stream, 1, p);
        } else if (logits_dtype == AJT_DT_F32) {
            if (V <= 2048) e = launch_dependent(loss_rows_generic<float, 32>, grid, 256, 0, stream, 1, p);
            else e = launch_dependent(loss_rows_generic<float, 256>, grid, 256, 0, stream, 1, p);
        } else {
            if (V <= 2048) e = launch_dependent(loss_rows_generic<__nv_bfloat16, 32>, grid, 256, 0, stream, 1, p);
            else e = launch_dependent(loss_rows_generic<__nv_bfloat16, 256>, grid, 256, 0, stream, 1, p);
        }
    }
    if (e != cudaSuccess) return AJT_ERR_CUDA;
    if (launch_dependent(loss_final_kernel, 1, 1024, 0, stream, 1, p, by_row) != cudaSuccess) return AJT_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? AJT_OK : AJT_ERR_CUDA;
}
}  // namespace

extern "C" int ajt_policy_loss_fwd_bwd(const void* logits, const int32_t* targets, const float* old_logp, const float* adv,
                                       const uint8_t* mask, const int32_t* seg_ids, float eps_lo, float eps_hi, int64_t T,
                                       int32_t V, int32_t S, int64_t ld_logits, int32_t logits_dtype, const float* seg_denom,
                                       float inv_num_segs, float grad_scale, void* dlogits, float* loss_out, float* logp_out,
                                       float* stats_out, void* workspace, size_t workspace_bytes, ajt_stream_t stream) {
    const LossExt x = {0, nullptr, 0.f, nullptr, nullptr, nullptr, 0.f};
    return loss_call(logits, targets, old_logp, adv, mask, seg_ids, eps_lo, eps_hi, T, V, S, ld_logits, logits_dtype, seg_denom,
                     inv_num_segs, grad_scale, dlogits, loss_out, logp_out, stats_out, x, workspace, workspace_bytes, stream);
}

extern "C" int ajt_policy_loss_fwd_bwd_ext(const void* logits, const int32_t* targets, const float* old_logp, const float* adv,
                                           const uint8_t* mask, const int32_t* seg_ids, float eps_lo, float eps_hi, int64_t T,
                                           int32_t V, int32_t S, int64_t ld_logits, int32_t logits_dtype, const float* seg_denom,
                                           float inv_num_segs, float grad_scale, const float* ref_logp, float kl_coef,
                                           float clip_c, void* dlogits, float* loss_out, float* logp_out, float* stats_out,
                                           float* k3_out, float* ent_out, float* ext_out, void* workspace, size_t workspace_bytes,
                                           ajt_stream_t stream) {
    const LossExt x = {1, ref_logp, kl_coef, k3_out, ent_out, ext_out, clip_c};
    return loss_call(logits, targets, old_logp, adv, mask, seg_ids, eps_lo, eps_hi, T, V, S, ld_logits, logits_dtype, seg_denom,
                     inv_num_segs, grad_scale, dlogits, loss_out, logp_out, stats_out, x, workspace, workspace_bytes, stream);
}

// ---- the loss call for callers that cannot allocate (CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc): the same kernels with their scratch in a file-scope device array instead of a caller-provided workspace.
// Every GPU that loads the library holds the array until exit.  Host code never passes the symbol itself to a kernel (in host
// code its name is a host-side stand-in, not a device address): its device address is looked up once per device with
// cudaGetSymbolAddress, that device being current.  The array keeps the last call's contents; what must start at zero (control
// block, tile states, per-segment counts) is cleared by loss_call's memset on the caller's stream as in every loss call.
constexpr size_t kStaticWsBytes = (size_t)4 << 20;   // 4 MiB: e.g. T = 40,960 rows with S = 4,096 (69 bytes per row + 4 S + 768)
static __device__ __align__(256) uint8_t g_loss_static_ws[kStaticWsBytes];
namespace {
constexpr int kStaticMaxDev = 64;
void* g_static_ws_addr[kStaticMaxDev];   // device address of g_loss_static_ws on device i, once looked up
std::mutex g_static_ws_mu;
}  // namespace

extern "C" size_t ajt_loss_static_scratch_bytes(void) { return kStaticWsBytes; }

extern "C" int ajt_policy_loss_fwd_bwd_static(const void* logits, const int32_t* targets, const float* old_logp, const float* adv,
                                              const uint8_t* mask, const int32_t* seg_ids, float eps_lo, float eps_hi, int64_t T,
                                              int32_t V, int32_t S, int64_t ld_logits, int32_t logits_dtype,
                                              const float* seg_denom, float inv_num_segs, float grad_scale, void* dlogits,
                                              float* loss_out, float* logp_out, float* stats_out, uint32_t* status_out,
                                              ajt_stream_t stream) {
    if (T < 0 || S <= 0) return AJT_ERR_INVALID_ARG;
    if (loss_ws_layout(T, S).total > kStaticWsBytes) return AJT_ERR_CAPACITY;   // beyond the static scratch: use the workspace call
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return AJT_ERR_CUDA;
    if (dev < 0 || dev >= kStaticMaxDev) return AJT_ERR_UNSUPPORTED;
    void* ws = nullptr;
    {
        std::lock_guard<std::mutex> lk(g_static_ws_mu);
        if (!g_static_ws_addr[dev]) {   // once per device, with that device current
            void* a = nullptr;
            if (cudaGetSymbolAddress(&a, g_loss_static_ws) != cudaSuccess || !a) return AJT_ERR_CUDA;
            g_static_ws_addr[dev] = a;
        }
        ws = g_static_ws_addr[dev];
    }
    const LossExt x = {0, nullptr, 0.f, nullptr, nullptr, nullptr, 0.f};
    const int rc = loss_call(logits, targets, old_logp, adv, mask, seg_ids, eps_lo, eps_hi, T, V, S, ld_logits, logits_dtype,
                             seg_denom, inv_num_segs, grad_scale, dlogits, loss_out, logp_out, stats_out, x, ws, kStaticWsBytes,
                             stream);
    if (rc != AJT_OK) return rc;
    if (status_out &&   // the status word is the first word of the scratch: handed to the caller on the same stream
        cudaMemcpyAsync(status_out, ws, sizeof(uint32_t), cudaMemcpyDeviceToDevice, reinterpret_cast<cudaStream_t>(stream)) !=
            cudaSuccess)
        return AJT_ERR_CUDA;
    return AJT_OK;
}

extern "C" int ajt_segment_counts(const uint8_t* mask, const int32_t* seg_ids, int64_t T, int32_t S, int32_t accumulate,
                                  float* seg_denom, uint32_t* status_bits, ajt_stream_t stream_) {
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    if (T < 0 || S <= 0 || !seg_denom) return AJT_ERR_INVALID_ARG;
    if (T > 0 && (!mask || !seg_ids)) return AJT_ERR_INVALID_ARG;
    int dev = 0, num_sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return AJT_ERR_CUDA;
    if (cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || num_sms < 1) return AJT_ERR_CUDA;
    if (!accumulate) {
        if (cudaMemsetAsync(seg_denom, 0, (size_t)S * sizeof(float), stream) != cudaSuccess) return AJT_ERR_CUDA;
        if (status_bits && cudaMemsetAsync(status_bits, 0, sizeof(uint32_t), stream) != cudaSuccess) return AJT_ERR_CUDA;
    }
    if (T == 0) return AJT_OK;
    const int64_t want = (T + 255) / 256;
    const int grid = (int)(want < (int64_t)num_sms * 8 ? want : (int64_t)num_sms * 8);
    AJT_LAUNCH(segment_counts_kernel<<<grid, 256, 0, stream>>>(mask, seg_ids, T, S, seg_denom, status_bits));
    return cudaGetLastError() == cudaSuccess ? AJT_OK : AJT_ERR_CUDA;
}
