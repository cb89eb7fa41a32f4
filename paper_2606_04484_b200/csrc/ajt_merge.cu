// Stage (a): timeline merging (Algorithm 1) on flat token streams, sm_100a.
//
// Definition: DESIGN.md "O-M".  Pipeline (rows M1-M7 of the scope table):
//   K1 merge_group_kernel    M1  stable grouping of timelines by traj_id: LSD radix sort of (traj_id - min, index),
//                                group ids, rank in group, entry / hash-segment offsets (prefix scans)
//   K2 merge_hash_kernel     M2  warp-cooperative prefix-hash scan, 128-bit loads.  The hash of the first p tokens of
//                                timeline i is F_i(p) = sum_{q<p} mix(x_q) B^(q+3) mod 2^64: a sum, hence a monoid, so
//                                every lane keeps its own partial and lanes are only combined (shuffles) where a key
//                                is emitted: at each length L_j of an earlier same-group timeline (probe key) and at
//                                L_i itself (full key)
//      merge_keys_kernel         per-timeline prefix over hash segments; final (hash, len) keys and 32-bit digests
//   K3 merge_select_kernel   M3  segmented radix sort: one CTA per group sorts its keys by digest (LSD, 8-bit digits,
//                                stable warp-match ranking) in shared memory (global ping-pong for huge groups)
//   K4   (same kernel)       M4  per full key: walk its equal-key run, pick the extender by the owner rule
//   K6 merge_compact_kernel  M6  survivors in original order, scans -> merged_offsets/origin/traj, owner, member lists
//   K5/K7 merge_scatter_kernel M5+M7  fused: every merged sequence is streamed once; each absorbed member is compared
//                                token-by-token against its owner (exact verification) while tokens / mask-OR / src /
//                                old_logp are written.  A mismatch (a hash collision) raises ctrl->collision.
//   Repair (enqueued always, exits at once unless ctrl->collision): K4 with exact comparison of every candidate it
//   accepts, then K6 and K7 again.  Hash collisions can therefore never change the result.
#include "ajt_common.cuh"

namespace {

using namespace ajt;

constexpr int kHSeg = 2048;        // hash-scan window: 2048 tokens = 16 steps x 32 lanes x 4 tokens
constexpr int kTile = 1024;        // scatter tile (positions per warp-task)
constexpr uint64_t kB = 0x9E3779B97F4A7C15ull;       // odd multiplier of the polynomial hash
constexpr uint64_t kMixAdd = 0x632BE59BD9B4E019ull;  // so that token 0 is not the additive identity
constexpr uint32_t kFatal = AJT_STATUS_BAD_OFFSETS | AJT_STATUS_ZERO_LEN | AJT_STATUS_PROBE_CAPACITY;
constexpr int kSelThreads = 256;
constexpr int kSelSmemKeys = 2048;  // groups with more keys than this sort through global memory

struct MergeParams {
    const int32_t* tokens;
    const int64_t* offsets;
    const int32_t* traj_ids;
    const int32_t* resp_start;
    const uint8_t* mask_in;
    const float* old_logp_in;
    int32_t n;
    int64_t N;
    int32_t owner_rule;
    uint32_t flags;
    int32_t* merged_tokens;
    uint8_t* merged_mask;
    int32_t* merged_src;
    float* merged_old_logp;
    int64_t* merged_offsets;
    int32_t* merged_origin;
    int32_t* merged_traj;
    int32_t* owner;
    int64_t* counts;
    // workspace
    AjtCtrl* ctrl;
    uint32_t* skey[2];     // [n] radix ping-pong keys (traj_id - min)
    uint32_t* sval[2];     // [n] radix ping-pong values (timeline index)
    int32_t* perm;         // [n] sorted position -> timeline index
    int32_t* gid_sorted;   // [n] group id of each sorted position
    int32_t* grp_start;    // [n+1] first sorted position of each group
    int32_t* grp_ent;      // [n+1] first entry of each group
    int32_t* t_rank;       // [n] rank of timeline i inside its group (input order)
    int32_t* t_gid;        // [n]
    int32_t* t_entbase;    // [n] first entry of timeline i: entries (i, a), a = 0..rank
    int32_t* seg_base;     // [n+1] first hash segment of timeline i
    uint64_t* seg_part;    // [nseg_cap] per-segment partial sums, then exclusive prefixes per timeline
    uint64_t* ent_hash;    // [E_cap]
    int32_t* ent_len;      // [E_cap] prefix length of the key, -1 if invalid (L_a > L_i)
    uint32_t* ent_dig;     // [E_cap] 32-bit digest of (hash, len)
    uint32_t* ent_idx;     // [E_cap] sorted order: local entry index inside the group
    uint32_t* tmp_dig;     // [E_cap]
    uint32_t* tmp_idx;     // [E_cap]
    uint8_t* absorbed;     // [n]
    int32_t* owner_tl;     // [n] owning timeline (itself for survivors)
    int32_t* midx;         // [n] merged index of survivors, -1 otherwise
    int32_t* mem_cnt;      // [n] number of absorbed members owned by timeline i
    int32_t* mem_off;      // [n+1] by merged index
    int32_t* mem_cur;      // [n] fill cursors by merged index
    int32_t* mem_list;     // [n] absorbed members, grouped by owner
    int32_t* tile_base;    // [n+1] by merged index
    int32_t E_cap;
    int32_t nseg_cap;
    int32_t mis;           // (address of tokens / 4) mod 4: element misalignment of the token array vs 16 bytes
};

struct MergeWs {
    size_t ctrl, skey0, skey1, sval0, sval1, gid_sorted, grp_start, grp_ent, t_rank, t_gid, t_entbase, seg_base, seg_part,
        absorbed, owner_tl, midx, mem_cnt, mem_off, mem_cur, mem_list, tile_base, ent, fixed_total;
};
__host__ inline size_t a256(size_t x) { return (x + 255) & ~(size_t)255; }
__host__ inline int32_t nseg_capacity(int32_t n, int64_t N) { return (int32_t)(N / kHSeg + 2 * (int64_t)n + 2); }

__host__ MergeWs merge_ws_layout(int32_t n, int64_t N) {
    MergeWs w;
    size_t o = 0;
    const size_t n4 = a256(((size_t)n + 1) * 4);
    w.ctrl = o; o += 256;
    w.skey0 = o; o += n4; w.skey1 = o; o += n4; w.sval0 = o; o += n4; w.sval1 = o; o += n4;
    w.gid_sorted = o; o += n4; w.grp_start = o; o += n4; w.grp_ent = o; o += n4;
    w.t_rank = o; o += n4; w.t_gid = o; o += n4; w.t_entbase = o; o += n4; w.seg_base = o; o += n4;
    w.seg_part = o; o += a256((size_t)nseg_capacity(n, N) * 8);
    w.absorbed = o; o += a256((size_t)n + 1);
    w.owner_tl = o; o += n4; w.midx = o; o += n4; w.mem_cnt = o; o += n4; w.mem_off = o; o += n4; w.mem_cur = o; o += n4;
    w.mem_list = o; o += n4; w.tile_base = o; o += n4;
    w.ent = o;
    w.fixed_total = o;
    return w;
}
constexpr size_t kEntBytes = 8 + 4 + 4 + 4 + 4 + 4;  // hash, len, dig, idx, tmp_dig, tmp_idx  (< 32, header promises 32)

__device__ __forceinline__ bool fatal(const MergeParams& p) { return (p.ctrl->status & kFatal) != 0; }

__device__ __forceinline__ uint64_t pow64(uint64_t b, uint64_t e) {
    uint64_t r = 1;
    while (e) {
        if (e & 1) r *= b;
        b *= b;
        e >>= 1;
    }
    return r;
}
__device__ __forceinline__ uint64_t mix_tok(int32_t x) { return (uint64_t)(uint32_t)x + kMixAdd; }
__device__ __forceinline__ uint32_t digest32(uint64_t h, int32_t len) {
    uint64_t z = h ^ ((uint64_t)(uint32_t)len * 0xD6E8FEB86659FD93ull);
    z ^= z >> 32;
    z *= 0xD6E8FEB86659FD93ull;
    z ^= z >> 32;
    return (uint32_t)z;
}
__device__ __forceinline__ uint64_t warp_sum_u64(uint64_t v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ---------------------------------------------------------------------------------------- block-level building blocks

// Exclusive scan of f(i), i in [0,n), by one CTA of NT threads; g(i, exclusive_prefix, value) consumes it.  Returns the
// total to every thread.  One __syncthreads per tile of NT (double-buffered warp totals).
template <int NT, class F, class G>
__device__ __forceinline__ int64_t block_scan(int n, F f, G g, int64_t (*s_w)[NT / 32]) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    int64_t base = 0;
    int buf = 0;
    for (int i0 = 0; i0 < n; i0 += NT, buf ^= 1) {
        const int i = i0 + tid;
        const int64_t v = i < n ? (int64_t)f(i) : 0;
        int64_t inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int64_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) s_w[buf][warp] = inc;
        __syncthreads();
        int64_t pre = 0, tot = 0;
#pragma unroll
        for (int w = 0; w < NT / 32; ++w) {
            const int64_t c = s_w[buf][w];
            if (w < warp) pre += c;
            tot += c;
        }
        if (i < n) g(i, base + pre + inc - v, v);
        base += tot;
    }
    __syncthreads();
    return base;
}

template <int NW>
struct RadixScratch {
    uint32_t cnt[NW][256];
    uint32_t off[256];
};

// One stable LSD pass (8-bit digit at `shift`) of (key, value) pairs by one CTA of NW warps.  Ranking inside a tile of
// NW*32 keys: lanes with equal digits find each other with match.any; the lowest lane of each peer set posts the set size
// in cnt[warp][digit]; one thread per digit turns the NW counts into running offsets; position = that + rank in peer set.
template <int NW>
__device__ void radix_pass(const uint32_t* kin, const uint32_t* vin, uint32_t* kout, uint32_t* vout, int n, int shift,
                           RadixScratch<NW>& sc) {
    constexpr int NT = NW * 32;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int d = tid; d < 256; d += NT) sc.off[d] = 0;
    for (int x = tid; x < NW * 256; x += NT) (&sc.cnt[0][0])[x] = 0;
    __syncthreads();
    for (int i = tid; i < n; i += NT) atomicAdd(&sc.off[(kin[i] >> shift) & 255u], 1u);
    __syncthreads();
    if (warp == 0) {  // exclusive scan of the 256-bin histogram: 8 bins per lane
        uint32_t loc[8], s = 0;
#pragma unroll
        for (int j = 0; j < 8; ++j) { loc[j] = sc.off[lane * 8 + j]; s += loc[j]; }
        uint32_t inc = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        uint32_t run = inc - s;
#pragma unroll
        for (int j = 0; j < 8; ++j) { sc.off[lane * 8 + j] = run; run += loc[j]; }
    }
    __syncthreads();
    for (int base = 0; base < n; base += NT) {
        const int i = base + tid;
        const bool valid = i < n;
        const uint32_t key = valid ? kin[i] : 0u;
        const uint32_t val = valid ? vin[i] : 0u;
        const uint32_t d = (key >> shift) & 255u;
        const unsigned peers = __match_any_sync(0xffffffffu, valid ? d : (0x100u | (uint32_t)lane));
        const int rk = __popc(peers & ((1u << lane) - 1u));
        if (valid && rk == 0) sc.cnt[warp][d] = (uint32_t)__popc(peers);
        __syncthreads();
        for (int d2 = tid; d2 < 256; d2 += NT) {
            uint32_t run = sc.off[d2];
#pragma unroll 8
            for (int w = 0; w < NW; ++w) {
                const uint32_t c = sc.cnt[w][d2];
                if (c) { sc.cnt[w][d2] = run; run += c; }
            }
            sc.off[d2] = run;
        }
        __syncthreads();
        if (valid) {
            const uint32_t pos = sc.cnt[warp][d] + (uint32_t)rk;
            kout[pos] = key;
            vout[pos] = val;
        }
        __syncthreads();
        if (valid && rk == 0) sc.cnt[warp][d] = 0;  // leave the table clean for the next tile
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------- K1: group (M1)

__global__ void __launch_bounds__(1024) merge_group_kernel(const MergeParams p) {
    __shared__ RadixScratch<32> sc;
    __shared__ int64_t s_w[2][32];
    __shared__ int s_min, s_max;
    __shared__ uint32_t s_bad;
    const int tid = threadIdx.x, n = p.n;
    if (tid == 0) { s_min = INT32_MAX; s_max = INT32_MIN; s_bad = 0; }
    __syncthreads();
    // validate offsets; min / max traj id
    int lmin = INT32_MAX, lmax = INT32_MIN;
    uint32_t bad = 0;
    for (int i = tid; i < n; i += 1024) {
        const int64_t a = p.offsets[i], b = p.offsets[i + 1];
        if (b < a || b - a > (int64_t)INT32_MAX) bad |= AJT_STATUS_BAD_OFFSETS;
        else if (b == a) bad |= AJT_STATUS_ZERO_LEN;
        const int t = p.traj_ids[i];
        lmin = min(lmin, t);
        lmax = max(lmax, t);
    }
    if (tid == 0 && (p.offsets[0] != 0 || p.offsets[n] != p.N)) bad |= AJT_STATUS_BAD_OFFSETS;
    if (bad) atomicOr(&s_bad, bad);
    if (lmin != INT32_MAX) { atomicMin(&s_min, lmin); atomicMax(&s_max, lmax); }
    __syncthreads();
    if (s_bad) {
        if (tid == 0) atomicOr(&p.ctrl->status, s_bad);
        return;
    }
    const int tmin = s_min;
    const uint32_t range = n ? (uint32_t)s_max - (uint32_t)tmin : 0u;
    for (int i = tid; i < n; i += 1024) {
        p.skey[0][i] = (uint32_t)p.traj_ids[i] - (uint32_t)tmin;
        p.sval[0][i] = (uint32_t)i;
    }
    __syncthreads();
    int cur = 0;
    for (int shift = 0; shift < 32 && (range >> shift) != 0; shift += 8) {
        radix_pass<32>(p.skey[cur], p.sval[cur], p.skey[cur ^ 1], p.sval[cur ^ 1], n, shift, sc);
        cur ^= 1;
        __syncthreads();
    }
    const uint32_t* key = p.skey[cur];
    const uint32_t* val = p.sval[cur];
    // group ids and group starts
    const int G = (int)block_scan<1024>(
        n, [&](int pos) { return (pos == 0 || key[pos] != key[pos - 1]) ? 1 : 0; },
        [&](int pos, int64_t ex, int64_t v) {
            const int g = (int)(ex + v) - 1;
            p.gid_sorted[pos] = g;
            p.perm[pos] = (int32_t)val[pos];
            if (v) p.grp_start[g] = pos;
        },
        s_w);
    if (tid == 0) p.grp_start[G] = n;
    __syncthreads();
    // rank in group; entries (i, a), a = 0..rank  ->  rank+1 entries per timeline
    const int64_t E = block_scan<1024>(
        n, [&](int pos) { return pos - p.grp_start[p.gid_sorted[pos]] + 1; },
        [&](int pos, int64_t ex, int64_t v) {
            const int i = p.perm[pos], g = p.gid_sorted[pos];
            p.t_rank[i] = (int)v - 1;
            p.t_gid[i] = g;
            p.t_entbase[i] = (int32_t)ex;
            if (v == 1) p.grp_ent[g] = (int32_t)ex;
        },
        s_w);
    // hash segments: aligned windows of kHSeg tokens intersected with each timeline (skipped for singleton groups)
    const int64_t nseg = block_scan<1024>(
        n,
        [&](int i) {
            const int g = p.t_gid[i];
            if (p.grp_start[g + 1] - p.grp_start[g] < 2) return 0;
            const int64_t a = p.offsets[i] + p.mis, b = p.offsets[i + 1] - 1 + p.mis;
            return (int)(b / kHSeg - a / kHSeg + 1);
        },
        [&](int i, int64_t ex, int64_t) { p.seg_base[i] = (int32_t)ex; }, s_w);
    if (tid == 0) {
        p.seg_base[n] = (int32_t)nseg;
        p.grp_ent[G] = (int32_t)min(E, (int64_t)INT32_MAX);
        p.ctrl->n_groups = G;
        p.ctrl->n_entries = (int32_t)min(E, (int64_t)INT32_MAX);
        p.ctrl->n_hash_segs = (int32_t)nseg;
        if (E > (int64_t)p.E_cap || nseg > (int64_t)p.nseg_cap) atomicOr(&p.ctrl->status, (uint32_t)AJT_STATUS_PROBE_CAPACITY);
    }
}

// ---------------------------------------------------------------------------------------- K2: prefix-hash scan (M2)

__global__ void __launch_bounds__(256) merge_hash_kernel(const MergeParams p) {
    if (fatal(p)) return;
    const int lane = threadIdx.x & 31;
    const int wglobal = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    const int nseg = p.ctrl->n_hash_segs, n = p.n;
    const uint64_t B2 = kB * kB, B3 = B2 * kB, B128 = pow64(kB, 128);
    for (int sidx = wglobal; sidx < nseg; sidx += nwarps) {
        // timeline of this segment: last i with seg_base[i] <= sidx
        int lo = 0, hi = n;
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (p.seg_base[mid] <= sidx) lo = mid; else hi = mid;
        }
        const int i = lo;
        const int64_t off = p.offsets[i];
        const int Li = (int)(p.offsets[i + 1] - off);
        const int64_t w = (off + p.mis) / kHSeg + (sidx - p.seg_base[i]);   // window index (virtual element space)
        const int64_t win0 = w * kHSeg - p.mis - off;                        // timeline position of the window's first slot
        const int g = p.t_gid[i], rank = p.t_rank[i];
        const int32_t* gl = p.perm + p.grp_start[g];
        const int ebase = p.t_entbase[i];
        // which 128-token steps of this window hold the end of a requested prefix (L_a of an earlier member, or L_i)
        uint32_t stepmask = 0;
        for (int a0 = 0; a0 <= rank; a0 += 32) {
            const int a = a0 + lane;
            if (a <= rank) {
                const int j = gl[a];
                const int64_t Lp = p.offsets[j + 1] - p.offsets[j];
                const int64_t rel = Lp - 1 - win0;
                if (Lp <= Li && rel >= 0 && rel < kHSeg) stepmask |= 1u << (int)(rel >> 7);
            }
        }
        stepmask = __reduce_or_sync(0xffffffffu, stepmask);

        // per-lane weight B^(q+3) of its first token slot, from the first step where q + 3 >= 0
        const int64_t q0 = win0 + lane * 4;
        const int s0 = q0 + 3 >= 0 ? 0 : (int)((-3 - q0 + 127) >> 7);
        uint64_t pw = pow64(kB, (uint64_t)(q0 + 128 * (int64_t)s0 + 3));
        uint64_t acc = 0;
        const int32_t* tok = p.tokens;
#pragma unroll 4
        for (int s = 0; s < kHSeg / 128; ++s) {
            if (win0 + 128 * (int64_t)s >= Li) break;  // warp-uniform: the whole step lies beyond the timeline
            const int64_t q = q0 + 128 * (int64_t)s;   // position of this lane's first slot
            const int64_t e = off + q;                  // element index, 16-byte aligned address
            int4 x = make_int4(0, 0, 0, 0);
            if (q + 3 >= 0 && q < Li) {
                if (e >= 0 && e + 3 < p.N) x = __ldg(reinterpret_cast<const int4*>(tok + e));
                else {
                    if (e >= 0 && e < p.N) x.x = tok[e];
                    if (e + 1 >= 0 && e + 1 < p.N) x.y = tok[e + 1];
                    if (e + 2 >= 0 && e + 2 < p.N) x.z = tok[e + 2];
                    if (e + 3 >= 0 && e + 3 < p.N) x.w = tok[e + 3];
                }
            }
            if (s > s0) pw *= B128;
            const bool v0 = q >= 0 && q < Li, v1 = q + 1 >= 0 && q + 1 < Li, v2 = q + 2 >= 0 && q + 2 < Li,
                       v3 = q + 3 >= 0 && q + 3 < Li;
            const uint64_t m0 = v0 ? mix_tok(x.x) : 0, m1 = v1 ? mix_tok(x.y) : 0, m2 = v2 ? mix_tok(x.z) : 0,
                           m3 = v3 ? mix_tok(x.w) : 0;
            if (stepmask & (1u << s)) {
                // emit every key whose prefix ends inside this step
                for (int a0 = 0; a0 <= rank; a0 += 32) {
                    const int a = a0 + lane;
                    int64_t Lp = -1;
                    if (a <= rank) {
                        const int j = gl[a];
                        Lp = p.offsets[j + 1] - p.offsets[j];
                        const int64_t rel = Lp - 1 - win0;
                        if (!(Lp <= Li && rel >= 0 && (rel >> 7) == s)) Lp = -1;
                    }
                    unsigned hits = __ballot_sync(0xffffffffu, Lp >= 0);
                    while (hits) {
                        const int src = __ffs(hits) - 1;
                        hits &= hits - 1;
                        const int64_t P = __shfl_sync(0xffffffffu, Lp, src);
                        uint64_t part = 0;
                        if (s >= s0) {
                            const uint64_t t0 = q < P ? m0 : 0, t1 = q + 1 < P ? m1 : 0, t2 = q + 2 < P ? m2 : 0,
                                           t3 = q + 3 < P ? m3 : 0;
                            part = (t0 + t1 * kB + t2 * B2 + t3 * B3) * pw;
                        }
                        const uint64_t tot = warp_sum_u64(acc + part);
                        if (lane == 0) p.ent_hash[ebase + a0 + src] = tot;
                    }
                }
            }
            if (s >= s0) acc += (m0 + m1 * kB + m2 * B2 + m3 * B3) * pw;
        }
        const uint64_t tot = warp_sum_u64(acc);
        if (lane == 0) p.seg_part[sidx] = tot;
    }
}

// per timeline: exclusive prefix over its hash segments, then the final keys of its entries (i, a), a = 0..rank
__global__ void __launch_bounds__(256) merge_keys_kernel(const MergeParams p) {
    if (fatal(p)) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.n) return;
    const int sb = p.seg_base[i], se = p.seg_base[i + 1];
    uint64_t run = 0;
    for (int s = sb; s < se; ++s) {
        const uint64_t v = p.seg_part[s];
        p.seg_part[s] = run;
        run += v;
    }
    if (se == sb) return;  // singleton group: no keys needed
    const int64_t off = p.offsets[i];
    const int Li = (int)(p.offsets[i + 1] - off);
    const int64_t w_first = (off + p.mis) / kHSeg;
    const int g = p.t_gid[i], rank = p.t_rank[i];
    const int32_t* gl = p.perm + p.grp_start[g];
    const int ebase = p.t_entbase[i];
    const bool weak = (p.flags & AJT_MERGE_WEAK_HASH) != 0;
    for (int a = 0; a <= rank; ++a) {
        const int j = gl[a];
        const int64_t Lp = p.offsets[j + 1] - p.offsets[j];
        const int e = ebase + a;
        if (Lp > Li) {
            p.ent_len[e] = -1;
            p.ent_hash[e] = 0;
            continue;
        }
        const int64_t widx = (off + Lp - 1 + p.mis) / kHSeg - w_first;
        uint64_t h = p.seg_part[sb + widx] + p.ent_hash[e];
        if (weak) h &= 0xFull;
        p.ent_hash[e] = h;
        p.ent_len[e] = (int32_t)Lp;
    }
}

// ---------------------------------------------------------------------------------------- K3 + K4: sort + select (M3, M4)

__device__ bool tokens_extend(const MergeParams& p, int i, int j) {  // exact: tokens_i[0:L_j] == tokens_j, L_i >= L_j
    const int64_t oi = p.offsets[i], oj = p.offsets[j];
    const int64_t Li = p.offsets[i + 1] - oi, Lj = p.offsets[j + 1] - oj;
    if (Li < Lj) return false;
    for (int64_t q = 0; q < Lj; ++q)
        if (p.tokens[oi + q] != p.tokens[oj + q]) return false;
    return true;
}

// local entry index -> rank of the probing timeline: entries of rank b occupy [b(b+1)/2, b(b+1)/2 + b]
__device__ __forceinline__ int rank_of_local(uint32_t l) {
    int b = (int)((sqrtf(8.f * (float)l + 1.f) - 1.f) * 0.5f);
    while ((uint64_t)(b + 1) * (uint64_t)(b + 2) / 2 <= l) ++b;
    while ((uint64_t)b * (uint64_t)(b + 1) / 2 > l) --b;
    return b;
}

// mode 0: trust hash-equal candidates (verified later by the scatter pass); mode 1: repair — runs only if the scatter pass
// found a collision, and accepts a candidate only after comparing tokens exactly.
__global__ void __launch_bounds__(kSelThreads) merge_select_kernel(const MergeParams p, int mode) {
    if (fatal(p)) return;
    if (mode == 1 && p.ctrl->collision == 0) return;
    __shared__ RadixScratch<kSelThreads / 32> sc;
    __shared__ uint32_t s_key[2][kSelSmemKeys];
    __shared__ uint32_t s_val[2][kSelSmemKeys];
    const int tid = threadIdx.x;
    const int G = p.ctrl->n_groups;
    for (int g = blockIdx.x; g < G; g += gridDim.x) {
        const int gs = p.grp_start[g], k = p.grp_start[g + 1] - gs;
        const int32_t* gl = p.perm + gs;
        if (k < 2) {
            if (tid == 0) { p.absorbed[gl[0]] = 0; p.owner_tl[gl[0]] = gl[0]; }
            continue;
        }
        const int eb = p.grp_ent[g], c = p.grp_ent[g + 1] - eb;
        // ---- M3: stable LSD radix sort of the group's keys by digest
        const uint32_t* sk;
        const uint32_t* sv;
        if (c <= kSelSmemKeys) {
            for (int x = tid; x < c; x += kSelThreads) {
                const int32_t L = p.ent_len[eb + x];
                s_key[0][x] = L < 0 ? 0xFFFFFFFFu : digest32(p.ent_hash[eb + x], L);
                s_val[0][x] = (uint32_t)x;
            }
            __syncthreads();
            int cur = 0;
            for (int shift = 0; shift < 32; shift += 8) {
                radix_pass<kSelThreads / 32>(s_key[cur], s_val[cur], s_key[cur ^ 1], s_val[cur ^ 1], c, shift, sc);
                cur ^= 1;
            }
            sk = s_key[cur];
            sv = s_val[cur];
        } else {
            uint32_t* kk[2] = {p.ent_idx + eb, p.tmp_idx + eb};
            uint32_t* dd[2] = {p.ent_dig + eb, p.tmp_dig + eb};
            for (int x = tid; x < c; x += kSelThreads) {
                const int32_t L = p.ent_len[eb + x];
                dd[0][x] = L < 0 ? 0xFFFFFFFFu : digest32(p.ent_hash[eb + x], L);
                kk[0][x] = (uint32_t)x;
            }
            __syncthreads();
            int cur = 0;
            for (int shift = 0; shift < 32; shift += 8) {
                radix_pass<kSelThreads / 32>(dd[cur], kk[cur], dd[cur ^ 1], kk[cur ^ 1], c, shift, sc);
                cur ^= 1;
                __syncthreads();
            }
            sk = dd[cur];   // after 4 passes cur == 0: digests are back in ent_dig (sorted), order in ent_idx
            sv = kk[cur];
        }
        __syncthreads();
        // ---- M4: survivors and the Algorithm-1 owner (latest extender)
        for (int b = tid; b < k; b += kSelThreads) {
            const int j = gl[b];
            const int ef = p.t_entbase[j] + b;          // full key of j
            const uint64_t H = p.ent_hash[ef];
            const int32_t L = p.ent_len[ef];
            const uint32_t dg = digest32(H, L);
            int lo = 0, hi = c;                          // lower bound of dg in the sorted digests
            while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if (sk[mid] < dg) lo = mid + 1; else hi = mid;
            }
            int best = -1;                               // max rank of an extender
            for (int x = lo; x < c && sk[x] == dg; ++x) {
                const uint32_t le = sv[x];
                const int rb = rank_of_local(le);
                if (rb <= b || rb <= best) continue;
                if (p.ent_len[eb + le] != L || p.ent_hash[eb + le] != H) continue;
                if (mode == 1 && !tokens_extend(p, gl[rb], j)) continue;
                best = rb;
            }
            p.absorbed[j] = best >= 0;
            p.owner_tl[j] = best >= 0 ? gl[best] : j;
        }
        __syncthreads();
        if (p.owner_rule == AJT_OWNER_LONGEST) {
            // the longest SURVIVING extender, then the lowest index (BASELINE.json north_star; reading M-3)
            for (int b = tid; b < k; b += kSelThreads) {
                const int j = gl[b];
                if (!p.absorbed[j]) continue;
                const int ef = p.t_entbase[j] + b;
                const uint64_t H = p.ent_hash[ef];
                const int32_t L = p.ent_len[ef];
                const uint32_t dg = digest32(H, L);
                int lo = 0, hi = c;
                while (lo < hi) {
                    const int mid = (lo + hi) >> 1;
                    if (sk[mid] < dg) lo = mid + 1; else hi = mid;
                }
                const int paper_rb = p.t_rank[p.owner_tl[j]];   // a surviving, (to be) verified extender: the fallback
                int best = paper_rb;
                int64_t bestL = p.offsets[gl[best] + 1] - p.offsets[gl[best]];
                for (int x = lo; x < c && sk[x] == dg; ++x) {
                    const uint32_t le = sv[x];
                    const int rb = rank_of_local(le);
                    if (rb <= b || rb == best) continue;
                    if (p.ent_len[eb + le] != L || p.ent_hash[eb + le] != H) continue;
                    const int i = gl[rb];
                    if (p.absorbed[i]) continue;
                    const int64_t Li = p.offsets[i + 1] - p.offsets[i];
                    if (!(Li > bestL || (Li == bestL && rb < best))) continue;
                    if (mode == 1 && !tokens_extend(p, i, j)) continue;
                    best = rb;
                    bestL = Li;
                }
                p.mem_cur[j] = gl[best];   // staged: owner_tl is still being read by other threads
            }
            __syncthreads();
            for (int b = tid; b < k; b += kSelThreads) {
                const int j = gl[b];
                if (p.absorbed[j]) p.owner_tl[j] = p.mem_cur[j];
            }
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------- K6: compact (M6)

__global__ void __launch_bounds__(1024) merge_compact_kernel(const MergeParams p, int mode) {
    if (fatal(p)) return;
    if (mode == 1 && p.ctrl->collision == 0) return;
    __shared__ int64_t s_w[2][32];
    const int tid = threadIdx.x, n = p.n;
    for (int i = tid; i < n; i += 1024) p.mem_cnt[i] = 0;
    __syncthreads();
    const int M = (int)block_scan<1024>(
        n, [&](int i) { return p.absorbed[i] ? 0 : 1; },
        [&](int i, int64_t ex, int64_t v) {
            p.midx[i] = v ? (int)ex : -1;
            if (v) { p.merged_origin[ex] = i; p.merged_traj[ex] = p.traj_ids[i]; }
            else atomicAdd(&p.mem_cnt[p.owner_tl[i]], 1);
        },
        s_w);
    const int64_t Nout = block_scan<1024>(
        M, [&](int m) { const int s = p.merged_origin[m]; return p.offsets[s + 1] - p.offsets[s]; },
        [&](int m, int64_t ex, int64_t) { p.merged_offsets[m] = ex; }, s_w);
    const int64_t ntiles = block_scan<1024>(
        M, [&](int m) { const int s = p.merged_origin[m]; return (p.offsets[s + 1] - p.offsets[s] + kTile - 1) / kTile; },
        [&](int m, int64_t ex, int64_t) { p.tile_base[m] = (int32_t)ex; }, s_w);
    block_scan<1024>(
        M, [&](int m) { return p.mem_cnt[p.merged_origin[m]]; },
        [&](int m, int64_t ex, int64_t) { p.mem_off[m] = (int32_t)ex; p.mem_cur[m] = (int32_t)ex; }, s_w);
    __syncthreads();
    for (int i = tid; i < n; i += 1024) {
        const int m = p.midx[p.owner_tl[i]];
        p.owner[i] = m;
        if (p.absorbed[i]) p.mem_list[atomicAdd(&p.mem_cur[m], 1)] = i;
    }
    if (tid == 0) {
        p.merged_offsets[M] = Nout;
        p.tile_base[M] = (int32_t)ntiles;
        p.mem_off[M] = n - M;
        p.counts[0] = M;
        p.counts[1] = Nout;
        p.ctrl->M = M;
        p.ctrl->N_out = Nout;
        p.ctrl->n_tiles = (int32_t)ntiles;
        if (mode == 1) {
            p.ctrl->collision = 2;   // repair in progress: the scatter pass must not find another mismatch
            atomicOr(&p.ctrl->status, (uint32_t)AJT_STATUS_HASH_COLLISION);
        }
    }
}

// ---------------------------------------------------------------------------------------- K5 + K7: verify + scatter (M5, M7)

__global__ void __launch_bounds__(256) merge_scatter_kernel(const MergeParams p, int mode) {
    if (fatal(p)) return;
    if (mode == 1 && p.ctrl->collision != 2) return;
    const int lane = threadIdx.x & 31;
    const int wglobal = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    const int ntiles = p.ctrl->n_tiles, M = p.ctrl->M;
    bool mismatch = false;
    for (int t = wglobal; t < ntiles; t += nwarps) {
        int lo = 0, hi = M;   // merged sequence of this tile: last m with tile_base[m] <= t
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (p.tile_base[mid] <= t) lo = mid; else hi = mid;
        }
        const int m = lo;
        const int s = p.merged_origin[m];
        const int64_t so = p.offsets[s];
        const int Ls = (int)(p.offsets[s + 1] - so);
        const int64_t mo = p.merged_offsets[m];
        const int p0 = (t - p.tile_base[m]) * kTile, p1 = min(Ls, p0 + kTile);
        const int mb = p.mem_off[m], me = p.mem_off[m + 1];
        const int rs_s = p.resp_start ? p.resp_start[s] : 0;
        for (int q = p0 + lane; q < p1; q += 32) {
            const int32_t x = p.tokens[so + q];
            int src = -1;
            if (p.mask_in ? (p.mask_in[so + q] != 0) : (q >= rs_s)) src = s;
            for (int u = mb; u < me; ++u) {
                const int j = p.mem_list[u];
                const int64_t jo = p.offsets[j];
                const int Lj = (int)(p.offsets[j + 1] - jo);
                if (q < Lj) {
                    if (p.tokens[jo + q] != x) mismatch = true;     // exact verification (M5)
                    const bool mk = p.mask_in ? (p.mask_in[jo + q] != 0) : (q >= p.resp_start[j]);
                    if (mk) src = max(src, j);
                }
            }
            p.merged_tokens[mo + q] = x;
            p.merged_mask[mo + q] = src >= 0;
            p.merged_src[mo + q] = src;
            if (p.merged_old_logp) p.merged_old_logp[mo + q] = src >= 0 ? p.old_logp_in[p.offsets[src] + q] : 0.f;
        }
    }
    if (__any_sync(0xffffffffu, mismatch) && lane == 0) {
        if (mode == 0) atomicExch(&p.ctrl->collision, 1);
        else atomicOr(&p.ctrl->status, (uint32_t)AJT_STATUS_INTERNAL);
    }
}

}  // namespace

extern "C" size_t ajt_merge_workspace_bytes(int32_t n, int64_t n_tokens) {
    if (n < 0 || n_tokens < 0) return 0;
    return merge_ws_layout(n, n_tokens).fixed_total + a256(((size_t)64 * (size_t)n + 4096) * 32);
}

extern "C" int ajt_merge_timelines(const int32_t* tokens, const int64_t* offsets, const int32_t* traj_ids,
                                   const int32_t* resp_start, const uint8_t* mask_in, const float* old_logp_in, int32_t n,
                                   int64_t n_tokens, int32_t owner_rule, uint32_t flags, int32_t* merged_tokens,
                                   uint8_t* merged_mask, int32_t* merged_src, float* merged_old_logp, int64_t* merged_offsets,
                                   int32_t* merged_origin, int32_t* merged_traj, int32_t* owner, int64_t* counts,
                                   void* workspace, size_t workspace_bytes, ajt_stream_t stream_) {
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    if (n < 0 || n_tokens < 0) return AJT_ERR_INVALID_ARG;
    if (owner_rule != AJT_OWNER_LONGEST && owner_rule != AJT_OWNER_PAPER) return AJT_ERR_INVALID_ARG;
    if (!offsets || !counts || !merged_offsets || !workspace) return AJT_ERR_INVALID_ARG;
    if (n > 0 && (!tokens || !traj_ids || (!resp_start && !mask_in) || !merged_tokens || !merged_mask || !merged_src ||
                  !merged_origin || !merged_traj || !owner))
        return AJT_ERR_INVALID_ARG;
    if ((old_logp_in == nullptr) != (merged_old_logp == nullptr)) return AJT_ERR_INVALID_ARG;
    if (((uintptr_t)workspace & 255) || ((uintptr_t)tokens & 3)) return AJT_ERR_INVALID_ARG;
    const MergeWs ws = merge_ws_layout(n, n_tokens);

    int dev = 0, num_sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return AJT_ERR_CUDA;
    if (cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || num_sms < 1) return AJT_ERR_CUDA;

    uint8_t* b = reinterpret_cast<uint8_t*>(workspace);
    MergeParams p;
    p.tokens = tokens; p.offsets = offsets; p.traj_ids = traj_ids; p.resp_start = resp_start; p.mask_in = mask_in;
    p.old_logp_in = old_logp_in; p.n = n; p.N = n_tokens; p.owner_rule = owner_rule; p.flags = flags;
    p.merged_tokens = merged_tokens; p.merged_mask = merged_mask; p.merged_src = merged_src; p.merged_old_logp = merged_old_logp;
    p.merged_offsets = merged_offsets; p.merged_origin = merged_origin; p.merged_traj = merged_traj; p.owner = owner;
    p.counts = counts;
    p.ctrl = reinterpret_cast<AjtCtrl*>(b + ws.ctrl);
    p.skey[0] = reinterpret_cast<uint32_t*>(b + ws.skey0); p.skey[1] = reinterpret_cast<uint32_t*>(b + ws.skey1);
    p.sval[0] = reinterpret_cast<uint32_t*>(b + ws.sval0); p.sval[1] = reinterpret_cast<uint32_t*>(b + ws.sval1);
    p.gid_sorted = reinterpret_cast<int32_t*>(b + ws.gid_sorted);
    p.grp_start = reinterpret_cast<int32_t*>(b + ws.grp_start);
    p.grp_ent = reinterpret_cast<int32_t*>(b + ws.grp_ent);
    p.t_rank = reinterpret_cast<int32_t*>(b + ws.t_rank);
    p.t_gid = reinterpret_cast<int32_t*>(b + ws.t_gid);
    p.t_entbase = reinterpret_cast<int32_t*>(b + ws.t_entbase);
    p.seg_base = reinterpret_cast<int32_t*>(b + ws.seg_base);
    p.seg_part = reinterpret_cast<uint64_t*>(b + ws.seg_part);
    p.absorbed = b + ws.absorbed;
    p.owner_tl = reinterpret_cast<int32_t*>(b + ws.owner_tl);
    p.midx = reinterpret_cast<int32_t*>(b + ws.midx);
    p.mem_cnt = reinterpret_cast<int32_t*>(b + ws.mem_cnt);
    p.mem_off = reinterpret_cast<int32_t*>(b + ws.mem_off);
    p.mem_cur = reinterpret_cast<int32_t*>(b + ws.mem_cur);
    p.mem_list = reinterpret_cast<int32_t*>(b + ws.mem_list);
    p.tile_base = reinterpret_cast<int32_t*>(b + ws.tile_base);
    // everything after the fixed part holds perm and the per-key arrays; their capacity follows from the size given
    size_t eo = ws.ent;
    p.perm = reinterpret_cast<int32_t*>(b + eo); eo += a256(((size_t)n + 1) * 4);
    if (workspace_bytes < eo + 6 * 256 + ((size_t)n + 1024) * kEntBytes) return AJT_ERR_WORKSPACE_TOO_SMALL;
    const size_t ecap = (workspace_bytes - eo - 6 * 256) / kEntBytes;
    p.E_cap = (int32_t)(ecap > (size_t)INT32_MAX ? (size_t)INT32_MAX : ecap);
    p.ent_hash = reinterpret_cast<uint64_t*>(b + eo); eo += a256((size_t)p.E_cap * 8);
    p.ent_len = reinterpret_cast<int32_t*>(b + eo); eo += a256((size_t)p.E_cap * 4);
    p.ent_dig = reinterpret_cast<uint32_t*>(b + eo); eo += a256((size_t)p.E_cap * 4);
    p.ent_idx = reinterpret_cast<uint32_t*>(b + eo); eo += a256((size_t)p.E_cap * 4);
    p.tmp_dig = reinterpret_cast<uint32_t*>(b + eo); eo += a256((size_t)p.E_cap * 4);
    p.tmp_idx = reinterpret_cast<uint32_t*>(b + eo); eo += a256((size_t)p.E_cap * 4);
    if (eo > workspace_bytes) return AJT_ERR_WORKSPACE_TOO_SMALL;
    p.nseg_cap = nseg_capacity(n, n_tokens);
    p.mis = (int32_t)(((uintptr_t)tokens >> 2) & 3);

    if (cudaMemsetAsync(p.ctrl, 0, sizeof(AjtCtrl), stream) != cudaSuccess) return AJT_ERR_CUDA;
    if (n == 0) {
        if (cudaMemsetAsync(counts, 0, 2 * sizeof(int64_t), stream) != cudaSuccess) return AJT_ERR_CUDA;
        if (cudaMemsetAsync(merged_offsets, 0, sizeof(int64_t), stream) != cudaSuccess) return AJT_ERR_CUDA;
        return AJT_OK;
    }
    const int wide = num_sms * 8;
    merge_group_kernel<<<1, 1024, 0, stream>>>(p);
    merge_hash_kernel<<<wide, 256, 0, stream>>>(p);
    merge_keys_kernel<<<(n + 255) / 256, 256, 0, stream>>>(p);
    merge_select_kernel<<<num_sms * 2, kSelThreads, 0, stream>>>(p, 0);
    merge_compact_kernel<<<1, 1024, 0, stream>>>(p, 0);
    merge_scatter_kernel<<<wide, 256, 0, stream>>>(p, 0);
    // exact repair path: each kernel returns at once unless the scatter pass saw a hash-equal, token-different pair
    merge_select_kernel<<<num_sms * 2, kSelThreads, 0, stream>>>(p, 1);
    merge_compact_kernel<<<1, 1024, 0, stream>>>(p, 1);
    merge_scatter_kernel<<<wide, 256, 0, stream>>>(p, 1);
    return cudaGetLastError() == cudaSuccess ? AJT_OK : AJT_ERR_CUDA;
}
