// Stage (a): timeline merging (Algorithm 1) on flat token streams, sm_100a.
//
// Definition: DESIGN.md "O-M".  Pipeline (rows M1-M7 of the scope table), 6 launches:
//   K1 merge_group_kernel    M1  one CTA, shared-memory resident for n <= 8192: validate offsets, stable LSD radix sort of
//                                (traj_id - min, index), group ids, rank in group, per-timeline record {first hash segment,
//                                group start, rank, first key slot}, lengths in group order
//   K2 merge_hash_kernel     M2  warp-cooperative prefix-hash scan, 128-bit loads, 4 vectors in flight per lane.  The hash of
//                                the first p tokens of timeline i is F_i(p) = sum_{q<p} x_q w(q) mod 2^64, w(q) = B^(q+3) mod 2^32: a sum, hence
//                                a monoid, so every lane keeps its own partial and lanes are only combined (three REDUX)
//                                where a key is emitted: at each length L_a of an earlier same-group timeline (probe key)
//                                and at L_i itself (full key).  The positions shared with the in-group predecessor are
//                                compared exactly on the way (the predecessor was just hashed: L2 hits)
//   K3 merge_select_kernel   M2  (one CTA per group) per-timeline prefix over its hash windows -> final (hash, len) keys
//                            M3  segmented radix sort of the group's keys by a 32-bit digest: one MSD pass on the top 11 bits
//                                in shared memory (<= 2048 keys: a bucket then holds the equal-key run, mean occupancy < 1,
//                                and keys inside it are compared exactly); 4 LSD passes through global memory above that
//   K4   (same kernel)       M4  per full key: walk its equal-key run, pick the extender by the owner rule
//   K6 merge_compact_kernel  M6  one CTA, one fused scan: survivors in original order -> merged_offsets/origin/traj, owner,
//                                tile table
//   K5/K7 merge_scatter_kernel M5+M7  fused: every merged sequence is streamed once in 256-position warp tiles; a member whose
//                                containment is not already implied by verified predecessor links (K2) is compared
//                                token-by-token against its owner (exact verification) while tokens / mask-OR / src /
//                                old_logp are written with 16-byte stores; tiles that every response region covers or
//                                misses are plain copies from one source.  A mismatch (a hash collision) raises
//                                ctrl->collision.
//   merge_repair_kernel      M5  one cooperative launch that exits at once unless ctrl->collision: K4 with exact comparison of
//                                every candidate it accepts, grid barrier, K6, grid barrier, K7.  Hash collisions can therefore
//                                never change the result.
#include <cooperative_groups.h>

#include "ajt_common.cuh"

namespace {

using namespace ajt;
namespace cg = cooperative_groups;

constexpr int kHSeg = 2048;        // hash-scan window: 2048 tokens = 16 steps x 32 lanes x 4 tokens
constexpr int kHSegLog = 11;
constexpr int kTile = 256;         // scatter tile (positions per warp task): 2 steps x 32 lanes x 4 tokens
constexpr uint32_t kW = 0x9E3779B1u;   // odd multiplier of the prefix hash's 32-bit position weights
constexpr uint32_t inv32(uint32_t b) {  // b^-1 mod 2^32 (b odd): Newton, 3 correct bits double every step
    uint32_t x = b;
    for (int i = 0; i < 5; ++i) x *= 2u - b * x;
    return x;
}
constexpr uint32_t cpow32(uint32_t b, uint32_t e) {
    uint32_t r = 1;
    for (; e; e >>= 1, b *= b)
        if (e & 1) r *= b;
    return r;
}
constexpr uint32_t kWinv = inv32(kW);
constexpr uint32_t kW128 = cpow32(kW, 128);
constexpr uint32_t kW2048 = cpow32(kW, 2048);
static_assert((uint32_t)(kW * kWinv) == 1u, "modular inverse");
constexpr uint32_t kFatal = AJT_STATUS_BAD_OFFSETS | AJT_STATUS_ZERO_LEN | AJT_STATUS_PROBE_CAPACITY;
constexpr int kSelThreads = 256;
constexpr int kSelSmemKeys = 2048;  // groups with more keys than this sort through global memory
constexpr int kSelBucketBits = 11;
constexpr int kSelBuckets = 1 << kSelBucketBits;
constexpr int kSelCacheK = 256;     // per-timeline facts of groups up to this size are staged in shared memory
constexpr int kGrpSmemN = 7936;     // batches up to this many timelines are grouped entirely in shared memory

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
    uint32_t* gbuf[6];     // [n+1] each: global stand-ins for the group kernel's shared arrays when n > kGrpSmemN
    int32_t* perm;         // [n] sorted position -> timeline index (groups contiguous, input order inside a group)
    int32_t* glen;         // [n] sorted position -> timeline length
    int32_t* grp_start;    // [G+1] first sorted position of each group
    int32_t* grp_ent;      // [G+1] first key slot of each group
    int4* tl_rec;          // [n] BY SORTED POSITION: {first hash segment, group start (sorted position), rank in group, first key slot}
    int32_t* tl_pos;       // [n] timeline index -> sorted position (written by the select kernel)
    uint64_t* seg_part;    // [nseg_cap] per-window partial sums, then exclusive prefixes per timeline
    uint64_t* ent_hash;    // [E_cap] key slot (i, a), a = 0..rank_i: in-window partial, then the final prefix hash
    uint32_t* ent_dig;     // [E_cap] global sort path: digests / order ping-pong
    uint32_t* ent_idx;     // [E_cap]
    uint32_t* tmp_dig;     // [E_cap]
    uint32_t* tmp_idx;     // [E_cap]
    uint8_t* absorbed;     // [n]
    uint8_t* link_bad;     // [n] 1: timeline i was compared with its in-group predecessor (hash pass) and is NOT an extension of it
    uint8_t* needv;        // [n] 1: absorbed timeline whose owner is not implied by a chain of verified predecessor links
    int32_t* owner_tl;     // [n] owning timeline (itself for survivors)
    int32_t* cand;         // [n] staging of the LONGEST owner while owner_tl is still being read
    int32_t* midx;         // [n] merged index of survivors, -1 otherwise
    int32_t* tile_base;    // [M+1] first scatter tile of each merged sequence
    int32_t E_cap;
    int32_t nseg_cap;
    int32_t mis;           // (address of tokens / 4) mod 4: element misalignment of the token array vs 16 bytes
};

struct MergeWs {
    size_t ctrl, gbuf[6], perm, glen, grp_start, grp_ent, tl_rec, tl_pos, seg_part, absorbed, link_bad, needv, owner_tl, cand, midx, tile_base, ent;
};
__host__ inline size_t a256(size_t x) { return (x + 255) & ~(size_t)255; }
__host__ inline int32_t nseg_capacity(int32_t n, int64_t N) { return (int32_t)(N / kHSeg + 2 * (int64_t)n + 2); }

__host__ MergeWs merge_ws_layout(int32_t n, int64_t N) {
    MergeWs w;
    size_t o = 0;
    const size_t n4 = a256(((size_t)n + 2) * 4);
    w.ctrl = o; o += 256;
    for (int k = 0; k < 6; ++k) { w.gbuf[k] = o; o += n4; }
    w.perm = o; o += n4; w.glen = o; o += n4; w.grp_start = o; o += n4; w.grp_ent = o; o += n4;
    w.tl_rec = o; o += a256(((size_t)n + 1) * 16);
    w.tl_pos = o; o += n4;
    w.seg_part = o; o += a256((size_t)nseg_capacity(n, N) * 8);
    w.absorbed = o; o += a256((size_t)n + 1);
    w.link_bad = o; o += a256((size_t)n + 1);
    w.needv = o; o += a256((size_t)n + 1);
    w.owner_tl = o; o += n4; w.cand = o; o += n4; w.midx = o; o += n4; w.tile_base = o; o += n4;
    w.ent = o;
    return w;
}
constexpr size_t kEntBytes = 32;  // per key slot: hash 8, dig 4, idx 4, tmp_dig 4, tmp_idx 4 = 24 used; ajt.h promises 32 per pair

__device__ __forceinline__ bool fatal(const MergeParams& p) { return (p.ctrl->status & kFatal) != 0; }

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
__device__ __forceinline__ int64_t tl_len(const MergeParams& p, int i) { return __ldg(p.offsets + i + 1) - __ldg(p.offsets + i); }

// Last index i in [0, n) with key(i) <= x, for a non-decreasing key with key(0) <= x: warp-cooperative 32-ary search
// (3 dependent loads for n <= 32768 instead of 15).
template <class F>
__device__ __forceinline__ int warp_search_last_le(int n, int64_t x, F key) {
    const int lane = threadIdx.x & 31;
    int lo = 0, hi = n;  // key(lo) <= x; hi == n or key(hi) > x
    while (hi - lo > 1) {
        const int step = (hi - lo + 31) >> 5;
        const int idx = lo + (lane + 1) * step;
        const bool le = idx < hi && (int64_t)key(idx) <= x;
        const int cnt = __popc(__ballot_sync(0xffffffffu, le));
        const int nlo = lo + cnt * step;
        hi = min(hi, nlo + step);
        lo = nlo;
    }
    return lo;
}

// ---------------------------------------------------------------------------------------- block-level building blocks

// Exclusive scan of the pair f(i) = (a, b), i in [0,n), by one CTA of NT threads; g(i, ex_a, ex_b, a, b) consumes it.
// Each thread owns kIpt consecutive items of a tile of NT * kIpt, so a tile costs one warp scan, one __syncthreads and one
// shuffle scan of the NT / 32 warp totals (double-buffered), whatever kIpt is.  Returns the totals to every thread.
struct I2 {
    int64_t a, b;
};
constexpr int kIpt = 4;
template <int NT, class F, class G>
__device__ __forceinline__ I2 block_scan2(int n, F f, G g, int64_t (*s_w)[2][NT / 32]) {
    static_assert(NT / 32 <= 32, "warp totals are scanned by one warp's lanes");
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    I2 base = {0, 0};
    int buf = 0;
    for (int i0 = 0; i0 < n; i0 += NT * kIpt, buf ^= 1) {
        const int b0 = i0 + tid * kIpt;
        I2 v[kIpt];
        int64_t sa = 0, sb = 0;
#pragma unroll
        for (int k = 0; k < kIpt; ++k) {
            v[k] = b0 + k < n ? f(b0 + k) : I2{0, 0};
            sa += v[k].a;
            sb += v[k].b;
        }
        int64_t ia = sa, ib = sb;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int64_t ta = __shfl_up_sync(0xffffffffu, ia, o), tb = __shfl_up_sync(0xffffffffu, ib, o);
            if (lane >= o) { ia += ta; ib += tb; }
        }
        if (lane == 31) { s_w[buf][0][warp] = ia; s_w[buf][1][warp] = ib; }
        __syncthreads();
        const int64_t wa = lane < NT / 32 ? s_w[buf][0][lane] : 0, wb = lane < NT / 32 ? s_w[buf][1][lane] : 0;
        int64_t ja = wa, jb = wb;
#pragma unroll
        for (int o = 1; o < NT / 32; o <<= 1) {
            const int64_t ta = __shfl_up_sync(0xffffffffu, ja, o), tb = __shfl_up_sync(0xffffffffu, jb, o);
            if (lane >= o) { ja += ta; jb += tb; }
        }
        const int64_t pa = __shfl_sync(0xffffffffu, ja - wa, warp), pb = __shfl_sync(0xffffffffu, jb - wb, warp);
        const int64_t ta = __shfl_sync(0xffffffffu, ja, NT / 32 - 1), tb = __shfl_sync(0xffffffffu, jb, NT / 32 - 1);
        int64_t ra = base.a + pa + ia - sa, rb = base.b + pb + ib - sb;
#pragma unroll
        for (int k = 0; k < kIpt; ++k) {
            if (b0 + k < n) g(b0 + k, ra, rb, v[k].a, v[k].b);
            ra += v[k].a;
            rb += v[k].b;
        }
        base.a += ta; base.b += tb;
    }
    __syncthreads();
    return base;
}
template <int NT, class F, class G>
__device__ __forceinline__ int64_t block_scan(int n, F f, G g, int64_t (*s_w)[2][NT / 32]) {
    return block_scan2<NT>(
               n, [&](int i) { return I2{(int64_t)f(i), 0}; }, [&](int i, int64_t ex, int64_t, int64_t v, int64_t) { g(i, ex, v); },
               s_w)
        .a;
}

// Lanes of the warp whose nbits-bit digit equals this lane's (and that are valid): one ballot per bit instead of match.any, whose
// cost grows with the number of distinct values in the warp (32 when trajectory ids arrive round-robin).
__device__ __forceinline__ unsigned peers8(uint32_t d, bool valid, int nbits) {
    unsigned m = __ballot_sync(0xffffffffu, valid);
#pragma unroll 1
    for (int b = 0; b < nbits; ++b) {
        const unsigned v = __ballot_sync(0xffffffffu, (d >> b) & 1u);
        m &= ((d >> b) & 1u) ? v : ~v;
    }
    return valid ? m : 0u;
}

template <int NW>
struct RadixScratch {
    uint32_t cnt[NW][256];
    uint32_t off[256];
};

// One stable LSD pass (digit of nbits <= 8 bits at `shift`) of (key, value) pairs by one CTA of NW warps.  Warp w owns the w-th
// contiguous chunk of the input, so "chunk, then round, then lane" is input order.  Count: per round, lanes with equal
// digits find each other with match.any and the lowest lane of each peer set adds the set size to cnt[w][digit].  Offsets:
// one thread per digit turns the NW counts into running offsets, one warp scans the 256 digit totals.  Scatter: the same
// rounds again, position = digit base + warp offset + rank in peer set.  Four __syncthreads per pass, whatever n is.
#ifdef AJT_TIMING
__device__ uint64_t g_rt[8];
#define AJT_RT(k) do { __syncthreads(); if (threadIdx.x == 0) { uint64_t t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); g_rt[k] = t_; } } while (0)
#else
#define AJT_RT(k) do { } while (0)
#endif
template <int NW>
__device__ __forceinline__ void radix_pass(const uint32_t* kin, const uint32_t* vin, uint32_t* kout, uint32_t* vout, int n,
                                           int shift, RadixScratch<NW>& sc, int nbits = 8) {
    const uint32_t dmask = (1u << nbits) - 1u;
    AJT_RT(0);
    constexpr int NT = NW * 32;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int x = tid; x < NW * 256; x += NT) (&sc.cnt[0][0])[x] = 0;
    __syncthreads();
    AJT_RT(1);
    const int per = ((n + NW - 1) / NW + 31) & ~31;
    const int c0 = min(n, warp * per), c1 = min(n, c0 + per);
    for (int base = c0; base < c1; base += 32) {
        const int i = base + lane;
        const bool valid = i < c1;
        const uint32_t d = valid ? (kin[i] >> shift) & dmask : 0u;
        const unsigned peers = peers8(d, valid, nbits);
        if (valid && lane == __ffs(peers) - 1) sc.cnt[warp][d] += (uint32_t)__popc(peers);
        __syncwarp();
    }
    __syncthreads();
    AJT_RT(2);
    for (int d2 = tid; d2 < 256; d2 += NT) {
        uint32_t run = 0;
#pragma unroll 4
        for (int w = 0; w < NW; ++w) {
            const uint32_t c = sc.cnt[w][d2];
            sc.cnt[w][d2] = run;
            run += c;
        }
        sc.off[d2] = run;
    }
    __syncthreads();
    AJT_RT(3);
    if (warp == 0) {  // exclusive scan of the 256 digit totals: 8 per lane
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
    AJT_RT(4);
    for (int base = c0; base < c1; base += 32) {
        const int i = base + lane;
        const bool valid = i < c1;
        const uint32_t key = valid ? kin[i] : 0u;
        const uint32_t val = valid ? vin[i] : 0u;
        const uint32_t d = (key >> shift) & dmask;
        const unsigned peers = peers8(d, valid, nbits);
        const int rk = __popc(peers & ((1u << lane) - 1u));
        if (valid) {
            const uint32_t pos = sc.off[d] + sc.cnt[warp][d] + (uint32_t)rk;
            kout[pos] = key;
            vout[pos] = val;
        }
        __syncwarp();
        if (valid && rk == 0) sc.cnt[warp][d] += (uint32_t)__popc(peers);
        __syncwarp();
    }
    __syncthreads();
    AJT_RT(5);
}

// ---------------------------------------------------------------------------------------- K1: group (M1)

#ifdef AJT_TIMING
#define AJT_TICK(k) do { __syncthreads(); if (threadIdx.x == 0) { uint64_t t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); tick_[k] = t_; } } while (0)
#else
#define AJT_TICK(k) do { } while (0)
#endif
template <bool kSmem>
__global__ void __launch_bounds__(1024) merge_group_kernel(const MergeParams p) {
#ifdef AJT_TIMING
    uint64_t tick_[10] = {0};
#endif
    AJT_TICK(0);
    extern __shared__ __align__(16) uint8_t g_dyn[];
    __shared__ RadixScratch<32> sc;
    __shared__ int64_t s_w[2][2][32];
    __shared__ int s_min, s_max;
    __shared__ uint32_t s_bad;
    const int tid = threadIdx.x, n = p.n;
    // five [n+1] work arrays: shared memory for n <= kGrpSmemN, the workspace otherwise
    const size_t nn = ((size_t)n + 4) & ~(size_t)3;   // (6 arrays of nn words)
    uint32_t* const sm32 = reinterpret_cast<uint32_t*>(g_dyn);
    uint32_t* kb[2] = {kSmem ? sm32 : p.gbuf[0], kSmem ? sm32 + nn : p.gbuf[1]};
    uint32_t* vb[2] = {kSmem ? sm32 + 2 * nn : p.gbuf[2], kSmem ? sm32 + 3 * nn : p.gbuf[3]};
    int32_t* nsg = reinterpret_cast<int32_t*>(kSmem ? sm32 + 4 * nn : p.gbuf[4]);   // [i] hash windows of timeline i
    int32_t* tln = reinterpret_cast<int32_t*>(kSmem ? sm32 + 5 * nn : p.gbuf[5]);   // [i] its length
    if (tid < (int)(sizeof(AjtCtrl) / 4)) reinterpret_cast<uint32_t*>(p.ctrl)[tid] = 0;   // fresh control block
    if (tid == 0) { s_min = INT32_MAX; s_max = INT32_MIN; s_bad = 0; }
    __syncthreads();
    // validate offsets; min / max traj id; hash windows per timeline
    int lmin = INT32_MAX, lmax = INT32_MIN;
    uint32_t bad = 0;
#pragma unroll 4
    for (int i = tid; i < n; i += 1024) {
        const int64_t a = __ldg(p.offsets + i), b = __ldg(p.offsets + i + 1);
        if (b < a || b - a > (int64_t)INT32_MAX) bad |= AJT_STATUS_BAD_OFFSETS;
        else if (b == a) bad |= AJT_STATUS_ZERO_LEN;
        const int t = __ldg(p.traj_ids + i);
        lmin = min(lmin, t);
        lmax = max(lmax, t);
        kb[0][i] = (uint32_t)t;
        vb[0][i] = (uint32_t)i;
        nsg[i] = (int32_t)(((b - 1 + p.mis) >> kHSegLog) - ((a + p.mis) >> kHSegLog) + 1);
        tln[i] = (int32_t)(b - a);
        p.link_bad[i] = 0;
    }
    AJT_TICK(1);
    if (tid == 0 && (p.offsets[0] != 0 || p.offsets[n] != p.N)) bad |= AJT_STATUS_BAD_OFFSETS;
    lmin = __reduce_min_sync(0xffffffffu, lmin);
    lmax = __reduce_max_sync(0xffffffffu, lmax);
    bad = __reduce_or_sync(0xffffffffu, bad);
    if ((tid & 31) == 0) {
        if (bad) atomicOr(&s_bad, bad);
        atomicMin(&s_min, lmin);
        atomicMax(&s_max, lmax);
    }
    __syncthreads();
    if (s_bad) {
        if (tid == 0) atomicOr(&p.ctrl->status, s_bad);
        return;
    }
    AJT_TICK(7);
    const int tmin = s_min;
    const uint32_t range = n ? (uint32_t)s_max - (uint32_t)tmin : 0u;
    for (int i = tid; i < n; i += 1024) kb[0][i] -= (uint32_t)tmin;
    __syncthreads();
    AJT_TICK(8);
    int cur = 0;
    for (int shift = 0; shift < 32 && (range >> shift) != 0; shift += 8) {
        radix_pass<32>(kb[cur], vb[cur], kb[cur ^ 1], vb[cur ^ 1], n, shift, sc);
        cur ^= 1;
        __syncthreads();
    }
    AJT_TICK(2);
    const uint32_t* key = kb[cur];
    const uint32_t* val = vb[cur];   // sorted position -> timeline index
    uint32_t* gid = kb[cur ^ 1];     // [pos] group id
    uint32_t* gsv = vb[cur ^ 1];     // [g]   first sorted position of group g
    // group ids and group starts
    const int G = (int)block_scan<1024>(
        n, [&](int pos) { return (pos == 0 || key[pos] != key[pos - 1]) ? 1 : 0; },
        [&](int pos, int64_t ex, int64_t v) {
            const int g = (int)(ex + v) - 1;
            gid[pos] = (uint32_t)g;
            if (v) { gsv[g] = (uint32_t)pos; p.grp_start[g] = pos; }
        },
        s_w);
    if (tid == 0) { gsv[G] = (uint32_t)n; p.grp_start[G] = n; }
    __syncthreads();
    AJT_TICK(3);
    // key slots (i, a), a = 0..rank_i: a group of k timelines has k(k+1)/2, the slots of rank r start r(r+1)/2 into it
    uint32_t* gent = kb[cur];        // [g] first key slot of group g (the sorted keys are no longer needed)
    const int64_t E = block_scan<1024>(
        G, [&](int g) { const int64_t k = gsv[g + 1] - gsv[g]; return k * (k + 1) / 2; },
        [&](int g, int64_t ex, int64_t) {
            gent[g] = (uint32_t)min(ex, (int64_t)INT32_MAX);
            p.grp_ent[g] = (int32_t)min(ex, (int64_t)INT32_MAX);
        },
        s_w);
    AJT_TICK(4);
    // hash segments: aligned windows of kHSeg tokens intersected with each timeline (none for singleton groups), numbered in
    // GROUP order, so that a timeline is hashed right after its in-group predecessor.  Everything the later kernels need
    // per timeline goes out by sorted position: coalesced, no scattered access from this one CTA.
    const int64_t nseg = block_scan<1024>(
        n, [&](int pos) { const int g = (int)gid[pos]; return gsv[g + 1] - gsv[g] < 2 ? 0 : nsg[val[pos]]; },
        [&](int pos, int64_t ex, int64_t) {
            const int i = (int)val[pos], g = (int)gid[pos];
            const int gs = (int)gsv[g], r = pos - gs;
            p.tl_rec[pos] = make_int4((int)ex, gs, r, (int)(gent[g] + (uint32_t)r * (uint32_t)(r + 1) / 2u));
            p.perm[pos] = i;
            p.glen[pos] = tln[i];
        },
        s_w);
    AJT_TICK(5);
    if (tid == 0) {
        p.grp_ent[G] = (int32_t)min(E, (int64_t)INT32_MAX);
        p.ctrl->n_groups = G;
        p.ctrl->n_entries = (int32_t)min(E, (int64_t)INT32_MAX);
        p.ctrl->n_hash_segs = (int32_t)nseg;
        if (E > (int64_t)p.E_cap || nseg > (int64_t)p.nseg_cap) atomicOr(&p.ctrl->status, (uint32_t)AJT_STATUS_PROBE_CAPACITY);
    }
    AJT_TICK(6);
#ifdef AJT_TIMING
    if (tid == 0) {
        for (int k = 0; k < 7; ++k) reinterpret_cast<uint64_t*>(p.ctrl->reserved)[k] = tick_[k];
        reinterpret_cast<uint64_t*>(p.ctrl->reserved)[14] = tick_[7];
        reinterpret_cast<uint64_t*>(p.ctrl->reserved)[15] = tick_[8];
        for (int k = 0; k < 6; ++k) reinterpret_cast<uint64_t*>(p.ctrl->reserved)[8 + k] = g_rt[k];
    }
#endif
}

// ---- K1 for batches that fit in shared memory (n <= kGrpSmemN): the same steps written for a SMALL CODE FOOTPRINT.  A
// merge call streams hundreds of MB through L2 between two launches of this kernel, so its instructions come from DRAM every
// time, and a one-CTA kernel that runs each line once pays for every 128-byte line it touches: loops are not unrolled, and
// the scans share one out-of-line routine working in place on shared arrays.

// In-place exclusive scan of a[0..n) by the CTA (1024 threads); returns the total to every thread.
__device__ __noinline__ uint32_t cta_scan_excl(uint32_t* a, int n, uint32_t* s_wt) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    uint32_t base = 0;
#pragma unroll 1
    for (int i0 = 0; i0 < n; i0 += 1024) {
        const int i = i0 + tid;
        const uint32_t v = i < n ? a[i] : 0u;
        uint32_t inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) s_wt[warp] = inc;
        __syncthreads();
        const uint32_t wv = s_wt[lane];
        uint32_t winc = wv;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += t;
        }
        const uint32_t pre = __shfl_sync(0xffffffffu, winc - wv, warp), tot = __shfl_sync(0xffffffffu, winc, 31);
        if (i < n) a[i] = base + pre + inc - v;
        base += tot;
        __syncthreads();
    }
    return base;
}

__global__ void __launch_bounds__(1024) merge_group_small_kernel(const MergeParams p) {
    extern __shared__ __align__(16) uint8_t g_dyn[];
    __shared__ RadixScratch<32> sc;
    __shared__ uint32_t s_wt[32];
    __shared__ int s_min, s_max;
    __shared__ uint32_t s_bad;
#ifdef AJT_TIMING
    uint64_t tick_[10] = {0};
#endif
    AJT_TICK(0);
    const int tid = threadIdx.x, n = p.n;
    const size_t nn = ((size_t)n + 32) & ~(size_t)31;   // 6 arrays of nn words
    // arrays read BY TIMELINE INDEX through the sorted order are swizzled: timelines of one group are often a power of two
    // apart (round-robin collection), which would put a warp's 32 gathers in one bank
    auto swz = [](int i) { return i ^ ((i >> 5) & 31) ^ ((i >> 10) & 31); };
    uint32_t* const sm32 = reinterpret_cast<uint32_t*>(g_dyn);
    uint32_t* kb[2] = {sm32, sm32 + nn};
    uint32_t* vb[2] = {sm32 + 2 * nn, sm32 + 3 * nn};
    uint32_t* nsg = sm32 + 4 * nn;   // [i] hash windows of timeline i
    uint32_t* tln = sm32 + 5 * nn;   // [i] its length; later [pos] windows by sorted position
    if (tid < (int)(sizeof(AjtCtrl) / 4)) reinterpret_cast<uint32_t*>(p.ctrl)[tid] = 0;   // fresh control block
    if (tid == 0) { s_min = INT32_MAX; s_max = INT32_MIN; s_bad = 0; }
    __syncthreads();
    // validate offsets; min / max traj id; hash windows per timeline
    int lmin = INT32_MAX, lmax = INT32_MIN;
    uint32_t bad = 0;
#pragma unroll 2
    for (int i = tid; i < n; i += 1024) {
        const int64_t a = __ldg(p.offsets + i), b = __ldg(p.offsets + i + 1);
        if (b < a || b - a > (int64_t)INT32_MAX) bad |= AJT_STATUS_BAD_OFFSETS;
        else if (b == a) bad |= AJT_STATUS_ZERO_LEN;
        const int t = __ldg(p.traj_ids + i);
        lmin = min(lmin, t);
        lmax = max(lmax, t);
        kb[0][i] = (uint32_t)t;
        vb[0][i] = (uint32_t)i;
        nsg[swz(i)] = (uint32_t)(((b - 1 + p.mis) >> kHSegLog) - ((a + p.mis) >> kHSegLog) + 1);
        tln[swz(i)] = (uint32_t)(b - a);
        p.link_bad[i] = 0;
    }
    if (tid == 0 && (__ldg(p.offsets) != 0 || __ldg(p.offsets + n) != p.N)) bad |= AJT_STATUS_BAD_OFFSETS;
    AJT_TICK(1);
    lmin = __reduce_min_sync(0xffffffffu, lmin);
    lmax = __reduce_max_sync(0xffffffffu, lmax);
    bad = __reduce_or_sync(0xffffffffu, bad);
    if ((tid & 31) == 0) {
        if (bad) atomicOr(&s_bad, bad);
        atomicMin(&s_min, lmin);
        atomicMax(&s_max, lmax);
    }
    __syncthreads();
    if (s_bad) {
        if (tid == 0) atomicOr(&p.ctrl->status, s_bad);
        return;
    }
    const uint32_t tmin = (uint32_t)s_min, range = (uint32_t)s_max - tmin;
#pragma unroll 1
    for (int i = tid; i < n; i += 1024) kb[0][i] -= tmin;
    __syncthreads();
    AJT_TICK(2);
    int cur = 0;
    {   // as few passes as the key range needs, digits of equal width (the ranking costs one ballot per digit bit)
        const int bits = 32 - __clz(range), npass = (bits + 7) / 8, w = npass ? (bits + npass - 1) / npass : 0;
#pragma unroll 1
        for (int shift = 0; shift < bits; shift += w) {
            radix_pass<32>(kb[cur], vb[cur], kb[cur ^ 1], vb[cur ^ 1], n, shift, sc, w);
            cur ^= 1;
        }
    }
    AJT_TICK(3);
    uint32_t* key = kb[cur];          // [pos] sorted keys; later [g] first key slot of group g
    const uint32_t* val = vb[cur];    // [pos] timeline index
    uint32_t* gid = kb[cur ^ 1];      // [pos] group id
    uint32_t* gsv = vb[cur ^ 1];      // [g]   first sorted position of group g
    // group ids and group starts
#pragma unroll 1
    for (int pos = tid; pos < n; pos += 1024) gid[pos] = (pos == 0 || key[pos] != key[pos - 1]) ? 1u : 0u;
    __syncthreads();
    const int G = (int)cta_scan_excl(gid, n, s_wt);   // gid[pos] = heads before pos
#pragma unroll 1
    for (int pos = tid; pos < n; pos += 1024) {
        const bool head = pos == 0 || key[pos] != key[pos - 1];
        const uint32_t g = gid[pos] + (head ? 1u : 0u) - 1u;
        gid[pos] = g;
        if (head) { gsv[g] = (uint32_t)pos; p.grp_start[g] = pos; }
    }
    if (tid == 0) { gsv[G] = (uint32_t)n; p.grp_start[G] = n; }
    __syncthreads();
    AJT_TICK(4);
    // key slots (i, a), a = 0..rank_i: a group of k timelines has k(k+1)/2 (at most n^2/2 < 2^25 here)
    uint32_t* gent = key;
#pragma unroll 1
    for (int g = tid; g < G; g += 1024) {
        const uint32_t k = gsv[g + 1] - gsv[g];
        gent[g] = k * (k + 1) / 2;
    }
    __syncthreads();
    const uint32_t E = cta_scan_excl(gent, G, s_wt);
    AJT_TICK(5);
    // lengths by sorted position; then the windows by sorted position (none for singleton groups) in the freed array
#pragma unroll 1
    for (int pos = tid; pos < n; pos += 1024) p.glen[pos] = (int32_t)tln[swz((int)val[pos])];
    __syncthreads();
    uint32_t* segs = tln;
#pragma unroll 1
    for (int pos = tid; pos < n; pos += 1024) {
        const uint32_t g = gid[pos];
        segs[pos] = gsv[g + 1] - gsv[g] < 2 ? 0u : nsg[swz((int)val[pos])];
    }
    __syncthreads();
    // hash segments numbered in GROUP order, so that a timeline is hashed right after its in-group predecessor
    const uint32_t nseg = cta_scan_excl(segs, n, s_wt);
    AJT_TICK(6);
#pragma unroll 1
    for (int pos = tid; pos < n; pos += 1024) {
        const uint32_t g = gid[pos], gs = gsv[g], r = (uint32_t)pos - gs;
        p.tl_rec[pos] = make_int4((int)segs[pos], (int)gs, (int)r, (int)(gent[g] + r * (r + 1) / 2u));
        p.perm[pos] = (int32_t)val[pos];
        if (r == 0) p.grp_ent[g] = (int32_t)gent[g];
    }
    if (tid == 0) {
        p.grp_ent[G] = (int32_t)E;
        p.ctrl->n_groups = G;
        p.ctrl->n_entries = (int32_t)E;
        p.ctrl->n_hash_segs = (int32_t)nseg;
        if ((int64_t)E > (int64_t)p.E_cap || (int64_t)nseg > (int64_t)p.nseg_cap)
            atomicOr(&p.ctrl->status, (uint32_t)AJT_STATUS_PROBE_CAPACITY);
    }
    AJT_TICK(7);
#ifdef AJT_TIMING
    if (tid == 0)
        for (int k = 0; k < 8; ++k) reinterpret_cast<uint64_t*>(p.ctrl->reserved)[k] = tick_[k];
#endif
}

// ---------------------------------------------------------------------------------------- K2: prefix-hash scan (M2)

// Prefix hash F_i(p) = sum_{q<p} x_q w(q) mod 2^64 with 32-bit weights w(q) = B^(q+3) mod 2^32: one IMAD.WIDE per token
// (32 x 32 -> 64 with a 64-bit addend).  A sum over positions, hence a monoid: per-lane partials, combined only where a key is
// emitted.  Weak by design (a 64-bit sum of 50-bit products); every accepted pair is verified exactly (M5).
__device__ __forceinline__ uint32_t pow32(uint32_t b, uint32_t e) {
    uint32_t r = 1;
    while (e) {
        if (e & 1) r *= b;
        b *= b;
        e >>= 1;
    }
    return r;
}
// Power tables (constant memory, warp-uniform reads): W^(win0 + 3) of a window that starts d = -win0 (mod 2048) slots before
// a multiple of 2048, j windows into its timeline, is W2048^j * Winv^(64 (d >> 6)) * Winv^(d & 63) * W^3.
template <int N>
struct PowTab {
    uint32_t v[N];
    constexpr PowTab() : v{} {}
    constexpr PowTab(uint32_t base) : v{} {
        uint32_t r = 1;
        for (int i = 0; i < N; ++i) { v[i] = r; r *= base; }
    }
};
__constant__ PowTab<64> c_w2048 = PowTab<64>(cpow32(kW, 2048));
__constant__ PowTab<32> c_winv64 = PowTab<32>(cpow32(kWinv, 64));
__constant__ PowTab<64> c_winv1 = PowTab<64>(kWinv);
__constant__ PowTab<16> c_w128 = PowTab<16>(kW128);
__constant__ PowTab<32> c_w4 = PowTab<32>(cpow32(kW, 4));
// weight of the first slot of window j of a timeline whose window grid starts d slots before its first token (0 <= d < 2048)
__device__ __forceinline__ uint32_t window_weight(int j, int d) {
    const uint32_t wj = j < 64 ? c_w2048.v[j] : pow32(kW2048, (uint32_t)j);
    return wj * c_winv64.v[d >> 6] * c_winv1.v[d & 63] * (kW * kW * kW);
}
__device__ __forceinline__ uint64_t mad_wide(uint32_t a, uint32_t b, uint64_t c) { return (uint64_t)a * b + c; }

constexpr int kHashThreads = 256;

// This lane's four tokens of step s of a window (positions q .. q+3 of the timeline whose tokens start at tl), zero outside
// the timeline.  16-byte aligned address.  lo / hi: how many elements may be read before tl / from tl (array bounds).
template <bool kInterior>
__device__ __forceinline__ int4 load_step(const int32_t* __restrict__ tl, int Li, int q, int64_t lo, int64_t hi) {
    if (kInterior) return __ldg(reinterpret_cast<const int4*>(tl + q));
    int4 x = make_int4(0, 0, 0, 0);
    if (q + 3 >= 0 && q < Li) {
        if (q >= -lo && q + 3 < hi) x = __ldg(reinterpret_cast<const int4*>(tl + q));
        else {
            if (q >= -lo && q < hi) x.x = tl[q];
            if (q + 1 >= -lo && q + 1 < hi) x.y = tl[q + 1];
            if (q + 2 >= -lo && q + 2 < hi) x.z = tl[q + 2];
            if (q + 3 >= -lo && q + 3 < hi) x.w = tl[q + 3];
        }
        if (!(q >= 0 && q < Li)) x.x = 0;
        if (!(q + 1 >= 0 && q + 1 < Li)) x.y = 0;
        if (!(q + 2 >= 0 && q + 2 < Li)) x.z = 0;
        if (!(q + 3 >= 0 && q + 3 < Li)) x.w = 0;
    }
    return x;
}

// One batch = 4 steps = 512 positions of a window: four 16-byte loads per lane in flight (plus 16 predecessor tokens when
// linked).  kInterior: the batch lies inside the timeline.  kLink: 0 no predecessor positions here, 1 some, 2 all of them.
// snap[s * 32] receives this lane's running sum BEFORE step s (the key-emission pass needs it); w are the lane's weights.
template <bool kInterior, int kLink>
__device__ __forceinline__ void hash_batch(const int32_t* __restrict__ tl, int Li, int qb, int64_t lo, int64_t hi,
                                           const int32_t* __restrict__ tprev, int Lprev, uint32_t (&w)[4], uint64_t& acc,
                                           uint32_t& diff, uint64_t* snap) {
    int4 x[4];
    int32_t y[4][4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int q = qb + 128 * u;
        x[u] = load_step<kInterior>(tl, Li, q, lo, hi);
        if (kLink == 2) {
#pragma unroll
            for (int k = 0; k < 4; ++k) y[u][k] = __ldg(tprev + q + k);
        } else if (kLink == 1) {
#pragma unroll
            for (int k = 0; k < 4; ++k) y[u][k] = (q + k >= 0 && q + k < Lprev) ? __ldg(tprev + q + k) : 0;
        }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int q = qb + 128 * u;
        if (kLink == 2) {
            diff |= (uint32_t)(y[u][0] ^ x[u].x) | (uint32_t)(y[u][1] ^ x[u].y);
            diff |= (uint32_t)(y[u][2] ^ x[u].z) | (uint32_t)(y[u][3] ^ x[u].w);
        } else if (kLink == 1) {
            if (q >= 0 && q < Lprev) diff |= (uint32_t)(y[u][0] ^ x[u].x);
            if (q + 1 >= 0 && q + 1 < Lprev) diff |= (uint32_t)(y[u][1] ^ x[u].y);
            if (q + 2 >= 0 && q + 2 < Lprev) diff |= (uint32_t)(y[u][2] ^ x[u].z);
            if (q + 3 >= 0 && q + 3 < Lprev) diff |= (uint32_t)(y[u][3] ^ x[u].w);
        }
        snap[u * 32] = acc;
        acc = mad_wide((uint32_t)x[u].x, w[0], acc);
        acc = mad_wide((uint32_t)x[u].y, w[1], acc);
        acc = mad_wide((uint32_t)x[u].z, w[2], acc);
        acc = mad_wide((uint32_t)x[u].w, w[3], acc);
        w[0] *= kW128; w[1] *= kW128; w[2] *= kW128; w[3] *= kW128;
    }
}

// Sum of a 64-bit value over the warp (mod 2^64) with three REDUX instead of ten shuffles: 22 + 22 + 20-bit slices, whose
// 32-term sums fit 32 bits.
__device__ __forceinline__ uint64_t warp_sum_u64_redux(uint64_t v) {
    const uint32_t a = (uint32_t)v & 0x3fffffu, b = (uint32_t)(v >> 22) & 0x3fffffu, c = (uint32_t)(v >> 44);
    const uint32_t sa = __reduce_add_sync(0xffffffffu, a), sb = __reduce_add_sync(0xffffffffu, b);
    const uint32_t sc = __reduce_add_sync(0xffffffffu, c);
    return (uint64_t)sa + ((uint64_t)sb << 22) + ((uint64_t)sc << 44);
}

// One key: F at prefix length (position r of the window) + 1.  Every lane adds to its running sum BEFORE step s = r >> 7 (its
// snapshot) the tokens of that step it holds at positions <= r (re-read: L1), and one warp sum gives the value.  ~40
// instructions per key; a window holds the end of 0-3 requested prefixes.
__device__ __forceinline__ uint64_t hash_key_value(const int32_t* __restrict__ tl, int Li, int64_t lo, int64_t hi, int win0, int r,
                                                   uint32_t w0_window, const uint64_t* snap) {
    const int lane = threadIdx.x & 31;
    const int s = r >> 7;
    const int4 x = load_step<false>(tl, Li, win0 + 128 * s + 4 * lane, lo, hi);
    const int c = (r & 127) - 4 * lane;   // tokens k <= c of this lane lie inside the prefix
    uint32_t w = w0_window * c_w128.v[s];
    uint64_t part = snap[s * 32];
    if (c >= 0) part = mad_wide((uint32_t)x.x, w, part);
    w *= kW;
    if (c >= 1) part = mad_wide((uint32_t)x.y, w, part);
    w *= kW;
    if (c >= 2) part = mad_wide((uint32_t)x.z, w, part);
    w *= kW;
    if (c >= 3) part = mad_wide((uint32_t)x.w, w, part);
    return warp_sum_u64_redux(part);
}

__global__ void __launch_bounds__(kHashThreads, 3) merge_hash_kernel(const MergeParams p) {
    __shared__ uint64_t s_snap[kHashThreads / 32][16 * 32];   // per warp: running sums before each step of the window
    if (fatal(p)) return;
    const int lane = threadIdx.x & 31;
    const int wglobal = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    const int nseg = p.ctrl->n_hash_segs, n = p.n;
    uint64_t* snap = s_snap[threadIdx.x >> 5] + lane;
    // Striped windows: at any moment the grid works on ~nwarps consecutive windows (a front of ~30 MB that sweeps the token
    // array once), so a timeline's in-group predecessor, hashed a little earlier, is still in L2 when it is compared.
    const uint32_t LW = c_w4.v[lane];
    auto seg_base = [&](int i) { return __ldg(reinterpret_cast<const int32_t*>(p.tl_rec) + 4 * i); };
    for (int sidx = wglobal; sidx < nseg; sidx += nwarps) {
        const int pos = warp_search_last_le(n, sidx, seg_base);   // sorted position of the window's timeline
        const int4 rec = __ldg(p.tl_rec + pos);
        const int i = __ldg(p.perm + pos);
        const int64_t off = __ldg(p.offsets + i);
        const int Li = (int)(__ldg(p.offsets + i + 1) - off);
        const int32_t* tl = p.tokens + off;
        const int64_t lo = off, hi = p.N - off;   // elements of the token array before / from tl
        // the in-group predecessor, if this timeline can extend it (the usual case: each call resends the context)
        int Lprev = 0;
        const int32_t* tprev = nullptr;
        if (rec.z > 0) {
            const int lp = __ldg(p.glen + pos - 1);
            if (lp <= Li) { Lprev = lp; tprev = p.tokens + __ldg(p.offsets + __ldg(p.perm + pos - 1)); }
        }
        const int d = (int)((off + p.mis) & (kHSeg - 1));   // the timeline starts d slots into its first window
        const int j = sidx - rec.x;                          // window index inside the timeline
        const int win0 = j * kHSeg - d;                      // timeline position of the window's first slot
        // pull the whole window (<= 8 KB = 64 lines) towards L2 now: the four batches below then wait on L2, not on DRAM
        for (int e = max(win0, 0) + 32 * lane; e < min(win0 + kHSeg, Li); e += 1024)
            asm volatile("prefetch.global.L2 [%0];" ::"l"(tl + e));
        const uint32_t w0 = window_weight(j, d) * LW;        // weight W^(q+3) of this lane's first slot q = win0 + 4 lane
        const int rank = rec.z, ebase = rec.w;
        const int32_t* gln = p.glen + rec.y;
        // ---- streaming pass: four batches of 512 positions
        uint32_t w[4] = {w0, w0 * kW, w0 * kW * kW, w0 * kW * kW * kW};
        uint32_t diff = 0;
        uint64_t acc = 0;
        const int q0 = win0 + lane * 4;
#pragma unroll 1
        for (int h = 0; h < 4; ++h) {
            const int b0 = win0 + 512 * h, b1 = b0 + 512;
            uint64_t* sn = snap + h * 4 * 32;
            if (b0 >= Li) {   // nothing of the timeline here
#pragma unroll
                for (int u = 0; u < 4; ++u) sn[u * 32] = acc;
                continue;
            }
            const bool interior = b0 >= 0 && b1 <= Li;
            const int qb = q0 + 512 * h;
#define AJT_HB(I, K) hash_batch<I, K>(tl, Li, qb, lo, hi, tprev, Lprev, w, acc, diff, sn)
            if (interior && b1 <= Lprev) AJT_HB(true, 2);
            else if (interior && b0 < Lprev) AJT_HB(true, 1);
            else if (interior) AJT_HB(true, 0);
            else if (b0 < Lprev) AJT_HB(false, 1);
            else AJT_HB(false, 0);
#undef AJT_HB
        }
        const uint64_t tot = warp_sum_u64(acc);
        if (lane == 0) p.seg_part[sidx] = tot;
        if (win0 < Lprev && __any_sync(0xffffffffu, diff != 0) && lane == 0) p.link_bad[i] = 1;
        // ---- key emission: the requested prefixes (L_a of an earlier member, or L_i) that end inside this window
        __syncwarp();
        for (int a0 = 0; a0 <= rank; a0 += 32) {
            const int a = a0 + lane;
            int rel = -1;
            if (a <= rank) {
                const int Lp = __ldg(gln + a);
                const int r = Lp - 1 - win0;
                if (Lp <= Li && r >= 0 && r < kHSeg) rel = r;
            }
            for (uint32_t m = __ballot_sync(0xffffffffu, rel >= 0); m; m &= m - 1) {
                const int b = __ffs(m) - 1;
                const uint64_t F = hash_key_value(tl, Li, lo, hi, win0, __shfl_sync(0xffffffffu, rel, b), w0, snap);
                if (lane == b) p.ent_hash[ebase + a] = F;
            }
        }
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------------- K3 + K4: keys, sort, select (M2-M4)

__device__ bool tokens_extend(const MergeParams& p, int i, int j) {  // exact: tokens_i[0:L_j] == tokens_j, L_i >= L_j
    const int64_t oi = p.offsets[i], oj = p.offsets[j];
    const int64_t Li = p.offsets[i + 1] - oi, Lj = p.offsets[j + 1] - oj;
    if (Li < Lj) return false;
    for (int64_t q = 0; q < Lj; ++q)
        if (p.tokens[oi + q] != p.tokens[oj + q]) return false;
    return true;
}

// local key slot -> rank of the probing timeline: slots of rank b occupy [b(b+1)/2, b(b+1)/2 + b]
__device__ __forceinline__ int rank_of_local(uint32_t l) {
    int b = (int)((sqrtf(8.f * (float)l + 1.f) - 1.f) * 0.5f);
    while ((uint64_t)(b + 1) * (uint64_t)(b + 2) / 2 <= l) ++b;
    while ((uint64_t)b * (uint64_t)(b + 1) / 2 > l) --b;
    return b;
}

struct SelectSmem {
    RadixScratch<kSelThreads / 32> sc;       // global LSD path
    uint32_t start[kSelBuckets + 1];         // MSD path: bucket starts, then fill cursors
    uint32_t sorted[kSelSmemKeys];           // MSD path: key slots grouped by bucket
    uint32_t dig[kSelSmemKeys];              // MSD path: digest of each key slot (0xFFFFFFFF: invalid)
    uint32_t wtot[kSelThreads / 32];
    int64_t t_off[kSelCacheK];               // per group member (by rank): token offset, first hash segment
    int32_t t_sb[kSelCacheK];
    uint8_t bad[kSelCacheK];                 // predecessor link of member r is broken (not an exact extension)
};

// mode 0: trust hash-equal candidates (verified later by the scatter pass); mode 1: repair — accepts a candidate only
// after comparing tokens exactly.  NT threads per CTA; CTAs stride over the groups.
template <int NT>
__device__ void select_body(const MergeParams& p, int mode, SelectSmem& sm) {
    static_assert(NT == kSelThreads, "select_body is written for kSelThreads");
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = p.ctrl->n_groups;
    const bool weak = (p.flags & AJT_MERGE_WEAK_HASH) != 0;
    for (int g = blockIdx.x; g < G; g += gridDim.x) {
        const int gs = p.grp_start[g], k = p.grp_start[g + 1] - gs;
        const int32_t* gl = p.perm + gs;
        const int32_t* gln = p.glen + gs;
        if (k < 2) {
            if (tid == 0) { p.absorbed[gl[0]] = 0; p.owner_tl[gl[0]] = gl[0]; p.needv[gl[0]] = 0; p.tl_pos[gl[0]] = gs; }
            continue;
        }
        const int eb = p.grp_ent[g], c = p.grp_ent[g + 1] - eb;
        const bool cached = k <= kSelCacheK, small = c <= kSelSmemKeys;
        // ---- M2 (end): per timeline, exclusive prefix over its hash windows (in place), one warp per timeline
        // (mode 1 finds seg_part and ent_hash already final)
        for (int r = warp; r < k; r += NT / 32) {
            const int i = gl[r];
            const int sb = p.tl_rec[gs + r].x;
            const int64_t off = p.offsets[i];
            const int ns = mode == 0 ? (int)(((off + gln[r] - 1 + p.mis) >> kHSegLog) - ((off + p.mis) >> kHSegLog) + 1) : 0;
            if (cached && lane == 0) {
                sm.t_off[r] = off;
                sm.t_sb[r] = sb;
                sm.bad[r] = r > 0 && (p.link_bad[i] != 0 || gln[r - 1] > gln[r]);
            }
            uint64_t carry = 0;
            for (int s0 = 0; s0 < ns; s0 += 32) {
                const int s = s0 + lane;
                const uint64_t v = s < ns ? p.seg_part[sb + s] : 0;
                uint64_t inc = v;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const uint64_t t = __shfl_up_sync(0xffffffffu, inc, o);
                    if (lane >= o) inc += t;
                }
                if (s < ns) p.seg_part[sb + s] = carry + inc - v;
                carry += __shfl_sync(0xffffffffu, inc, 31);
            }
        }
        if (small)
            for (int b = tid; b <= kSelBuckets; b += NT) sm.start[b] = 0;
        __syncthreads();
        // ---- final keys: hash of T_i[0:L_a] = prefix of the windows before the one holding position L_a - 1 + its partial
        uint32_t* gdig = p.ent_dig + eb;
        uint32_t* gidx = p.ent_idx + eb;
        for (int x = tid; x < c; x += NT) {
            const int r = rank_of_local((uint32_t)x), a = x - r * (r + 1) / 2;
            const int64_t Lp = gln[a];
            uint32_t dg = 0xFFFFFFFFu;
            if (Lp <= gln[r]) {
                uint64_t h = p.ent_hash[eb + x];
                if (mode == 0) {
                    int64_t off;
                    int sb;
                    if (cached) { off = sm.t_off[r]; sb = sm.t_sb[r]; }
                    else { const int i = gl[r]; off = p.offsets[i]; sb = p.tl_rec[gs + r].x; }
                    const int64_t widx = ((off + Lp - 1 + p.mis) >> kHSegLog) - ((off + p.mis) >> kHSegLog);
                    h += p.seg_part[sb + widx];
                    if (weak) h &= 0xFull;
                    p.ent_hash[eb + x] = h;
                }
                dg = digest32(h, (int32_t)Lp);
                if (dg == 0xFFFFFFFFu) dg = 0xFFFFFFFEu;
            }
            if (small) {
                sm.dig[x] = dg;
                if (dg != 0xFFFFFFFFu) atomicAdd(&sm.start[dg >> (32 - kSelBucketBits)], 1u);
            } else {
                gdig[x] = dg;
                gidx[x] = (uint32_t)x;
            }
        }
        __syncthreads();
        // ---- M3: segmented radix sort of the group's keys by digest
        const uint32_t* sk = nullptr;   // global path: sorted digests / order
        const uint32_t* sv = nullptr;
        if (small) {
            // one MSD pass on the top 11 bits: exclusive scan of the 2048-bin histogram (8 bins per thread), then scatter
            uint32_t loc[kSelBuckets / NT], s = 0;
#pragma unroll
            for (int j = 0; j < kSelBuckets / NT; ++j) { loc[j] = sm.start[tid * (kSelBuckets / NT) + j]; s += loc[j]; }
            uint32_t inc = s;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += t;
            }
            if (lane == 31) sm.wtot[warp] = inc;
            __syncthreads();
            uint32_t run = inc - s;
#pragma unroll
            for (int w = 0; w < NT / 32; ++w)
                if (w < warp) run += sm.wtot[w];
#pragma unroll
            for (int j = 0; j < kSelBuckets / NT; ++j) { sm.start[tid * (kSelBuckets / NT) + j] = run; run += loc[j]; }
            if (tid == NT - 1) sm.start[kSelBuckets] = run;
            __syncthreads();
            for (int x = tid; x < c; x += NT) {
                const uint32_t dg = sm.dig[x];
                if (dg != 0xFFFFFFFFu) sm.sorted[atomicAdd(&sm.start[dg >> (32 - kSelBucketBits)], 1u)] = (uint32_t)x;
            }
            __syncthreads();   // start[b] now holds the END of bucket b (= start of b + 1)
        } else {
            uint32_t* kk[2] = {gidx, p.tmp_idx + eb};
            uint32_t* dd[2] = {gdig, p.tmp_dig + eb};
            int cur = 0;
            for (int shift = 0; shift < 32; shift += 8) {
                radix_pass<NT / 32>(dd[cur], kk[cur], dd[cur ^ 1], kk[cur ^ 1], c, shift, sm.sc);
                cur ^= 1;
                __syncthreads();
            }
            sk = dd[cur];   // after 4 passes cur == 0: digests are back in ent_dig (sorted), order in ent_idx
            sv = kk[cur];
        }
        // visit(dg, fn): fn(le) for every key slot of this group whose digest is dg (the equal-key run)
        auto visit = [&](uint32_t dg, auto fn) {
            if (small) {
                const uint32_t b = dg >> (32 - kSelBucketBits);
                const uint32_t x1 = sm.start[b], x0 = b ? sm.start[b - 1] : 0u;
                for (uint32_t x = x0; x < x1; ++x) {
                    const uint32_t le = sm.sorted[x];
                    if (sm.dig[le] == dg) fn(le);
                }
            } else {
                int lo = 0, hi = c;   // lower bound of dg in the sorted digests
                while (lo < hi) {
                    const int mid = (lo + hi) >> 1;
                    if (sk[mid] < dg) lo = mid + 1; else hi = mid;
                }
                for (int x = lo; x < c && sk[x] == dg; ++x) fn(sv[x]);
            }
        };
        // ---- M4: survivors and the Algorithm-1 owner (latest extender)
        for (int b = tid; b < k; b += NT) {
            const int j = gl[b];
            const int ef = eb + b * (b + 1) / 2 + b;        // full key of j
            const uint64_t H = p.ent_hash[ef];
            const int32_t L = gln[b];
            uint32_t dg = digest32(H, L);
            if (dg == 0xFFFFFFFFu) dg = 0xFFFFFFFEu;
            int best = -1;                                   // max rank of an extender
            visit(dg, [&](uint32_t le) {
                const int rb = rank_of_local(le);
                if (rb <= b || rb <= best) return;
                const int a = (int)le - rb * (rb + 1) / 2;
                if (gln[a] != L || p.ent_hash[eb + le] != H) return;
                if (mode == 1 && !tokens_extend(p, gl[rb], j)) return;
                best = rb;
            });
            p.absorbed[j] = best >= 0;
            p.owner_tl[j] = best >= 0 ? gl[best] : j;
            p.tl_pos[j] = gs + b;
        }
        __syncthreads();
        if (p.owner_rule == AJT_OWNER_LONGEST) {
            // the longest SURVIVING extender, then the lowest index (BASELINE.json north_star; reading M-3)
            for (int b = tid; b < k; b += NT) {
                const int j = gl[b];
                if (!p.absorbed[j]) continue;
                const int ef = eb + b * (b + 1) / 2 + b;
                const uint64_t H = p.ent_hash[ef];
                const int32_t L = gln[b];
                uint32_t dg = digest32(H, L);
                if (dg == 0xFFFFFFFFu) dg = 0xFFFFFFFEu;
                int best = p.tl_pos[p.owner_tl[j]] - gs;   // a surviving, (to be) verified extender: the fallback
                int32_t bestL = gln[best];
                visit(dg, [&](uint32_t le) {
                    const int rb = rank_of_local(le);
                    if (rb <= b || rb == best) return;
                    const int a = (int)le - rb * (rb + 1) / 2;
                    if (gln[a] != L || p.ent_hash[eb + le] != H) return;
                    const int i = gl[rb];
                    if (p.absorbed[i]) return;
                    const int32_t Li = gln[rb];
                    if (!(Li > bestL || (Li == bestL && rb < best))) return;
                    if (mode == 1 && !tokens_extend(p, i, j)) return;
                    best = rb;
                    bestL = Li;
                });
                p.cand[j] = gl[best];   // staged: owner_tl is still being read by other threads
            }
            __syncthreads();
            for (int b = tid; b < k; b += NT) {
                const int j = gl[b];
                if (p.absorbed[j]) p.owner_tl[j] = p.cand[j];
            }
        }
        // ---- M5, first half: T_j is a prefix of its owner T_o for certain if every predecessor link between them was
        // verified by the hash pass (prefix-of is transitive); only the other members are re-read by the scatter pass
        for (int b = tid; b < k; b += NT) {
            const int j = gl[b];
            bool nv = p.absorbed[j] != 0;
            if (nv && cached) {
                const int o = p.tl_pos[p.owner_tl[j]] - gs;
                nv = false;
                for (int r = b + 1; r <= o; ++r) nv |= sm.bad[r] != 0;
            }
            p.needv[j] = nv;
        }
        __syncthreads();
    }
}

__global__ void __launch_bounds__(kSelThreads) merge_select_kernel(const MergeParams p) {
    __shared__ SelectSmem sm;
    if (fatal(p)) return;
    select_body<kSelThreads>(p, 0, sm);
}

// ---------------------------------------------------------------------------------------- K6: compact (M6)

template <int NT>
__device__ void compact_body(const MergeParams& p, int mode, int64_t (*s_w)[2][NT / 32]) {
    const int tid = threadIdx.x, n = p.n;
    // one fused scan over the timelines: survivors (-> merged index), their scatter tiles, their lengths (-> offsets).
    // A merged sequence starting at merged offset mo is tiled on the 4-element grid of the OUTPUT arrays, so it needs
    // ceil((L + (mo & 3)) / kTile) tiles; (L + 3) bounds that without knowing mo (an empty extra tile exits at once).
    const I2 tot = block_scan2<NT>(
        n,
        [&](int i) {
            if (mode == 0 ? __ldg(p.absorbed + i) : p.absorbed[i]) return I2{0, 0};   // (mode 1: written earlier in this launch)
            const int64_t L = tl_len(p, i);
            return I2{((int64_t)1 << 32) | ((L + 3 + kTile - 1) / kTile), L};
        },
        [&](int i, int64_t exa, int64_t exb, int64_t va, int64_t) {
            if (!va) { p.midx[i] = -1; return; }
            const int m = (int)(exa >> 32);
            p.midx[i] = m;
            p.merged_origin[m] = i;
            p.merged_traj[m] = __ldg(p.traj_ids + i);
            p.merged_offsets[m] = exb;
            p.tile_base[m] = (int32_t)(exa & 0xffffffff);
        },
        s_w);
    const int M = (int)(tot.a >> 32);
    const int32_t ntiles = (int32_t)(tot.a & 0xffffffff);
#pragma unroll 4
    for (int i = tid; i < n; i += NT) p.owner[i] = p.midx[mode == 0 ? __ldg(p.owner_tl + i) : p.owner_tl[i]];
    if (tid == 0) {
        p.merged_offsets[M] = tot.b;
        p.tile_base[M] = ntiles;
        p.counts[0] = M;
        p.counts[1] = tot.b;
        p.ctrl->M = M;
        p.ctrl->N_out = tot.b;
        p.ctrl->n_tiles = ntiles;
        if (mode == 1) {
            p.ctrl->collision = 2;   // repair in progress: the scatter pass must not find another mismatch
            atomicOr(&p.ctrl->status, (uint32_t)AJT_STATUS_HASH_COLLISION);
        }
    }
}

__global__ void __launch_bounds__(1024) merge_compact_kernel(const MergeParams p) {
    __shared__ int64_t s_w[2][2][32];
    if (fatal(p)) {   // outputs are unspecified after a fatal status, but the counts a caller may chain on are not garbage
        if (threadIdx.x == 0) { p.counts[0] = 0; p.counts[1] = 0; }
        return;
    }
    compact_body<1024>(p, 0, s_w);
}

// ---------------------------------------------------------------------------------------- K5 + K7: verify + scatter (M5, M7)

// Warp task = one tile of kTile positions of one merged sequence, laid on the 4-element grid of the OUTPUT arrays so that
// tokens / src / old_logp leave as 16-byte stores and the mask as 4-byte stores.  Lane l holds positions
// qbase + 128 u + 4 l + e (u < 4, e < 4).  A warp takes a contiguous run of tiles, so the members of a merged sequence (the
// absorbed timelines it owns, found among the earlier timelines of its group) are gathered once per sequence into a
// per-warp shared-memory list {index, length, resp_start, token offset}, ascending.  Each member is compared against the
// survivor exactly (M5) and painted into the slot map in ascending order; slot 0 = nobody, c + 1 = member c, 33 = survivor.
constexpr int kMemCap = 32;
struct MemberList {
    int64_t jo[kMemCap];
    int32_t j[kMemCap], L[kMemCap], rs[kMemCap];
    uint8_t nv[kMemCap];
};

struct TileCtx {
    int s, Ls, rs_s, gs, rank_s;
    int64_t so, mo;
};

// Slow path for a sequence with more than kMemCap members: walks the group's earlier timelines for every tile.
template <bool kExplicit>
__device__ __noinline__ bool scatter_tile_generic(const MergeParams& p, const TileCtx c, int qbase, bool vec_ok) {
    constexpr int kU = kTile / 128;
    const int lane = threadIdx.x & 31;
    const int ql = qbase + 4 * lane;
    const int s = c.s, Ls = c.Ls;
    bool mismatch = false;
    int32_t x[kU][4], src[kU][4];
#pragma unroll
    for (int u = 0; u < kU; ++u)
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int q = ql + 128 * u + e;
            const bool v = q >= 0 && q < Ls;
            x[u][e] = v ? p.tokens[c.so + q] : 0;
            bool mk = false;
            if (v) mk = kExplicit ? (p.mask_in[c.so + q] != 0) : (q >= c.rs_s);
            src[u][e] = mk ? s : -1;
        }
    const int qlo = max(qbase, 0);
    for (int a0 = 0; a0 < c.rank_s; a0 += 32) {
        const int a = a0 + lane;
        int j = -1, Lj = 0;
        if (a < c.rank_s) {
            Lj = p.glen[c.gs + a];
            if (Lj > qlo) {
                j = p.perm[c.gs + a];
                if (p.owner_tl[j] != s) j = -1;
            }
        }
        unsigned hits = __ballot_sync(0xffffffffu, j >= 0);
        while (hits) {
            const int sl = __ffs(hits) - 1;
            hits &= hits - 1;
            const int jj = __shfl_sync(0xffffffffu, j, sl), Ljj = __shfl_sync(0xffffffffu, Lj, sl);
            const int64_t jo = p.offsets[jj];
            const int rs_j = kExplicit ? 0 : p.resp_start[jj];
#pragma unroll
            for (int u = 0; u < kU; ++u) {
                if (qbase + 128 * u >= Ljj) break;   // warp-uniform: the member ends before this step
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int q = ql + 128 * u + e;
                    if (q >= 0 && q < Ljj) {
                        if (p.tokens[jo + q] != x[u][e]) mismatch = true;     // exact verification (M5)
                        const bool mk = kExplicit ? (p.mask_in[jo + q] != 0) : (q >= rs_j);
                        if (mk) src[u][e] = max(src[u][e], jj);
                    }
                }
            }
        }
    }
    const int64_t dbase = c.mo + ql;   // multiple of 4
#pragma unroll
    for (int u = 0; u < kU; ++u) {
        const int q = ql + 128 * u;
        if (q >= Ls || q + 3 < 0) continue;
        const int64_t d = dbase + 128 * u;
        float lp[4] = {0.f, 0.f, 0.f, 0.f};
        if (p.merged_old_logp) {
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int sj = src[u][e];
                if (sj >= 0) lp[e] = p.old_logp_in[(sj == s ? c.so : p.offsets[sj]) + q + e];
            }
        }
        if (vec_ok && q >= 0 && q + 3 < Ls) {
            *reinterpret_cast<int4*>(p.merged_tokens + d) = make_int4(x[u][0], x[u][1], x[u][2], x[u][3]);
            *reinterpret_cast<int4*>(p.merged_src + d) = make_int4(src[u][0], src[u][1], src[u][2], src[u][3]);
            *reinterpret_cast<uint32_t*>(p.merged_mask + d) = (src[u][0] >= 0 ? 1u : 0u) | (src[u][1] >= 0 ? 0x100u : 0u) |
                                                              (src[u][2] >= 0 ? 0x10000u : 0u) | (src[u][3] >= 0 ? 0x1000000u : 0u);
            if (p.merged_old_logp) *reinterpret_cast<float4*>(p.merged_old_logp + d) = make_float4(lp[0], lp[1], lp[2], lp[3]);
        } else {
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                if (q + e >= 0 && q + e < Ls) {
                    p.merged_tokens[d + e] = x[u][e];
                    p.merged_src[d + e] = src[u][e];
                    p.merged_mask[d + e] = src[u][e] >= 0;
                    if (p.merged_old_logp) p.merged_old_logp[d + e] = lp[e];
                }
            }
        }
    }
    return mismatch;
}

template <bool kExplicit>
__device__ __forceinline__ bool scatter_tile_fast(const MergeParams& p, const TileCtx& c, int qbase, bool vec_ok,
                                                  const MemberList& ml, int cnt) {
    constexpr int kU = kTile / 128;
    constexpr int kSurv = kMemCap + 1;
    const int lane = threadIdx.x & 31;
    const int ql = qbase + 4 * lane;
    const int s = c.s, Ls = c.Ls;
    bool mismatch = false;
    const bool full = qbase >= 0 && qbase + kTile <= Ls;   // warp-uniform: every slot of the tile is a position of the sequence
    const int32_t* __restrict__ tok = p.tokens + c.so;
    // ---- uniform tile: every response region [rs_m, L_m) of a member (and the survivor's own) either covers the whole tile
    // or misses it, and nobody needs verifying here: one source for the whole tile.  Regions are hundreds of tokens long, so
    // most tiles are of this kind; they cost a plain copy instead of a per-element walk over the members.
    if (!kExplicit && full && vec_ok) {
        const int qhi = qbase + kTile;
        bool covers = false, partial = false;
        if (lane < cnt) {
            const int Lm = ml.L[lane], rsm = ml.rs[lane];
            covers = rsm <= qbase && Lm >= qhi;
            partial = (!covers && Lm > qbase && rsm < qhi) || (ml.nv[lane] && Lm > qbase);
        }
        const bool s_covers = c.rs_s <= qbase;
        if (!__any_sync(0xffffffffu, partial) && (s_covers || c.rs_s >= qhi)) {
            const unsigned cb = __ballot_sync(0xffffffffu, covers);
            const int sl = s_covers ? kSurv : (cb ? 32 - __clz(cb) : 0);
            const int32_t sj = sl == 0 ? -1 : (sl == kSurv ? s : ml.j[sl - 1]);
            const float* __restrict__ lps = p.old_logp_in + (sl == kSurv ? c.so : (sl ? ml.jo[sl - 1] : 0));
            const bool want_lp = p.merged_old_logp != nullptr && sl != 0;
            const bool tvec = (((uintptr_t)(tok + qbase)) & 15) == 0, lvec = want_lp && (((uintptr_t)(lps + qbase)) & 15) == 0;
            int4 xv[kU];
            float4 lv[kU];
#pragma unroll
            for (int u = 0; u < kU; ++u) {
                const int q = ql + 128 * u;
                if (tvec) xv[u] = __ldg(reinterpret_cast<const int4*>(tok + q));
                else xv[u] = make_int4(__ldg(tok + q), __ldg(tok + q + 1), __ldg(tok + q + 2), __ldg(tok + q + 3));
                lv[u] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (lvec) lv[u] = __ldg(reinterpret_cast<const float4*>(lps + q));
                else if (want_lp) lv[u] = make_float4(__ldg(lps + q), __ldg(lps + q + 1), __ldg(lps + q + 2), __ldg(lps + q + 3));
            }
            const int64_t d0 = c.mo + ql;
#pragma unroll
            for (int u = 0; u < kU; ++u) {
                const int64_t d = d0 + 128 * u;
                *reinterpret_cast<int4*>(p.merged_tokens + d) = xv[u];
                *reinterpret_cast<int4*>(p.merged_src + d) = make_int4(sj, sj, sj, sj);
                *reinterpret_cast<uint32_t*>(p.merged_mask + d) = sl ? 0x01010101u : 0u;
                if (p.merged_old_logp) *reinterpret_cast<float4*>(p.merged_old_logp + d) = lv[u];
            }
            return false;
        }
    }
    int32_t x[kU][4];
    int32_t slot[kU][4];
#pragma unroll
    for (int u = 0; u < kU; ++u)
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int q = ql + 128 * u + e;
            const bool v = full || (q >= 0 && q < Ls);
            x[u][e] = v ? tok[q] : 0;
            bool mk = false;
            if (v) mk = kExplicit ? (p.mask_in[c.so + q] != 0) : (q >= c.rs_s);
            slot[u][e] = mk ? kSurv : 0;
        }
    const int qlo = max(qbase, 0);
    for (int m = 0; m < cnt; ++m) {
        const int Lj = ml.L[m];
        if (Lj <= qlo) continue;                 // warp-uniform: the member ends before this tile
        const int rs_j = ml.rs[m];
        const int32_t* __restrict__ tj = p.tokens + ml.jo[m];
        const uint8_t* mkj = kExplicit ? p.mask_in + ml.jo[m] : nullptr;
        // all of the member's loads first (independent), then the compares: one memory latency per member, not one per element
        if (kExplicit || ml.nv[m]) {   // warp-uniform
            int32_t y[kU][4];
            uint8_t ym[kU][4];
#pragma unroll
            for (int u = 0; u < kU; ++u)
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int q = ql + 128 * u + e;
                    const bool in = q >= 0 && q < Lj;
                    y[u][e] = in ? tj[q] : x[u][e];
                    if (kExplicit) ym[u][e] = in ? mkj[q] : (uint8_t)0;
                }
#pragma unroll
            for (int u = 0; u < kU; ++u)
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int q = ql + 128 * u + e;
                    mismatch |= y[u][e] != x[u][e];     // exact verification (M5, second half)
                    const bool mk = kExplicit ? (ym[u][e] != 0) : (q >= rs_j && q < Lj);
                    if (mk) slot[u][e] = max(slot[u][e], m + 1);
                }
        } else {
#pragma unroll
            for (int u = 0; u < kU; ++u)
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int q = ql + 128 * u + e;
                    if (q >= rs_j && q < Lj) slot[u][e] = max(slot[u][e], m + 1);
                }
        }
    }
    // ---- outputs
    const int64_t dbase = c.mo + ql;   // multiple of 4
    float lp[kU][4];
    if (p.merged_old_logp) {
#pragma unroll
        for (int u = 0; u < kU; ++u)
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int sl = slot[u][e];
                lp[u][e] = 0.f;
                if (sl) lp[u][e] = p.old_logp_in[(sl == kSurv ? c.so : ml.jo[sl - 1]) + ql + 128 * u + e];
            }
    }
#pragma unroll
    for (int u = 0; u < kU; ++u) {
        const int q = ql + 128 * u;
        if (!full && (q >= Ls || q + 3 < 0)) continue;
        const int64_t d = dbase + 128 * u;
        int32_t sj[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int sl = slot[u][e];
            sj[e] = sl == 0 ? -1 : (sl == kSurv ? s : ml.j[sl - 1]);
        }
        if (vec_ok && (full || (q >= 0 && q + 3 < Ls))) {
            *reinterpret_cast<int4*>(p.merged_tokens + d) = make_int4(x[u][0], x[u][1], x[u][2], x[u][3]);
            *reinterpret_cast<int4*>(p.merged_src + d) = make_int4(sj[0], sj[1], sj[2], sj[3]);
            *reinterpret_cast<uint32_t*>(p.merged_mask + d) =
                (sj[0] >= 0 ? 1u : 0u) | (sj[1] >= 0 ? 0x100u : 0u) | (sj[2] >= 0 ? 0x10000u : 0u) | (sj[3] >= 0 ? 0x1000000u : 0u);
            if (p.merged_old_logp)
                *reinterpret_cast<float4*>(p.merged_old_logp + d) = make_float4(lp[u][0], lp[u][1], lp[u][2], lp[u][3]);
        } else {
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                if (q + e >= 0 && q + e < Ls) {
                    p.merged_tokens[d + e] = x[u][e];
                    p.merged_src[d + e] = sj[e];
                    p.merged_mask[d + e] = sj[e] >= 0;
                    if (p.merged_old_logp) p.merged_old_logp[d + e] = lp[u][e];
                }
            }
        }
    }
    return mismatch;
}

template <bool kExplicit>
__device__ void scatter_body(const MergeParams& p, int mode, MemberList* lists) {
    const int lane = threadIdx.x & 31;
    const int wglobal = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    const int ntiles = p.ctrl->n_tiles, M = p.ctrl->M;
    const int per = (ntiles + nwarps - 1) / nwarps;
    const int t_begin = wglobal * per, t_end = min(ntiles, t_begin + per);
    if (t_begin >= t_end) return;
    MemberList& ml = lists[threadIdx.x >> 5];
    const bool vec_ok = ((((uintptr_t)p.merged_tokens | (uintptr_t)p.merged_src | (uintptr_t)p.merged_old_logp) & 15) == 0) &&
                        (((uintptr_t)p.merged_mask & 3) == 0);
    bool mismatch = false;
    int m = warp_search_last_le(M, t_begin, [&](int x) { return p.tile_base[x]; });
    int cur_m = -1, cnt = 0, tb = 0;
    int tb_next = p.tile_base[m + 1];   // first tile of the next sequence: kept in a register, so that a tile inside a
                                        // sequence does not start with a dependent global load
    TileCtx c = {};
    for (int t = t_begin; t < t_end; ++t) {
        while (tb_next <= t) {
            ++m;
            tb_next = p.tile_base[m + 1];
        }
        if (m != cur_m) {
            cur_m = m;
            tb = p.tile_base[m];
            c.s = p.merged_origin[m];
            c.mo = p.merged_offsets[m];
            const int4 rec = p.tl_rec[p.tl_pos[c.s]];
            c.gs = rec.y;
            c.rank_s = rec.z;
            c.so = p.offsets[c.s];
            c.Ls = (int)(p.offsets[c.s + 1] - c.so);
            c.rs_s = kExplicit ? 0 : p.resp_start[c.s];
            // members of s: earlier timelines of its group that it owns, ascending
            __syncwarp();
            cnt = 0;
            for (int a0 = 0; a0 < c.rank_s; a0 += 32) {
                const int a = a0 + lane;
                int j = -1;
                if (a < c.rank_s) {
                    j = p.perm[c.gs + a];
                    if (p.owner_tl[j] != c.s) j = -1;
                }
                const unsigned bal = __ballot_sync(0xffffffffu, j >= 0);
                const int pos = cnt + __popc(bal & ((1u << lane) - 1u));
                if (j >= 0 && pos < kMemCap) {
                    ml.j[pos] = j;
                    ml.L[pos] = p.glen[c.gs + a];
                    ml.rs[pos] = kExplicit ? 0 : p.resp_start[j];
                    ml.jo[pos] = p.offsets[j];
                    ml.nv[pos] = p.needv[j];
                }
                cnt += __popc(bal);
            }
            __syncwarp();
        }
        const int qbase = (t - tb) * kTile - (int)(c.mo & 3);   // position of the tile's first slot (may be -3..-1)
        if (qbase >= c.Ls) continue;
        if (cnt <= kMemCap) mismatch |= scatter_tile_fast<kExplicit>(p, c, qbase, vec_ok, ml, cnt);
        else mismatch |= scatter_tile_generic<kExplicit>(p, c, qbase, vec_ok);
    }
    if (__any_sync(0xffffffffu, mismatch) && lane == 0) {
        if (mode == 0) atomicExch(&p.ctrl->collision, 1);
        else atomicOr(&p.ctrl->status, (uint32_t)AJT_STATUS_INTERNAL);
    }
}

constexpr int kScatThreads = 256;
__global__ void __launch_bounds__(kScatThreads, 4) merge_scatter_kernel(const MergeParams p) {
    __shared__ MemberList lists[kScatThreads / 32];
    if (fatal(p)) return;
    if (p.mask_in) scatter_body<true>(p, 0, lists);
    else scatter_body<false>(p, 0, lists);
}

// ---------------------------------------------------------------------------------------- exact repair (M5)

// Cooperative launch; every CTA returns at once unless the scatter pass saw a hash-equal, token-different pair.
__global__ void __launch_bounds__(kSelThreads) merge_repair_kernel(const MergeParams p) {
    __shared__ SelectSmem sm;
    __shared__ int64_t s_w[2][2][kSelThreads / 32];
    if (fatal(p) || p.ctrl->collision == 0) return;
    cg::grid_group grid = cg::this_grid();
    select_body<kSelThreads>(p, 1, sm);
    grid.sync();
    if (blockIdx.x == 0) compact_body<kSelThreads>(p, 1, s_w);
    grid.sync();
    MemberList* lists = reinterpret_cast<MemberList*>(&sm);   // the select scratch is free again
    static_assert(sizeof(SelectSmem) >= sizeof(MemberList) * (kSelThreads / 32), "member lists fit in the select scratch");
    if (p.mask_in) scatter_body<true>(p, 1, lists);
    else scatter_body<false>(p, 1, lists);
}

}  // namespace

extern "C" size_t ajt_merge_workspace_bytes(int32_t n, int64_t n_tokens) {
    if (n < 0 || n_tokens < 0) return 0;
    return merge_ws_layout(n, n_tokens).ent + a256(((size_t)64 * (size_t)n + 4096) * 32);
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
    for (int k = 0; k < 6; ++k) p.gbuf[k] = reinterpret_cast<uint32_t*>(b + ws.gbuf[k]);
    p.perm = reinterpret_cast<int32_t*>(b + ws.perm);
    p.glen = reinterpret_cast<int32_t*>(b + ws.glen);
    p.grp_start = reinterpret_cast<int32_t*>(b + ws.grp_start);
    p.grp_ent = reinterpret_cast<int32_t*>(b + ws.grp_ent);
    p.tl_rec = reinterpret_cast<int4*>(b + ws.tl_rec);
    p.tl_pos = reinterpret_cast<int32_t*>(b + ws.tl_pos);
    p.seg_part = reinterpret_cast<uint64_t*>(b + ws.seg_part);
    p.absorbed = b + ws.absorbed;
    p.link_bad = b + ws.link_bad;
    p.needv = b + ws.needv;
    p.owner_tl = reinterpret_cast<int32_t*>(b + ws.owner_tl);
    p.cand = reinterpret_cast<int32_t*>(b + ws.cand);
    p.midx = reinterpret_cast<int32_t*>(b + ws.midx);
    p.tile_base = reinterpret_cast<int32_t*>(b + ws.tile_base);
    // everything after the fixed part holds the per-key arrays; their capacity follows from the size given
    size_t eo = ws.ent;
    if (workspace_bytes < eo + 5 * 256 + ((size_t)n + 1024) * kEntBytes) return AJT_ERR_WORKSPACE_TOO_SMALL;
    const size_t ecap = (workspace_bytes - eo - 5 * 256) / kEntBytes;
    p.E_cap = (int32_t)(ecap > (size_t)INT32_MAX ? (size_t)INT32_MAX : ecap);
    p.ent_hash = reinterpret_cast<uint64_t*>(b + eo); eo += a256((size_t)p.E_cap * 8);
    p.ent_dig = reinterpret_cast<uint32_t*>(b + eo); eo += a256((size_t)p.E_cap * 4);
    p.ent_idx = reinterpret_cast<uint32_t*>(b + eo); eo += a256((size_t)p.E_cap * 4);
    p.tmp_dig = reinterpret_cast<uint32_t*>(b + eo); eo += a256((size_t)p.E_cap * 4);
    p.tmp_idx = reinterpret_cast<uint32_t*>(b + eo); eo += a256((size_t)p.E_cap * 4);
    if (eo > workspace_bytes) return AJT_ERR_WORKSPACE_TOO_SMALL;
    p.nseg_cap = nseg_capacity(n, n_tokens);
    p.mis = (int32_t)(((uintptr_t)tokens >> 2) & 3);

    if (n == 0) {
        if (cudaMemsetAsync(p.ctrl, 0, sizeof(AjtCtrl), stream) != cudaSuccess) return AJT_ERR_CUDA;
        if (cudaMemsetAsync(counts, 0, 2 * sizeof(int64_t), stream) != cudaSuccess) return AJT_ERR_CUDA;
        if (cudaMemsetAsync(merged_offsets, 0, sizeof(int64_t), stream) != cudaSuccess) return AJT_ERR_CUDA;
        return AJT_OK;
    }
    // per-device launch facts (attribute opt-in, co-resident grid of the cooperative repair kernel): looked up once
    static int s_repair_grid[64] = {0};
    if (dev < 0 || dev >= 64) return AJT_ERR_UNSUPPORTED;
    if (s_repair_grid[dev] == 0) {
        if (cudaFuncSetAttribute(merge_group_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 6 * ((kGrpSmemN + 32) & ~31) * 4) !=
            cudaSuccess)
            return AJT_ERR_CUDA;
        int per_sm = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, merge_repair_kernel, kSelThreads, 0) != cudaSuccess || per_sm < 1)
            return AJT_ERR_CUDA;
        s_repair_grid[dev] = num_sms * (per_sm < 4 ? per_sm : 4);
    }
    if (n <= kGrpSmemN) merge_group_small_kernel<<<1, 1024, 6 * (((size_t)n + 32) & ~(size_t)31) * 4, stream>>>(p);
    else merge_group_kernel<false><<<1, 1024, 0, stream>>>(p);
    merge_hash_kernel<<<num_sms * 3, 256, 0, stream>>>(p);
    merge_select_kernel<<<num_sms * 4, kSelThreads, 0, stream>>>(p);
    merge_compact_kernel<<<1, 1024, 0, stream>>>(p);
    merge_scatter_kernel<<<num_sms * 4, kScatThreads, 0, stream>>>(p);
    void* args[] = {(void*)&p};
    if (cudaLaunchCooperativeKernel((const void*)merge_repair_kernel, dim3((unsigned)s_repair_grid[dev]), dim3(kSelThreads), args, 0,
                                    stream) != cudaSuccess)
        return AJT_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? AJT_OK : AJT_ERR_CUDA;
}
