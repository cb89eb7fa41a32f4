// Stage (a): timeline merging (Algorithm 1) on flat token streams, sm_100a.
//
// Definition: DESIGN.md "O-M".  Pipeline (rows M1-M7 of the scope table), 7 launches on one
// stream, no host round trip, no cooperative launch (the call can be captured in a CUDA graph); kernels 2-7 are programmatic
// dependents of their predecessor (griddepcontrol), so their launch latency overlaps its tail:
//   K1  merge_group_fast_kernel  M1  one CTA, everything in shared memory (n <= 7936): trajectory ids go through a hash
//                                    table (atomicCAS), groups are laid out by a scan over its slots, members are placed
//                                    with an atomic cursor and put in input order by a bitonic network per warp.  Emits, by
//                                    SORTED POSITION, {timeline, length, token offset, first hash slice, group start, group
//                                    size, first key slot}.  merge_group_radix_kernel (stable LSD radix sort through the
//                                    workspace) does the same for larger batches.
//   K1b merge_units_kernel       M1  the hash pass's work list, built over the whole GPU: chunks of 8 consecutive ranks of a
//                                    group x slices of 508 positions up to the chunk's longest member.
//   K2  merge_hash_kernel        M2  warp per unit (dynamic ticket): the warp streams the SAME 508 positions of the chunk's
//                                    members, in rank order, through a warp-private ring of 2 KB slots, one bulk async copy
//                                    (TMA, 1-D) of the aligned superset each.  Prefix hash in the ring mod 2^32,
//                                    F_i(p) = sum_{q<p} x_q W^q: weights per slot element, one REDUX per slice total, the
//                                    member's shift applied afterwards; keys = masked partial sums where an earlier
//                                    member's length falls into the slice.
//                                M5  (first half) member r is compared EXACTLY with member r - 1 on the way, slot against
//                                    slot: a difference marks the link r-1 -> r broken.  Every token is loaded from DRAM
//                                    once.
//   K3  merge_select_kernel      M2  (end) one CTA per group: exclusive prefix of each member's slice totals -> final keys
//                                M3  segmented radix sort of the group's (hash, length) keys by a 32-bit digest: one MSD
//                                    pass on the top 11 bits in shared memory (<= 2048 keys), 4 LSD passes through global
//                                    memory above that
//                                M4  per timeline: its equal-key run gives the hash-equal extenders; survivor flag,
//                                    Algorithm-1 owner (latest extender), under LONGEST the longest surviving extender
//                                M5  (second half) a candidate is ACCEPTED only if an unbroken chain of verified links
//                                    leads to it (prefix-of is transitive) or after an exact warp-cooperative token
//                                    comparison; a hash-equal candidate that fails is skipped
//                                    (AJT_STATUS_HASH_COLLISION, informational).  Results are exact whatever the hash
//                                    does (AJT_MERGE_WEAK_HASH degrades it to 4 bits to test this).  Then per survivor:
//                                    its member list and its SEGMENTS (maximal runs of positions with one source of mask /
//                                    log-prob), warp-cooperatively.
//   K4  merge_compact_kernel     M6  one CTA scans the timelines once: survivors in original order -> merged_offsets /
//                                    origin / traj, owner, first segment of every merged sequence
//   K5  merge_plan_kernel        M7  segments rebased to output positions (one 32-byte record each), and for every tile
//                                    of 512 OUTPUT positions the first segment that touches it
//   K6  merge_scatter_kernel     M7  warp per output tile: bulk async copies of the tile's source pieces into shared
//                                    memory, then 16-byte stores of tokens / old_logp / src / mask straight from registers
//                                    -- whatever the alignment of the sources
#include "ajt_common.cuh"
#include "../../include/ajt_test.h"

namespace {

using namespace ajt;

constexpr int kVT = 4;              // 16-byte vectors of a hash slot per lane (8 = 4 KB slots of 1,020 positions: 127 registers,
                                   // 2 CTAs per SM, hash pass 70 instead of 72-76 us, the merge inside the bench step unchanged)
constexpr int kSl = 128 * kVT - 4;           // hash slice: 508 token positions; with up to 3 elements of misalignment a slice is
                                   // exactly 128 aligned 16-byte vectors = 4 per lane
__host__ __device__ __forceinline__ int slices_of(int L) { return (L + kSl - 1) / kSl; }
__host__ __device__ __forceinline__ int slice_at(int pos) { return pos / kSl; }
constexpr int kTS = 512;           // scatter tile: 512 output positions = 16 per lane
constexpr int kTSLog = 9;
constexpr uint32_t kW = 0x9E3779B1u;   // odd multiplier of the prefix hash's 32-bit position weights
constexpr uint32_t cpow32(uint32_t b, uint32_t e) {
    uint32_t r = 1;
    for (; e; e >>= 1, b *= b)
        if (e & 1) r *= b;
    return r;
}
constexpr uint32_t kW128 = cpow32(kW, 128);
constexpr uint32_t kWSl = cpow32(kW, kSl);
constexpr uint32_t kWinv = cpow32(kW, 0x7fffffffu);   // W^-1 mod 2^32 (the odd residues have exponent 2^30)
static_assert(kW * kWinv == 1u, "inverse of the hash multiplier");
constexpr uint32_t kFatal = AJT_STATUS_BAD_OFFSETS | AJT_STATUS_ZERO_LEN | AJT_STATUS_PROBE_CAPACITY;
constexpr int kSelThreads = 256;
constexpr int kSelSmemKeys = 2048;  // groups with more keys than this sort through global memory
constexpr int kSelBucketBits = 11;
constexpr int kSelBuckets = 1 << kSelBucketBits;
constexpr int kSelCacheK = 256;     // per-member decision state of groups up to this size lives in shared memory
constexpr int kGrpSmemN = 7936;     // batches up to this many timelines are grouped entirely in shared memory
constexpr int32_t kSrcNone = -1;      // segment source: nobody (mask 0)
constexpr int32_t kSrcExplicit = -2;  // segment source: decided per token from the explicit masks of the members

struct __align__(16) GSeg {   // one constant-source run of the merged output
    int64_t out_start;        // first output position
    int64_t tok_delta;        // token source index = output position + tok_delta
    int64_t lp_delta;         // log-prob source index = output position + lp_delta (src >= 0); explicit: first member slot
    int32_t src;              // supplying timeline, kSrcNone or kSrcExplicit
    int32_t aux;              // explicit: number of members
};
static_assert(sizeof(GSeg) == 32, "GSeg is one 32-byte record");

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
    uint32_t* gbuf[6];     // [n+2] each: the radix group kernel's work arrays (n > kGrpSmemN)
    int32_t* perm;         // [n] sorted position -> timeline index (groups contiguous, input order inside a group)
    int32_t* glen;         // [n] sorted position -> timeline length
    int64_t* goff;         // [n] sorted position -> token offset
    int4* tl_rec;          // [n] BY SORTED POSITION: {first hash slice, group start (sorted position), members of the group, first key slot of the timeline}
    uint8_t* lbad;         // [n] BY SORTED POSITION: the member differs from its in-group predecessor on that one's positions (exact)
    int4* grp_rec;         // [G+1] {group start, members, first key slot, first hash unit}
    int4* unit_rec;        // [slice_cap] hash units {group start (sorted position), first rank of the chunk, members of the group, slice}
    uint64_t* seg_part;    // [slice_cap] per (member, slice) hash totals, then exclusive prefixes per member
    uint64_t* ent_hash;    // [E_cap] key slot (r, a), a = 0..r: in-slice partial, then the final prefix hash
    uint32_t* ent_dig;     // [E_cap] global sort path: digests / order ping-pong
    uint32_t* ent_idx;     // [E_cap]
    uint32_t* tmp_dig;     // [E_cap]
    uint32_t* tmp_idx;     // [E_cap]
    uint2* cinfo;          // [n] by timeline, for the compaction: {1 << 24 | segments, length} of a survivor, {0, 0} of an absorbed one
    int32_t* owner_tl;     // [n] owning timeline (itself for survivors)
    int32_t* midx;         // [n] merged index of survivors, -1 otherwise
    int32_t* sel[8];       // [n] each, by sorted position: decision state of groups larger than kSelCacheK
    int2* sel_q;           // [n] by sorted position: their verification queue
    int32_t* mem_list;     // [n] members of every survivor (timeline indices, ascending), grouped by survivor
    int4* sv_rec;          // [n] by timeline, survivors only: {first member slot, members, first relative segment, segments}
    int2* rseg;            // [2n] relative segments {first position, source}
    int32_t* gseg_base;    // [M+1] first global segment of each merged sequence
    GSeg* gseg;            // [2n+1] global segments, ascending output position; the last one is a sentinel at N_out
    int32_t* tile_seg;     // [tile_cap] segment holding the first position of each output tile
    int32_t E_cap;
    int32_t slice_cap;
    int32_t mis;           // (address of tokens / 4) mod 4: element misalignment of the token array vs 16 bytes
    int32_t slim;          // the group kernel left {timeline | group << 16, first slice} in sel_q: the units kernel writes the records
};

struct MergeWs {
    size_t ctrl, gbuf[6], perm, glen, goff, tl_rec, lbad, grp_rec, unit_rec, seg_part, absorbed, owner_tl, midx, sel[8],
        sel_q, mem_list, sv_rec, rseg, gseg_base, gseg, tile_seg, ent;
};
__host__ inline size_t a256(size_t x) { return (x + 255) & ~(size_t)255; }
__host__ inline int64_t slice_capacity(int32_t n, int64_t N) { return N / kSl + (int64_t)n + 2; }

__host__ MergeWs merge_ws_layout(int32_t n, int64_t N) {
    MergeWs w;
    size_t o = 0;
    const size_t n4 = a256(((size_t)n + 2) * 4), n8 = a256(((size_t)n + 2) * 8), n16 = a256(((size_t)n + 2) * 16);
    const size_t sc = (size_t)slice_capacity(n, N);
    w.ctrl = o; o += 256;
    for (int k = 0; k < 6; ++k) { w.gbuf[k] = o; o += n > kGrpSmemN ? n4 : 0; }
    w.perm = o; o += n4; w.glen = o; o += n4; w.goff = o; o += n8;
    w.tl_rec = o; o += n16;
    w.lbad = o; o += a256((size_t)n + 2);
    w.grp_rec = o; o += n16;
    w.unit_rec = o; o += a256(sc * 16);
    w.seg_part = o; o += a256(sc * 8);
    w.absorbed = o; o += n8;   // (cinfo)
    w.owner_tl = o; o += n4; w.midx = o; o += n4;
    for (int k = 0; k < 8; ++k) { w.sel[k] = o; o += n4; }
    w.sel_q = o; o += n8;
    w.mem_list = o; o += n4;
    w.sv_rec = o; o += n16;
    w.rseg = o; o += a256(((size_t)n + 1) * 16);
    w.gseg_base = o; o += n4;
    w.gseg = o; o += a256(((size_t)2 * n + 2) * sizeof(GSeg));
    w.tile_seg = o; o += a256(((size_t)(N >> kTSLog) + 2) * 4);
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
__device__ __forceinline__ int64_t shfl_i64(int64_t v, int src) {
    const uint32_t lo = __shfl_sync(0xffffffffu, (uint32_t)v, src), hi = __shfl_sync(0xffffffffu, (uint32_t)((uint64_t)v >> 32), src);
    return (int64_t)(((uint64_t)hi << 32) | lo);
}
template <class T>
__device__ __forceinline__ T ldcg(const T* p) { return __ldcg(p); }

// ---------------------------------------------------------------------------------------- block-level building blocks

// Exclusive scan of the pair f(i) = (a, b), i in [0,n), by one CTA of NT threads; g(i, ex_a, ex_b, a, b) consumes it.
// Each thread owns IPT consecutive items of a tile of NT * IPT (their loads are independent: one memory round trip per
// tile), so a tile costs one warp scan, one __syncthreads and one shuffle scan of the NT / 32 warp totals (double-buffered).
// Returns the totals to every thread.
struct I2 {
    int64_t a, b;
};
template <int NT, int IPT, class F, class G>
__device__ __forceinline__ I2 block_scan2(int n, F f, G g, int64_t (*s_w)[2][NT / 32]) {
    static_assert(NT / 32 <= 32, "warp totals are scanned by one warp's lanes");
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    I2 base = {0, 0};
    int buf = 0;
    for (int i0 = 0; i0 < n; i0 += NT * IPT, buf ^= 1) {
        const int b0 = i0 + tid * IPT;
        I2 v[IPT];
        int64_t sa = 0, sb = 0;
#pragma unroll
        for (int k = 0; k < IPT; ++k) v[k] = b0 + k < n ? f(b0 + k) : I2{0, 0};
#pragma unroll
        for (int k = 0; k < IPT; ++k) {
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
        for (int k = 0; k < IPT; ++k) {
            if (b0 + k < n) g(b0 + k, ra, rb, v[k].a, v[k].b);
            ra += v[k].a;
            rb += v[k].b;
        }
        base.a += ta; base.b += tb;
    }
    __syncthreads();
    return base;
}
template <int NT, int IPT, class F, class G>
__device__ __forceinline__ int64_t block_scan(int n, F f, G g, int64_t (*s_w)[2][NT / 32]) {
    return block_scan2<NT, IPT>(
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
// digits find each other (peers8) and the lowest lane of each peer set adds the set size to cnt[w][digit].  Offsets:
// one thread per digit turns the NW counts into running offsets, one warp scans the 256 digit totals.  Scatter: the same
// rounds again, position = digit base + warp offset + rank in peer set.  Four __syncthreads per pass, whatever n is.
template <int NW>
__device__ __forceinline__ void radix_pass(const uint32_t* kin, const uint32_t* vin, uint32_t* kout, uint32_t* vout, int n,
                                           int shift, RadixScratch<NW>& sc, int nbits = 8) {
    const uint32_t dmask = (1u << nbits) - 1u;
    constexpr int NT = NW * 32;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int x = tid; x < NW * 256; x += NT) (&sc.cnt[0][0])[x] = 0;
    __syncthreads();
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
}

// Fatal status found while grouping: the later kernels return at once; the counts a caller may chain on are not garbage.
__device__ __forceinline__ void group_fail(const MergeParams& p, uint32_t bits) {
    atomicOr(&p.ctrl->status, bits);
    p.counts[0] = 0;
    p.counts[1] = 0;
    p.merged_offsets[0] = 0;
}

constexpr int kChunk = 8;      // hash units: a group's members are cut into chunks of this many consecutive ranks ...
constexpr int kSliceBlk = 1;   // ... and every slice of a chunk is a unit of its own: one warp's critical path is ~9 member-slices
static_assert(kSliceBlk == 1, "the hash kernel takes one slice per unit");

// ---------------------------------------------------------------------------------------- K1: group (M1)

constexpr uint32_t kEmpty = 0xFFFFFFFFu;

// n <= kGrpSmemN.  Dynamic shared memory (H = hash-table slots, passed by the host; G <= n groups):
//   B1 [H+2] u32  table keys              -> members per group -> group starts (sorted position, exclusive scan)
//   B2 [H+2] u16  group of each table slot -> timeline by sorted position
//   B3 [n+2] u32  length by timeline
//   B4 [n+2] u32  per-group cursor        -> key slots per group (-> exclusive scan)
//   B5 [n+2] u32  longest member of group -> hash units per group (-> exclusive scan)
//   B6 [n]   u16  table slot by timeline  -> group by timeline
//   B7 [n]   u16  members as placed (unordered inside a group)
//   B9 [n+2] u32  first hash slice by sorted position
// One SM does all of this, so what counts is shared-memory wavefronts and dependent global round trips (~0.8 us each): the
// members of a group are put in order by a warp-wide bitonic network (shuffles), and every global store is coalesced.
__global__ void __launch_bounds__(1024) merge_group_fast_kernel(const MergeParams p, const int H) {
    extern __shared__ __align__(16) uint8_t g_dyn[];
    __shared__ int64_t s_w[2][2][32];
    __shared__ uint32_t s_bad, s_ng;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, n = p.n;
    uint32_t* const B1 = reinterpret_cast<uint32_t*>(g_dyn);
    uint16_t* const B2 = reinterpret_cast<uint16_t*>(B1 + (H + 2));
    uint32_t* const B3 = reinterpret_cast<uint32_t*>(B2 + ((H + 3) & ~1));
    uint32_t* const B4 = B3 + (n + 2);
    uint32_t* const B5 = B4 + (n + 2);
    uint32_t* const B9 = B5 + (n + 2);
    uint16_t* const B6 = reinterpret_cast<uint16_t*>(B9 + (n + 2));
    uint16_t* const B7 = B6 + ((n + 1) & ~1);
    uint16_t* const B8 = B2;
    if (tid < (int)(sizeof(AjtCtrl) / 4)) reinterpret_cast<uint32_t*>(p.ctrl)[tid] = 0;   // fresh control block
    if (tid == 0) { s_bad = 0; s_ng = 0; }
#pragma unroll 1
    for (int s = tid; s < H + 2; s += 1024) B1[s] = kEmpty;
#pragma unroll 1
    for (int g = tid; g < n + 2; g += 1024) { B4[g] = 0; B5[g] = 0; }
    __syncthreads();
    // ---- validate offsets; trajectory id -> table slot; the thread that claims a slot numbers the group
    uint32_t bad = 0;
#pragma unroll 1
    for (int i0 = tid; i0 < n; i0 += 8 * 1024) {
        int64_t a[8], b[8];
        uint32_t t[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {   // all loads of eight timelines in flight at once: one cold round trip (~2 us)
            const int i = i0 + u * 1024;
            const bool v = i < n;
            a[u] = v ? __ldg(p.offsets + i) : 0;
            b[u] = v ? __ldg(p.offsets + i + 1) : 1;
            t[u] = v ? (uint32_t)__ldg(p.traj_ids + i) : 0u;
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int i = i0 + u * 1024;
            if (i >= n) break;
            if (b[u] < a[u] || b[u] - a[u] > (int64_t)INT32_MAX) bad |= AJT_STATUS_BAD_OFFSETS;
            else if (b[u] == a[u]) bad |= AJT_STATUS_ZERO_LEN;
            uint32_t h = (uint32_t)H;   // the id that doubles as the empty marker has a slot of its own
            uint32_t prev = kEmpty;
            if (t[u] != kEmpty) {
                h = __umulhi(t[u] * 0x9E3779B1u, (uint32_t)H);
                while (true) {
                    prev = atomicCAS(&B1[h], kEmpty, t[u]);
                    if (prev == kEmpty || prev == t[u]) break;
                    h = h + 1 == (uint32_t)H ? 0u : h + 1;
                }
            } else {
                prev = atomicCAS(&B1[h], kEmpty, 0u);
            }
            if (prev == kEmpty) B2[h] = (uint16_t)atomicAdd(&s_ng, 1u);
            B6[i] = (uint16_t)h;
            B3[i] = (uint32_t)a[u];
        }
    }
    if (tid == 0 && (__ldg(p.offsets) != 0 || __ldg(p.offsets + n) != p.N)) bad |= AJT_STATUS_BAD_OFFSETS;
    if (tid == 0) B3[n] = (uint32_t)p.N;
    bad = __reduce_or_sync(0xffffffffu, bad);
    if ((tid & 31) == 0 && bad) atomicOr(&s_bad, bad);
    __syncthreads();
    if (s_bad) {
        if (tid == 0) group_fail(p, s_bad);
        return;
    }
    const int G = (int)s_ng;
    // ---- the table keys are done: B1 becomes the per-group member count
#pragma unroll 1
    for (int i = tid; i < n; i += 1024) B6[i] = B2[B6[i]];
#pragma unroll 1
    for (int g = tid; g <= G; g += 1024) B1[g] = 0;
    __syncthreads();
#pragma unroll 1
    for (int i = tid; i < n; i += 1024) {
        const uint32_t g = B6[i];
        atomicAdd(&B1[g], 1u);
    }
    __syncthreads();
    block_scan<1024, 8>(
        G + 1, [&](int g) { return g < G ? B1[g] : 0u; }, [&](int g, int64_t ex, int64_t) { B1[g] = (uint32_t)ex; }, s_w);
    // ---- place the members (any order inside a group) ...
#pragma unroll 1
    for (int i = tid; i < n; i += 1024) {
        const uint32_t g = B6[i];
        B7[B1[g] + atomicAdd(&B4[g], 1u)] = (uint16_t)i;
    }
    __syncthreads();
    // ---- ... and put them in input order, one warp per group: a bitonic network over the lanes for groups of up to 32
    // (15 shuffles), ranking by counting (members are read as broadcasts) for larger ones
#pragma unroll 1
    for (int g0 = warp; g0 < G; g0 += 2 * 32) {   // two groups per warp at a time: two independent shuffle chains
        uint32_t gs[2], k[2], v0[2], v1[2];       // a group of up to 64: elements lane and lane + 32
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const int g = g0 + 32 * u;
            gs[u] = g < G ? B1[g] : 0u;
            k[u] = g < G ? B1[g + 1] - gs[u] : 0u;
            const bool net = k[u] <= 64;
            v0[u] = net && (uint32_t)lane < k[u] ? B7[gs[u] + lane] : 0xFFFFu;
            v1[u] = net && (uint32_t)lane + 32 < k[u] ? B7[gs[u] + lane + 32] : 0xFFFFu;
        }
        const bool wide = k[0] > 32 || k[1] > 32;   // warp-uniform: the 32-wide network is enough otherwise
#pragma unroll
        for (int sz = 2; sz <= 64; sz <<= 1) {
            if (sz == 64 && !wide) break;
#pragma unroll
            for (int st = sz >> 1; st > 0; st >>= 1) {
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    if (st == 32) {   // partner of element e is e ^ 32: the lane's other register; block of 64 ascending
                        const uint32_t lo = min(v0[u], v1[u]), hi = max(v0[u], v1[u]);
                        v0[u] = lo; v1[u] = hi;
                    } else {
                        const uint32_t o0 = __shfl_xor_sync(0xffffffffu, v0[u], st), o1 = __shfl_xor_sync(0xffffffffu, v1[u], st);
                        const bool lower = (lane & st) == 0;
                        // direction of the block of size sz that holds the element: ascending iff (e & sz) == 0
                        const bool up0 = sz == 64 ? true : (lane & sz) == 0;
                        const bool up1 = sz == 64 ? true : (sz == 32 ? false : (lane & sz) == 0);
                        v0[u] = (lower == up0) ? min(v0[u], o0) : max(v0[u], o0);
                        v1[u] = (lower == up1) ? min(v1[u], o1) : max(v1[u], o1);
                    }
                }
            }
        }
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            if (k[u] <= 64) {
                if ((uint32_t)lane < k[u]) B8[gs[u] + lane] = (uint16_t)v0[u];
                if ((uint32_t)lane + 32 < k[u]) B8[gs[u] + lane + 32] = (uint16_t)v1[u];
            } else {
                for (uint32_t m = lane; m < k[u]; m += 32) {
                    const uint32_t i = B7[gs[u] + m];
                    uint32_t r = 0;
#pragma unroll 4
                    for (uint32_t x = 0; x < k[u]; ++x) r += B7[gs[u] + x] < i ? 1u : 0u;
                    B8[gs[u] + r] = (uint16_t)i;
                }
            }
        }
    }
    __syncthreads();
    // ---- key slots and hash units by group (two scans), hash slices by sorted position (one scan)
    const int64_t E = block_scan<1024, 8>(
        G + 1, [&](int g) { const int64_t k = g < G ? B1[g + 1] - B1[g] : 0; return k * (k + 1) / 2; },
        [&](int g, int64_t ex, int64_t) { B4[g] = (uint32_t)min(ex, (int64_t)INT32_MAX); }, s_w);
    if (E > (int64_t)p.E_cap) {   // (slices and units always fit: the workspace is sized for their worst case)
        if (tid == 0) group_fail(p, (uint32_t)AJT_STATUS_PROBE_CAPACITY);
        return;
    }
    const int64_t nslice = block_scan<1024, 8>(
        n,
        [&](int pos) {
            const uint32_t i = B8[pos], g = B6[i];
            return B1[g + 1] - B1[g] < 2 ? 0u : (uint32_t)slices_of((int)(B3[i + 1] - B3[i]));
        },
        [&](int pos, int64_t ex, int64_t) { B9[pos] = (uint32_t)ex; }, s_w);
    // ---- by sorted position: {timeline | group << 16, first hash slice}, 8 bytes.  One SM stores slowly (the full 37-byte
    // records cost 8 us here), so merge_units_kernel expands these into tl_rec / perm / glen / goff / lbad over the whole GPU.
#pragma unroll 2
    for (int pos = tid; pos < n; pos += 1024) {
        const uint32_t i = B8[pos], g = B6[i];
        p.sel_q[pos] = make_int2((int)(i | (g << 16)), (int)B9[pos]);   // n <= 7936 < 2^13: both fit 16 bits
    }
#pragma unroll 1
    for (int g = tid; g <= G; g += 1024)
        p.grp_rec[g] = make_int4((int)B1[g], g < G ? (int)(B1[g + 1] - B1[g]) : 0, (int)B4[g], 0);
    if (tid == 0) {
        p.ctrl->n_groups = G;
        p.ctrl->n_entries = (int32_t)E;
        p.ctrl->n_hash_segs = (int32_t)nslice;
    }
}

// The same for any n: a stable LSD radix sort of (traj_id - min, index) and block scans, through arrays in the workspace.
__global__ void __launch_bounds__(1024) merge_group_radix_kernel(const MergeParams p) {
    __shared__ RadixScratch<32> sc;
    __shared__ int64_t s_w[2][2][32];
    __shared__ int s_min, s_max;
    __shared__ uint32_t s_bad;
    const int tid = threadIdx.x, n = p.n;
    uint32_t* kb[2] = {p.gbuf[0], p.gbuf[1]};
    uint32_t* vb[2] = {p.gbuf[2], p.gbuf[3]};
    int32_t* tln = reinterpret_cast<int32_t*>(p.gbuf[5]);        // [i] length of timeline i
    if (tid < (int)(sizeof(AjtCtrl) / 4)) reinterpret_cast<uint32_t*>(p.ctrl)[tid] = 0;   // fresh control block
    if (tid == 0) { s_min = INT32_MAX; s_max = INT32_MIN; s_bad = 0; }
    __syncthreads();
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
        tln[i] = (int32_t)(b - a);
    }
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
        if (tid == 0) group_fail(p, s_bad);
        return;
    }
    const int tmin = s_min;
    const uint32_t range = n ? (uint32_t)s_max - (uint32_t)tmin : 0u;
    for (int i = tid; i < n; i += 1024) kb[0][i] -= (uint32_t)tmin;
    __syncthreads();
    int cur = 0;
    for (int shift = 0; shift < 32 && (range >> shift) != 0; shift += 8) {
        radix_pass<32>(kb[cur], vb[cur], kb[cur ^ 1], vb[cur ^ 1], n, shift, sc);
        cur ^= 1;
        __syncthreads();
    }
    const uint32_t* key = kb[cur];
    const uint32_t* val = vb[cur];   // sorted position -> timeline index
    uint32_t* gid = kb[cur ^ 1];     // [pos] group id
    uint32_t* gsv = vb[cur ^ 1];     // [g]   first sorted position of group g
    const int G = (int)block_scan<1024, 4>(
        n, [&](int pos) { return (pos == 0 || key[pos] != key[pos - 1]) ? 1 : 0; },
        [&](int pos, int64_t ex, int64_t v) {
            const int g = (int)(ex + v) - 1;
            gid[pos] = (uint32_t)g;
            if (v) gsv[g] = (uint32_t)pos;
        },
        s_w);
    if (tid == 0) gsv[G] = (uint32_t)n;
    __syncthreads();
    // key slots (r, a), a = 0..r: a group of k timelines has k(k+1)/2, the slots of rank r start r(r+1)/2 into it
    uint32_t* gent = kb[cur];        // [g] first key slot of group g (the sorted keys are no longer needed)
    const int64_t E = block_scan<1024, 4>(
        G, [&](int g) { const int64_t k = gsv[g + 1] - gsv[g]; return k * (k + 1) / 2; },
        [&](int g, int64_t ex, int64_t) { gent[g] = (uint32_t)min(ex, (int64_t)INT32_MAX); }, s_w);
    if (tid == 0) gent[G] = (uint32_t)min(E, (int64_t)INT32_MAX);
    // hash slices: numbered in GROUP order, by sorted position
    const int64_t nslice = block_scan<1024, 4>(
        n, [&](int pos) { const int g = (int)gid[pos]; return gsv[g + 1] - gsv[g] < 2 ? 0 : slices_of((int)tln[val[pos]]); },
        [&](int pos, int64_t ex, int64_t) {
            const int i = (int)val[pos], g = (int)gid[pos];
            const int gs = (int)gsv[g], r = pos - gs;
            p.tl_rec[pos] = make_int4((int)ex, gs, (int)(gsv[g + 1] - gsv[g]), (int)(gent[g] + (uint32_t)r * (uint32_t)(r + 1) / 2u));
            p.perm[pos] = i;
            p.glen[pos] = tln[i];
            p.goff[pos] = __ldg(p.offsets + i);
            p.lbad[pos] = 0;
        },
        s_w);
    if (E > (int64_t)p.E_cap || nslice > (int64_t)p.slice_cap) {   // (units <= slices)
        if (tid == 0) group_fail(p, (uint32_t)AJT_STATUS_PROBE_CAPACITY);
        return;
    }
    for (int g = tid; g <= G; g += 1024)
        p.grp_rec[g] = make_int4((int)gsv[g], g < G ? (int)(gsv[g + 1] - gsv[g]) : 0, (int)gent[g], 0);
    if (tid == 0) {
        p.ctrl->n_groups = G;
        p.ctrl->n_entries = (int32_t)E;
        p.ctrl->n_hash_segs = (int32_t)nslice;
    }
}

// ---------------------------------------------------------------------------------------- K1b: hash units

// Hash units, in parallel over the whole GPU (the group kernel is one SM): thread per sorted position; the thread of a rank
// that is a multiple of kChunk in a group of at least two emits one unit {group start, first rank, members of the group, slice}
// per slice up to the longest member of its chunk.  Unit slots come from one counter (one atomic per warp); units are short
// (<= kChunk + 1 member-slices), so their order does not matter.
__global__ void __launch_bounds__(256) merge_units_kernel(const MergeParams p) {
    pdl_wait();
    if (fatal(p)) return;
    const int lane = threadIdx.x & 31, n = p.n;
    const int npad = (n + 31) & ~31;
    for (int pos = blockIdx.x * blockDim.x + threadIdx.x; pos < npad; pos += gridDim.x * blockDim.x) {
        int4 t = make_int4(0, 0, 0, 0);
        int cnt = 0;
        bool open = false;
        if (p.slim) {
            // expand the group kernel's slim record into the per-position records, and take the lengths from the offsets
            int2 sr = make_int2(0, 0);
            int4 gr = make_int4(0, 0, 0, 0);
            if (pos < n) {
                sr = __ldg(p.sel_q + pos);
                gr = __ldg(p.grp_rec + ((uint32_t)sr.x >> 16));   // {group start, members, first key slot}
            }
            const int i = sr.x & 0xffff, gs = gr.x, k = gr.y, r = pos - gs;
            open = pos < n && k >= 2 && r % kChunk == 0;
            int64_t o0 = 0, o1 = 0;
            if (pos < n) { o0 = __ldg(p.offsets + i); o1 = __ldg(p.offsets + i + 1); }
            int mx = 0;
            if (open) {   // the chunk's other members: their lengths straight from the offsets (their records are being written now)
                int ix[kChunk];
#pragma unroll
                for (int x = 1; x < kChunk; ++x) ix[x] = x < k - r ? (__ldg(p.sel_q + pos + x).x & 0xffff) : -1;
#pragma unroll
                for (int x = 1; x < kChunk; ++x)
                    if (ix[x] >= 0) mx = max(mx, (int)(__ldg(p.offsets + ix[x] + 1) - __ldg(p.offsets + ix[x])));
            }
            if (pos < n) {
                t = make_int4(sr.y, gs, k, gr.z + (int)((uint32_t)r * (uint32_t)(r + 1) / 2u));
                p.tl_rec[pos] = t;
                p.perm[pos] = i;
                p.glen[pos] = (int32_t)(o1 - o0);
                p.goff[pos] = o0;
                p.lbad[pos] = 0;
            }
            if (open) cnt = slices_of(max(mx, (int)(o1 - o0)));
        } else {
            if (pos < n) t = __ldg(p.tl_rec + pos);
            const int k = t.z, r = pos - t.y;
            open = pos < n && k >= 2 && r % kChunk == 0;
            if (open) {
                int mx = 0;
                for (int x = 0; x < min(kChunk, k - r); ++x) mx = max(mx, __ldg(p.glen + pos + x));
                cnt = slices_of(mx);
            }
        }
        const int gs = t.y, k = t.z, r = pos - gs;
        if (!__any_sync(0xffffffffu, open)) continue;
        int inc = cnt;   // inclusive scan of the unit counts over the warp
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += v;
        }
        const int tot = __shfl_sync(0xffffffffu, inc, 31);
        int ub = 0;
        if (lane == 0) ub = atomicAdd(&p.ctrl->n_units, tot);
        ub = __shfl_sync(0xffffffffu, ub, 0);
        if (open) {
            int4* const ur = p.unit_rec + ub + inc - cnt;
            for (int j = 0; j < cnt; ++j) ur[j] = make_int4(gs, r, k, j);
        }
    }
}

// ---------------------------------------------------------------------------------------- K2: prefix-hash scan (M2, M5 first half)

// Prefix hash F_i(p) = sum_{q<p} x_q w(q) mod 2^64 with 32-bit weights w(q) = W^(q+3) mod 2^32: one IMAD.WIDE per token
// (32 x 32 -> 64 with a 64-bit addend).  A sum over positions, hence a monoid: per-lane partials, combined only where a value
// leaves the warp.  Weak by design (a 64-bit sum of 50-bit products); every accepted pair is verified exactly (M5).
__device__ __forceinline__ uint32_t pow32(uint32_t b, uint32_t e) {
    uint32_t r = 1;
    while (e) {
        if (e & 1) r *= b;
        b *= b;
        e >>= 1;
    }
    return r;
}
template <int N>
struct PowTab {
    uint32_t v[N];
    constexpr PowTab() : v{} {}
    constexpr PowTab(uint32_t base) : v{} {
        uint32_t r = 1;
        for (int i = 0; i < N; ++i) { v[i] = r; r *= base; }
    }
};

// Last index i in [0, n) with key(i) <= x, for a non-decreasing key with key(0) <= x: warp-cooperative 32-ary search
// (2 dependent loads for n <= 1024 instead of 10).
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

__device__ __forceinline__ bool mbar_wait_bounded(uint64_t* bar, uint32_t parity) {
    for (int spin = 0; spin < (1 << 22); ++spin)
        if (mbar_try_wait(bar, parity)) return true;
    return false;
}
__device__ __forceinline__ uint32_t lds32(uint32_t saddr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(saddr));
    return v;
}
__device__ __forceinline__ void sts32(uint32_t saddr, uint32_t v) { asm volatile("st.shared.u32 [%0], %1;" ::"r"(saddr), "r"(v) : "memory"); }

constexpr int kHashThreads = 256;
constexpr int kHashStages = 3;          // the member in flight, the member at work, its predecessor
constexpr int kSlotBytes = 512 * kVT;                                    // 128 aligned vectors: the slice + its misalignment
constexpr int kStageBytes = 16 + kSlotBytes + 16;                   // a zero vector on either side (reads at e + delta, |delta| <= 3)
constexpr int kHashWarpBytes = kHashStages * kStageBytes + 128;     // + mbarriers (padded to 64 B) + descriptors
constexpr int kHashSmem = (kHashThreads / 32) * kHashWarpBytes + 128;
__constant__ PowTab<128> c_wsl = PowTab<128>(kWSl);     // W^(508 j): slice j of a timeline (65k tokens before the slow path)
__constant__ PowTab<4> c_winv = PowTab<4>(kWinv);       // W^-D: undoes the misalignment of a member in its slot

__device__ __forceinline__ uint4 lds128(uint32_t saddr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(saddr));
    return v;
}

// Warp per hash unit = (chunk of <= kChunk consecutive ranks of a group, block of kSliceBlk slices of 508 positions), taken
// from an atomic ticket, largest first.  The chunk's members -- preceded by the last member of the previous chunk, which is
// only there to be compared with -- sit one per lane; for every slice of the block the warp streams the members that reach
// it, in rank order.  A member's slice arrives as ONE bulk async copy (TMA, 1-D) of the 16-byte-aligned superset of its
// bytes -- exactly 128 vectors, whatever the member's misalignment D -- launched by the lane that holds the member and
// counted on a warp-private mbarrier.  Lane l owns vectors l + 32 t (t < 4) of EVERY slot, i.e. slot elements
// e = 4 (l + 32 t) + i: four conflict-free 16-byte shared-memory loads per member.  The hash is a polynomial in the ring mod
// 2^32, F(p) = sum_{q<p} x_q W^q: a lane's weights belong to the SLOT elements and never change, and the member's shift
// (slice start, misalignment) is one multiplication by W^(S0 - D) after the warp reduction (one REDUX: the sum wraps mod 2^32
// by itself).  Elements outside the member (before D, behind its end) are zeroed in shared memory on arrival, and every
// slot sits between two zero vectors, so member r is compared with member r - 1 slot against slot at an element shift
// delta = D' - D without masks; when the two agree over a whole slice the slice total is inherited and nothing is
// multiplied at all.  Slices in which a member or its predecessor ends take a masked path.  Why chunks: one warp works
// through its members one after the other (~2 us each), so a unit of 40 members would take as long as the whole kernel.
__global__ void __launch_bounds__(kHashThreads, kVT > 4 ? 2 : 3) merge_hash_kernel(const MergeParams p) {
    pdl_wait();
    extern __shared__ __align__(128) uint8_t h_dyn[];
    if (fatal(p)) return;
    const int lane = threadIdx.x & 31, wic = threadIdx.x >> 5;
    uint8_t* const wbuf = reinterpret_cast<uint8_t*>(((uintptr_t)h_dyn + 127) & ~(uintptr_t)127) + (size_t)wic * kHashWarpBytes;
    uint64_t* const full = reinterpret_cast<uint64_t*>(wbuf + kHashStages * kStageBytes);
    const uint32_t sdesc = smem_u32(wbuf + kHashStages * kStageBytes + 64);
    const uint32_t sbuf = smem_u32(wbuf) + 16;   // element 0 of stage 0
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < kHashStages; ++s) mbar_init(&full[s], 1);
        fence_mbar_init();
    }
    if (lane < 2 * kHashStages) {   // the zero vectors around every slot (never written again)
        const uint32_t a = smem_u32(wbuf) + (lane >> 1) * kStageBytes + (lane & 1) * (16 + kSlotBytes);
        asm volatile("st.shared.v4.u32 [%0], {%1,%1,%1,%1};" ::"r"(a), "r"(0u) : "memory");
    }
    __syncwarp();
    uint32_t phases = 0;   // bit s: the parity stage s completes next
    const int U = p.ctrl->n_units;
    const int32_t* __restrict__ tokens = p.tokens;
    const int64_t N = p.N;
    const int mis = p.mis;
    // weights of this lane's vectors: slot elements e = 4 (lane + 32 t) + i weigh W^e = bt[t] W^i (Horner inside a vector)
    uint32_t bt[kVT];
    bt[0] = pow32(kW, 4u * (uint32_t)lane);
#pragma unroll
    for (int t = 1; t < kVT; ++t) bt[t] = bt[t - 1] * kW128;
    auto dot = [&](const uint32_t* y) {
        uint32_t g = 0;
#pragma unroll
        for (int t = 0; t < kVT; ++t) g += (((y[4 * t + 3] * kW + y[4 * t + 2]) * kW + y[4 * t + 1]) * kW + y[4 * t]) * bt[t];
        return g;
    };
    bool dead = false;
    int next = 0;
    if (lane == 0) next = atomicAdd(&p.ctrl->unit_ticket, 1);
    next = __shfl_sync(0xffffffffu, next, 0);
    while (next < U) {
        const int u = next;
        if (lane == 0) next = atomicAdd(&p.ctrl->unit_ticket, 1);   // needed only after this unit: the round trip is hidden
        const int4 ur = __ldg(p.unit_rec + u);                      // {group start, first rank, members of the group, slice}
        const int gs = ur.x, r0 = ur.y, k = ur.z, w = ur.w;
        const int rlo = r0 - (r0 > 0 ? 1 : 0);                      // lane i holds rank rlo + i: the predecessor of the chunk first
        const int rhi = min(k, r0 + kChunk);
        const int32_t* __restrict__ gln = p.glen + gs;
        const int S0 = w * kSl;                                     // first position of the slice
        // ---- each lane's member and its slot in this slice
        const bool mine = rlo + lane < rhi;
        const int myr = rlo + lane;
        const int iL = mine ? __ldg(gln + myr) : 0;
        const int64_t ioff = mine ? __ldg(p.goff + gs + myr) : 0;
        const int4 trec = mine ? __ldg(p.tl_rec + gs + myr) : make_int4(0, 0, 0, 0);   // .x first slice, .w first key slot
        const int L0 = lane < k ? __ldg(gln + lane) : 0;   // lengths of the group's first 32 ranks: where prefixes end
        const int iD = (int)((ioff + mis + S0) & 3);               // slot element of position S0
        const int64_t ig0 = ioff + S0 - iD;                        // array index of slot element 0
        const int inv = (min(iL - S0, kSl) + iD + 3) >> 2;         // vectors holding positions < min(L, S0 + 508): at most 128
        const bool iedge = !(ig0 >= 0 && ig0 + 4 * (int64_t)inv <= N);
        uint64_t* const my_tot = p.seg_part + trec.x + w;          // where this member's slice total goes
        uint64_t* const my_keys = p.ent_hash + trec.w;             // its key slots (myr, a), a <= myr
        unsigned preach = __ballot_sync(0xffffffffu, iL > S0);     // members still to be fetched / still to be worked on
        unsigned creach = preach;
        const unsigned edges = __ballot_sync(0xffffffffu, iedge) & preach;
        const uint32_t wS0 = w < 128 ? c_wsl.v[w] : pow32(kWSl, (uint32_t)w);   // W^S0
        const uint32_t fD_mine = wS0 * c_winv.v[iD];               // W^(S0 - D)
        const unsigned end0 = __ballot_sync(0xffffffffu, L0 > 0 && slice_at(L0 - 1) == w);
        bool end_hi = false;   // does a member of rank >= 32 end in this slice?  (groups of more than 32 only)
        for (int a0 = 32; a0 < k && !end_hi; a0 += 32) {
            const int La = a0 + lane < k ? __ldg(gln + a0 + lane) : 0;
            end_hi = __any_sync(0xffffffffu, La > 0 && slice_at(La - 1) == w);
        }
        int istage = 0, st = 0, pst = 0;
        // launches the next member's copy into stage `istage` (if there is one)
        auto issue_next = [&]() {
            if (preach == 0) return;
            const int b = __ffs(preach) - 1;
            preach &= preach - 1;
            const int stage = istage;
            if ((edges >> b) & 1u) {   // first / last vectors of the token array: element-wise, inside the array only
                const int64_t gb = shfl_i64(ig0, b);
                const int nvb = __shfl_sync(0xffffffffu, inv, b);
                for (int e = lane; e < 4 * nvb; e += 32) {
                    const int64_t gi = gb + e;
                    sts32(sbuf + stage * kStageBytes + 4 * e, gi >= 0 && gi < N ? (uint32_t)tokens[gi] : 0u);
                }
                __syncwarp();
                if (lane == b) mbar_arrive(&full[stage]);
            } else if (lane == b) {
                mbar_arrive_expect_tx(&full[stage], 16u * (uint32_t)inv);
                fence_proxy_async_smem();   // the stage's last user zeroed a few of its elements with ordinary stores
                bulk_load(wbuf + 16 + stage * kStageBytes, tokens + ig0, 16u * (uint32_t)inv, &full[stage]);
            }
            if (++istage == kHashStages) istage = 0;
        };
        int prev_r = -2, prev_L = 0, prev_D = 0;
        uint32_t prev_tot = 0;
        bool prev_hashed = false;
        uint32_t Fk = 0;        // lane a: the partial of the prefix ending at member a's last token, for the latest member
        unsigned fvalid = 0;    // ranks whose Fk belongs to the latest member
        issue_next();           // one member ahead: the predecessor's stage stays intact while a member is compared with it
#pragma unroll 1
        while (creach) {
            issue_next();
            const int b = __ffs(creach) - 1;   // the member at work sits in lane b
            creach &= creach - 1;
            const int r = rlo + b;
            const int Lr = __shfl_sync(0xffffffffu, iL, b), D = __shfl_sync(0xffffffffu, iD, b);
            if (!mbar_wait_bounded(&full[st], (phases >> st) & 1u)) dead = true;   // never in practice: a lost copy must not hang the GPU
            phases ^= 1u << st;
            const uint32_t slot = sbuf + st * kStageBytes;
            const int len = min(Lr - S0, kSl);           // positions of the member in this slice
            // zero what is not the member's: elements [0, D) and [D + len, end of the last vector) -- for a whole slice up to
            // the end of the slot (with D = 0 the copy is 127 vectors and the 128th holds an earlier member's data)
            if (lane < D) sts32(slot + 4 * lane, 0u);
            if (lane < 4 && D + len + lane < (len == kSl ? kSlotBytes / 4 : (len + D + 3) & ~3)) sts32(slot + 4 * (D + len + lane), 0u);
            __syncwarp();
            if (r < r0) {   // the previous chunk's last member: here to be compared with, nothing else
                prev_hashed = false;
            } else {
                const bool have_prev = prev_r == r - 1;
                const int plen = min(prev_L - S0, kSl);
                const uint32_t pslot = sbuf + pst * kStageBytes;
                const int delta = prev_D - D;                 // position p: own element p + D, predecessor's element p + D + delta
                uint32_t y[4 * kVT];
                bool same = false;   // the two agree on every position of the slice below prev_L
                if (len == kSl && (!have_prev || plen == kSl)) {
                    // ---- whole slices: no masks anywhere
#pragma unroll
                    for (int t = 0; t < kVT; ++t) {
                        const uint4 v = lds128(slot + 16 * (lane + 32 * t));
                        y[4 * t] = v.x; y[4 * t + 1] = v.y; y[4 * t + 2] = v.z; y[4 * t + 3] = v.w;
                    }
                    if (have_prev) {
                        uint32_t diff = 0;
                        if (delta == 0) {
#pragma unroll
                            for (int t = 0; t < kVT; ++t) {
                                const uint4 z = lds128(pslot + 16 * (lane + 32 * t));
                                diff |= (y[4 * t] ^ z.x) | (y[4 * t + 1] ^ z.y) | (y[4 * t + 2] ^ z.z) | (y[4 * t + 3] ^ z.w);
                            }
                        } else {
                            const uint32_t pa = pslot + 4 * delta + 16 * lane;
#pragma unroll
                            for (int t = 0; t < kVT; ++t)
#pragma unroll
                                for (int i = 0; i < 4; ++i) diff |= y[4 * t + i] ^ lds32(pa + 512 * t + 4 * i);
                        }
                        same = !__any_sync(0xffffffffu, diff != 0);
                    }
                } else {
                    // ---- the member or its predecessor ends in this slice: element by element
                    const int cmp = have_prev ? min(len, plen) : 0;   // positions to compare
                    uint32_t diff = 0;
#pragma unroll
                    for (int t = 0; t < kVT; ++t)
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            const int e = 4 * (lane + 32 * t) + i, pos = e - D;
                            const uint32_t v = pos >= 0 && pos < len ? lds32(slot + 4 * e) : 0u;
                            y[4 * t + i] = v;
                            if (pos >= 0 && pos < cmp) diff |= v ^ lds32(pslot + 4 * (e + delta));
                        }
                    if (have_prev) same = !__any_sync(0xffffffffu, diff != 0);
                }
                if (have_prev && !same && lane == b) p.lbad[gs + r] = 1;
                const uint32_t fD = __shfl_sync(0xffffffffu, fD_mine, b);
                uint32_t tot;
                if (have_prev && same && prev_hashed && len == kSl && plen == kSl) tot = prev_tot;   // the same 508 tokens
                else tot = __reduce_add_sync(0xffffffffu, dot(y)) * fD;
                if (lane == b) *my_tot = tot;
                // keys: the prefixes (L_a of an earlier member, or L_r itself) that end inside this slice
                if (!same) fvalid = 0;
                if (end0) {
                    unsigned m0 = end0 & (r >= 31 ? 0xffffffffu : (2u << r) - 1u);
                    if (m0) m0 &= __ballot_sync(0xffffffffu, L0 <= Lr);
                    for (; m0; m0 &= m0 - 1) {
                        const int a = __ffs(m0) - 1;
                        const int La = __shfl_sync(0xffffffffu, L0, a);
                        uint32_t F;
                        if (((fvalid >> a) & 1u) && La <= prev_L) {
                            F = __shfl_sync(0xffffffffu, Fk, a);   // member r - 1 has the same tokens up to there
                        } else {
                            if (a == r) {
                                F = tot;   // its own last token: everything beyond is zero already
                            } else {
                                const int rem = La - S0 + D - 4 * lane;   // slot elements 128 t + i < rem are inside the prefix
                                uint32_t z[4 * kVT];
#pragma unroll
                                for (int j = 0; j < 4 * kVT; ++j) z[j] = 128 * (j >> 2) + (j & 3) < rem ? y[j] : 0u;
                                F = __reduce_add_sync(0xffffffffu, dot(z)) * fD;
                            }
                            if (lane == a) Fk = F;
                            fvalid |= 1u << a;
                        }
                        if (lane == b) my_keys[a] = F;
                    }
                }
                if (end_hi && r >= 32) {   // groups of more than 32: ends of ranks >= 32, no caching
                    for (int a0r = 32; a0r <= r; a0r += 32) {
                        const int a = a0r + lane;
                        const int La = a < k ? __ldg(gln + a) : 0;
                        const bool hit = a <= r && La > 0 && La <= Lr && slice_at(La - 1) == w;
                        for (unsigned m = __ballot_sync(0xffffffffu, hit); m; m &= m - 1) {
                            const int a1 = __ffs(m) - 1;
                            const int rem = __shfl_sync(0xffffffffu, La, a1) - S0 + D - 4 * lane;
                            uint32_t z[4 * kVT];
#pragma unroll
                            for (int j = 0; j < 4 * kVT; ++j) z[j] = 128 * (j >> 2) + (j & 3) < rem ? y[j] : 0u;
                            const uint32_t F = __reduce_add_sync(0xffffffffu, dot(z)) * fD;
                            if (lane == b) my_keys[a0r + a1] = F;
                        }
                    }
                }
                prev_tot = tot;
                prev_hashed = true;
            }
            prev_r = r;
            prev_L = Lr;
            prev_D = D;
            pst = st;
            if (++st == kHashStages) st = 0;
            __syncwarp();   // every lane is done with the stage before a later issue refills it
        }
        next = __shfl_sync(0xffffffffu, next, 0);
        if (__any_sync(0xffffffffu, dead)) break;
    }
    if (dead && lane == 0) atomicOr(&p.ctrl->status, (uint32_t)AJT_STATUS_INTERNAL);
}

// ---------------------------------------------------------------------------------------- K3: keys, sort, select, verify, segments, compact (M2-M6)

// Exact: tokens[oa .. oa + L) == tokens[ob .. ob + L), by one warp.  128-bit loads when the two ranges are co-aligned
// (after a scalar head), coalesced 32-bit loads otherwise; leaves at the first block that differs.
__device__ __noinline__ bool warp_tokens_equal(const int32_t* __restrict__ tokens, int64_t oa, int64_t ob, int L, int mis) {
    const int lane = threadIdx.x & 31;
    const int32_t* __restrict__ A = tokens + oa;
    const int32_t* __restrict__ B = tokens + ob;
    int q = 0;
    if (((oa ^ ob) & 3) == 0) {
        const int head = min(L, (int)((4 - ((oa + mis) & 3)) & 3));
        bool bad = lane < head && A[lane] != B[lane];
        if (__any_sync(0xffffffffu, bad)) return false;
        const int nvec = (L - head) >> 2;
        const int4* __restrict__ A4 = reinterpret_cast<const int4*>(A + head);
        const int4* __restrict__ B4 = reinterpret_cast<const int4*>(B + head);
        for (int v0 = 0; v0 < nvec; v0 += 128) {
            uint32_t diff = 0;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int v = v0 + lane + 32 * j;
                if (v < nvec) {
                    const int4 x = __ldg(A4 + v), y = __ldg(B4 + v);
                    diff |= (uint32_t)(x.x ^ y.x) | (uint32_t)(x.y ^ y.y) | (uint32_t)(x.z ^ y.z) | (uint32_t)(x.w ^ y.w);
                }
            }
            if (__any_sync(0xffffffffu, diff != 0)) return false;
        }
        q = head + 4 * nvec;   // at most 3 tokens left
    }
    for (; q < L; q += 256) {
        uint32_t diff = 0;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const int e = q + lane + 32 * j;
            if (e < L) diff |= (uint32_t)(__ldg(A + e) ^ __ldg(B + e));
        }
        if (__any_sync(0xffffffffu, diff != 0)) return false;
    }
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
    int64_t s_w[2][2][kSelThreads / 32];     // block scans
    int32_t st[8][kSelCacheK];               // per-member decision state (groups up to kSelCacheK)
    int2 q[kSelCacheK];                      // verification queue {member, candidate}
    int32_t qn;
    int32_t coll;
};
// Staged copy of one group (dynamic shared memory): a CTA pays ~1 us per dependent global round trip, so a group of up to
// kSelCacheK members, kSelSmemKeys keys and kSelSlices hash slices is fetched in three batched round trips and decided from
// shared memory; larger groups work through the workspace.
constexpr int kSelSlices = 2048;
struct SelectStage {
    uint64_t eh[kSelSmemKeys];               // key slots: in-slice partial, then the final prefix hash
    uint64_t sp[kSelSlices];                 // slice totals of the group's members, then exclusive prefixes per member
    int64_t off[kSelCacheK];                 // by rank: token offset
    int32_t L[kSelCacheK], sb[kSelCacheK], idx[kSelCacheK], rs[kSelCacheK];   // length, first slice, timeline, response start
    int32_t mj[kSelCacheK], mL[kSelCacheK], mR[kSelCacheK];                   // by member slot: timeline, length, response start
    uint8_t bad[kSelCacheK];                 // the exact comparison with the predecessor found a difference
};

// The segments of one surviving timeline, by one warp: maximal runs [p0, p1) of positions whose mask / log-prob come from one
// member (the largest member index j with rs_j <= p < L_j, Algorithm 1 lines 10-17; kSrcNone if there is none).  The run
// boundaries are response starts and ends of members, at most 2c of them.  mj / mL / mR: timeline, length and response
// start (clamped to [0, L]) of the c members, ascending, the survivor last.  With explicit masks the source is decided
// per token by the scatter pass: one segment.  Returns the number of segments written to out[].
__device__ __noinline__ int build_segments(bool explicit_masks, const int32_t* mj, const int32_t* mL, const int32_t* mR, int c,
                                           int2* out) {
    const int lane = threadIdx.x & 31;
    if (explicit_masks) {
        if (lane == 0) out[0] = make_int2(0, kSrcExplicit);
        return 1;
    }
    const int Ls = mL[c - 1];
    int cnt = 0, last = INT32_MIN, pos = 0;
    // members of the first 32 stay in registers; longer lists are re-read per step
    int j0 = -1, L0 = 0, r0 = 0;
    if (lane < c) { j0 = mj[lane]; L0 = mL[lane]; r0 = mR[lane]; }
    while (pos < Ls) {
        int src = kSrcNone, nxt = Ls;
        if (j0 >= 0) {
            if (r0 <= pos && pos < L0) src = j0;
            if (r0 > pos) nxt = min(nxt, r0);
            if (L0 > pos) nxt = min(nxt, L0);
        }
        for (int m0 = 32; m0 < c; m0 += 32) {
            if (m0 + lane < c) {
                const int j = mj[m0 + lane], Lj = mL[m0 + lane], rj = mR[m0 + lane];
                if (rj <= pos && pos < Lj) src = max(src, j);
                if (rj > pos) nxt = min(nxt, rj);
                if (Lj > pos) nxt = min(nxt, Lj);
            }
        }
        src = __reduce_max_sync(0xffffffffu, src);
        nxt = __reduce_min_sync(0xffffffffu, nxt);
        if (src != last) {
            if (lane == 0) out[cnt] = make_int2(pos, src);
            ++cnt;
            last = src;
        }
        pos = nxt;
    }
    return cnt;
}

// M6.  One CTA, one fused scan over the timelines (original order): survivors -> merged index, offsets, origin, traj, first
// global segment; then owner[].  A lone SM pays ~1-2 us per dependent global round trip and handles only so many memory
// sectors per cycle, so every global access is coalesced (lane = consecutive timeline) and issued 8 deep, and the scan --
// which wants 8 CONSECUTIVE timelines per thread -- runs on a copy in shared memory.  Two round trips in all.
constexpr int kCompactChunk = 8192;
constexpr int kCompactSmem = kCompactChunk * 16;
__global__ void __launch_bounds__(1024) merge_compact_kernel(const MergeParams p) {
    pdl_wait();
    extern __shared__ __align__(16) uint8_t c_dyn[];
    __shared__ int64_t s_wa[32], s_wb[32];
    if (fatal(p)) return;
    constexpr int NT = 1024;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, n = p.n;
    uint2* const prA = reinterpret_cast<uint2*>(c_dyn);                         // in: {survivor << 24 | segments, length}; out: {merged index, first segment}
    int64_t* const prB = reinterpret_cast<int64_t*>(c_dyn + kCompactChunk * 8);  // out: merged offset
    int64_t base_a = 0, base_b = 0;   // {survivors << 32 | segments}, tokens, before this chunk
    for (int c0 = 0; c0 < n; c0 += kCompactChunk) {
        const int cn = min(kCompactChunk, n - c0);
        uint32_t sv[8];
        // ---- A: coalesced loads, 8 timelines per thread in flight: one 8-byte record each, written by the select pass
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int j = u * NT + tid, i = c0 + j;
            uint2 v = make_uint2(0u, 0u);
            if (j < cn) v = __ldg(p.cinfo + i);
            sv[u] = v.x;
            prA[j] = v;
        }
        __syncthreads();
        // ---- B: thread t scans timelines 8 t .. 8 t + 7 of the chunk
        uint2 it[8];
        int64_t sa = 0, sb = 0;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            it[q] = prA[8 * tid + q];
            sa += ((int64_t)(it[q].x >> 24) << 32) | (it[q].x & 0xffffffu);
            sb += it[q].y;
        }
        int64_t ia = sa, ib = sb;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int64_t ta = __shfl_up_sync(0xffffffffu, ia, o), tb = __shfl_up_sync(0xffffffffu, ib, o);
            if (lane >= o) { ia += ta; ib += tb; }
        }
        if (lane == 31) { s_wa[warp] = ia; s_wb[warp] = ib; }
        __syncthreads();
        int64_t wa = s_wa[lane], wb = s_wb[lane], ja = wa, jb = wb;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int64_t ta = __shfl_up_sync(0xffffffffu, ja, o), tb = __shfl_up_sync(0xffffffffu, jb, o);
            if (lane >= o) { ja += ta; jb += tb; }
        }
        int64_t ra = base_a + __shfl_sync(0xffffffffu, ja - wa, warp) + ia - sa;
        int64_t rb = base_b + __shfl_sync(0xffffffffu, jb - wb, warp) + ib - sb;
        const int64_t ta = __shfl_sync(0xffffffffu, ja, 31), tb = __shfl_sync(0xffffffffu, jb, 31);
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            prA[8 * tid + q] = make_uint2((uint32_t)(ra >> 32), (uint32_t)(ra & 0xffffffff));
            prB[8 * tid + q] = rb;
            ra += ((int64_t)(it[q].x >> 24) << 32) | (it[q].x & 0xffffffu);
            rb += it[q].y;
        }
        base_a += ta;
        base_b += tb;
        __syncthreads();
        // ---- C: coalesced outputs
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int j = u * NT + tid, i = c0 + j;
            if (j >= cn) break;
            int32_t m = -1;
            if (sv[u]) {
                const uint2 e = prA[j];
                m = (int32_t)e.x;
                p.merged_origin[m] = i;
                p.merged_offsets[m] = prB[j];
                p.gseg_base[m] = (int32_t)e.y;
            }
            p.midx[i] = m;
        }
        __syncthreads();
    }
    const int M = (int)(base_a >> 32);
    const int32_t nseg = (int32_t)(base_a & 0xffffffff);
    // (owner[] = merged index of every timeline's owner is a gather over all timelines: merge_plan_kernel does it GPU-wide)
    if (tid == 0) {
        p.merged_offsets[M] = base_b;
        p.gseg_base[M] = nseg;
        p.counts[0] = M;
        p.counts[1] = base_b;
        p.ctrl->M = M;
        p.ctrl->N_out = base_b;
        p.ctrl->n_gsegs = nseg;
        p.ctrl->n_tiles = (int32_t)((base_b + kTS - 1) >> kTSLog);
    }
}

__global__ void __launch_bounds__(kSelThreads, 2) merge_select_kernel(const MergeParams p) {
    pdl_wait();
    __shared__ SelectSmem sm;
    extern __shared__ __align__(16) uint8_t sel_dyn[];
    SelectStage& sg = *reinterpret_cast<SelectStage*>(sel_dyn);
    constexpr int NT = kSelThreads;
    if (fatal(p)) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = p.ctrl->n_groups;
    const bool weak = (p.flags & AJT_MERGE_WEAK_HASH) != 0;
    const bool longest = p.owner_rule == AJT_OWNER_LONGEST;
    const bool explicit_masks = p.mask_in != nullptr;
    if (tid == 0) sm.coll = 0;
    for (int g = blockIdx.x; g < G; g += gridDim.x) {
        const int4 gr = __ldg(p.grp_rec + g);
        const int gs = gr.x, k = gr.y, eb = gr.z;
        const int c = (int)min((int64_t)k * (k + 1) / 2, (int64_t)INT32_MAX);   // key slots (fits: checked against E_cap)
        int2* const rs_out = p.rseg + 2 * (int64_t)gs;
        int32_t* const mem = p.mem_list + gs;
        if (k < 2) {   // a group of one: it survives and is its own only member
            if (warp == 0) {
                const int i = __ldg(p.perm + gs), L = __ldg(p.glen + gs);
                const int rs = explicit_masks ? 0 : min(max(__ldg(p.resp_start + i), 0), L);
                if (lane == 0) {
                    p.owner_tl[i] = i; mem[0] = i;
                    p.sel[3][gs] = L; p.sel[4][gs] = rs;
                }
                __syncwarp();
                const int sc = build_segments(explicit_masks, mem, p.sel[3] + gs, p.sel[4] + gs, 1, rs_out);
                if (lane == 0) {
                    p.sv_rec[i] = make_int4(gs, 1, 2 * gs, sc);
                    p.cinfo[i] = make_uint2((1u << 24) | (uint32_t)sc, (uint32_t)L);
                }
            }
            continue;
        }
        const bool cached = k <= kSelCacheK, small = c <= kSelSmemKeys;
        // ---- stage-in, round trip 2 (the group record was 1): per-member facts and the key partials, all independent loads
        bool fast = cached && small;
        if (fast) {
            if (tid < k) {
                const int i = __ldg(p.perm + gs + tid);
                sg.idx[tid] = i;
                sg.L[tid] = __ldg(p.glen + gs + tid);
                sg.off[tid] = __ldg(p.goff + gs + tid);
                sg.sb[tid] = __ldg(reinterpret_cast<const int32_t*>(p.tl_rec + gs + tid));
                sg.bad[tid] = p.lbad[gs + tid];
            }
            for (int x = tid; x < c; x += NT) sg.eh[x] = p.ent_hash[eb + x];
            __syncthreads();
            const int sb0 = sg.sb[0], nsl = sg.sb[k - 1] + slices_of(sg.L[k - 1]) - sb0;
            fast = nsl <= kSelSlices;
            if (fast) {   // round trip 3: the slice totals (contiguous: slices are numbered in group order), response starts
                for (int x = tid; x < nsl; x += NT) sg.sp[x] = p.seg_part[sb0 + x];
                if (tid < k) sg.rs[tid] = explicit_masks ? 0 : min(max(__ldg(p.resp_start + sg.idx[tid]), 0), sg.L[tid]);
            }
            __syncthreads();
        }
        const int32_t* const gl = fast ? sg.idx : p.perm + gs;
        const int32_t* const gln = fast ? sg.L : p.glen + gs;
        const int64_t* const gof = fast ? sg.off : p.goff + gs;
        uint64_t* const eh = fast ? sg.eh : p.ent_hash + eb;
        uint64_t* const sp = fast ? sg.sp - sg.sb[0] : p.seg_part;   // sp[first slice of member r + s]
        auto sb_of = [&](int r) { return fast ? sg.sb[r] : p.tl_rec[gs + r].x; };
        // per-member decision state, by rank
        int32_t* const own = cached ? sm.st[0] : p.sel[0] + gs;    // -2 undecided, -1 survivor, else rank of the owner
        int32_t* const lim = cached ? sm.st[1] : p.sel[1] + gs;    // PAPER: candidates below this rank only
        int32_t* const badc = cached ? sm.st[2] : p.sel[2] + gs;   // broken links among ranks <= r
        int32_t* const exL = cached ? sm.st[3] : p.sel[3] + gs;    // LONGEST: the last candidate that failed (length, rank)
        int32_t* const exR = cached ? sm.st[4] : p.sel[4] + gs;
        int32_t* const fin = cached ? sm.st[5] : p.sel[5] + gs;    // LONGEST: the owner, -2 while undecided
        int32_t* const mcnt = cached ? sm.st[6] : p.sel[6] + gs;   // members per survivor
        int32_t* const mbase = cached ? sm.st[7] : p.sel[7] + gs;  // its first member slot
        int2* const vq = cached ? sm.q : p.sel_q + gs;
        // ---- M2 (end): per member, exclusive prefix over its slice totals (in place), one warp per member
        for (int r = warp; r < k; r += NT / 32) {
            const int sb = sb_of(r);
            const int ns = slices_of(gln[r]);
            uint64_t carry = 0;
            for (int s0 = 0; s0 < ns; s0 += 32) {
                const int s = s0 + lane;
                const uint64_t v = s < ns ? sp[sb + s] : 0;
                uint64_t inc = v;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const uint64_t t = __shfl_up_sync(0xffffffffu, inc, o);
                    if (lane >= o) inc += t;
                }
                if (s < ns) sp[sb + s] = carry + inc - v;
                carry += __shfl_sync(0xffffffffu, inc, 31);
            }
        }
        // broken links up to each rank: link r is broken when the exact comparison of the hash pass found a difference, or
        // when the predecessor is longer (it cannot be a prefix then)
        block_scan<NT, 1>(
            k, [&](int r) { return r > 0 && ((fast ? sg.bad[r] : p.lbad[gs + r]) != 0 || gln[r - 1] > gln[r]) ? 1 : 0; },
            [&](int r, int64_t ex, int64_t v) { badc[r] = (int32_t)(ex + v); own[r] = -2; lim[r] = k; mcnt[r] = 0; }, sm.s_w);
        if (small)
            for (int b = tid; b <= kSelBuckets; b += NT) sm.start[b] = 0;
        if (tid == 0) sm.qn = 0;
        __syncthreads();
        // ---- final keys: hash of T_r[0:L_a] = prefix of the slices before the one holding position L_a - 1 + its partial
        uint32_t* gdig = p.ent_dig + eb;
        uint32_t* gidx = p.ent_idx + eb;
        for (int x = tid; x < c; x += NT) {
            const int r = rank_of_local((uint32_t)x), a = x - r * (r + 1) / 2;
            const int32_t Lp = gln[a];
            uint32_t dg = 0xFFFFFFFFu;
            if (Lp <= gln[r]) {
                uint64_t h = (eh[x] + sp[sb_of(r) + slice_at(Lp - 1)]) & 0xFFFFFFFFull;   // the hash lives in the ring mod 2^32
                if (weak) h &= 0xFull;
                eh[x] = h;
                dg = digest32(h, Lp);
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
        // visit(dg, fn): one warp; fn(le) for every key slot of this group whose digest is dg (the equal-key run), a lane each
        auto visit = [&](uint32_t dg, auto fn) {
            if (small) {
                const uint32_t b = dg >> (32 - kSelBucketBits);
                const uint32_t x1 = sm.start[b], x0 = b ? sm.start[b - 1] : 0u;
                for (uint32_t x = x0 + lane; x < x1; x += 32) {
                    const uint32_t le = sm.sorted[x];
                    if (sm.dig[le] == dg) fn(le);
                }
            } else {
                int lo = 0, hi = c;   // lower bound of dg in the sorted digests
                while (lo < hi) {
                    const int mid = (lo + hi) >> 1;
                    if (sk[mid] < dg) lo = mid + 1; else hi = mid;
                }
                for (int x0 = lo;; x0 += 32) {
                    const int x = x0 + lane;
                    const bool in = x < c && sk[x] == dg;
                    if (in) fn(sv[x]);
                    if (!__all_sync(0xffffffffu, in)) break;
                }
            }
        };
        // Verification rounds.  pick(b) proposes a candidate for every undecided member (or decides it); proposals that no
        // chain of verified links implies are compared exactly, one warp per pair; a failure excludes the candidate.
        auto run_queue = [&](auto accept, auto reject) {
            __syncthreads();
            const int nq = sm.qn;
            for (int qi = warp; qi < nq; qi += NT / 32) {
                const int2 e = vq[qi];
                const bool ok = warp_tokens_equal(p.tokens, gof[e.y], gof[e.x], gln[e.x], p.mis);
                if (lane == 0) {
                    if (ok) accept(e.x, e.y);
                    else { reject(e.x, e.y); sm.coll = 1; }
                }
            }
            __syncthreads();
            if (tid == 0) sm.qn = 0;
            __syncthreads();
            return nq;
        };
        // ---- M4 + M5: survivors and the Algorithm-1 owner = the latest extender
        while (true) {
            for (int b = warp; b < k; b += NT / 32) {   // a warp per member: the lanes share its equal-key run
                if (own[b] != -2) continue;
                const uint64_t H = eh[b * (b + 1) / 2 + b];   // full key of member b
                const int32_t L = gln[b];
                uint32_t dg = digest32(H, L);
                if (dg == 0xFFFFFFFFu) dg = 0xFFFFFFFEu;
                const int lm = lim[b];
                int best = -1;
                visit(dg, [&](uint32_t le) {
                    const int rb = rank_of_local(le);
                    if (rb <= b || rb >= lm || rb <= best) return;
                    const int a = (int)le - rb * (rb + 1) / 2;
                    if (gln[a] != L || eh[le] != H) return;
                    best = rb;
                });
                best = __reduce_max_sync(0xffffffffu, best);
                if (lane == 0) {
                    if (best < 0) own[b] = -1;
                    else if (badc[best] == badc[b]) own[b] = best;   // every link b+1 .. best was verified by the hash pass
                    else vq[atomicAdd(&sm.qn, 1)] = make_int2(b, best);
                }
            }
            if (run_queue([&](int b, int cd) { own[b] = cd; }, [&](int b, int cd) { lim[b] = cd; }) == 0) break;
        }
        if (longest) {
            // the longest SURVIVING extender, then the lowest index (BASELINE.json north_star; reading M-3)
            for (int b = tid; b < k; b += NT) { fin[b] = own[b] >= 0 ? -2 : -1; exL[b] = INT32_MAX; exR[b] = -1; }
            __syncthreads();
            while (true) {
                for (int b = warp; b < k; b += NT / 32) {
                    if (fin[b] != -2) continue;
                    const uint64_t H = eh[b * (b + 1) / 2 + b];
                    const int32_t L = gln[b];
                    uint32_t dg = digest32(H, L);
                    if (dg == 0xFFFFFFFFu) dg = 0xFFFFFFFEu;
                    const int xL = exL[b], xR = exR[b];
                    int best = -1;
                    int32_t bestL = -1;
                    visit(dg, [&](uint32_t le) {
                        const int rb = rank_of_local(le);
                        if (rb <= b || own[rb] >= 0) return;                       // survivors only
                        const int32_t Li = gln[rb];
                        if (!(Li < xL || (Li == xL && rb > xR))) return;            // after the last failure in (length desc, rank asc)
                        if (!(Li > bestL || (Li == bestL && rb < best))) return;
                        const int a = (int)le - rb * (rb + 1) / 2;
                        if (gln[a] != L || eh[le] != H) return;
                        best = rb;
                        bestL = Li;
                    });
                    // the longest over the lanes, then the lowest rank among those
                    const int32_t topL = __reduce_max_sync(0xffffffffu, bestL);
                    best = (int)__reduce_min_sync(0xffffffffu, best >= 0 && bestL == topL ? (unsigned)best : 0xFFFFFFFFu);
                    if (lane == 0) {
                        if (best < 0 || best == own[b]) fin[b] = own[b];            // the Algorithm-1 owner is verified already
                        else if (badc[best] == badc[b]) fin[b] = best;
                        else vq[atomicAdd(&sm.qn, 1)] = make_int2(b, best);
                    }
                }
                if (run_queue([&](int b, int cd) { fin[b] = cd; }, [&](int b, int cd) { exL[b] = gln[cd]; exR[b] = cd; }) == 0) break;
            }
            for (int b = tid; b < k; b += NT)
                if (own[b] >= 0) own[b] = fin[b];
            __syncthreads();
        }
        // ---- outputs by timeline; members of every survivor, ascending
        for (int b = tid; b < k; b += NT) {
            const int j = gl[b], o = own[b] < 0 ? b : own[b];
            if (own[b] >= 0) p.cinfo[j] = make_uint2(0u, 0u);
            p.owner_tl[j] = gl[o];
            atomicAdd(&mcnt[o], 1);
        }
        __syncthreads();
        block_scan<NT, 1>(
            k, [&](int r) { return mcnt[r]; }, [&](int r, int64_t ex, int64_t) { mbase[r] = (int32_t)ex; }, sm.s_w);
        // member slots: timeline, length, response start (exL / exR are free again: they hold the last two when the group
        // works through the workspace)
        int32_t* const mj = fast ? sg.mj : mem;
        int32_t* const mL = fast ? sg.mL : exL;
        int32_t* const mR = fast ? sg.mR : exR;
        __syncthreads();
        for (int b = tid; b < k; b += NT) {
            const int o = own[b] < 0 ? b : own[b];
            int at = 0;
            for (int x = 0; x < b; ++x) at += (own[x] < 0 ? x : own[x]) == o ? 1 : 0;
            const int slot = mbase[o] + at, j = gl[b], L = gln[b];
            mem[slot] = j;
            mj[slot] = j;
            mL[slot] = L;
            mR[slot] = fast ? sg.rs[b] : (explicit_masks ? 0 : min(max(__ldg(p.resp_start + j), 0), L));
        }
        __syncthreads();
        // ---- segments of every survivor, one warp each
        for (int b = warp; b < k; b += NT / 32) {
            if (own[b] >= 0) continue;
            const int mb = mbase[b], mc = mcnt[b];
            const int sc = build_segments(explicit_masks, mj + mb, mL + mb, mR + mb, mc, rs_out + 2 * mb);
            if (lane == 0) {
                p.sv_rec[gl[b]] = make_int4(gs + mb, mc, 2 * (gs + mb), sc);
                p.cinfo[gl[b]] = make_uint2((1u << 24) | (uint32_t)sc, (uint32_t)gln[b]);
            }
        }
        __syncthreads();
    }
    if (tid == 0 && sm.coll) {
        atomicOr(&p.ctrl->status, (uint32_t)AJT_STATUS_HASH_COLLISION);
        p.ctrl->collision = 1;
    }
}

// ---------------------------------------------------------------------------------------- K4: plan (M7, records)

// (a) one warp per merged sequence: its relative segments -> global segment records at output positions;
// (b) one thread per output tile: the segment that holds the tile's first position.
__global__ void __launch_bounds__(256) merge_plan_kernel(const MergeParams p) {
    pdl_wait();
    if (fatal(p)) return;
    const int lane = threadIdx.x & 31;
    const int wglobal = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    const int M = p.ctrl->M;
    const int64_t N_out = p.ctrl->N_out;
    for (int m = wglobal; m < M; m += nwarps) {
        const int s = __ldg(p.merged_origin + m);
        const int4 sr = __ldg(p.sv_rec + s);
        const int64_t mo = __ldg(p.merged_offsets + m), mo1 = __ldg(p.merged_offsets + m + 1), so = __ldg(p.offsets + s);
        const int gb = __ldg(p.gseg_base + m);
        if (lane == 0) p.merged_traj[m] = __ldg(p.traj_ids + s);
        for (int li = lane; li < sr.w; li += 32) {
            const int2 rs = __ldg(p.rseg + sr.z + li);
            GSeg o;
            o.out_start = mo + rs.x;
            o.tok_delta = so - mo;
            o.src = rs.y;
            o.aux = 0;
            if (rs.y >= 0) o.lp_delta = __ldg(p.offsets + rs.y) - mo;
            else if (rs.y == kSrcExplicit) { o.lp_delta = sr.x; o.aux = sr.y; }
            else o.lp_delta = 0;
            p.gseg[gb + li] = o;
        }
        // the tiles whose first position lies in this sequence: a lane each; the last relative segment that starts at or
        // before it (the sequence's segment list was read a moment ago: these searches hit L1)
        const int64_t t0 = (mo + kTS - 1) >> kTSLog, t1 = (mo1 + kTS - 1) >> kTSLog;   // tiles t0 .. t1 - 1 start in [mo, mo1)
        for (int64_t t = t0 + lane; t < t1; t += 32) {
            const int64_t pr = (t << kTSLog) - mo;
            int a = 0, b = sr.w - 1;
            while (a < b) {
                const int mid = (a + b + 1) >> 1;
                if ((int64_t)__ldg(p.rseg + sr.z + mid).x <= pr) a = mid; else b = mid - 1;
            }
            p.tile_seg[t] = gb + a;
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        GSeg o;
        o.out_start = N_out; o.tok_delta = 0; o.lp_delta = 0; o.src = kSrcNone; o.aux = 0;
        p.gseg[p.ctrl->n_gsegs] = o;
    }
    // owner[j] = merged index of the timeline that owns j (index map, reading M-12)
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < p.n; j += gridDim.x * blockDim.x)
        p.owner[j] = __ldg(p.midx + __ldg(p.owner_tl + j));
}

// ---------------------------------------------------------------------------------------- K5: scatter (M7)

// The source of one token under explicit masks: the largest member index whose mask is 1 at position q (reading M-7).
__device__ __noinline__ int32_t explicit_src(const int32_t* __restrict__ mem, const int64_t* __restrict__ offsets,
                                             const uint8_t* __restrict__ mask_in, int cnt, int64_t q) {
    // eight members at a time, largest first: their three loads each are independent, so a batch costs three round trips
    // instead of twenty-four
    for (int x0 = cnt - 1; x0 >= 0; x0 -= 8) {
        int j[8];
        int64_t oj[8], len[8];
        uint8_t mk[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) j[i] = x0 - i >= 0 ? __ldg(mem + x0 - i) : -1;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            oj[i] = j[i] >= 0 ? __ldg(offsets + j[i]) : 0;
            len[i] = j[i] >= 0 ? __ldg(offsets + j[i] + 1) - oj[i] : 0;
        }
#pragma unroll
        for (int i = 0; i < 8; ++i) mk[i] = q < len[i] ? __ldg(mask_in + oj[i] + q) : (uint8_t)0;
#pragma unroll
        for (int i = 0; i < 8; ++i)
            if (mk[i] != 0) return j[i];
    }
    return kSrcNone;
}

__device__ __forceinline__ GSeg load_gseg(const GSeg* g) {
    const int4 a = __ldg(reinterpret_cast<const int4*>(g)), b = __ldg(reinterpret_cast<const int4*>(g) + 1);
    GSeg o;
    o.out_start = (int64_t)(((uint64_t)(uint32_t)a.y << 32) | (uint32_t)a.x);
    o.tok_delta = (int64_t)(((uint64_t)(uint32_t)a.w << 32) | (uint32_t)a.z);
    o.lp_delta = (int64_t)(((uint64_t)(uint32_t)b.y << 32) | (uint32_t)b.x);
    o.src = b.z;
    o.aux = b.w;
    return o;
}

// One tile moved position by position through registers, walking the segment records from the tile's first one: the path
// for explicit masks, for the last (partial) tile, for tiles cut into more than 8 pieces and for pieces at the very ends
// of the input arrays.  Lane l owns positions l + 32 j of the tile.
struct ScatPtrs {   // what the walk needs, passed by value (a reference to the kernel parameters would copy all of them to the stack)
    const int32_t* tokens; const float* old_logp_in; const int64_t* offsets; const uint8_t* mask_in; const int32_t* mem_list;
    const GSeg* gseg; const int32_t* tile_seg;
    int32_t* merged_tokens; uint8_t* merged_mask; int32_t* merged_src; float* merged_old_logp;
};
__device__ __noinline__ void scatter_tile_walk(const ScatPtrs p, int t, int64_t N_out, int j_begin = 0, int j_end = 16) {
    const int lane = threadIdx.x & 31;
    const int32_t* __restrict__ tokens = p.tokens;
    const float* __restrict__ lps = p.old_logp_in;
    const bool want_lp = p.merged_old_logp != nullptr;
    const int64_t d0 = ((int64_t)t << kTSLog) + lane;
    int idx = __ldg(p.tile_seg + t);
    GSeg cur = load_gseg(p.gseg + idx);
    int64_t nxt = __ldg(&p.gseg[idx + 1].out_start);
#pragma unroll 1
    for (int j0 = j_begin; j0 < j_end; j0 += 4) {
        uint32_t xg[4], lg[4];
        int32_t sg[4];
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) {
            const int64_t d = d0 + 32 * (j0 + jj);
            xg[jj] = 0u; lg[jj] = 0u; sg[jj] = kSrcNone;
            if (d < N_out) {
                while (d >= nxt) {
                    ++idx;
                    cur = load_gseg(p.gseg + idx);
                    nxt = __ldg(&p.gseg[idx + 1].out_start);
                }
                xg[jj] = (uint32_t)__ldg(tokens + (d + cur.tok_delta));
                int32_t sj = cur.src;
                if (sj == kSrcExplicit) {
                    const int64_t q = d - cur.out_start;
                    sj = explicit_src(p.mem_list + cur.lp_delta, p.offsets, p.mask_in, cur.aux, q);
                    if (want_lp && sj >= 0) lg[jj] = __float_as_uint(__ldg(lps + (__ldg(p.offsets + sj) + q)));
                } else if (want_lp && sj >= 0) {
                    lg[jj] = __float_as_uint(__ldg(lps + (d + cur.lp_delta)));
                }
                sg[jj] = sj;
            }
        }
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) {
            const int64_t d = d0 + 32 * (j0 + jj);
            if (d < N_out) {
                p.merged_tokens[d] = (int32_t)xg[jj];
                p.merged_src[d] = sg[jj];
                p.merged_mask[d] = sg[jj] >= 0 ? 1 : 0;
                if (want_lp) p.merged_old_logp[d] = __uint_as_float(lg[jj]);
            }
        }
    }
}

constexpr int kScatThreads = 512;                                   // 16 warps: 118 registers without spills (20 warps fit the shared memory but spill at 96)
constexpr int kScatInBytes = 2560;                                   // one input array of a tile: 2 KB + 16-byte slack of up to 8 pieces
constexpr int kScatWarpBytes = 2 * 2 * kScatInBytes + 2 * 8 * 32 + 128;   // 2 input stages (tokens, old_logp), piece tables, barriers
constexpr int kScatSmem = (kScatThreads / 32) * kScatWarpBytes + 128;
static_assert(kScatWarpBytes % 128 == 0, "warp regions stay 128-byte aligned");

// Warp per tile of 512 OUTPUT positions, all bulk data through the TMA engine: a tile is cut at segment boundaries into
// at most 8 pieces; the lane that owns a piece launches one bulk async copy of the 16-byte-aligned superset of its token
// source (and one of its log-prob source) into the warp's input stage, one tile ahead; the warp then rewrites the pieces at
// the output's alignment into a staging copy of the four output rows (32-bit shared-memory accesses, conflict-free) and one
// lane sends them off with four bulk stores.  Requests of kilobytes instead of 128 bytes: what it takes to fill HBM.
__global__ void __launch_bounds__(kScatThreads, 1) merge_scatter_kernel(const MergeParams p) {
    pdl_wait();
    extern __shared__ __align__(128) uint8_t sc_dyn[];
    if (fatal(p)) return;
    const int lane = threadIdx.x & 31, wic = threadIdx.x >> 5;
    const int wglobal = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    const int ntiles = p.ctrl->n_tiles, nseg = p.ctrl->n_gsegs;
    const int64_t N_out = p.ctrl->N_out, N = p.N;
    const bool want_lp = p.merged_old_logp != nullptr;
    const int mis_t = p.mis, mis_l = (int)(((uintptr_t)p.old_logp_in >> 2) & 3);
    uint8_t* const wb = reinterpret_cast<uint8_t*>(((uintptr_t)sc_dyn + 127) & ~(uintptr_t)127) + (size_t)wic * kScatWarpBytes;
    uint8_t* const in_base = wb;                                            // [stage][tok | lp]
    int4* const tbl = reinterpret_cast<int4*>(wb + 4 * kScatInBytes);   // [stage][8 pieces][2]
    uint64_t* const full = reinterpret_cast<uint64_t*>(wb + 4 * kScatInBytes + 2 * 8 * 32);
    const ScatPtrs sp = {p.tokens, p.old_logp_in, p.offsets, p.mask_in, p.mem_list, p.gseg, p.tile_seg,
                         p.merged_tokens, p.merged_mask, p.merged_src, p.merged_old_logp};
    if (lane == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        fence_mbar_init();
    }
    __syncwarp();
    uint32_t phases = 0;
    // plan(t, stage): cuts tile t into pieces, launches their copies into input stage `stage`; returns the number of pieces,
    // or -1 when the tile takes the register walk.  rec = this lane's segment record of the tile (lane l: record s0 + l).
    auto plan = [&](int t, int stage, const GSeg& rec) -> int {
        const int64_t dt = (int64_t)t << kTSLog;
        const int64_t rel64 = rec.out_start - dt;
        const int rel = (int)max((int64_t)-1, min(rel64, (int64_t)kTS));           // lane 0: <= 0; later lanes: > 0, kTS = beyond
        const int reln = __shfl_down_sync(0xffffffffu, rel, 1);
        const bool valid = lane < 8 && (lane == 0 || rel < kTS);
        const int np = __popc(__ballot_sync(0xffffffffu, valid));
        const int rel8 = __shfl_sync(0xffffffffu, rel, 8);
        const int q0 = max(rel, 0), q1 = min(reln, kTS);
        bool bad = false;
        uint32_t tb = 0, lb = 0;
        int64_t tg0 = 0, lg0 = 0;
        int tw = 0, lw = -1;
        if (valid) {
            bad = rec.src == kSrcExplicit;
            const int pb = ((4 * q0) & ~15) + 48 * lane;                           // byte offset of the piece in the input stage
            const int64_t e0 = dt + q0 + rec.tok_delta;
            const int a = (int)((e0 + mis_t) & 3);
            tg0 = e0 - a;
            tb = (uint32_t)(((q1 - q0 + a + 3) >> 2) << 4);
            tw = (pb >> 2) + a;
            bad = bad || tg0 < 0 || tg0 + (tb >> 2) > N;
            if (want_lp && rec.src >= 0) {
                const int64_t f0 = dt + q0 + rec.lp_delta;
                const int al = (int)((f0 + mis_l) & 3);
                lg0 = f0 - al;
                lb = (uint32_t)(((q1 - q0 + al + 3) >> 2) << 4);
                lw = (pb >> 2) + al;
                bad = bad || lg0 < 0 || lg0 + (lb >> 2) > N;
            }
        }
        if (__any_sync(0xffffffffu, bad) || rel8 < kTS || dt + kTS > N_out) return -1;
        uint8_t* const ib = in_base + stage * 2 * kScatInBytes;
        const uint32_t total = __reduce_add_sync(0xffffffffu, valid ? tb + lb : 0u);
        if (valid) {
            tbl[(stage * 8 + lane) * 2] = make_int4(q0, q1, tw, lw);
            tbl[(stage * 8 + lane) * 2 + 1] = make_int4(rec.src, 0, 0, 0);
            bulk_load(ib + (((4 * q0) & ~15) + 48 * lane), p.tokens + tg0, tb, &full[stage]);
            if (lb) bulk_load(ib + kScatInBytes + (((4 * q0) & ~15) + 48 * lane), p.old_logp_in + lg0, lb, &full[stage]);
        }
        if (lane == 0) mbar_arrive_expect_tx(&full[stage], total);
        return np;
    };
    auto load_rec = [&](int t) -> GSeg {
        const int s0 = __ldg(p.tile_seg + t);
        return load_gseg(p.gseg + min(s0 + lane, nseg));   // lanes beyond the last record read the sentinel (starts at N_out)
    };
    const bool out_ok = ((((uintptr_t)p.merged_tokens | (uintptr_t)p.merged_src | (uintptr_t)p.merged_old_logp | (uintptr_t)p.merged_mask) & 15) == 0);
    if ((int64_t)ntiles * 4 <= nwarps) {   // few tiles (latency, not bandwidth): a quarter of a tile per warp, position by position
        if (wglobal < ntiles * 4) scatter_tile_walk(sp, wglobal >> 2, N_out, (wglobal & 3) * 4, (wglobal & 3) * 4 + 4);
        return;
    }
    if (wglobal >= ntiles) return;
    // Tiles go round the warps with a fixed stride.  (Handing them out by an atomic ticket evens out the warps' finishing
    // times -- tiles cut into several pieces take longer -- but 45 k same-address atomics cost more than that: 256 against
    // 235 us for the whole merge inside the bench step.)  tA: at work; tB: its copies are in flight; tC: its segment record
    // is being loaded.
    int tA = wglobal, tB = wglobal + nwarps, tC = wglobal + 2 * nwarps, pend = 0;
    pend = wglobal + 3 * nwarps;
    GSeg rec = load_rec(tA);
    int np_cur = out_ok ? plan(tA, 0, rec) : -1;
    if (tB < ntiles) rec = load_rec(tB);
    int it = 0;
    bool dead = false;
#pragma unroll 1
    for (; tA < ntiles; ++it) {
        const int t = tA;
        const int st = it & 1;
        int np_next = -1;
        if (tB < ntiles) {   // next tile: its copies fly while this one is rewritten; the tile after: its record
            if (out_ok) np_next = plan(tB, st ^ 1, rec);
            if (tC < ntiles) rec = load_rec(tC);
        }
        if (np_cur < 0) {
            scatter_tile_walk(sp, t, N_out);
        } else {
            const int64_t dt = (int64_t)t << kTSLog;
            const uint32_t in_tok = smem_u32(in_base + st * 2 * kScatInBytes), in_lp = in_tok + kScatInBytes;
            if (!mbar_wait_bounded(&full[st], (phases >> st) & 1u)) dead = true;
            phases ^= 1u << st;
            if (np_cur == 1) {
                // one source: lane l writes positions 4 l + 128 j .. + 3 (16-byte stores, 512 contiguous bytes per instruction),
                // read from the input stage at the source's own misalignment
                const int4 e0 = tbl[(st * 8) * 2], e1 = tbl[(st * 8) * 2 + 1];
                const uint32_t a0 = in_tok + 4 * (e0.z + 4 * lane);
                uint4* const gt4 = reinterpret_cast<uint4*>(p.merged_tokens + dt) + lane;
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    gt4[32 * j] = make_uint4(lds32(a0 + 512 * j), lds32(a0 + 512 * j + 4), lds32(a0 + 512 * j + 8), lds32(a0 + 512 * j + 12));
                if (want_lp) {
                    uint4* const gl4 = reinterpret_cast<uint4*>(p.merged_old_logp + dt) + lane;
                    if (e0.w >= 0) {
                        const uint32_t b0 = in_lp + 4 * (e0.w + 4 * lane);
#pragma unroll
                        for (int j = 0; j < 4; ++j)
                            gl4[32 * j] = make_uint4(lds32(b0 + 512 * j), lds32(b0 + 512 * j + 4), lds32(b0 + 512 * j + 8), lds32(b0 + 512 * j + 12));
                    } else {
#pragma unroll
                        for (int j = 0; j < 4; ++j) gl4[32 * j] = make_uint4(0u, 0u, 0u, 0u);
                    }
                }
                const uint32_t sv = (uint32_t)e1.x, mk = e1.x >= 0 ? 0x01010101u : 0u;
                uint4* const gs4 = reinterpret_cast<uint4*>(p.merged_src + dt) + lane;
#pragma unroll
                for (int j = 0; j < 4; ++j) gs4[32 * j] = make_uint4(sv, sv, sv, sv);
                reinterpret_cast<uint4*>(p.merged_mask + dt)[lane] = make_uint4(mk, mk, mk, mk);
            } else {
#pragma unroll 1
                for (int pi = 0; pi < np_cur; ++pi) {
                    const int4 e0 = tbl[(st * 8 + pi) * 2], e1 = tbl[(st * 8 + pi) * 2 + 1];
                    for (int q = e0.x + lane; q < e0.y; q += 32) {
                        p.merged_tokens[dt + q] = (int32_t)lds32(in_tok + 4 * (e0.z + q - e0.x));
                        if (want_lp) p.merged_old_logp[dt + q] = e0.w >= 0 ? __uint_as_float(lds32(in_lp + 4 * (e0.w + q - e0.x))) : 0.f;
                        p.merged_src[dt + q] = e1.x;
                        p.merged_mask[dt + q] = e1.x >= 0 ? (uint8_t)1 : (uint8_t)0;
                    }
                }
            }
        }
        np_cur = np_next;
        tA = tB;
        tB = tC;
        tC = pend;
        pend += nwarps;
        if (__any_sync(0xffffffffu, dead)) break;
    }
    if (dead && lane == 0) atomicOr(&p.ctrl->status, (uint32_t)AJT_STATUS_INTERNAL);
}
}  // namespace

// Per-device launch facts: the SM count and the one-time opt-in to large dynamic shared memory.  A process-wide table that
// is written once per device (idempotent values, so a race between two first calls is benign); nothing else is kept
// between calls.
namespace {
struct DevFacts {
    int num_sms;
    bool ready;
};
DevFacts g_dev[64] = {};
size_t group_fast_smem(int n) {
    const size_t H = (size_t)n + n / 8 + 16;
    return (H + 2) * 4 + ((H + 3) & ~(size_t)1) * 2 + 4 * ((size_t)n + 2) * 4 + 2 * (((size_t)n + 1) & ~(size_t)1) * 2 + 16;
}

int merge_dev_facts(int* num_sms) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return AJT_ERR_CUDA;
    if (dev < 0 || dev >= 64) return AJT_ERR_UNSUPPORTED;
    if (!g_dev[dev].ready) {
        int sms = 0;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) return AJT_ERR_CUDA;
        const int grp_smem = (int)group_fast_smem(kGrpSmemN);
        if (cudaFuncSetAttribute(merge_group_fast_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, grp_smem) != cudaSuccess)
            return AJT_ERR_CUDA;
        if (cudaFuncSetAttribute(merge_hash_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kHashSmem) != cudaSuccess)
            return AJT_ERR_CUDA;
        if (cudaFuncSetAttribute(merge_select_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SelectStage)) != cudaSuccess)
            return AJT_ERR_CUDA;
        if (cudaFuncSetAttribute(merge_scatter_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kScatSmem) != cudaSuccess)
            return AJT_ERR_CUDA;
        if (cudaFuncSetAttribute(merge_compact_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kCompactSmem) != cudaSuccess)
            return AJT_ERR_CUDA;
        g_dev[dev].num_sms = sms;
        g_dev[dev].ready = true;
    }
    *num_sms = g_dev[dev].num_sms;
    return AJT_OK;
}

}  // namespace

extern "C" size_t ajt_merge_workspace_bytes(int32_t n, int64_t n_tokens) {
    if (n < 0 || n_tokens < 0) return 0;
    return merge_ws_layout(n, n_tokens).ent + 5 * 256 + a256(((size_t)64 * (size_t)n + 4096) * kEntBytes);
}

extern "C" size_t ajt_merge_workspace_bytes_for_pairs(int32_t n, int64_t n_tokens, int64_t n_pairs) {
    if (n < 0 || n_tokens < 0 || n_pairs < 0) return 0;
    const size_t pairs = (size_t)n_pairs > (size_t)n + 1024 ? (size_t)n_pairs : (size_t)n + 1024;
    return merge_ws_layout(n, n_tokens).ent + 5 * 256 + a256(pairs * kEntBytes);
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

    int num_sms = 0;
    const int frc = merge_dev_facts(&num_sms);
    if (frc != AJT_OK) return frc;

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
    p.goff = reinterpret_cast<int64_t*>(b + ws.goff);
    p.tl_rec = reinterpret_cast<int4*>(b + ws.tl_rec);
    p.lbad = b + ws.lbad;
    p.grp_rec = reinterpret_cast<int4*>(b + ws.grp_rec);
    p.unit_rec = reinterpret_cast<int4*>(b + ws.unit_rec);
    p.seg_part = reinterpret_cast<uint64_t*>(b + ws.seg_part);
    p.cinfo = reinterpret_cast<uint2*>(b + ws.absorbed);
    p.owner_tl = reinterpret_cast<int32_t*>(b + ws.owner_tl);
    p.midx = reinterpret_cast<int32_t*>(b + ws.midx);
    for (int k = 0; k < 8; ++k) p.sel[k] = reinterpret_cast<int32_t*>(b + ws.sel[k]);
    p.sel_q = reinterpret_cast<int2*>(b + ws.sel_q);
    p.mem_list = reinterpret_cast<int32_t*>(b + ws.mem_list);
    p.sv_rec = reinterpret_cast<int4*>(b + ws.sv_rec);
    p.rseg = reinterpret_cast<int2*>(b + ws.rseg);
    p.gseg_base = reinterpret_cast<int32_t*>(b + ws.gseg_base);
    p.gseg = reinterpret_cast<GSeg*>(b + ws.gseg);
    p.tile_seg = reinterpret_cast<int32_t*>(b + ws.tile_seg);
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
    const int64_t sc = slice_capacity(n, n_tokens);
    if (sc > (int64_t)INT32_MAX) return AJT_ERR_UNSUPPORTED;
    p.slice_cap = (int32_t)sc;
    p.mis = (int32_t)(((uintptr_t)tokens >> 2) & 3);
    p.slim = n <= kGrpSmemN ? 1 : 0;

    if (n == 0) {
        if (cudaMemsetAsync(p.ctrl, 0, sizeof(AjtCtrl), stream) != cudaSuccess) return AJT_ERR_CUDA;
        if (cudaMemsetAsync(counts, 0, 2 * sizeof(int64_t), stream) != cudaSuccess) return AJT_ERR_CUDA;
        if (cudaMemsetAsync(merged_offsets, 0, sizeof(int64_t), stream) != cudaSuccess) return AJT_ERR_CUDA;
        return AJT_OK;
    }
    if (n <= kGrpSmemN) AJT_LAUNCH(merge_group_fast_kernel<<<1, 1024, group_fast_smem(n), stream>>>(p, n + n / 8 + 16));
    else AJT_LAUNCH(merge_group_radix_kernel<<<1, 1024, 0, stream>>>(p));
    // kernels 2..6 are launched as programmatic dependents: resident and waiting when their predecessor ends
    const int64_t want = ((int64_t)n * 32 + 255) / 256;   // a warp per merged sequence (at most n)
    const int plan_grid = (int)(want < (int64_t)num_sms * 8 ? (want < 1 ? 1 : want) : (int64_t)num_sms * 8);
    const int64_t uwant = ((int64_t)n + 255) / 256;
    if (launch_dependent(merge_units_kernel, (int)(uwant < (int64_t)num_sms * 4 ? uwant : (int64_t)num_sms * 4), 256, 0, stream, 1, p) != cudaSuccess ||
        launch_dependent(merge_hash_kernel, num_sms * (kVT > 4 ? 2 : 3), kHashThreads, kHashSmem, stream, 1, p) != cudaSuccess ||
        launch_dependent(merge_select_kernel, num_sms * 4, kSelThreads, sizeof(SelectStage), stream, 1, p) != cudaSuccess ||
        launch_dependent(merge_compact_kernel, 1, 1024, kCompactSmem, stream, 1, p) != cudaSuccess ||
        launch_dependent(merge_plan_kernel, plan_grid, 256, 0, stream, 1, p) != cudaSuccess ||
        launch_dependent(merge_scatter_kernel, num_sms, kScatThreads, kScatSmem, stream, 1, p) != cudaSuccess)
        return AJT_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? AJT_OK : AJT_ERR_CUDA;
}
