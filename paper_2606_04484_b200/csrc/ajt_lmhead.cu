// Log-prob and entropy of the target token straight from the hidden states: logits = H W^T are produced tile by tile on the
// 5th-generation tensor cores (tcgen05.mma, bf16 x bf16 -> fp32 in TMEM) and reduced on the fly (online max / sum-exp /
// sum e (z - m) / target gather), so the [T, V] logits never reach HBM.  This is the forward half of SURVEY.md §8(f) f3: the pass
// that produces the old / reference log-probs the loss consumes.  DESIGN.md "O-H".
//
// Work unit = (a block of 128 or 256 rows of H) x (one of 4 vocabulary ranges), striped over the SMs (one CTA, or one CTA pair, per
// SM / pair of SMs).  Inside a unit the range is walked in tiles of 256 columns; per tile the K loop streams 64-wide slabs of H
// and W through a TMA ring (SWIZZLE_128B, K-major), one elected thread issues 4 x tcgen05.mma per slab, and the two 256-column
// TMEM accumulators alternate so that the epilogue warps (one row per thread: tcgen05.ld 32 columns at a time) reduce tile n
// while the tensor cores fill tile n+1.  The work groups that run at the same time share the W ranges (L2).
// Per (row, range) the epilogue leaves {m, s, u, z_y}; lm_head_combine_kernel folds the range partials of a row.
// With a mask, the unmasked rows are compacted first (lm_compact_kernel, lm_gather_kernel) so that masked rows cost no flops.
#include <cuda.h>

#include "ajt_common.cuh"
#include "ajt_token.cuh"

namespace {

using namespace ajt;

constexpr int kBM = 128, kBN = 256, kBK = 64, kVS = 16;
constexpr int kABytes = kBM * kBK * 2;
constexpr int kLmThreads = 192;   // warp 0: TMA producer, warp 1: MMA issuer + TMEM owner, warps 2-5: epilogue
constexpr float kLog2e = 1.4426950408889634f;
// NCTA = 1: one CTA per 128-row block, the whole 256-column W tile in its shared memory (16 + 32 KB per slab, 4 stages).
// NCTA = 2: a CTA pair (cluster of 2, tcgen05 cta_group::2) per 256-row block: each CTA stages its own 128 rows of H and
// HALF of the W tile (16 + 16 KB per slab, 6 stages); the leader issues 256 x 256 x 16 MMAs that read both CTAs' shared
// memory and fill both CTAs' tensor memory.  Less shared-memory traffic per flop and a deeper ring.
template <int NCTA> struct LmCfg {
    static constexpr int kBRows = kBN / NCTA;                      // W rows (vocabulary columns) staged per CTA
    static constexpr int kBBytes = kBRows * kBK * 2;
    static constexpr int kStageBytes = kABytes + kBBytes;
    static constexpr int kStages = NCTA == 1 ? 4 : 6;
    static constexpr size_t kSmem = (size_t)kStages * kStageBytes + 1024 /* alignment slack */ + 256 /* barriers */;
    // instruction descriptor (kind::f16): D = F32, A = B = BF16, both K-major, N = 256, M = 128 per CTA
    static constexpr uint32_t kIdesc =
        (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(kBN >> 3) << 17) | ((uint32_t)((kBM * NCTA) >> 4) << 24);
};
constexpr uint32_t kPeerBitMask = 0xFEFFFFFFu;   // shared::cluster address of the same location in the pair's CTA 0

struct LmParams {
    const int32_t* targets;     // per row of the (possibly compacted) hidden matrix the kernel sees
    const uint8_t* mask;
    const int32_t* n_rows;      // DEVICE: rows to process when the masked rows were compacted away, else NULL (then T)
    const int32_t* row_idx;     // [n_rows] original row of compacted row k, or NULL
    int64_t T;
    int32_t round_bf16;          // AJT_LM_ROUND_LOGITS_BF16: logits rounded to bf16 (RNE) before the softmax
    int32_t d, V, vs_len, nvs;   // vs_len: columns per vocabulary range (multiple of kBN); nvs: ranges in use (<= kVS)
    float4* part;                             // [T][kVS] {m, s, u, z_y (or -inf)}
    float* logp_out;
    float* ent_out;
    float* lse_out;
    uint32_t* status;            // first word of the workspace: AJT_STATUS_BAD_TARGET when a processed row's target is outside [0, V)
    // ---- backward (ajt_lm_head_loss_bwd): the same mainloop with other epilogues
    int64_t row0;                // first (compacted) row of the chunk this launch works on; rows are counted from it
    const float* g_row;          // kDz: [rows] d loss / d logp of every (compacted) row (0: nothing to propagate)
    const float* lse_row;        // kDz: [rows] log-sum-exp of the row's logits (forward pass)
    __nv_bfloat16* dz;           // kDz: [chunk rows, ld_dz] dZ of the chunk, row-major
    __nv_bfloat16* dzt;          // kDz: [ld_dz, ld_dzt] its transpose (vocabulary-major)
    int64_t ld_dz, ld_dzt;
    __nv_bfloat16* out_bf16;     // kStoreBf16: [*, ld_out] rows scattered through row_idx (dH)
    float* out_f32;              // kAccF32: [n_out_rows, ld_out] += (dW)
    int64_t ld_out;
    int64_t n_out_rows;          // kAccF32: rows that exist (the operand is zero-padded beyond)
};
// Epilogue of the tile kernel.  kReduce: the forward pass (online log-sum-exp / entropy / target gather).  kDz: the tile of
// logits becomes dZ = g (1[v = y] - exp(z - lse)) in bf16, stored row-major and transposed.  kStoreBf16 / kAccF32: a plain
// product A B^T written as bf16 rows (dH) or added to an fp32 matrix (dW).
enum { kReduce = 0, kDz = 1, kStoreBf16 = 2, kAccF32 = 3 };

__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(
                     smem_u32(smem_dst)),
                 "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
                 : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// pair: the copy lands in this CTA's shared memory, its bytes are counted on CTA 0's barrier
__device__ __forceinline__ void tma_load_2d_pair(void* smem_dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(
            smem_u32(smem_dst)),
        "l"(map), "r"(smem_u32(bar) & kPeerBitMask), "r"(c0), "r"(c1)
        : "memory");
}
template <int NCTA>
__device__ __forceinline__ void tc_commit(uint64_t* bar) {
    if (NCTA == 1)
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
    else   // arrives on the barrier at this offset in BOTH CTAs of the pair
        asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(
                         smem_u32(bar)),
                     "h"((uint16_t)3)
                     : "memory");
}
// arrive on the barrier at this offset in CTA `rank` of the cluster
__device__ __forceinline__ void mbar_arrive_remote(uint64_t* bar, uint32_t rank) {
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(mapa(smem_u32(bar), rank)) : "memory");
}
// K-major operand tile, rows of 128 bytes (64 bf16), 8-row groups 1024 bytes apart, SWIZZLE_128B
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr) {
    const uint64_t lo = (uint64_t)((addr >> 4) & 0x3FFFu);
    const uint64_t hi = (uint64_t)((1024u >> 4) & 0x3FFFu) | (1ull << 14) /* descriptor version */ | (2ull << 29) /* SWIZZLE_128B */;
    return lo | (hi << 32);
}
template <int NCTA>
__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t accumulate) {
    if (NCTA == 1)
        asm volatile(
            "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
            "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem_d),
            "l"(da), "l"(db), "r"(LmCfg<1>::kIdesc), "r"(accumulate)
            : "memory");
    else
        asm volatile(
            "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
            "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem_d),
            "l"(da), "l"(db), "r"(LmCfg<2>::kIdesc), "r"(accumulate)
            : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
          "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]),
          "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]),
          "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr)
        : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// How many vocabulary ranges to cut the columns into, given the row blocks there really are (known only on the device when
// masked rows were compacted away) and the G work groups of the launch: every group walks `rounds` items of `len` column
// tiles each, so the launch takes ~ rounds x len tile times; the fewest ranges with the smallest product win.  (61 row
// blocks on 74 groups: 4 ranges = 4 rounds x 149 tiles, 6 ranges = 5 x 99: 17 % less.)  Host and device, forward kernel and
// combine kernel all call this with the same arguments.
__host__ __device__ inline void choose_ranges(int64_t n_mtiles, int G, int V, int& nvs, int& vs_len) {
    const int ncol = (V + kBN - 1) / kBN;
    int64_t best = INT64_MAX;
    nvs = 1;
    vs_len = ncol * kBN;
    for (int s = 1; s <= kVS && s <= ncol; ++s) {
        const int len = (ncol + s - 1) / s, se = (ncol + len - 1) / len;   // se <= s ranges are not empty
        const int64_t rounds = (n_mtiles * se + G - 1) / G, cost = rounds * len;
        if (cost < best) { best = cost; nvs = se; vs_len = len * kBN; }
    }
}

// Work unit u = (row block u / nvs, vocabulary range u % nvs); work group g (a CTA, or a CTA pair) takes units g, g + G, ...
// Groups that run together hold neighbouring units: a few row blocks times all ranges, so the W ranges are shared through L2.
template <int NCTA>
__device__ __forceinline__ bool item_of(int nvs, int n_mtiles, int it, int& mt, int& vs) {
    const int G = (int)gridDim.x / NCTA, g = (int)blockIdx.x / NCTA;
    const int64_t u = (int64_t)it * G + g;
    mt = (int)(u / nvs);
    vs = (int)(u % nvs);
    return mt < n_mtiles;
}

// Row blocks are 128 * NCTA rows.
template <int NCTA, int MODE>
__global__ void __launch_bounds__(kLmThreads, 1) lm_head_kernel(const __grid_constant__ CUtensorMap map_h,
                                                                const __grid_constant__ CUtensorMap map_w, const LmParams p) {
    using Cfg = LmCfg<NCTA>;
    constexpr int kStages = Cfg::kStages, kStageBytes = Cfg::kStageBytes;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + (size_t)kStages * kStageBytes);
    uint64_t* empty = full + kStages;
    uint64_t* tfull = empty + kStages;    // [2] accumulator ready
    uint64_t* tempty = tfull + 2;         // [2] accumulator drained (pair: CTA 0's counts both CTAs' epilogue warps)
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty + 2);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = NCTA > 1 ? cluster_ctarank() : 0u;
    const int nk = p.d / kBK;
    // rows actually present: all of them, or (masked rows compacted away) the device-side count; a backward launch works on the
    // chunk of p.T rows that starts at row0 and has nothing to do beyond the count
    int64_t Teff = p.n_rows ? (int64_t)*p.n_rows : p.T;
    if (MODE != kReduce) {
        const int64_t left = p.n_rows ? Teff - p.row0 : p.T;   // unmasked rows from this chunk on
        if (left <= 0) return;   // uniform over the grid: before any barrier / tensor-memory allocation
        Teff = MODE == kAccF32 ? p.T : (left < p.T ? left : p.T);
    }
    const int n_mtiles = (int)((Teff + kBM * NCTA - 1) / (kBM * NCTA));
    const int n_groups = (int)gridDim.x / NCTA;
    int nvs = p.nvs, vs_len = p.vs_len;
    if (nvs == 0) choose_ranges(n_mtiles, n_groups, p.V, nvs, vs_len);   // ranges fitted to the rows there are
    const int n_items = (int)(((int64_t)n_mtiles * nvs + n_groups - 1) / n_groups);

    if (threadIdx.x == 0) {
        for (int i = 0; i < kStages; ++i) {
            mbar_init(&full[i], 1);
            mbar_init(&empty[i], 1);
        }
        for (int i = 0; i < 2; ++i) {
            mbar_init(&tfull[i], 1);
            mbar_init(&tempty[i], 4 * NCTA);
        }
        fence_mbar_init();
    }
    if (warp == 1) {   // TMEM: all 512 columns (two 256-column fp32 accumulators of this CTA's 128 rows)
        if (NCTA == 1) {
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
        } else {
            asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
        }
    }
    tc_fence_before();
    if (NCTA > 1) cluster_sync_all(); else __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        // ===== TMA producer (every CTA: its own rows of H, its share of the W tile) =====
        if (lane == 0) {
            int stage = 0;
            uint32_t ph = 0;
            for (int it = 0; it < n_items; ++it) {
                int mt, vs;
                if (!item_of<NCTA>(nvs, n_mtiles, it, mt, vs)) continue;
                const int v0 = vs * vs_len, v1 = min(p.V, v0 + vs_len);
                const int row0 = (mt * NCTA + (int)rank) * kBM;
                for (int n0 = v0; n0 < v1; n0 += kBN) {
                    for (int k = 0; k < nk; ++k) {
                        mbar_wait(&empty[stage], ph ^ 1u);
                        uint8_t* sa = smem + (size_t)stage * kStageBytes;
                        if (NCTA == 1) {
                            mbar_arrive_expect_tx(&full[stage], kStageBytes);
                            tma_load_2d(sa, &map_h, k * kBK, row0, &full[stage]);
                            tma_load_2d(sa + kABytes, &map_w, k * kBK, n0, &full[stage]);
                        } else {
                            if (rank == 0) mbar_arrive_expect_tx(&full[stage], 2 * kStageBytes);   // both CTAs' bytes land on CTA 0's barrier
                            tma_load_2d_pair(sa, &map_h, k * kBK, row0, &full[stage]);
                            tma_load_2d_pair(sa + kABytes, &map_w, k * kBK, n0 + (int)rank * Cfg::kBRows, &full[stage]);
                        }
                        if (++stage == kStages) { stage = 0; ph ^= 1u; }
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer (pair: the leader CTA only) =====
        if (rank == 0) {
            int stage = 0, as = 0;
            uint32_t ph = 0, aph = 0;
            for (int it = 0; it < n_items; ++it) {
                int mt, vs;
                if (!item_of<NCTA>(nvs, n_mtiles, it, mt, vs)) continue;
                const int v0 = vs * vs_len, v1 = min(p.V, v0 + vs_len);
                for (int n0 = v0; n0 < v1; n0 += kBN) {
                    mbar_wait(&tempty[as], aph ^ 1u);
                    tc_fence_after();
                    const uint32_t tacc = tmem_base + (uint32_t)(as * kBN);
                    for (int k = 0; k < nk; ++k) {
                        mbar_wait(&full[stage], ph);
                        tc_fence_after();
                        if (lane == 0) {
                            const uint32_t sa = smem_u32(smem + (size_t)stage * kStageBytes), sb = sa + kABytes;
#pragma unroll
                            for (int kk = 0; kk < kBK / 16; ++kk)   // 16 bf16 = 32 bytes along K inside the 128-byte swizzled row
                                umma_bf16<NCTA>(tacc, smem_desc(sa + kk * 32), smem_desc(sb + kk * 32), (uint32_t)((k | kk) != 0));
                            tc_commit<NCTA>(&empty[stage]);               // frees the smem slot (in both CTAs) once read
                            if (k == nk - 1) tc_commit<NCTA>(&tfull[as]); // accumulator complete
                        }
                        __syncwarp();
                        if (++stage == kStages) { stage = 0; ph ^= 1u; }
                    }
                    if (++as == 2) { as = 0; aph ^= 1u; }
                }
            }
        }
    } else {
        // ===== epilogue: thread <-> one row of this CTA's 128 (TMEM lane); warp w may touch lanes 32 (w % 4) .. +31 =====
        const int quad = warp & 3;
        const int rloc = quad * 32 + lane;
        int as = 0;
        uint32_t aph = 0;
        for (int it = 0; it < n_items; ++it) {
            int mt, vs;
            if (!item_of<NCTA>(nvs, n_mtiles, it, mt, vs)) continue;
            const int64_t row = (int64_t)(mt * NCTA + (int)rank) * kBM + rloc;
            const bool live = row < Teff;
            const int v0 = vs * vs_len, v1 = min(p.V, v0 + vs_len);
            if (MODE != kReduce) {
                // ---- backward epilogues: one row of the tile per thread, 32 columns at a time
                int y = -1;
                float g = 0.f, klse = 0.f;
                int64_t orow = row;
                if (MODE == kDz && live) {
                    y = p.targets[p.row0 + row];
                    g = p.g_row[p.row0 + row];
                    klse = -p.lse_row[p.row0 + row] * kLog2e;
                }
                if (MODE == kStoreBf16 && live && p.row_idx) orow = p.row_idx[p.row0 + row];
                for (int n0 = v0; n0 < v1; n0 += kBN) {
                    mbar_wait(&tfull[as], aph);
                    tc_fence_after();
                    const uint32_t tacc = tmem_base + ((uint32_t)(quad * 32) << 16) + (uint32_t)(as * kBN);
#pragma unroll 1
                    for (int c = 0; c < kBN; c += 32) {
                        uint32_t v[32];
                        tmem_ld32(tacc + (uint32_t)c, v);
                        const int col0 = n0 + c;
                        if (MODE == kDz) {
                            uint32_t w2[16];
#pragma unroll
                            for (int e = 0; e < 32; e += 2) {
                                float x0 = __uint_as_float(v[e]), x1 = __uint_as_float(v[e + 1]);
                                if (p.round_bf16) {
                                    x0 = __bfloat162float(__float2bfloat16_rn(x0));
                                    x1 = __bfloat162float(__float2bfloat16_rn(x1));
                                }
                                float d0 = -g * ex2(fmaf(x0, kLog2e, klse)), d1 = -g * ex2(fmaf(x1, kLog2e, klse));
                                if (col0 + e == y) d0 += g;
                                if (col0 + e + 1 == y) d1 += g;
                                if (col0 + e >= p.V || g == 0.f) d0 = 0.f;        // padding columns of the operand are zeros
                                if (col0 + e + 1 >= p.V || g == 0.f) d1 = 0.f;
                                w2[e >> 1] = pack_bf16x2(d0, d1);
                            }
                            // row-major: this thread's 32 columns are 64 contiguous bytes (rows beyond the chunk do not exist)
                            if (row < p.T) {
                                uint4* dst = reinterpret_cast<uint4*>(p.dz + row * p.ld_dz + col0);
#pragma unroll
                                for (int q = 0; q < 4; ++q) dst[q] = make_uint4(w2[4 * q], w2[4 * q + 1], w2[4 * q + 2], w2[4 * q + 3]);
                                // transposed: for one column the warp's 32 rows are 64 contiguous bytes
                                unsigned short* dt = reinterpret_cast<unsigned short*>(p.dzt) + (int64_t)col0 * p.ld_dzt + row;
#pragma unroll
                                for (int e = 0; e < 32; ++e)
                                    dt[(int64_t)e * p.ld_dzt] = (unsigned short)((e & 1) ? (w2[e >> 1] >> 16) : (w2[e >> 1] & 0xffffu));
                            }
                        } else if (MODE == kStoreBf16) {
                            if (live && col0 < p.V) {
                                uint4* dst = reinterpret_cast<uint4*>(p.out_bf16 + orow * p.ld_out + col0);
#pragma unroll
                                for (int q = 0; q < 4; ++q)
                                    dst[q] = make_uint4(pack_bf16x2(__uint_as_float(v[8 * q]), __uint_as_float(v[8 * q + 1])),
                                                        pack_bf16x2(__uint_as_float(v[8 * q + 2]), __uint_as_float(v[8 * q + 3])),
                                                        pack_bf16x2(__uint_as_float(v[8 * q + 4]), __uint_as_float(v[8 * q + 5])),
                                                        pack_bf16x2(__uint_as_float(v[8 * q + 6]), __uint_as_float(v[8 * q + 7])));
                            }
                        } else {   // kAccF32
                            if (row < p.n_out_rows && col0 < p.V) {
                                float4* dst = reinterpret_cast<float4*>(p.out_f32 + row * p.ld_out + col0);
#pragma unroll
                                for (int q = 0; q < 8; ++q) {
                                    float4 a = dst[q];
                                    a.x += __uint_as_float(v[4 * q]); a.y += __uint_as_float(v[4 * q + 1]);
                                    a.z += __uint_as_float(v[4 * q + 2]); a.w += __uint_as_float(v[4 * q + 3]);
                                    dst[q] = a;
                                }
                            }
                        }
                    }
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) {
                        if (NCTA == 1) mbar_arrive(&tempty[as]);
                        else mbar_arrive_remote(&tempty[as], 0);
                    }
                    if (++as == 2) { as = 0; aph ^= 1u; }
                }
                continue;
            }
            const int y = live ? p.targets[row] : -1;
            float m = -INFINITY, s = 0.f, u = 0.f, zy = -INFINITY;
            for (int n0 = v0; n0 < v1; n0 += kBN) {
                mbar_wait(&tfull[as], aph);
                tc_fence_after();
                const uint32_t tacc = tmem_base + ((uint32_t)(quad * 32) << 16) + (uint32_t)(as * kBN);
#pragma unroll 1
                for (int c = 0; c < kBN; c += 32) {
                    uint32_t v[32];
                    tmem_ld32(tacc + (uint32_t)c, v);
                    if (p.round_bf16) {   // what a forward pass that stores bf16 logits (the loss call's input) would see
#pragma unroll
                        for (int e = 0; e < 32; ++e) v[e] = __float_as_uint(__bfloat162float(__float2bfloat16_rn(__uint_as_float(v[e]))));
                    }
                    const int col0 = n0 + c;
                    if (col0 >= v1) continue;
                    const int nval = min(32, v1 - col0);
                    float cm = -INFINITY;
#pragma unroll
                    for (int e = 0; e < 32; ++e)
                        if (e < nval) cm = fmaxf(cm, __uint_as_float(v[e]));
                    if (cm > m) {   // re-base the running partial onto the new maximum
                        const float f = m == -INFINITY ? 0.f : ex2((m - cm) * kLog2e);
                        const float dm = m == -INFINITY ? 0.f : m - cm;
                        u = f * fmaf(dm, s, u);
                        s = f * s;
                        m = cm;
                    }
                    const float km = -m * kLog2e;
                    float es = 0.f, eu = 0.f;
#pragma unroll
                    for (int e = 0; e < 32; ++e) {
                        if (e < nval) {
                            const float x = __uint_as_float(v[e]);
                            const float ex = ex2(fmaf(x, kLog2e, km));
                            es += ex;
                            eu = fmaf(ex, x - m, eu);
                        }
                    }
                    s += es;
                    u += eu;
                    if (y >= col0 && y < col0 + nval) {
#pragma unroll
                        for (int e = 0; e < 32; ++e)
                            if (e == y - col0) zy = __uint_as_float(v[e]);
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) {
                    if (NCTA == 1) mbar_arrive(&tempty[as]);
                    else mbar_arrive_remote(&tempty[as], 0);   // the leader's MMA warp waits for both CTAs' epilogues
                }
                if (++as == 2) { as = 0; aph ^= 1u; }
            }
            if (live) p.part[row * kVS + vs] = make_float4(m, s, u, zy);
        }
    }
    tc_fence_before();
    if (NCTA > 1) cluster_sync_all(); else __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        if (NCTA == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
        else asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
    }
}

// Folds the range partials of every processed row and writes the outputs at the row's ORIGINAL position (the outputs of
// masked rows were zeroed beforehand when the rows were compacted).
__global__ void __launch_bounds__(256) lm_head_combine_kernel(const LmParams p, int groups, int ncta) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t Teff = p.n_rows ? (int64_t)*p.n_rows : p.T;
    int nvs, vs_len;   // the ranges the tile kernel chose: same function, same arguments
    choose_ranges((Teff + kBM * ncta - 1) / (kBM * ncta), groups, p.V, nvs, vs_len);
    for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < Teff; t += stride) {
        float lp = 0.f, H = 0.f, lse = 0.f;
        {
            const float4* q = p.part + t * kVS;
            float M = -INFINITY, zy = -INFINITY;
            for (int k = 0; k < nvs; ++k) {
                M = fmaxf(M, q[k].x);
                zy = fmaxf(zy, q[k].w);   // exactly one range holds the target; the others left -inf
            }
            float S = 0.f, U = 0.f;
            for (int k = 0; k < nvs; ++k) {
                const float4 v = q[k];
                const float f = v.x == -INFINITY ? 0.f : ex2((v.x - M) * kLog2e);
                const float dm = v.x == -INFINITY ? 0.f : v.x - M;
                U += f * fmaf(dm, v.y, v.z);
                S += f * v.y;
            }
            const float logS = logf(S);
            lp = (zy - M) - logS;
            H = logS - U / S;
            lse = M + logS;
        }
        const int y = p.targets[t];
        if (y < 0 || y >= p.V) {   // no column matched: report it instead of returning -inf (the row's outputs are 0)
            atomicOr(p.status, (uint32_t)AJT_STATUS_BAD_TARGET);
            lp = 0.f; H = 0.f; lse = 0.f;
        }
        const int64_t o = p.row_idx ? (int64_t)p.row_idx[t] : t;
        p.logp_out[o] = lp;
        if (p.ent_out) p.ent_out[o] = H;
        if (p.lse_out) p.lse_out[o] = lse;
    }
}

// ---- masked rows are not worth a single flop: compact the unmasked rows first (stable, one pass: tiles of 1,024 rows handed out
// by an atomic ticket, each publishes its count and adds up its predecessors'), gather their hidden rows and targets into a
// dense matrix, run the tiles on that, scatter the results back.
constexpr int kCompactTile = 1024;
__global__ void __launch_bounds__(256) lm_compact_kernel(const uint8_t* __restrict__ mask, int64_t T, uint64_t* tile_state, int32_t* ticket,
                                                         int32_t* row_idx, int32_t* n_rows) {
    __shared__ int s_w[8];
    __shared__ int s_tile, s_base;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int ntiles = (int)((T + kCompactTile - 1) / kCompactTile);
    for (;;) {
        if (tid == 0) s_tile = atomicAdd(ticket, 1);
        __syncthreads();
        const int tile = s_tile;
        if (tile >= ntiles) break;
        const int64_t t0 = (int64_t)tile * kCompactTile + tid * 4;
        bool on[4];
        int cnt = 0;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            on[e] = t0 + e < T && mask[t0 + e] != 0;
            cnt += on[e];
        }
        int inc = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += v;
        }
        if (lane == 31) s_w[warp] = inc;
        __syncthreads();
        int wbase = 0, total = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) {
            if (w < warp) wbase += s_w[w];
            total += s_w[w];
        }
        if (tid == 0) {
            __threadfence();
            atomicExch(reinterpret_cast<unsigned long long*>(&tile_state[tile]), (1ull << 63) | (unsigned long long)total);
        }
        int pre = 0;
        for (int t = tid; t < tile; t += 256) {
            unsigned long long st;
            do {
                st = *reinterpret_cast<volatile unsigned long long*>(&tile_state[t]);
            } while (!(st >> 63));
            pre += (int)(st & 0x7fffffffull);
        }
#pragma unroll
        for (int o = 16; o; o >>= 1) pre += __shfl_xor_sync(0xffffffffu, pre, o);
        __syncthreads();
        if (lane == 0) s_w[warp] = pre;
        __syncthreads();
        if (tid == 0) {
            int b = 0;
            for (int w = 0; w < 8; ++w) b += s_w[w];
            s_base = b;
        }
        __syncthreads();
        int k = s_base + wbase + inc - cnt;
#pragma unroll
        for (int e = 0; e < 4; ++e)
            if (on[e]) row_idx[k++] = (int32_t)(t0 + e);
        if (tile == ntiles - 1 && tid == 255) *n_rows = s_base + total;
        __syncthreads();
    }
}
__global__ void __launch_bounds__(256) lm_gather_kernel(const uint4* __restrict__ hidden, int64_t ld16, int32_t d16, const int32_t* __restrict__ targets,
                                                        const int32_t* __restrict__ row_idx, const int32_t* __restrict__ n_rows, uint4* hidden_c,
                                                        int32_t* targets_c) {
    const int64_t n = (int64_t)*n_rows * d16, stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const int64_t k = i / d16;
        const int c = (int)(i - k * d16);
        const int64_t r = row_idx[k];
        hidden_c[i] = __ldg(hidden + r * ld16 + c);
        if (c == 0) targets_c[k] = targets[r];
    }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// [rows, d] row-major bf16 with row stride ld (elements); box = 64 columns x box_rows rows, 128-byte swizzle
bool make_map(EncodeTiledFn fn, CUtensorMap* map, const void* base, int64_t rows, int32_t d, int64_t ld, int box_rows) {
    const cuuint64_t dims[2] = {(cuuint64_t)d, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)ld * 2};
    const cuuint32_t box[2] = {(cuuint32_t)kBK, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1, 1};
    return fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

namespace {
struct LmWs { size_t status, part, n_rows, tile_state, row_idx, targets_c, hidden_c, total; };
inline size_t lm_a256(size_t x) { return (x + 255) & ~(size_t)255; }
LmWs lm_ws_layout(int64_t T, int32_t d) {
    LmWs w;
    size_t o = 0;
    w.status = o; o += 256;                                  // status word first (ajt_last_status)
    w.part = o; o += lm_a256((size_t)T * kVS * sizeof(float4));
    w.n_rows = o; o += 256;                                  // {n_rows, ticket}
    w.tile_state = o; o += lm_a256((size_t)((T + kCompactTile - 1) / kCompactTile + 1) * 8);
    w.row_idx = o; o += lm_a256((size_t)T * 4);
    w.targets_c = o; o += lm_a256((size_t)T * 4);
    w.hidden_c = o; o += lm_a256((size_t)T * d * 2);
    w.total = o;
    return w;
}
}  // namespace

extern "C" size_t ajt_lm_head_workspace_bytes(int64_t T, int32_t d, int32_t V) {
    if (T < 0 || d <= 0 || V <= 0) return 0;
    return lm_ws_layout(T, d).total;
}

extern "C" int ajt_lm_head_logp(const void* hidden, const void* weight, const int32_t* targets, const uint8_t* mask, int64_t T,
                                int32_t d, int32_t V, int64_t ld_hidden, int64_t ld_weight, float* logp_out, float* ent_out,
                                float* lse_out, uint32_t flags, void* workspace, size_t workspace_bytes, ajt_stream_t stream_) {
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    if (T < 0 || d <= 0 || V <= 0 || ld_hidden < d || ld_weight < d) return AJT_ERR_INVALID_ARG;
    if (!logp_out || !workspace) return AJT_ERR_INVALID_ARG;
    if (T > 0 && (!hidden || !weight || !targets)) return AJT_ERR_INVALID_ARG;
    if (d % kBK != 0 || (ld_hidden % 8) != 0 || (ld_weight % 8) != 0 || (((uintptr_t)hidden | (uintptr_t)weight) & 15) ||
        T >= ((int64_t)1 << 31))
        return AJT_ERR_UNSUPPORTED;   // K slabs of 64, 16-byte aligned rows (TMA)
    if (((uintptr_t)workspace & 255) || workspace_bytes < ajt_lm_head_workspace_bytes(T, d, V)) return AJT_ERR_WORKSPACE_TOO_SMALL;
    if (T == 0) return AJT_OK;
    const LmWs ws = lm_ws_layout(T, d);
    uint8_t* wsb = reinterpret_cast<uint8_t*>(workspace);

    int dev = 0, num_sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return AJT_ERR_CUDA;
    if (cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || num_sms < kVS) return AJT_ERR_CUDA;
    static EncodeTiledFn encode = nullptr;
    if (!encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) return AJT_ERR_CUDA;
        encode = reinterpret_cast<EncodeTiledFn>(fn);
    }
    const int ncta = T > kBM ? 2 : 1;   // CTA pairs (256-row blocks) unless a single 128-row block holds everything
    LmParams p;
    p.targets = targets; p.mask = mask; p.T = T; p.d = d; p.V = V;
    p.n_rows = nullptr; p.row_idx = nullptr;
    p.status = reinterpret_cast<uint32_t*>(wsb + ws.status);
    if (cudaMemsetAsync(p.status, 0, 256, stream) != cudaSuccess) return AJT_ERR_CUDA;
    p.round_bf16 = (flags & AJT_LM_ROUND_LOGITS_BF16) ? 1 : 0;
    const void* h_src = hidden;
    int64_t h_ld = ld_hidden;
    if (mask) {
        int32_t* n_rows = reinterpret_cast<int32_t*>(wsb + ws.n_rows);
        int32_t* row_idx = reinterpret_cast<int32_t*>(wsb + ws.row_idx);
        int32_t* targets_c = reinterpret_cast<int32_t*>(wsb + ws.targets_c);
        if (cudaMemsetAsync(wsb + ws.n_rows, 0, ws.row_idx - ws.n_rows, stream) != cudaSuccess) return AJT_ERR_CUDA;   // count, ticket, tile states
        if (cudaMemsetAsync(logp_out, 0, (size_t)T * 4, stream) != cudaSuccess) return AJT_ERR_CUDA;
        if (ent_out && cudaMemsetAsync(ent_out, 0, (size_t)T * 4, stream) != cudaSuccess) return AJT_ERR_CUDA;
        if (lse_out && cudaMemsetAsync(lse_out, 0, (size_t)T * 4, stream) != cudaSuccess) return AJT_ERR_CUDA;
        const int ntiles = (int)((T + kCompactTile - 1) / kCompactTile);
        AJT_LAUNCH(lm_compact_kernel<<<ntiles < num_sms ? ntiles : num_sms, 256, 0, stream>>>(mask, T, reinterpret_cast<uint64_t*>(wsb + ws.tile_state),
                                                                                 n_rows + 1, row_idx, n_rows));
        AJT_LAUNCH(lm_gather_kernel<<<num_sms * 8, 256, 0, stream>>>(reinterpret_cast<const uint4*>(hidden), ld_hidden / 8, d / 8, targets, row_idx, n_rows,
                                                         reinterpret_cast<uint4*>(wsb + ws.hidden_c), targets_c));
        p.targets = targets_c; p.n_rows = n_rows; p.row_idx = row_idx;
        h_src = wsb + ws.hidden_c;
        h_ld = d;
    }
    CUtensorMap map_h, map_w;
    if (!make_map(encode, &map_h, h_src, T, d, h_ld, kBM) || !make_map(encode, &map_w, weight, V, d, ld_weight, kBN / ncta))
        return AJT_ERR_CUDA;

    const int64_t n_mtiles = (T + kBM * ncta - 1) / (kBM * ncta);   // row blocks of 128 * ncta rows (upper bound when rows are compacted)
    p.nvs = 0;                                  // the kernel fits the vocabulary ranges to the rows there really are
    p.vs_len = 0;
    int groups = num_sms / ncta;                // one work group per SM (pair of SMs)
    if ((int64_t)groups > n_mtiles * kVS) groups = (int)(n_mtiles * kVS);
    p.part = reinterpret_cast<float4*>(wsb + ws.part);
    p.logp_out = logp_out; p.ent_out = ent_out; p.lse_out = lse_out;

    if (ncta == 1) {
        if (cudaFuncSetAttribute(lm_head_kernel<1, kReduce>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)LmCfg<1>::kSmem) != cudaSuccess)
            return AJT_ERR_CUDA;
        AJT_LAUNCH(lm_head_kernel<1, kReduce><<<groups, kLmThreads, LmCfg<1>::kSmem, stream>>>(map_h, map_w, p));
    } else {
        if (cudaFuncSetAttribute(lm_head_kernel<2, kReduce>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)LmCfg<2>::kSmem) != cudaSuccess)
            return AJT_ERR_CUDA;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)(groups * 2));
        cfg.blockDim = dim3(kLmThreads);
        cfg.dynamicSmemBytes = LmCfg<2>::kSmem;
        cfg.stream = stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 2;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        ajt::note_launch();
        if (cudaLaunchKernelEx(&cfg, lm_head_kernel<2, kReduce>, map_h, map_w, p) != cudaSuccess) return AJT_ERR_CUDA;
    }
    const int64_t want = (T + 255) / 256;
    AJT_LAUNCH(lm_head_combine_kernel<<<(int)(want < (int64_t)num_sms * 4 ? want : (int64_t)num_sms * 4), 256, 0, stream>>>(p, groups, ncta));
    return cudaGetLastError() == cudaSuccess ? AJT_OK : AJT_ERR_CUDA;
}

// ================================================================================================ backward
//
// ajt_lm_head_loss_bwd: loss, dH and dW straight from the hidden states.  The [T, V] logits are recomputed
// tile by tile on the tensor cores and turned into dZ = g (1[v = y] - exp(z - lse)) in the epilogue; the two follow-on
// contractions dH = dZ W and dW = dZ^T H run through the SAME TMA / tcgen05 mainloop with a store / accumulate epilogue.
// dZ cannot stay on chip between them: its consumers' accumulators (rows x d fp32 for dH, V x d fp32 for dW) are 30-1000x the
// tensor memory of the whole GPU, so dZ is staged in bf16, a CHUNK of rows at a time (row-major for dH, transposed for dW),
// in the workspace.  Per chunk of R compacted rows: [R, V] bf16 is written twice and read once each: 4 R V bytes of traffic
// against 6 R V d flops (d = 4096: 0.016 % of the time at the roofs).  Masked rows cost nothing (they are compacted away).
namespace {

constexpr int kBwdChunk = 4096;   // rows of dZ staged at a time (multiple of 256); 9,472 (8 full rounds of dH tiles) measured 5 % slower

// d loss / d logp of every compacted row k (original row t = row_idx[k], or k), the row's lse, and the loss: steps 2-6 of O-L
// on the forward pass's log-probs (ajt_token.cuh).  Block partials in fp64, summed in block order by the last kernel.
__global__ void __launch_bounds__(256) lm_token_grad_kernel(const float* __restrict__ logp, const float* __restrict__ lse,
                                                            const float* __restrict__ old_logp, const float* __restrict__ adv,
                                                            const int32_t* __restrict__ seg_ids, const float* __restrict__ seg_denom,
                                                            const int32_t* __restrict__ row_idx, const int32_t* __restrict__ n_rows,
                                                            int64_t T, int32_t S, float inv_num_segs, float eps_lo, float eps_hi,
                                                            float grad_scale, float* __restrict__ g_row, float* __restrict__ lse_row,
                                                            double* __restrict__ partials, uint32_t* status) {
    __shared__ double s_red[8];
    __shared__ float s_inv;
    if (threadIdx.x == 0) s_inv = inv_num_segs;
    if (inv_num_segs == 0.f) {   // 1 / S' from the normalisers (reading L-3): every block counts the live trajectories itself
        int live = 0;
        for (int x = threadIdx.x; x < S; x += 256) live += seg_denom[x] > 0.f ? 1 : 0;
        live = __reduce_add_sync(0xffffffffu, live);
        __shared__ int s_live[8];
        if ((threadIdx.x & 31) == 0) s_live[threadIdx.x >> 5] = live;
        __syncthreads();
        if (threadIdx.x == 0) {
            int tot = 0;
            for (int w = 0; w < 8; ++w) tot += s_live[w];
            s_inv = tot > 0 ? 1.f / (float)tot : 0.f;
        }
    }
    __syncthreads();
    const int64_t Teff = n_rows ? (int64_t)*n_rows : T;
    const int64_t k = (int64_t)blockIdx.x * 256 + threadIdx.x;
    double wl = 0.0;
    if (k < T) {
        float g = 0.f, ls = 0.f;
        if (k < Teff) {
            const int64_t t = row_idx ? (int64_t)row_idx[k] : k;
            const int sg = seg_ids[t];
            if (sg < 0 || sg >= S) {
                atomicOr(status, (uint32_t)AJT_STATUS_BAD_SEG);
            } else {
                const float Ns = seg_denom[sg];
                const float w = Ns > 0.f ? s_inv / Ns : 0.f;
                const TokScalars ts = token_scalars(0.f, 1.f, logp[t], old_logp[t], adv[t], w, eps_lo, eps_hi, grad_scale);
                g = ts.g;
                wl = ts.wl;
                ls = lse[t];
            }
        }
        g_row[k] = g;
        lse_row[k] = ls;
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) wl += __shfl_xor_sync(0xffffffffu, wl, o);
    if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = wl;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int w = 0; w < 8; ++w) tot += s_red[w];
        partials[blockIdx.x] = tot;
    }
}
__global__ void lm_loss_sum_kernel(const double* partials, int n, float* loss_out) {
    double tot = 0.0;
    for (int i = 0; i < n; ++i) tot += partials[i];
    *loss_out = (float)tot;
}

// out[c, r] = in[r, c] for r < rows, c < cols (zeros elsewhere up to out_rows x ld_out): 64 x 64 tiles through shared memory.
// `n_rows` (DEVICE, or NULL): rows that exist in `in` counted from row0; rows beyond are written as zeros.
__global__ void __launch_bounds__(256) lm_transpose_kernel(const __nv_bfloat16* __restrict__ in, int64_t ld_in, int64_t rows, int64_t cols,
                                                           __nv_bfloat16* __restrict__ out, int64_t ld_out, int64_t out_rows, int64_t out_cols,
                                                           const int32_t* __restrict__ n_rows, int64_t row0) {
    __shared__ __nv_bfloat16 tile[64][66];
    if (n_rows) rows = min(rows, max((int64_t)0, (int64_t)*n_rows - row0));
    const int64_t r0 = (int64_t)blockIdx.y * 64, c0 = (int64_t)blockIdx.x * 64;   // tile of `in`: rows r0.., cols c0..
    for (int x = threadIdx.x; x < 64 * 64; x += 256) {
        const int rr = x >> 6, cc = x & 63;
        const int64_t r = r0 + rr, c = c0 + cc;
        tile[rr][cc] = (r < rows && c < cols) ? in[r * ld_in + c] : __float2bfloat16(0.f);
    }
    __syncthreads();
    for (int x = threadIdx.x; x < 64 * 64; x += 256) {
        const int cc = x >> 6, rr = x & 63;
        const int64_t r = r0 + rr, c = c0 + cc;
        if (c < out_rows && r < out_cols) out[c * ld_out + r] = tile[rr][cc];
    }
}

struct LmBwdWs { size_t fwd, logp, lse, g_row, lse_row, ns, partials, ones, wt, dz, dzt, hct, total; };
LmBwdWs lm_bwd_ws_layout(int64_t T, int32_t d, int32_t V, int32_t S) {
    LmBwdWs w;
    size_t o = 0;
    const size_t Vp = ((size_t)V + 255) / 256 * 256, R = kBwdChunk;
    w.fwd = o; o += lm_a256(lm_ws_layout(T, d).total);
    w.logp = o; o += lm_a256((size_t)T * 4);
    w.lse = o; o += lm_a256((size_t)T * 4);
    w.g_row = o; o += lm_a256((size_t)T * 4);
    w.lse_row = o; o += lm_a256((size_t)T * 4);
    w.ns = o; o += lm_a256((size_t)S * 4);
    w.partials = o; o += lm_a256(((size_t)T / 256 + 2) * 8);
    w.ones = o; o += lm_a256((size_t)T);
    w.wt = o; o += lm_a256((size_t)d * Vp * 2);
    w.dz = o; o += lm_a256(R * Vp * 2);
    w.dzt = o; o += lm_a256(Vp * R * 2);
    w.hct = o; o += lm_a256((size_t)d * R * 2);
    w.total = o;
    return w;
}

// one launch of the tile kernel: C[M, N] (epilogue MODE) from A [M, K] and B [N, K], both K-major bf16
template <int MODE>
int lm_launch(EncodeTiledFn encode, int num_sms, const void* A, int64_t M, int64_t lda, const void* Bm, int64_t N, int64_t ldb, int64_t K,
              LmParams p, bool ranges, cudaStream_t stream) {
    constexpr int ncta = 2;
    CUtensorMap map_a, map_b;
    if (!make_map(encode, &map_a, A, M, (int32_t)K, lda, kBM) || !make_map(encode, &map_b, Bm, N, (int32_t)K, ldb, kBN / ncta)) return AJT_ERR_CUDA;
    p.T = M; p.d = (int32_t)K; p.V = (int32_t)N;
    if (ranges) {   // the forward's decomposition: vocabulary ranges walked tile by tile
        p.nvs = 0;   // fitted on the device
        p.vs_len = 0;
    } else {        // one output tile per work item
        p.nvs = (int32_t)((N + kBN - 1) / kBN);
        p.vs_len = kBN;
    }
    const int64_t n_mtiles = (M + kBM * ncta - 1) / (kBM * ncta);
    int groups = num_sms / ncta;
    if ((int64_t)groups > n_mtiles * (p.nvs ? p.nvs : kVS)) groups = (int)(n_mtiles * (p.nvs ? p.nvs : kVS));
    if (cudaFuncSetAttribute(lm_head_kernel<ncta, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)LmCfg<ncta>::kSmem) != cudaSuccess)
        return AJT_ERR_CUDA;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(groups * 2));
    cfg.blockDim = dim3(kLmThreads);
    cfg.dynamicSmemBytes = LmCfg<ncta>::kSmem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    ajt::note_launch();
    return cudaLaunchKernelEx(&cfg, lm_head_kernel<ncta, MODE>, map_a, map_b, p) == cudaSuccess ? AJT_OK : AJT_ERR_CUDA;
}

}  // namespace

extern "C" size_t ajt_lm_head_bwd_workspace_bytes(int64_t T, int32_t d, int32_t V, int32_t S) {
    if (T < 0 || d <= 0 || V <= 0 || S <= 0) return 0;
    return lm_bwd_ws_layout(T, d, V, S).total;
}

extern "C" int ajt_lm_head_loss_bwd(const void* hidden, const void* weight, const int32_t* targets, const float* old_logp,
                                    const float* adv, const uint8_t* mask, const int32_t* seg_ids, float eps_lo, float eps_hi,
                                    int64_t T, int32_t d, int32_t V, int32_t S, int64_t ld_hidden, int64_t ld_weight,
                                    const float* seg_denom, float inv_num_segs, float grad_scale, void* dH, int64_t ld_dh,
                                    float* dW, int64_t ld_dw, int32_t accumulate_dw, float* loss_out, float* logp_out,
                                    uint32_t flags, void* workspace, size_t workspace_bytes, ajt_stream_t stream_) {
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    if (T < 0 || d <= 0 || V <= 0 || S <= 0 || !workspace || !loss_out) return AJT_ERR_INVALID_ARG;
    if (T > 0 && (!hidden || !weight || !targets || !old_logp || !adv || !seg_ids || !dH || !dW)) return AJT_ERR_INVALID_ARG;
    if (!(eps_lo >= 0.f) || !(eps_hi >= 0.f) || inv_num_segs < 0.f) return AJT_ERR_INVALID_ARG;
    if ((d % 64) || (ld_hidden % 8) || (ld_weight % 8) || (ld_dh % 8) || (ld_dw % 4) || ld_dh < d || ld_dw < d) return AJT_ERR_UNSUPPORTED;
    if (((uintptr_t)hidden | (uintptr_t)weight | (uintptr_t)dH | (uintptr_t)dW) & 15) return AJT_ERR_UNSUPPORTED;
    if ((uintptr_t)workspace & 255) return AJT_ERR_INVALID_ARG;
    if (T >= ((int64_t)1 << 31)) return AJT_ERR_INVALID_ARG;
    const LmBwdWs ws = lm_bwd_ws_layout(T, d, V, S);
    if (workspace_bytes < ws.total) return AJT_ERR_WORKSPACE_TOO_SMALL;
    uint8_t* b = reinterpret_cast<uint8_t*>(workspace);
    int dev = 0, num_sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return AJT_ERR_CUDA;
    if (cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || num_sms < kVS) return AJT_ERR_CUDA;
    static EncodeTiledFn encode = nullptr;
    if (!encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) return AJT_ERR_CUDA;
        encode = reinterpret_cast<EncodeTiledFn>(fn);
    }
    if (T == 0) {
        if (cudaMemsetAsync(loss_out, 0, 4, stream) != cudaSuccess) return AJT_ERR_CUDA;
        if (!accumulate_dw && cudaMemsetAsync(dW, 0, (size_t)V * ld_dw * 4, stream) != cudaSuccess) return AJT_ERR_CUDA;
        return AJT_OK;
    }
    float* logp = reinterpret_cast<float*>(b + ws.logp);
    float* lse = reinterpret_cast<float*>(b + ws.lse);
    float* g_row = reinterpret_cast<float*>(b + ws.g_row);
    float* lse_row = reinterpret_cast<float*>(b + ws.lse_row);
    float* ns = reinterpret_cast<float*>(b + ws.ns);
    double* partials = reinterpret_cast<double*>(b + ws.partials);
    __nv_bfloat16* wt = reinterpret_cast<__nv_bfloat16*>(b + ws.wt);
    __nv_bfloat16* dz = reinterpret_cast<__nv_bfloat16*>(b + ws.dz);
    __nv_bfloat16* dzt = reinterpret_cast<__nv_bfloat16*>(b + ws.dzt);
    __nv_bfloat16* hct = reinterpret_cast<__nv_bfloat16*>(b + ws.hct);
    uint32_t* status = reinterpret_cast<uint32_t*>(b + ws.fwd);   // the forward's status word is the call's
    const int64_t Vp = ((int64_t)V + 255) / 256 * 256, R = kBwdChunk;

    // ---- forward half: log-probs and log-sum-exp of every unmasked row (compacts the unmasked rows into the workspace)
    int rc = ajt_lm_head_logp(hidden, weight, targets, mask, T, d, V, ld_hidden, ld_weight, logp, nullptr, lse, flags, b + ws.fwd,
                              lm_a256(lm_ws_layout(T, d).total), stream_);
    if (rc != AJT_OK) return rc;
    if (logp_out && cudaMemcpyAsync(logp_out, logp, (size_t)T * 4, cudaMemcpyDeviceToDevice, stream) != cudaSuccess) return AJT_ERR_CUDA;
    const LmWs fw = lm_ws_layout(T, d);
    const int32_t* n_rows = mask ? reinterpret_cast<const int32_t*>(b + ws.fwd + fw.n_rows) : nullptr;
    const int32_t* row_idx = mask ? reinterpret_cast<const int32_t*>(b + ws.fwd + fw.row_idx) : nullptr;
    const int32_t* targets_c = mask ? reinterpret_cast<const int32_t*>(b + ws.fwd + fw.targets_c) : targets;
    const __nv_bfloat16* hc = mask ? reinterpret_cast<const __nv_bfloat16*>(b + ws.fwd + fw.hidden_c) : reinterpret_cast<const __nv_bfloat16*>(hidden);
    const int64_t ld_hc = mask ? d : ld_hidden;
    // ---- per-trajectory normalisers, then d loss / d logp per compacted row and the loss
    if (!seg_denom) {
        const uint8_t* mk = mask;
        if (!mk) {
            if (cudaMemsetAsync(b + ws.ones, 1, (size_t)T, stream) != cudaSuccess) return AJT_ERR_CUDA;
            mk = b + ws.ones;
        }
        rc = ajt_segment_counts(mk, seg_ids, T, S, 0, ns, nullptr, stream_);
        if (rc != AJT_OK) return rc;
        seg_denom = ns;
    }
    const int nblk = (int)((T + 255) / 256);
    AJT_LAUNCH(lm_token_grad_kernel<<<nblk, 256, 0, stream>>>(logp, lse, old_logp, adv, seg_ids, seg_denom, row_idx, n_rows, T, S, inv_num_segs,
                                                   eps_lo, eps_hi, grad_scale, g_row, lse_row, partials, status));
    AJT_LAUNCH(lm_loss_sum_kernel<<<1, 1, 0, stream>>>(partials, nblk, loss_out));
    // ---- outputs start from zero (masked rows of dH stay zero); W^T once
    if (cudaMemsetAsync(dH, 0, (size_t)T * ld_dh * 2, stream) != cudaSuccess) return AJT_ERR_CUDA;
    if (!accumulate_dw && cudaMemsetAsync(dW, 0, (size_t)V * ld_dw * 4, stream) != cudaSuccess) return AJT_ERR_CUDA;
    AJT_LAUNCH(lm_transpose_kernel<<<dim3((unsigned)((d + 63) / 64), (unsigned)((Vp + 63) / 64)), 256, 0, stream>>>(
        reinterpret_cast<const __nv_bfloat16*>(weight), ld_weight, V, d, wt, Vp, d, Vp, nullptr, 0));
    // the staging buffers never hold anything but finite numbers (a chunk may leave parts of them untouched)
    if (cudaMemsetAsync(dz, 0, (size_t)R * Vp * 2, stream) != cudaSuccess || cudaMemsetAsync(dzt, 0, (size_t)Vp * R * 2, stream) != cudaSuccess)
        return AJT_ERR_CUDA;
    LmParams p = {};
    p.targets = targets_c; p.n_rows = n_rows; p.row_idx = row_idx; p.round_bf16 = (flags & AJT_LM_ROUND_LOGITS_BF16) ? 1 : 0;
    p.status = status; p.g_row = g_row; p.lse_row = lse_row; p.dz = dz; p.dzt = dzt; p.ld_dz = Vp; p.ld_dzt = R;
    p.out_bf16 = reinterpret_cast<__nv_bfloat16*>(dH); p.out_f32 = dW; p.n_out_rows = V;
    for (int64_t c0 = 0; c0 < T; c0 += R) {   // chunks beyond the number of unmasked rows (known on the device only) exit at once
        const int64_t rows = T - c0 < R ? T - c0 : R;
        p.row0 = c0;
        // dZ of the chunk (row-major and transposed) from recomputed logits tiles
        rc = lm_launch<kDz>(encode, num_sms, hc + c0 * ld_hc, rows, ld_hc, weight, V, ld_weight, d, p, true, stream);
        if (rc != AJT_OK) return rc;
        // H_chunk^T (rows beyond the unmasked count: zeros)
        AJT_LAUNCH(lm_transpose_kernel<<<dim3((unsigned)((d + 63) / 64), (unsigned)(R / 64)), 256, 0, stream>>>(hc + c0 * ld_hc, ld_hc, rows, d, hct, R, d, R,
                                                                                              n_rows, c0));
        // dH_chunk = dZ_chunk W  (rows scattered to their original positions)
        p.ld_out = ld_dh;
        rc = lm_launch<kStoreBf16>(encode, num_sms, dz, rows, Vp, wt, d, Vp, Vp, p, false, stream);
        if (rc != AJT_OK) return rc;
        // dW += dZ_chunk^T H_chunk
        p.ld_out = ld_dw;
        rc = lm_launch<kAccF32>(encode, num_sms, dzt, Vp, R, hct, d, R, R, p, false, stream);
        if (rc != AJT_OK) return rc;
    }
    return cudaGetLastError() == cudaSuccess ? AJT_OK : AJT_ERR_CUDA;
}
