// Text-level (block-level) timeline merging: Algorithm 1 on timelines of message blocks.
//
// Match = text compares the blocks' texts, represented by caller-supplied 64-bit ids (reading B-1), so the prefix relation
// between timelines is the token-level one on the id streams: the ids are handed to the token-level pipeline of
// ajt_merge.cu as pairs of 32-bit "tokens" (all lengths even, so prefixes end on pair boundaries), with mask = (author is
// llm) and Algorithm 1's own owner rule.  Its outputs already say, per block position k of a survivor, whether any member
// has an llm block there and which is the latest such member (Alg. 1 lines 6-17: j runs downwards and only fills blocks
// that are not llm yet).  What is left is to MATERIALISE the survivors: block k of survivor s takes tokens, log-probs and
// mask from block k of that member (lines 12-14), else from s itself.
//
//   blocks_prep_kernel     offsets in id-words, mask per id-word                                     tiny
//   (7 launches of the token-level merge on 8 B per block)
//   blocks_info_kernel     per merged block: supplying timeline, source block, length, author        tiny (per block)
//   blocks_scan_kernel     single-pass exclusive scan of the block lengths -> token offsets          tiny
//   blocks_offsets_kernel  merged_offsets / merged_block_offsets / counts                            tiny
//   blocks_copy_kernel     gathers tokens / log-probs / mask of every merged block                   HBM: 4-9 B read, 9-13 B written per token
#include "ajt_common.cuh"

namespace {

constexpr int kAuthorLlm = AJT_AUTHOR_LLM;
constexpr int kScanTile = 2048;   // blocks per scan tile (256 threads x 8)

struct BlockParams {
    const int64_t* block_ids;
    const int64_t* block_offsets;
    const int32_t* traj_ids;
    const uint8_t* author;
    const int64_t* tok_off;
    const int32_t* tokens;
    const float* logp;
    const uint8_t* tok_mask;
    int32_t n;
    int64_t B, N;
    int32_t* merged_tokens;
    uint8_t* merged_mask;
    float* merged_logp;
    int32_t* merged_tok_src;
    int64_t* merged_offsets;
    int64_t* merged_block_offsets;
    int32_t* merged_block_src;
    uint8_t* merged_block_author;
    int64_t* merged_block_tok_off;
    int32_t* merged_origin;
    int64_t* counts;
    // workspace
    AjtCtrl* ctrl;            // the token-level merge's control block (status word first)
    int64_t* offsets2;        // [n+1] timeline offsets in id-words
    uint8_t* mask2;           // [2B]
    int32_t* ids_out;         // [2B] merged id-words (not returned)
    uint8_t* mask2_out;       // [2B]
    int32_t* src2_out;        // [2B]
    int64_t* offs2_out;       // [n+1]
    int64_t* counts2;         // [2] {M, 2 B_out}
    int64_t* blk_srcblk;      // [B] source block of merged block b
    uint64_t* tile_state;     // [ntiles] scan: bit 63 valid, low bits the tile's sum
    int32_t* tile_counter;    // [1]
};

struct BlockWs {
    size_t inner, offsets2, mask2, ids_out, mask2_out, src2_out, offs2_out, counts2, blk_srcblk, tile_state, tile_counter, total;
};

__host__ inline size_t a256(size_t x) { return (x + 255) & ~(size_t)255; }

// The id-level merge's workspace comes first (its status word is the call's status word) and takes whatever the caller
// provides beyond the minimum: more room for candidate pairs (AJT_STATUS_PROBE_CAPACITY), as for ajt_merge_timelines.
__host__ BlockWs block_ws_layout(int32_t n, int64_t B, size_t inner_bytes = 0) {
    BlockWs w;
    size_t o = 0;
    const size_t inner_min = a256(ajt_merge_workspace_bytes(n, 2 * B));
    w.inner = o; o += inner_bytes > inner_min ? (inner_bytes & ~(size_t)255) : inner_min;
    w.offsets2 = o; o += a256(((size_t)n + 1) * 8);
    w.mask2 = o; o += a256((size_t)2 * B + 16);
    w.ids_out = o; o += a256((size_t)2 * B * 4 + 16);
    w.mask2_out = o; o += a256((size_t)2 * B + 16);
    w.src2_out = o; o += a256((size_t)2 * B * 4 + 16);
    w.offs2_out = o; o += a256(((size_t)n + 1) * 8);
    w.counts2 = o; o += 256;
    w.blk_srcblk = o; o += a256((size_t)B * 8 + 8);
    w.tile_state = o; o += a256((size_t)((B + kScanTile - 1) / kScanTile + 1) * 8);
    w.tile_counter = o; o += 256;
    w.total = o;
    return w;
}

__global__ void __launch_bounds__(256) blocks_prep_kernel(const BlockParams p, int ntiles) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x, t0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (int64_t i = t0; i <= p.n; i += stride) p.offsets2[i] = 2 * p.block_offsets[i];
    uint16_t* m2 = reinterpret_cast<uint16_t*>(p.mask2);
    for (int64_t b = t0; b < p.B; b += stride) m2[b] = p.author[b] == kAuthorLlm ? (uint16_t)0x0101 : (uint16_t)0;
    for (int64_t t = t0; t < ntiles; t += stride) p.tile_state[t] = 0;
    if (t0 == 0) *p.tile_counter = 0;
}

__device__ __forceinline__ bool fatal(const BlockParams& p) {
    return (p.ctrl->status & (AJT_STATUS_BAD_OFFSETS | AJT_STATUS_ZERO_LEN | AJT_STATUS_PROBE_CAPACITY)) != 0;
}
// {M, B_out} of the id-level merge; nothing when it stopped on a fatal status (its counts are then unspecified)
__device__ __forceinline__ void merged_counts(const BlockParams& p, int64_t& M, int64_t& Bout) {
    const bool bad = fatal(p);
    M = bad ? 0 : p.counts2[0];
    Bout = bad ? 0 : (p.counts2[1] >> 1);
}

// last index i in [0, n) with a[i] <= x (a non-decreasing, a[0] <= x)
__device__ __forceinline__ int64_t search_last_le(const int64_t* __restrict__ a, int64_t n, int64_t x) {
    int64_t lo = 0, hi = n - 1;
    while (lo < hi) {
        const int64_t mid = (lo + hi + 1) >> 1;
        if (__ldg(a + mid) <= x) lo = mid;
        else hi = mid - 1;
    }
    return lo;
}

// Per merged block b = (survivor m, position k): the timeline that supplies it (Alg. 1 lines 11-14), its source block, its
// author after merging, and its length (left in merged_block_tok_off[b] for the scan).
__global__ void __launch_bounds__(256) blocks_info_kernel(const BlockParams p) {
    int64_t M, Bout;
    merged_counts(p, M, Bout);
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; b < Bout; b += stride) {
        const int64_t m = search_last_le(p.offs2_out, M, 2 * b);
        const int64_t k = b - (p.offs2_out[m] >> 1);
        const int32_t s = p.merged_origin[m];
        const int32_t sj2 = p.src2_out[2 * b];               // latest member with an llm block here, or -1
        const int32_t sj = sj2 >= 0 ? sj2 : s;
        const int64_t sb = p.block_offsets[sj] + k;
        const int64_t len = p.tok_off[sb + 1] - p.tok_off[sb];
        if (len < 0 || len > (int64_t)INT32_MAX) {
            atomicOr(&p.ctrl->status, (uint32_t)AJT_STATUS_BAD_OFFSETS);
        }
        p.blk_srcblk[b] = sb;
        p.merged_block_src[b] = sj;
        p.merged_block_author[b] = sj2 >= 0 ? (uint8_t)kAuthorLlm : p.author[p.block_offsets[s] + k];
        p.merged_block_tok_off[b] = len < 0 ? 0 : len;
    }
}

// Exclusive scan of merged_block_tok_off[0 .. B_out) in place, one pass: tiles are handed out by an atomic ticket (every
// predecessor of a tile has started), a tile publishes its sum, then adds up the sums of all its predecessors.
__global__ void __launch_bounds__(256) blocks_scan_kernel(const BlockParams p) {
    __shared__ int64_t s_w[8];
    __shared__ int64_t s_base;
    __shared__ int s_tile;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    int64_t M, Bout;
    merged_counts(p, M, Bout);
    const int ntiles = (int)((Bout + kScanTile - 1) / kScanTile);
    for (;;) {
        if (tid == 0) s_tile = atomicAdd(p.tile_counter, 1);
        __syncthreads();
        const int tile = s_tile;
        if (tile >= ntiles) break;
        const int64_t b0 = (int64_t)tile * kScanTile + tid * 8;
        int64_t v[8], sum = 0;
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            v[e] = b0 + e < Bout ? p.merged_block_tok_off[b0 + e] : 0;
            sum += v[e];
        }
        int64_t inc = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int64_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) s_w[warp] = inc;
        __syncthreads();
        int64_t wbase = 0, total = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) {
            if (w < warp) wbase += s_w[w];
            total += s_w[w];
        }
        if (tid == 0) {
            __threadfence();
            atomicExch(reinterpret_cast<unsigned long long*>(&p.tile_state[tile]), (1ull << 63) | (unsigned long long)total);
        }
        // sum of the predecessors' totals (spin until each is published)
        int64_t pre = 0;
        for (int t = tid; t < tile; t += 256) {
            unsigned long long st;
            do {
                st = *reinterpret_cast<volatile unsigned long long*>(&p.tile_state[t]);
            } while (!(st >> 63));
            pre += (int64_t)(st & ~(1ull << 63));
        }
#pragma unroll
        for (int o = 16; o; o >>= 1) pre += __shfl_xor_sync(0xffffffffu, pre, o);
        __syncthreads();   // s_w reads above are done
        if (lane == 0) s_w[warp] = pre;
        __syncthreads();
        if (tid == 0) {
            int64_t b = 0;
            for (int w = 0; w < 8; ++w) b += s_w[w];
            s_base = b;
        }
        __syncthreads();
        int64_t run = s_base + wbase + inc - sum;
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            if (b0 + e < Bout) p.merged_block_tok_off[b0 + e] = run;
            run += v[e];
        }
        if (tile == ntiles - 1 && tid == 255) {
            p.merged_block_tok_off[Bout] = s_base + total;
        }
        __syncthreads();
    }
    if (ntiles == 0 && blockIdx.x == 0 && tid == 0) p.merged_block_tok_off[0] = 0;
}

__global__ void __launch_bounds__(256) blocks_offsets_kernel(const BlockParams p) {
    int64_t M, Bout;
    merged_counts(p, M, Bout);
    if (fatal(p)) {   // the id-level merge stopped: its outputs are unspecified and must not be used as indices
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            p.merged_offsets[0] = 0;
            p.merged_block_offsets[0] = 0;
            p.counts[0] = p.counts[1] = p.counts[2] = 0;
        }
        return;
    }
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t m = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; m <= M; m += stride) {
        const int64_t bo = p.offs2_out[m] >> 1;
        p.merged_block_offsets[m] = bo;
        p.merged_offsets[m] = p.merged_block_tok_off[bo];
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        p.counts[0] = M;
        p.counts[1] = Bout;
        p.counts[2] = p.merged_block_tok_off[Bout];
    }
}

// Gather: a warp takes a tile of 512 consecutive output tokens (4 steps of 32 lanes x 4 tokens, 16-byte stores where the
// output arrays allow it).  The block that holds the tile's first token is found once per tile (a binary search whose loads
// are warp-uniform); from there every lane walks forward over the block boundaries it meets (blocks are tens to thousands
// of tokens long).  All of a step's loads are issued before its stores.
constexpr int kCopyTile = 512;

struct BlkCursor {   // the block a lane is in: where it ends, where its tokens come from, who supplied it
    int64_t b, bend, delta;
    int32_t sj;
    bool llm;
};
__device__ __forceinline__ void cursor_load(const BlockParams& p, BlkCursor& c) {
    c.bend = __ldg(p.merged_block_tok_off + c.b + 1);
    c.delta = __ldg(p.tok_off + __ldg(p.blk_srcblk + c.b)) - __ldg(p.merged_block_tok_off + c.b);   // source = output + delta
    c.sj = p.merged_block_src[c.b];
    c.llm = p.merged_block_author[c.b] == kAuthorLlm;
}

__global__ void __launch_bounds__(256) blocks_copy_kernel(const BlockParams p) {
    int64_t M, Bout;
    merged_counts(p, M, Bout);
    if (Bout == 0) return;
    const int64_t Nout = p.merged_block_tok_off[Bout];
    const bool vec_ok = ((((uintptr_t)p.merged_tokens | (uintptr_t)p.merged_tok_src | (uintptr_t)p.merged_logp) & 15) == 0) &&
                        (((uintptr_t)p.merged_mask & 3) == 0);
    const int lane = threadIdx.x & 31;
    const int64_t wglobal = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    const int64_t ntiles = (Nout + kCopyTile - 1) / kCopyTile;
    for (int64_t tile = wglobal; tile < ntiles; tile += nwarps) {
        const int64_t t0 = tile * kCopyTile;
        BlkCursor c;
        c.b = search_last_le(p.merged_block_tok_off, Bout, t0);
        cursor_load(p, c);
#pragma unroll 2
        for (int u = 0; u < kCopyTile / 128; ++u) {
            const int64_t q0 = t0 + 128 * u + 4 * lane;
            if (q0 >= Nout) break;
            int32_t x[4], sr[4];
            float lp[4];
            uint32_t mk = 0;
            if (q0 + 3 < c.bend) {   // the four tokens lie in the lane's current block (the usual case)
                const int64_t sq = q0 + c.delta;
#pragma unroll
                for (int e = 0; e < 4; ++e) x[e] = __ldg(p.tokens + sq + e);
                uint32_t m4 = c.llm ? 0x01010101u : 0u;
                if (p.tok_mask) {
                    m4 = 0;
#pragma unroll
                    for (int e = 0; e < 4; ++e) m4 |= (__ldg(p.tok_mask + sq + e) != 0 ? 1u : 0u) << (8 * e);
                }
                mk = m4;
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const bool m = (m4 >> (8 * e)) & 1u;
                    sr[e] = m ? c.sj : -1;
                    lp[e] = (m && p.logp) ? __ldg(p.logp + sq + e) : 0.f;
                }
            } else {
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int64_t q = q0 + e;
                    x[e] = 0; sr[e] = -1; lp[e] = 0.f;
                    if (q < Nout) {
                        while (q >= c.bend) {   // next block (blocks may be empty)
                            ++c.b;
                            cursor_load(p, c);
                        }
                        const int64_t sq = q + c.delta;
                        x[e] = __ldg(p.tokens + sq);
                        const bool m = p.tok_mask ? (__ldg(p.tok_mask + sq) != 0) : c.llm;
                        if (m) {
                            mk |= 1u << (8 * e);
                            sr[e] = c.sj;
                            if (p.logp) lp[e] = __ldg(p.logp + sq);
                        }
                    }
                }
            }
            if (vec_ok && q0 + 3 < Nout) {
                *reinterpret_cast<int4*>(p.merged_tokens + q0) = make_int4(x[0], x[1], x[2], x[3]);
                *reinterpret_cast<int4*>(p.merged_tok_src + q0) = make_int4(sr[0], sr[1], sr[2], sr[3]);
                *reinterpret_cast<uint32_t*>(p.merged_mask + q0) = mk;
                if (p.merged_logp) *reinterpret_cast<float4*>(p.merged_logp + q0) = make_float4(lp[0], lp[1], lp[2], lp[3]);
            } else {
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    if (q0 + e < Nout) {
                        p.merged_tokens[q0 + e] = x[e];
                        p.merged_tok_src[q0 + e] = sr[e];
                        p.merged_mask[q0 + e] = (uint8_t)((mk >> (8 * e)) & 1u);
                        if (p.merged_logp) p.merged_logp[q0 + e] = lp[e];
                    }
                }
            }
            // the lane's next step starts 128 tokens further: catch up with the blocks in between
            const int64_t qn = q0 + 128;
            while (qn < Nout && qn >= c.bend) {
                ++c.b;
                cursor_load(p, c);
            }
        }
    }
}

}  // namespace

extern "C" size_t ajt_merge_blocks_workspace_bytes(int32_t n, int64_t n_blocks) {
    if (n < 0 || n_blocks < 0 || n_blocks >= ((int64_t)1 << 30)) return 0;
    return block_ws_layout(n, n_blocks).total;
}

extern "C" int ajt_merge_blocks(const int64_t* block_ids, const int64_t* block_offsets, const int32_t* traj_ids,
                                const uint8_t* author, const int64_t* tok_off, const int32_t* tokens, const float* logp,
                                const uint8_t* tok_mask, int32_t n, int64_t n_blocks, int64_t n_tokens, uint32_t flags,
                                int32_t* merged_tokens, uint8_t* merged_mask, float* merged_logp, int32_t* merged_tok_src,
                                int64_t* merged_offsets, int64_t* merged_block_offsets, int32_t* merged_block_src,
                                uint8_t* merged_block_author, int64_t* merged_block_tok_off, int32_t* merged_origin,
                                int32_t* merged_traj, int32_t* owner, int64_t* counts, void* workspace, size_t workspace_bytes,
                                ajt_stream_t stream_) {
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    if (n < 0 || n_blocks < 0 || n_tokens < 0 || n_blocks >= ((int64_t)1 << 30)) return AJT_ERR_INVALID_ARG;
    if (!block_offsets || !tok_off || !counts || !merged_offsets || !merged_block_offsets || !merged_block_tok_off || !workspace)
        return AJT_ERR_INVALID_ARG;
    if (n > 0 && (!block_ids || !traj_ids || !author || !merged_block_src || !merged_block_author || !merged_origin ||
                  !merged_traj || !owner))
        return AJT_ERR_INVALID_ARG;
    if (n_tokens > 0 && (!tokens || !merged_tokens || !merged_mask || !merged_tok_src)) return AJT_ERR_INVALID_ARG;
    if ((logp == nullptr) != (merged_logp == nullptr)) return AJT_ERR_INVALID_ARG;
    if (((uintptr_t)workspace & 255) || ((uintptr_t)block_ids & 7)) return AJT_ERR_INVALID_ARG;
    const BlockWs ws0 = block_ws_layout(n, n_blocks);
    if (workspace_bytes < ws0.total) return AJT_ERR_WORKSPACE_TOO_SMALL;
    const BlockWs ws = block_ws_layout(n, n_blocks, ws0.offsets2 + (workspace_bytes - ws0.total));   // the surplus goes to the pairs

    int dev = 0, num_sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return AJT_ERR_CUDA;
    if (cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || num_sms < 1) return AJT_ERR_CUDA;

    uint8_t* b = reinterpret_cast<uint8_t*>(workspace);
    BlockParams p;
    p.block_ids = block_ids; p.block_offsets = block_offsets; p.traj_ids = traj_ids; p.author = author; p.tok_off = tok_off;
    p.tokens = tokens; p.logp = logp; p.tok_mask = tok_mask; p.n = n; p.B = n_blocks; p.N = n_tokens;
    p.merged_tokens = merged_tokens; p.merged_mask = merged_mask; p.merged_logp = merged_logp; p.merged_tok_src = merged_tok_src;
    p.merged_offsets = merged_offsets; p.merged_block_offsets = merged_block_offsets; p.merged_block_src = merged_block_src;
    p.merged_block_author = merged_block_author; p.merged_block_tok_off = merged_block_tok_off; p.merged_origin = merged_origin;
    p.counts = counts;
    p.ctrl = reinterpret_cast<AjtCtrl*>(b + ws.inner);
    p.offsets2 = reinterpret_cast<int64_t*>(b + ws.offsets2);
    p.mask2 = b + ws.mask2;
    p.ids_out = reinterpret_cast<int32_t*>(b + ws.ids_out);
    p.mask2_out = b + ws.mask2_out;
    p.src2_out = reinterpret_cast<int32_t*>(b + ws.src2_out);
    p.offs2_out = reinterpret_cast<int64_t*>(b + ws.offs2_out);
    p.counts2 = reinterpret_cast<int64_t*>(b + ws.counts2);
    p.blk_srcblk = reinterpret_cast<int64_t*>(b + ws.blk_srcblk);
    p.tile_state = reinterpret_cast<uint64_t*>(b + ws.tile_state);
    p.tile_counter = reinterpret_cast<int32_t*>(b + ws.tile_counter);

    const int ntiles = (int)((n_blocks + kScanTile - 1) / kScanTile);
    const int64_t want = (n_blocks + 255) / 256 + 1;
    const int grid_b = (int)(want < (int64_t)num_sms * 8 ? want : (int64_t)num_sms * 8);
    AJT_LAUNCH(blocks_prep_kernel<<<grid_b, 256, 0, stream>>>(p, ntiles));
    // Algorithm 1 on the id streams: text-level Match, its own owner rule (the latest extender absorbs)
    const int rc = ajt_merge_timelines(reinterpret_cast<const int32_t*>(block_ids), p.offsets2, traj_ids, nullptr, p.mask2, nullptr,
                                       n, 2 * n_blocks, AJT_OWNER_PAPER, flags, p.ids_out, p.mask2_out, p.src2_out, nullptr,
                                       p.offs2_out, merged_origin, merged_traj, owner, p.counts2, b + ws.inner,
                                       ws.offsets2 - ws.inner, stream_);
    if (rc != AJT_OK) return rc;
    AJT_LAUNCH(blocks_info_kernel<<<grid_b, 256, 0, stream>>>(p));
    AJT_LAUNCH(blocks_scan_kernel<<<max(1, min(ntiles, num_sms)), 256, 0, stream>>>(p));
    AJT_LAUNCH(blocks_offsets_kernel<<<max(1, min((n + 256) / 256, num_sms)), 256, 0, stream>>>(p));
    const int64_t wantc = (n_tokens + 8 * kCopyTile - 1) / (8 * kCopyTile) + 1;   // 8 warps per CTA, one tile per warp and turn
    AJT_LAUNCH(blocks_copy_kernel<<<(int)(wantc < (int64_t)num_sms * 8 ? wantc : (int64_t)num_sms * 8), 256, 0, stream>>>(p));
    return cudaGetLastError() == cudaSuccess ? AJT_OK : AJT_ERR_CUDA;
}
