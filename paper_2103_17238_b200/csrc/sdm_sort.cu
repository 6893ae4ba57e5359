// Row a3 of SURVEY.md section 8(a): stable LSD radix sort passes, 8-bit digits, one launch per digit
// ("Onesweep" structure: the digit histograms of ALL passes are built up-front -- k_keys_hist for the
// general path, k_cell_digit_hist for the hybrid path -- so each pass reads its input once and scatters
// it once; the global offsets travel between tiles by decoupled look-back).
//
// Three element flows share one kernel template:
//   MODE_KEY_FIRST   general path, pass 0.  in: u64 sortkey = (cell_id << 32 | Philox key), index implicit
//                    in the position.  out: packed = ((sortkey >> 8) << idxbits) | index.
//   MODE_CELL_FIRST  hybrid path, pass 0.  in: int32 cell_id, index implicit.  out: (cell_id << idxbits) | index
//                    in a u64 or (when it fits) u32 word.
//   MODE_LATER       every later pass: reads and writes the same word, digit at `shift`.
// One word per element per pass: a single LDG / STS / LDS / STG per element.
//
// Stability (required: ties between equal keys must keep index order, R4): within a tile
// the elements are ranked warp by warp in load order -- warp w owns the contiguous slab
// [w*32*ITEMS, (w+1)*32*ITEMS), round k covers 32 consecutive elements.  The peers of a lane (lanes of
// the same round with the same digit) are gathered as a lane mask by one shared-memory atomic OR per
// element (MATCH.ANY costs grow with the number of distinct digits in the warp, eight ballots per round
// cost ~45 instructions per element: profiles/).  Ranks follow (warp, round, lane) = memory order.
#include "sdm_internal.h"

namespace sdm {

constexpr u32 FLAG_AGG = 1u << 30;     // tile aggregate available
constexpr u32 FLAG_PREFIX = 2u << 30;  // inclusive prefix (with the global digit base) available
constexpr u32 VALUE_MASK = (1u << 30) - 1u;
constexpr int SORT_WARPS = SORT_BLOCK / 32;
constexpr int LOOK_WINDOW = 8;
static_assert((1 << SORT_TILE_BITS) == SORT_TILE, "tile-local index width");
static_assert(SORT_BLOCK >= RADIX && SORT_BLOCK % RADIX == 0, "the first RADIX threads own one digit each");
#ifndef SORT_MIN_BLOCKS
#define SORT_MIN_BLOCKS (1024 / SORT_BLOCK_THREADS)
#endif

enum { MODE_KEY_FIRST = 0, MODE_CELL_FIRST = 1, MODE_LATER = 2 };

// Block-wide exclusive scan of one value per digit thread (the first RADIX threads; the others pass 0 and get nothing).
__device__ __forceinline__ u32 block_excl_scan_256(u32 x, u32* s_warp /*[SORT_WARPS]*/, int lane, int warp) {
    u32 incl = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const u32 y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += y;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    u32 woff = 0;
#pragma unroll
    for (int w = 0; w < RADIX / 32; ++w)
        if (w < warp) woff += s_warp[w];
    __syncthreads();  // s_warp reusable afterwards
    return woff + incl - x;
}

template <typename T>
__device__ __forceinline__ T ld_stream(const T* p);
template <>
__device__ __forceinline__ u64 ld_stream<u64>(const u64* p) { return ld_stream_u64(p); }
template <>
__device__ __forceinline__ u32 ld_stream<u32>(const u32* p) {
    u32 v;
    asm volatile("ld.global.L1::no_allocate.u32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}

template <typename TIn, typename TW, int MODE>
__global__ void __launch_bounds__(SORT_BLOCK, SORT_MIN_BLOCKS)
k_radix_pass(const TIn* __restrict__ in, TW* __restrict__ out, u32 n_sd, int shift, int idxbits, int n_cell,
             const u32* __restrict__ ghist /*[RADIX] global histogram of this digit*/,
             u32* __restrict__ ticket, u32* __restrict__ tile_state /*[n_tiles][RADIX]*/) {
    static_assert(sizeof(TW) * SORT_TILE >= (size_t)SORT_WARPS * RADIX * 4, "the lane-mask table aliases the staging buffer");
    __shared__ TW s_stage[SORT_TILE];
    __shared__ u32 s_whist[SORT_WARPS][RADIX];
    __shared__ u32 s_goff[RADIX];
    __shared__ u32 s_warp[SORT_WARPS];
    __shared__ u32 s_tile;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
#pragma unroll
    for (int i = 0; i < SORT_WARPS * RADIX / SORT_BLOCK; ++i) (&s_whist[0][0])[i * SORT_BLOCK + tid] = 0;
#pragma unroll
    for (int i = 0; i < SORT_WARPS * RADIX / SORT_BLOCK; ++i)
        reinterpret_cast<u32*>(s_stage)[i * SORT_BLOCK + tid] = 0;  // the lane-mask table of the ranking phase
    __syncthreads();
    const u32 tile = s_tile;
    const u32 base = tile * (u32)SORT_TILE;
    const u32 n_valid = min((u32)SORT_TILE, n_sd - base);
    // where the digit sits in the staged word (first passes stage `word << SORT_TILE_BITS | tile-local index`)
    const int dshift = (MODE == MODE_LATER) ? shift : SORT_TILE_BITS + shift;

    // ---- load (warp-striped: round k of warp w = 32 consecutive elements) ----
    TW item[SORT_ITEMS];
    const u32 wbase = warp * 32u * SORT_ITEMS + lane;
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k) {
        const u32 off = wbase + k * 32u;
        TW x = (TW)~(TW)0;  // out-of-range elements sort to the end of the last tile (digit 255)
        if (off < n_valid) {
            if constexpr (MODE == MODE_CELL_FIRST) {
                int c = (int)ld_stream<u32>(reinterpret_cast<const u32*>(in) + base + off);
                c = c < 0 ? 0 : (c >= n_cell ? n_cell - 1 : c);  // bad data was flagged by the histogram kernel
                x = ((TW)(u32)c << SORT_TILE_BITS) | (TW)off;
            } else if constexpr (MODE == MODE_KEY_FIRST) {
                x = ((TW)ld_stream<TIn>(in + base + off) << SORT_TILE_BITS) | (TW)off;  // tile-local index below the key
            } else {
                x = (TW)ld_stream<TIn>(in + base + off);
            }
        }
        item[k] = x;
    }

    // ---- stable ranks inside the warp, round by round (32 consecutive elements each) ----
    // The peers of a lane (lanes of the round with the same digit) are collected in a per-warp table of
    // lane masks: one shared-memory atomic OR per element instead of eight ballots and their selects; the
    // first peer then advances the warp's running digit counter and clears the mask for the next use.
    // The table aliases the staging buffer, which is not written before every warp has finished ranking.
    u32 (*s_mask)[RADIX] = reinterpret_cast<u32 (*)[RADIX]>(s_stage);
    u32 info[SORT_ITEMS];  // [23:16] digit, [15:0] rank among this warp's elements with that digit
    const u32 lt = lanemask_lt();
    const u32 me = 1u << lane;
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k) {
        const u32 d = (u32)(item[k] >> dshift) & 0xFFu;
        u32 peers, old;
        if (__all_sync(0xffffffffu, d == __shfl_sync(0xffffffffu, d, 0))) {
            // one digit in the whole round (cell digits of an already grouped array): no table traffic,
            // and none of the 32-way same-address serialisation the atomic would see
            peers = 0xffffffffu;
            old = s_whist[warp][d];
            __syncwarp();
            if (lane == 0) s_whist[warp][d] = old + 32u;
        } else {
            atomicOr(&s_mask[warp][d], me);
            __syncwarp();
            peers = s_mask[warp][d];
            __syncwarp();  // every lane has its mask before the first peer clears it
            // the first peer takes the warp's running count of the digit forward and hands the old value to the others
            // (one atomic by the first peers and a shuffle instead of a load by every lane and a store by the first
            // peers: the pass is bound by the shared-memory pipe, profiles/r2d_README.md)
            old = 0;
            if ((peers & lt) == 0) {
                old = atomicAdd(&s_whist[warp][d], (u32)__popc(peers));
                s_mask[warp][d] = 0u;
            }
            old = __shfl_sync(0xffffffffu, old, __ffs(peers) - 1);
        }
        __syncwarp();
        const u32 pre = __popc(peers & lt);
        info[k] = (d << 16) | (old + pre);
    }
    __syncthreads();

    // ---- per-digit (the first RADIX threads): scan over warps, tile totals, tile-local digit starts ----
    const u32 d_mine = tid & (RADIX - 1);
    const bool digit_thread = SORT_BLOCK == RADIX || tid < RADIX;
    u32 total = 0;
    if (digit_thread) {
#pragma unroll
        for (int w = 0; w < SORT_WARPS; ++w) {
            const u32 t = s_whist[w][d_mine];
            s_whist[w][d_mine] = total;
            total += t;
        }
    }
    // publish the aggregate as early as possible (tile 0 publishes its inclusive prefix below)
    u32* my_state = tile_state + (size_t)tile * RADIX + d_mine;
    if (digit_thread && tile != 0) st_relaxed_u32(my_state, FLAG_AGG | total);
    const u32 lstart = block_excl_scan_256(total, s_warp, lane, warp);  // tile-local start of digit
    if (digit_thread) {
#pragma unroll
        for (int w = 0; w < SORT_WARPS; ++w) s_whist[w][d_mine] += lstart;
    }
    __syncthreads();

    // ---- stage in shared memory in sorted order ----
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k) s_stage[s_whist[warp][info[k] >> 16] + (info[k] & 0xFFFFu)] = item[k];

    // ---- decoupled look-back: global position of this tile's first element of digit d ----
    u32 gexcl = 0;
    if (tile == 0) {
        gexcl = block_excl_scan_256(digit_thread ? ghist[d_mine] : 0u, s_warp, lane, warp);  // global digit base
    } else if (digit_thread) {
        // a window of LOOK_WINDOW predecessors per round trip to L2 (the tiles of a launch wave publish their
        // aggregates at about the same time, so the walk back to the nearest inclusive prefix is a dozen tiles long
        // on average: one dependent load per tile made the walk the longest stall of the pass)
        int t = (int)tile - 1;
        bool done = false;
        while (!done) {
            u32 s[LOOK_WINDOW];
#pragma unroll
            for (int w = 0; w < LOOK_WINDOW; ++w)
                s[w] = (t - w >= 0) ? ld_relaxed_u32(tile_state + (size_t)(t - w) * RADIX + d_mine) : 0u;
#pragma unroll
            for (int w = 0; w < LOOK_WINDOW; ++w) {
                const u32 flag = s[w] & ~VALUE_MASK;
                if (done || flag == 0) break;  // not published yet: poll again from this tile on
                gexcl += s[w] & VALUE_MASK;
                --t;
                done = flag == FLAG_PREFIX;  // tile 0 always publishes its prefix: the walk ends there at the latest
            }
        }
    }
    if (digit_thread) {
        st_relaxed_u32(my_state, FLAG_PREFIX | (gexcl + total));
        s_goff[d_mine] = gexcl - lstart;
    }
    __syncthreads();

    // ---- coalesced scatter: consecutive staged positions of one digit are consecutive in `out` ----
#pragma unroll
    for (int j = 0; j < SORT_ITEMS; ++j) {
        const u32 p = j * SORT_BLOCK + tid;
        if (p < n_valid) {
            TW x = s_stage[p];
            const u32 d = (u32)(x >> dshift) & 0xFFu;
            if (MODE == MODE_KEY_FIRST) {
                const TW idx = (TW)base + (x & (TW)(SORT_TILE - 1));
                x = ((x >> (SORT_TILE_BITS + 8)) << idxbits) | idx;  // drop digit 0, append the global index
            } else if (MODE == MODE_CELL_FIRST) {
                const TW idx = (TW)base + (x & (TW)(SORT_TILE - 1));
                x = ((x >> SORT_TILE_BITS) << idxbits) | idx;  // keep the whole cell_id above the global index
            }
            out[s_goff[d] + p] = x;
        }
    }
}

// General path (north_star (b)): pass 0 reads the 8-byte sort keys, later passes the packed words.  Executed
// pass p sorts digit q = plan.skip + p of (cell_id << 32 | key); the skipped low key digits are left to
// k_tie_repair.
cudaError_t launch_sort_pass(sdm_ctx* ctx, int pass, const u64* in, u64* out, int64_t n_sd,
                             const Plan& plan) {
    const int q = plan.skip + pass;
    u32* ticket = ctx->ws.ctl + CTL_TICKET0 + pass;
    u32* state = ctx->ws.tile_state + (size_t)pass * (size_t)plan.n_tiles * RADIX;
    const u32* ghist = ctx->ws.digit_hist + q * RADIX;
    LaunchScope scope(ctx, PROF_RADIX_PASS);
    if (pass == 0) {
        k_radix_pass<u64, u64, MODE_KEY_FIRST><<<plan.n_tiles, SORT_BLOCK, 0, ctx->stream>>>(
            in, out, (u32)n_sd, 8 * q, plan.idxbits, 0, ghist, ticket, state);
    } else {
        const int shift = plan.idxbits + 8 * (q - 1);
        k_radix_pass<u64, u64, MODE_LATER><<<plan.n_tiles, SORT_BLOCK, 0, ctx->stream>>>(
            in, out, (u32)n_sd, shift, plan.idxbits, 0, ghist, ticket, state);
    }
    return cudaGetLastError();
}

// Exact order inside the runs of equal sorted digits.  After the passes the words are ordered by
// (cell_id, key >> 8 skip); members of a run that ties on that are still in index order (LSD stability).
// The thread at a run's first position sorts the run by (full Philox key, index) -- the order the
// remaining passes would have produced.  Runs are disjoint, so the repair is race-free and in place;
// with kb sorted key bits a super-droplet sits in such a run with probability ~ n_c / 2^kb.
__device__ __noinline__ void repair_run(u64* __restrict__ sorted, u32 s, u32 n_sd, int idxbits, int tshift,
                                        const PhiloxKeys* __restrict__ pkp /* the kernel's __grid_constant__ parameter */) {
    const PhiloxKeys& pk = *pkp;
    const u64 tag = sorted[s] >> tshift;
    u32 e = s + 2;
    while (e < n_sd && (sorted[e] >> tshift) == tag) ++e;
    const u64 idx_mask = (1ull << idxbits) - 1ull;
    for (u32 a = s + 1; a < e; ++a) {  // insertion sort by (key, index)
        const u64 wa = sorted[a];
        const u64 ia = wa & idx_mask;
        const u64 ka = ((u64)philox_perm_key(pk, ia) << 32) | ia;
        u32 b = a;
        while (b > s) {
            const u64 wb = sorted[b - 1];
            const u64 ib = wb & idx_mask;
            const u64 kb = ((u64)philox_perm_key(pk, ib) << 32) | ib;
            if (kb < ka) break;
            sorted[b] = wb;
            --b;
        }
        sorted[b] = wa;
    }
}

constexpr int TR_ITEMS = 4;

__global__ void __launch_bounds__(256)
k_tie_repair(u64* __restrict__ sorted, u32 n_sd, int idxbits, int tshift, const __grid_constant__ PhiloxKeys pk) {
    const u64 none = ~0ull;  // a tag no real word has (tshift >= 1): stands in where the array ends
    const u32 stride = gridDim.x * 256u * TR_ITEMS;
    for (u32 s0 = (blockIdx.x * 256u + threadIdx.x) * TR_ITEMS; s0 < n_sd; s0 += stride) {
        // tags of positions s0 - 1 .. s0 + TR_ITEMS
        u64 t[TR_ITEMS + 2];
        if (s0 + TR_ITEMS <= n_sd) {
            const ulonglong2 p = *reinterpret_cast<const ulonglong2*>(sorted + s0);
            const ulonglong2 q = *reinterpret_cast<const ulonglong2*>(sorted + s0 + 2);
            t[1] = p.x >> tshift; t[2] = p.y >> tshift; t[3] = q.x >> tshift; t[4] = q.y >> tshift;
        } else {
#pragma unroll
            for (int k = 0; k < TR_ITEMS; ++k) t[1 + k] = (s0 + k < n_sd) ? (sorted[s0 + k] >> tshift) : none;
        }
        t[0] = s0 > 0 ? (sorted[s0 - 1] >> tshift) : none;
        t[TR_ITEMS + 1] = (s0 + TR_ITEMS < n_sd) ? (sorted[s0 + TR_ITEMS] >> tshift) : none;
        // a run starts where the tag differs from the predecessor's and equals the successor's; its first
        // position repairs it (runs are disjoint: a run reaching into another thread's positions does not
        // start there, and its members keep their common tag while they are being permuted)
        u32 starts = 0;
#pragma unroll
        for (int k = 0; k < TR_ITEMS; ++k)
            if (t[1 + k] != none && t[1 + k] != t[k] && t[1 + k] == t[2 + k]) starts |= 1u << k;
        while (starts) {
            const int k = __ffs(starts) - 1;
            starts &= starts - 1u;
            repair_run(sorted, s0 + k, n_sd, idxbits, tshift, &pk);
        }
    }
}

cudaError_t launch_tie_repair(sdm_ctx* ctx, u64* sorted, int64_t n_sd, const Plan& plan, const PhiloxKeys& pk) {
    LaunchScope scope(ctx, PROF_TIE_REPAIR);
    // the words hold (sortkey >> 8) above the index: sorted key bit 8 skip sits at idxbits + 8 (skip - 1)
    const u32 need = (u32)((n_sd + 256 * TR_ITEMS - 1) / (256 * TR_ITEMS));
    const u32 resident = (u32)ctx->sm_count * 8u;
    k_tie_repair<<<need < resident ? need : resident, 256, 0, ctx->stream>>>(sorted, (u32)n_sd, plan.idxbits,
                                                                           plan.idxbits + 8 * (plan.skip - 1), pk);
    return cudaGetLastError();
}

// Hybrid path: LSD passes over the cell_id digits only; words are (cell_id << idxbits | index).
// `narrow` selects 4-byte words (legal when cbits + idxbits <= 32 and cbits + 12 <= 32).
cudaError_t launch_cell_sort_pass(sdm_ctx* ctx, int pass, bool narrow, const int32_t* cell_id, const void* in,
                                  void* out, int64_t n_sd, int32_t n_cell, const Plan& plan) {
    u32* ticket = ctx->ws.ctl + CTL_TICKET0 + pass;
    u32* state = ctx->ws.tile_state + (size_t)pass * (size_t)plan.n_tiles * RADIX;
    const u32* ghist = ctx->ws.digit_hist + (4 + pass) * RADIX;  // cell digits live after the four key digits
    LaunchScope scope(ctx, PROF_RADIX_PASS);
    const int shift = plan.idxbits + 8 * pass;
    if (narrow) {
        if (pass == 0)
            k_radix_pass<int32_t, u32, MODE_CELL_FIRST><<<plan.n_tiles, SORT_BLOCK, 0, ctx->stream>>>(
                cell_id, reinterpret_cast<u32*>(out), (u32)n_sd, 0, plan.idxbits, n_cell, ghist, ticket, state);
        else
            k_radix_pass<u32, u32, MODE_LATER><<<plan.n_tiles, SORT_BLOCK, 0, ctx->stream>>>(
                reinterpret_cast<const u32*>(in), reinterpret_cast<u32*>(out), (u32)n_sd, shift, plan.idxbits, n_cell,
                ghist, ticket, state);
    } else {
        if (pass == 0)
            k_radix_pass<int32_t, u64, MODE_CELL_FIRST><<<plan.n_tiles, SORT_BLOCK, 0, ctx->stream>>>(
                cell_id, reinterpret_cast<u64*>(out), (u32)n_sd, 0, plan.idxbits, n_cell, ghist, ticket, state);
        else
            k_radix_pass<u64, u64, MODE_LATER><<<plan.n_tiles, SORT_BLOCK, 0, ctx->stream>>>(
                reinterpret_cast<const u64*>(in), reinterpret_cast<u64*>(out), (u32)n_sd, shift, plan.idxbits, n_cell,
                ghist, ticket, state);
    }
    return cudaGetLastError();
}

}  // namespace sdm
