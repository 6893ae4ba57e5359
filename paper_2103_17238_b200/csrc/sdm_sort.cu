// Row a3 of SURVEY.md section 8(a): the per-cell shuffle as a stable LSD radix sort of
// (cell_id << 32 | Philox key), 8-bit digits, one kernel launch per digit ("Onesweep" structure:
// the digit histograms of ALL passes were built up-front by k_keys_hist, so each pass reads its
// input once and scatters it once; the global offsets travel between tiles by decoupled look-back).
//
// Element format.  Pass 1 reads sortkey = (cell_id << 32 | key) (48 significant bits) with the
// super-droplet index implicit in the position, and writes
//      packed = ((sortkey >> 8) << idxbits) | index              (needs 40 + cbits-16.. <= 64 bits)
// every later pass reads and writes `packed`, taking its digit at bit idxbits + 8 (pass - 1).
// One 8-byte word per element per pass: a single LDG.64 / STS.64 / LDS.64 / STG.64 per element.
//
// Stability (required: ties between equal keys must keep index order, R4): within a tile
// the elements are ranked warp by warp in load order -- warp w owns the contiguous slab
// [w*32*ITEMS, (w+1)*32*ITEMS), round k covers 32 consecutive elements -- with
// __match_any_sync peer masks; ranks follow (warp, round, lane) = memory order.
#include "sdm_internal.h"

namespace sdm {

constexpr u32 FLAG_AGG = 1u << 30;     // tile aggregate available
constexpr u32 FLAG_PREFIX = 2u << 30;  // inclusive prefix (with the global digit base) available
constexpr u32 VALUE_MASK = (1u << 30) - 1u;
constexpr int SORT_WARPS = SORT_BLOCK / 32;
constexpr int SORT_TILE_BITS = 12;
static_assert((1 << SORT_TILE_BITS) == SORT_TILE, "tile-local index width");
static_assert(SORT_BLOCK == RADIX, "one thread per digit");

// Block-wide exclusive scan of one value per thread (SORT_BLOCK == RADIX threads).
__device__ __forceinline__ u32 block_excl_scan_256(u32 x, u32* s_warp /*[8]*/, int lane, int warp) {
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
    for (int w = 0; w < SORT_WARPS; ++w)
        if (w < warp) woff += s_warp[w];
    __syncthreads();  // s_warp reusable afterwards
    return woff + incl - x;
}

template <bool FIRST>
__global__ void __launch_bounds__(SORT_BLOCK, 3)
k_radix_pass(const u64* __restrict__ in, u64* __restrict__ out, u32 n_sd, int shift, int idxbits,
             const u32* __restrict__ ghist /*[RADIX] global histogram of this digit*/,
             u32* __restrict__ ticket, u32* __restrict__ tile_state /*[n_tiles][RADIX]*/) {
    __shared__ u64 s_stage[SORT_TILE];
    __shared__ u32 s_whist[SORT_WARPS][RADIX];
    __shared__ u32 s_goff[RADIX];
    __shared__ u32 s_warp[SORT_WARPS];
    __shared__ u32 s_tile;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) s_whist[w][tid] = 0;
    __syncthreads();
    const u32 tile = s_tile;
    const u32 base = tile * (u32)SORT_TILE;
    const u32 n_valid = min((u32)SORT_TILE, n_sd - base);

    // ---- load (warp-striped: round k of warp w = 32 consecutive elements) ----
    u64 item[SORT_ITEMS];
    const u32 wbase = warp * 32u * SORT_ITEMS + lane;
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k) {
        const u32 off = wbase + k * 32u;
        u64 x = ~0ull;  // out-of-range elements sort to the end of the last tile (digit 255)
        if (off < n_valid) {
            x = ld_stream_u64(in + base + off);
            if (FIRST) x = (x << SORT_TILE_BITS) | (u64)off;  // tile-local index below the sort key
        }
        item[k] = x;
    }

    // ---- rank within the warp, round by round (stable) ----
    u32 rank[SORT_ITEMS];
    const u32 lt = lanemask_lt();
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k) {
        const u32 d = (u32)(item[k] >> shift) & 0xFFu;
        const u32 peers = __match_any_sync(0xffffffffu, d);
        const u32 pre = __popc(peers & lt);
        u32 old = 0;
        if (pre == 0) {
            old = s_whist[warp][d];
            s_whist[warp][d] = old + __popc(peers);
        }
        old = __shfl_sync(0xffffffffu, old, __ffs(peers) - 1);
        rank[k] = old + pre;
        __syncwarp();
    }
    __syncthreads();

    // ---- per-digit: scan over warps, tile totals, tile-local digit starts ----
    const u32 d_mine = tid;  // one thread per digit
    u32 total = 0;
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) {
        const u32 t = s_whist[w][d_mine];
        s_whist[w][d_mine] = total;
        total += t;
    }
    // publish the aggregate as early as possible (tile 0 publishes its inclusive prefix below)
    u32* my_state = tile_state + (size_t)tile * RADIX + d_mine;
    if (tile != 0) st_relaxed_u32(my_state, FLAG_AGG | total);
    const u32 lstart = block_excl_scan_256(total, s_warp, lane, warp);  // tile-local start of digit
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) s_whist[w][d_mine] += lstart;
    __syncthreads();

    // ---- stage in shared memory in sorted order ----
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k) {
        const u32 d = (u32)(item[k] >> shift) & 0xFFu;
        s_stage[s_whist[warp][d] + rank[k]] = item[k];
    }

    // ---- decoupled look-back: global position of this tile's first element of digit d ----
    u32 gexcl;
    if (tile == 0) {
        gexcl = block_excl_scan_256(ghist[d_mine], s_warp, lane, warp);  // global digit base
    } else {
        gexcl = 0;
        int t = (int)tile - 1;
        while (true) {
            const u32 s = ld_relaxed_u32(tile_state + (size_t)t * RADIX + d_mine);
            const u32 flag = s & ~VALUE_MASK;
            if (flag == 0) continue;  // predecessor not published yet
            gexcl += s & VALUE_MASK;
            if (flag == FLAG_PREFIX) break;
            --t;
        }
    }
    st_relaxed_u32(my_state, FLAG_PREFIX | (gexcl + total));
    s_goff[d_mine] = gexcl - lstart;
    __syncthreads();

    // ---- coalesced scatter: consecutive staged positions of one digit are consecutive in `out` ----
#pragma unroll
    for (int j = 0; j < SORT_ITEMS; ++j) {
        const u32 p = j * SORT_BLOCK + tid;
        if (p < n_valid) {
            u64 x = s_stage[p];
            const u32 d = (u32)(x >> shift) & 0xFFu;
            if (FIRST) {
                const u64 idx = (u64)base + (x & (u64)(SORT_TILE - 1));
                x = ((x >> (SORT_TILE_BITS + 8)) << idxbits) | idx;  // drop digit 0, append the global index
            }
            out[s_goff[d] + p] = x;
        }
    }
}

cudaError_t launch_sort_pass(sdm_ctx* ctx, int pass, const u64* in, u64* out, int64_t n_sd,
                             const Plan& plan) {
    u32* ticket = ctx->ws.ctl + CTL_TICKET0 + pass;
    u32* state = ctx->ws.tile_state + (size_t)pass * (size_t)plan.n_tiles * RADIX;
    const u32* ghist = ctx->ws.digit_hist + pass * RADIX;
    LaunchScope scope(ctx, PROF_RADIX_PASS);
    if (pass == 0) {
        k_radix_pass<true><<<plan.n_tiles, SORT_BLOCK, 0, ctx->stream>>>(in, out, (u32)n_sd, SORT_TILE_BITS, plan.idxbits,
                                                                          ghist, ticket, state);
    } else {
        const int shift = plan.idxbits + 8 * (pass - 1);
        k_radix_pass<false><<<plan.n_tiles, SORT_BLOCK, 0, ctx->stream>>>(in, out, (u32)n_sd, shift,
                                                                           plan.idxbits, ghist, ticket, state);
    }
    return cudaGetLastError();
}

}  // namespace sdm
