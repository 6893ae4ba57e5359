// Rows a1 + a2 of SURVEY.md section 8(a): Philox permutation keys, the radix-digit histograms of
// the composite sort key (cell_id << 32 | key), the per-cell histogram and its exclusive scan.
//
//   k_keys_hist  reads cell_id (4 B/SD), writes sortkey u64 (8 B/SD)            -> HBM bound, 12 B/SD
//   k_cell_scan  one CTA per slab of 4096 counts, decoupled look-back over slab totals -> latency bound
#include "sdm_internal.h"

namespace sdm {

constexpr int HIST_BLOCK = 256;
constexpr int HIST_ROUNDS = 4;        // items per thread per chunk
constexpr int SMEM_CELLS = 2048;      // cell histograms this small are built in shared memory

template <bool HAS_CELLS>
__global__ void __launch_bounds__(HIST_BLOCK)
k_keys_hist(const int32_t* __restrict__ cell_id, u32 n_sd /* < 2^30 */, int n_cell, int n_cpass, int skip,
            PhiloxKeys pk, u64* __restrict__ sortkey, u32* __restrict__ digit_hist,
            u32* __restrict__ cell_count, u32* __restrict__ ctl, u32* __restrict__ sticky) {
    __shared__ u32 s_hist[MAX_PASSES][RADIX];
    __shared__ u32 s_cells[HAS_CELLS ? SMEM_CELLS : 1];
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const bool smem_cells = HAS_CELLS && n_cell <= SMEM_CELLS;

    for (int q = tid; q < MAX_PASSES * RADIX; q += HIST_BLOCK) (&s_hist[0][0])[q] = 0;
    if (smem_cells)
        for (int q = tid; q < n_cell; q += HIST_BLOCK) s_cells[q] = 0;
    __syncthreads();

    const u32 chunk = HIST_BLOCK * HIST_ROUNDS;
    const u32 n_chunks = (n_sd + chunk - 1) / chunk;
    bool bad = false, unsorted = false;
    for (u32 ch = blockIdx.x; ch < n_chunks; ch += gridDim.x) {
        const u32 base = ch * chunk;
        int c[HIST_ROUNDS], c_before[HIST_ROUNDS];  // c_before: lane 0's predecessor, loaded with the rest (no dependent load later)
#pragma unroll
        for (int r = 0; r < HIST_ROUNDS; ++r) {
            const u32 i = base + (u32)r * HIST_BLOCK + tid;
            c[r] = 0;
            c_before[r] = -1;
            if (HAS_CELLS && i < n_sd) {
                c[r] = __ldg(cell_id + i);
                if (lane == 0 && i > 0) c_before[r] = __ldg(cell_id + i - 1);
            }
        }
#pragma unroll
        for (int r = 0; r < HIST_ROUNDS; ++r) {
            const u32 i = base + (u32)r * HIST_BLOCK + tid;
            const bool valid = i < n_sd;
            int cc = c[r];
            if (HAS_CELLS) {
                if (valid && (cc < 0 || cc >= n_cell)) { bad = true; cc = cc < 0 ? 0 : n_cell - 1; }
                // cell_id non-decreasing?  (selects the cell-sorted fast path)
                int prev = __shfl_up_sync(0xffffffffu, cc, 1);
                if (lane == 0) prev = c_before[r];  // -1 at the array start and past its end: never > cc
                if (valid && prev > cc) unsorted = true;
            }
            const u32 active = __ballot_sync(0xffffffffu, valid);
            if (valid) {
                const u32 key = philox_perm_key(pk, (u64)i);
                sortkey[i] = ((u64)(u32)cc << 32) | (u64)key;
                if (skip < 1) atomicAdd(&s_hist[0][key & 0xFF], 1u);  // skipped digits are never sorted on
                if (skip < 2) atomicAdd(&s_hist[1][(key >> 8) & 0xFF], 1u);
                if (skip < 3) atomicAdd(&s_hist[2][(key >> 16) & 0xFF], 1u);
                atomicAdd(&s_hist[3][key >> 24], 1u);
                if (HAS_CELLS) {
                    // warp-aggregated: one leader per distinct cell in this warp round
                    const u32 peers = __match_any_sync(active, cc);
                    if ((peers & lanemask_lt()) == 0) {
                        const u32 cnt = __popc(peers);
                        if (smem_cells) atomicAdd(&s_cells[cc], cnt);
                        else atomicAdd(&cell_count[cc], cnt);
                        for (int q = 0; q < n_cpass; ++q)
                            atomicAdd(&s_hist[4 + q][((u32)cc >> (8 * q)) & 0xFF], cnt);
                    }
                }
            }
        }
    }
    __syncthreads();
    for (int q = tid; q < (4 + n_cpass) * RADIX; q += HIST_BLOCK) {
        const u32 h = (&s_hist[0][0])[q];
        if (h) atomicAdd(&digit_hist[q], h);
    }
    if (smem_cells)
        for (int q = tid; q < n_cell; q += HIST_BLOCK) {
            const u32 h = s_cells[q];
            if (h) atomicAdd(&cell_count[q], h);
        }
    if (bad) sticky[STICKY_BAD_DATA] = 1u;
    if (unsorted) ctl[CTL_UNSORTED] = 1u;
}

// Exclusive scan of the per-cell counts -> cell_start[0..n_cell].  Slabs of 4096 counts, one CTA of 1024
// threads per slab (at most one CTA per SM, so every CTA of a round is resident), chained by a decoupled
// look-back over 64-bit slab states {epoch << 2 | kind, value}: kind 1 = slab total, 2 = inclusive prefix.
// The epoch tag (one per step) makes stale states of earlier steps invisible without a memset.
constexpr int SCAN_BLOCK = 1024;
constexpr int SCAN_SLAB = SCAN_BLOCK * 4;

__device__ __forceinline__ u64 ld_relaxed_u64(const u64* p) {
    u64 v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed_u64(u64* p, u64 v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

__global__ void __launch_bounds__(SCAN_BLOCK)
k_cell_scan(const u32* __restrict__ cell_count, u32* __restrict__ cell_start, int n_cell, u32 n_sd_total,
            int32_t* __restrict__ dbg_cell_start, u32* __restrict__ ctl, u64* __restrict__ slab_state, u32 epoch) {
    __shared__ u32 s_warp[32];
    __shared__ u32 s_carry;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (n_cell == 1) {  // box model: the single cell holds every super-droplet
        if (tid == 0 && blockIdx.x == 0) {
            cell_start[0] = 0;
            cell_start[1] = n_sd_total;
            if (dbg_cell_start) { dbg_cell_start[0] = 0; dbg_cell_start[1] = (int32_t)n_sd_total; }
            ctl[CTL_MAX_COUNT] = n_sd_total;
        }
        return;
    }
    const int n_slabs = (n_cell + SCAN_SLAB - 1) / SCAN_SLAB;
    const u64 tag_total = ((u64)epoch << 2 | 1ull) << 32, tag_prefix = ((u64)epoch << 2 | 2ull) << 32;
    u32 my_max = 0;
    for (int slab = blockIdx.x; slab < n_slabs; slab += gridDim.x) {
        const int c0 = slab * SCAN_SLAB + tid * 4;
        u32 x[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) x[j] = (c0 + j < n_cell) ? cell_count[c0 + j] : 0u;
        const u32 tsum = x[0] + x[1] + x[2] + x[3];
        my_max = max(my_max, max(max(x[0], x[1]), max(x[2], x[3])));
        u32 incl = tsum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const u32 y = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += y;
        }
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            const u32 w = s_warp[lane];
            u32 wi = w;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const u32 y = __shfl_up_sync(0xffffffffu, wi, o);
                if (lane >= o) wi += y;
            }
            s_warp[lane] = wi - w;  // exclusive warp offsets
            const u32 total = __shfl_sync(0xffffffffu, wi, 31);
            if (lane == 0 && slab != 0) st_relaxed_u64(slab_state + slab, tag_total | total);
            // look-back, a window of 32 predecessors at a time (lane l inspects slab j - l)
            u32 excl = 0;
            for (int j = slab - 1; j >= 0; j -= 32) {
                const int q = j - lane;
                u64 st = tag_prefix;  // before slab 0: prefix 0
                if (q >= 0) {
                    do st = ld_relaxed_u64(slab_state + q);
                    while ((u32)(st >> 34) != epoch);
                }
                const bool is_prefix = ((st >> 32) & 3ull) == 2ull;
                const u32 pm = __ballot_sync(0xffffffffu, is_prefix);
                const int first = pm ? __ffs(pm) - 1 : 32;
                excl += __reduce_add_sync(0xffffffffu, lane <= first ? (u32)st : 0u);
                if (pm) break;
            }
            if (lane == 0) {
                st_relaxed_u64(slab_state + slab, tag_prefix | (u64)(excl + total));
                s_carry = excl;
            }
        }
        __syncthreads();
        u32 run = s_carry + s_warp[warp] + (incl - tsum);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            if (c0 + j < n_cell) {
                cell_start[c0 + j] = run;
                if (dbg_cell_start) dbg_cell_start[c0 + j] = (int32_t)run;
            }
            run += x[j];
        }
        __syncthreads();  // s_warp / s_carry are rewritten by the next slab
    }
    my_max = __reduce_max_sync(0xffffffffu, my_max);
    if (lane == 0 && my_max) atomicMax(&ctl[CTL_MAX_COUNT], my_max);
    if (tid == 0 && blockIdx.x == 0) {
        cell_start[n_cell] = n_sd_total;
        if (dbg_cell_start) dbg_cell_start[n_cell] = (int32_t)n_sd_total;
    }
}

// Hybrid path: histograms of the cell_id digits alone (no Philox keys, no per-cell counts): reads cell_id
// once (4 B/SD).  Digit q of cell_id lands in digit_hist[(4 + q) * RADIX ...] (after the four key digits).
constexpr int CDH_ITEMS = 4;

__global__ void __launch_bounds__(HIST_BLOCK)
k_cell_digit_hist(const int32_t* __restrict__ cell_id, u32 n_sd, int n_cell, int n_cpass, int vec_ok,
                  u32* __restrict__ digit_hist, u32* __restrict__ sticky) {
    __shared__ u32 s_hist[4][RADIX];
    const int tid = threadIdx.x;
    for (int q = tid; q < 4 * RADIX; q += HIST_BLOCK) (&s_hist[0][0])[q] = 0;
    __syncthreads();
    bool bad = false;
    const u32 chunk = HIST_BLOCK * CDH_ITEMS;
    for (u32 base = blockIdx.x * chunk; base < n_sd; base += gridDim.x * chunk) {
        const u32 i0 = base + tid * CDH_ITEMS;
        int c[CDH_ITEMS];
        if (vec_ok && i0 + CDH_ITEMS <= n_sd) {
            const int4 v = __ldg(reinterpret_cast<const int4*>(cell_id + i0));
            c[0] = v.x; c[1] = v.y; c[2] = v.z; c[3] = v.w;
        } else {
#pragma unroll
            for (int k = 0; k < CDH_ITEMS; ++k) c[k] = (i0 + k < n_sd) ? __ldg(cell_id + i0 + k) : -1;
        }
        // grouped input (whole warp inside one cell): one add of 32 x CDH_ITEMS per digit instead of 128
        // same-address atomics, which shared memory would serialise
        const bool full = i0 + CDH_ITEMS <= n_sd;
        const bool same = full && c[0] == c[1] && c[0] == c[2] && c[0] == c[3] && (u32)c[0] < (u32)n_cell;
        const int c_first = __shfl_sync(0xffffffffu, c[0], 0);  // every lane takes part, whatever `same` says
        if (__all_sync(0xffffffffu, same && c[0] == c_first)) {
            if ((tid & 31) == 0)
                for (int q = 0; q < n_cpass; ++q) atomicAdd(&s_hist[q][((u32)c[0] >> (8 * q)) & 0xFFu], 32u * CDH_ITEMS);
            continue;
        }
#pragma unroll
        for (int k = 0; k < CDH_ITEMS; ++k) {
            if (i0 + k < n_sd) {
                int cc = c[k];
                if (cc < 0 || cc >= n_cell) { bad = true; cc = cc < 0 ? 0 : n_cell - 1; }
                for (int q = 0; q < n_cpass; ++q) atomicAdd(&s_hist[q][((u32)cc >> (8 * q)) & 0xFFu], 1u);
            }
        }
    }
    __syncthreads();
    for (int q = tid; q < n_cpass * RADIX; q += HIST_BLOCK) {
        const u32 h = (&s_hist[0][0])[q];
        if (h) atomicAdd(&digit_hist[4 * RADIX + q], h);
    }
    if (bad) sticky[STICKY_BAD_DATA] = 1u;
}

cudaError_t launch_cell_digit_hist(sdm_ctx* ctx, const int32_t* cell_id, int64_t n_sd, int32_t n_cell,
                                   const Plan& plan) {
    const long long chunk = (long long)HIST_BLOCK * CDH_ITEMS;
    long long n_chunks = (n_sd + chunk - 1) / chunk;
    int grid = (int)(n_chunks < (long long)ctx->sm_count * 8 ? n_chunks : (long long)ctx->sm_count * 8);
    if (grid < 1) grid = 1;
    const int vec_ok = (reinterpret_cast<uintptr_t>(cell_id) & 15u) == 0;
    LaunchScope scope(ctx, PROF_CELL_DIGIT_HIST);
    k_cell_digit_hist<<<grid, HIST_BLOCK, 0, ctx->stream>>>(cell_id, (u32)n_sd, n_cell, plan.n_cpass, vec_ok,
                                                            ctx->ws.digit_hist, ctx->ws.sticky);
    return cudaGetLastError();
}

cudaError_t launch_keys_hist(sdm_ctx* ctx, const int32_t* cell_id, int64_t n_sd, int32_t n_cell,
                             const Plan& plan, const PhiloxKeys& pk, u64* sortkey_out) {
    const long long chunk = (long long)HIST_BLOCK * HIST_ROUNDS;
    long long n_chunks = (n_sd + chunk - 1) / chunk;
    int grid = (int)(n_chunks < (long long)ctx->sm_count * 8 ? n_chunks : (long long)ctx->sm_count * 8);
    if (grid < 1) grid = 1;
    const int n_cpass = plan.n_cpass;
    LaunchScope scope(ctx, PROF_KEYS_HIST);
    if (n_cell > 1)
        k_keys_hist<true><<<grid, HIST_BLOCK, 0, ctx->stream>>>(cell_id, (u32)n_sd, n_cell, n_cpass, plan.skip, pk, sortkey_out,
                                                                 ctx->ws.digit_hist, ctx->ws.cell_count,
                                                                 ctx->ws.ctl, ctx->ws.sticky);
    else
        k_keys_hist<false><<<grid, HIST_BLOCK, 0, ctx->stream>>>(cell_id, (u32)n_sd, n_cell, n_cpass, plan.skip, pk, sortkey_out,
                                                                  ctx->ws.digit_hist, ctx->ws.cell_count,
                                                                  ctx->ws.ctl, ctx->ws.sticky);
    return cudaGetLastError();
}

cudaError_t launch_cell_scan(sdm_ctx* ctx, int32_t n_cell, int64_t n_sd) {
    LaunchScope scope(ctx, PROF_CELL_SCAN);
    const int n_slabs = (n_cell + SCAN_SLAB - 1) / SCAN_SLAB;
    const int grid = n_slabs < ctx->sm_count ? n_slabs : ctx->sm_count;  // all CTAs of a round resident (look-back)
    k_cell_scan<<<grid, SCAN_BLOCK, 0, ctx->stream>>>(ctx->ws.cell_count, ctx->ws.cell_start, n_cell, (u32)n_sd,
                                                      ctx->dbg_cell_start, ctx->ws.ctl, ctx->ws.scan_state, ctx->epoch);
    return cudaGetLastError();
}

}  // namespace sdm
