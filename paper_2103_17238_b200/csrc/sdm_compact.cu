// Rows a5 and a6 of SURVEY.md section 8(a): stable in-place removal of zero-multiplicity super-
// droplets (north_star (d)) and the per-cell statistics (O6); plus the two test
// hooks that expose the a1 generator and the kernel function on their own.
//
// Compaction = (1) k_count_zero reads xi once (8 B/SD) and counts the zeros; the host needs that
// count anyway (*n_sd_out), and when it is 0 nothing else runs.  (2) k_compact: single-pass chained
// scan (decoupled look-back on one counter per tile) + scatter, IN PLACE.  In-place is safe because a
// tile publishes its count only after all of its loads have completed (bar.sync + release), a
// successor stores only after it has acquired every predecessor's count, and destinations never lie
// beyond the tile's own end: a store can only land where the owning tile has already read.
#include "sdm_internal.h"

namespace sdm {

constexpr u32 CMP_FLAG_AGG = 1u << 30;
constexpr u32 CMP_FLAG_PREFIX = 2u << 30;
constexpr u32 CMP_VALUE_MASK = (1u << 30) - 1u;

__global__ void __launch_bounds__(256) k_count_zero(const long long* __restrict__ xi, long long n_sd,
                                                    u32* __restrict__ ctl) {
    u32 zeros = 0;
    const long long stride = (long long)gridDim.x * blockDim.x * 2;
    for (long long i = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * 2; i < n_sd; i += stride) {
        if (i + 1 < n_sd) {
            const longlong2 x = *reinterpret_cast<const longlong2*>(xi + i);
            zeros += (x.x == 0) + (x.y == 0);
        } else {
            zeros += (xi[i] == 0);
        }
    }
    zeros = __reduce_add_sync(0xffffffffu, zeros);
    __shared__ u32 s_sum;
    if (threadIdx.x == 0) s_sum = 0;
    __syncthreads();
    if ((threadIdx.x & 31) == 0 && zeros) atomicAdd(&s_sum, zeros);
    __syncthreads();
    if (threadIdx.x == 0 && s_sum) atomicAdd(&ctl[CTL_ZERO_COUNT], s_sum);
}

__global__ void __launch_bounds__(CMP_BLOCK)
k_compact(long long* __restrict__ xi, double* __restrict__ v, int* __restrict__ cell_id, u32 n_sd,
          u32* __restrict__ ticket, u32* __restrict__ state) {
    __shared__ u32 s_tile;
    __shared__ u32 s_wcount[CMP_BLOCK / 32];
    __shared__ u32 s_prefix;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    __syncthreads();
    const u32 tile = s_tile;
    const u32 base = tile * (u32)CMP_TILE;

    long long x[CMP_ITEMS];
    double vv[CMP_ITEMS];
    int cc[CMP_ITEMS];
    u32 rank[CMP_ITEMS];
    u32 keepmask = 0;
    const u32 wbase = base + warp * 32u * CMP_ITEMS + lane;
#pragma unroll
    for (int k = 0; k < CMP_ITEMS; ++k) {
        const u32 i = wbase + k * 32u;
        x[k] = 0; vv[k] = 0.0; cc[k] = 0;
        if (i < n_sd) { x[k] = xi[i]; vv[k] = v[i]; cc[k] = cell_id[i]; }
    }
    u32 wrun = 0;  // survivors of this warp so far (rounds in memory order)
#pragma unroll
    for (int k = 0; k < CMP_ITEMS; ++k) {
        const bool keep = x[k] != 0;  // out-of-range entries were loaded as 0
        const u32 b = __ballot_sync(0xffffffffu, keep);
        rank[k] = wrun + __popc(b & lanemask_lt());
        wrun += __popc(b);
        keepmask |= (keep ? 1u : 0u) << k;
    }
    if (lane == 0) s_wcount[warp] = wrun;
    __syncthreads();  // every load of this CTA has completed (values were consumed by the ballots)
    u32 woff = 0, total = 0;
#pragma unroll
    for (int w = 0; w < CMP_BLOCK / 32; ++w) {
        const u32 cnt = s_wcount[w];
        if (w < warp) woff += cnt;
        total += cnt;
    }
    if (warp == 0) {
        // decoupled look-back by one warp, a window of 32 predecessors per round trip (lane l inspects tile - 1 - l):
        // with thousands of tiles in flight a single thread walking back one tile per L2 round trip was the whole
        // kernel (167 us for 8.4 M entries; 110 us now -- four windows per round trip measured slower, 127 us: what
        // remains is the wait for the predecessors' own loads, during which a tile holds its slot with nothing in flight)
        u32 excl = 0;
        if (tile == 0) {
            if (lane == 0) st_release_u32(state + tile, CMP_FLAG_PREFIX | total);
        } else {
            if (lane == 0) st_release_u32(state + tile, CMP_FLAG_AGG | total);
            for (int j = (int)tile - 1; j >= 0; j -= 32) {
                const int q = j - lane;
                u32 sv = CMP_FLAG_PREFIX;  // before tile 0: prefix 0
                if (q >= 0) {
                    do sv = ld_relaxed_u32(state + q);  // relaxed polling; one fence below is the acquire side
                    while ((sv & ~CMP_VALUE_MASK) == 0u);
                }
                const u32 pm = __ballot_sync(0xffffffffu, (sv & ~CMP_VALUE_MASK) == CMP_FLAG_PREFIX);
                const int first = pm ? __ffs(pm) - 1 : 32;  // nearest predecessor that already knows its prefix
                excl += __reduce_add_sync(0xffffffffu, lane <= first ? (sv & CMP_VALUE_MASK) : 0u);
                if (pm) break;
            }
            __threadfence();  // acquire side of the predecessors' releases: relaxed polling, one fence at the end
            if (lane == 0) st_release_u32(state + tile, CMP_FLAG_PREFIX | (excl + total));
        }
        if (lane == 0) s_prefix = excl;
    }
    __syncthreads();
    const u32 dst0 = s_prefix + woff;
    // nothing was removed before or inside this tile: every survivor is already in place
    if (s_prefix == base && total == min((u32)CMP_TILE, n_sd - base)) return;
#pragma unroll
    for (int k = 0; k < CMP_ITEMS; ++k) {
        if ((keepmask >> k) & 1u) {
            const u32 dst = dst0 + rank[k];
            xi[dst] = x[k];
            v[dst] = vv[k];
            cell_id[dst] = cc[k];
        }
    }
}

// ------------------------------------------------------------------------------------------
// a6: per-cell count, sum xi, sum xi v, sum xi v^2.  Warp-aggregated atomics: one leader per
// distinct cell in each warp round adds the warp's partial sums.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_cell_stats(const long long* __restrict__ xi, const double* __restrict__ v, const int* __restrict__ cell_id,
             long long n_sd, int n_cell, int* __restrict__ count, unsigned long long* __restrict__ sum_xi,
             double* __restrict__ sum_xi_v, double* __restrict__ sum_xi_v2, u32* __restrict__ sticky) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    const int lane = threadIdx.x & 31;
    for (long long i0 = (long long)blockIdx.x * blockDim.x; i0 < n_sd; i0 += stride) {
        const long long i = i0 + threadIdx.x;
        const bool valid = i < n_sd;
        int c = valid ? cell_id[i] : 0;
        const bool ok = valid && c >= 0 && c < n_cell;
        if (valid && !ok) sticky[STICKY_BAD_DATA] = 1u;
        const u32 okmask = __ballot_sync(0xffffffffu, ok);
        if (!ok) continue;
        const long long x = xi[i];
        const double xd = (double)x;
        const double xv = __dmul_rn(xd, v[i]);
        const double xv2 = __dmul_rn(xv, v[i]);
        // peers: the lanes of this warp round that hold the same cell
        const u32 here = __match_any_sync(okmask, c);
        const int leader = __ffs(here) - 1;
        u32 cnt = __popc(here);
        long long sx = 0;
        double sxv = 0.0, sxv2 = 0.0;
        // leader accumulates its peers in lane order (deterministic within the warp)
        for (u32 m = here; m; m &= m - 1) {
            const int src = __ffs(m) - 1;
            sx += __shfl_sync(here, x, src);
            sxv = __dadd_rn(sxv, __shfl_sync(here, xv, src));
            sxv2 = __dadd_rn(sxv2, __shfl_sync(here, xv2, src));
        }
        if (lane == leader) {
            if (count) atomicAdd(&count[c], (int)cnt);
            if (sum_xi) atomicAdd(&sum_xi[c], (unsigned long long)sx);
            if (sum_xi_v) atomicAdd(&sum_xi_v[c], sxv);
            if (sum_xi_v2) atomicAdd(&sum_xi_v2[c], sxv2);
        }
    }
}

// ------------------------------------------------------------------------------------------
// Test hooks
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_philox_fill(PhiloxKeys pk, u64 i0, long long n, u32* __restrict__ key_out,
                                                     double* __restrict__ u_out) {
    const long long t = (long long)blockIdx.x * 256 + threadIdx.x;
    if (t >= n) return;
    const PhiloxOut w = philox4x32_10(pk, i0 + (u64)t);
    if (key_out) key_out[t] = w.w0;
    if (u_out) u_out[t] = uniform_from_words(w.w2, w.w3);
}

__global__ void __launch_bounds__(256) k_kernel_eval(KernelParams kp, const double* __restrict__ vj,
                                                     const double* __restrict__ vk, long long n,
                                                     double* __restrict__ K_out) {
    const long long t = (long long)blockIdx.x * 256 + threadIdx.x;
    if (t < n) K_out[t] = coalescence_kernel(kp, vj[t], vk[t]);
}

cudaError_t launch_count_zero(sdm_ctx* ctx, const int64_t* xi, int64_t n_sd) {
    long long want = (n_sd / 2 + 255) / 256;
    int grid = (int)(want < (long long)ctx->sm_count * 8 ? want : (long long)ctx->sm_count * 8);
    if (grid < 1) grid = 1;
    LaunchScope scope(ctx, PROF_COUNT_ZERO);
    k_count_zero<<<grid, 256, 0, ctx->stream>>>(reinterpret_cast<const long long*>(xi), n_sd, ctx->ws.ctl);
    return cudaGetLastError();
}

cudaError_t launch_compact(sdm_ctx* ctx, int64_t* xi, double* v, int32_t* cell_id, int64_t n_sd) {
    const u32 n_tiles = (u32)((n_sd + CMP_TILE - 1) / CMP_TILE);
    LaunchScope scope(ctx, PROF_COMPACT);
    k_compact<<<n_tiles, CMP_BLOCK, 0, ctx->stream>>>(reinterpret_cast<long long*>(xi), v, cell_id, (u32)n_sd,
                                                      ctx->ws.ctl + CTL_CMP_TICKET, ctx->ws.cmp_state);
    return cudaGetLastError();
}

cudaError_t launch_cell_stats(sdm_ctx* ctx, const int64_t* xi, const double* v, const int32_t* cell_id,
                              int64_t n_sd, int32_t n_cell, int32_t* count, int64_t* sum_xi,
                              double* sum_xi_v, double* sum_xi_v2) {
    long long want = (n_sd + 255) / 256;
    int grid = (int)(want < (long long)ctx->sm_count * 16 ? want : (long long)ctx->sm_count * 16);
    if (grid < 1) grid = 1;
    LaunchScope scope(ctx, PROF_CELL_STATS);
    k_cell_stats<<<grid, 256, 0, ctx->stream>>>(reinterpret_cast<const long long*>(xi), v, cell_id, n_sd, n_cell,
                                                count, reinterpret_cast<unsigned long long*>(sum_xi), sum_xi_v,
                                                sum_xi_v2, ctx->ws.sticky);
    return cudaGetLastError();
}

cudaError_t launch_philox_fill(sdm_ctx* ctx, const PhiloxKeys& pk, u64 i0, int64_t n, u32* key_out,
                               double* u_out) {
    const u32 grid = (u32)((n + 255) / 256);
    LaunchScope scope(ctx, PROF_OTHER);
    k_philox_fill<<<grid, 256, 0, ctx->stream>>>(pk, i0, n, key_out, u_out);
    return cudaGetLastError();
}

cudaError_t launch_kernel_eval(sdm_ctx* ctx, const KernelParams& kp, const double* vj, const double* vk,
                               int64_t n, double* K_out) {
    const u32 grid = (u32)((n + 255) / 256);
    LaunchScope scope(ctx, PROF_OTHER);
    k_kernel_eval<<<grid, 256, 0, ctx->stream>>>(kp, vj, vk, n, K_out);
    return cudaGetLastError();
}

}  // namespace sdm
