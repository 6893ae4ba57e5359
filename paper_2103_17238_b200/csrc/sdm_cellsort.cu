// Cell-sorted fast path: when cell_id is non-decreasing, every cell
// is a contiguous run of the arrays, so the global LSD radix sort can be replaced by a per-cell sort
// held entirely in registers and fused with the pair kernel.  The order produced is the same total
// order (cell, Philox key, index) the general path and the oracle's stable sort produce, hence the
// output is bit-identical -- at 36 B/SD of HBM traffic instead of 156.
//
//   k_cell_bounds  reads cell_id once (4 B/SD): verifies order and range, writes cell_start[0..n_cell]
//   k_cell_fused   one WARP per cell (n_c <= 32*R, R in {1,2,4,8}): Philox keys -> bitonic sort of
//                  (key << 32 | local index) across the warp's registers (shuffles) -> both members of
//                  a pair sit in one lane -> probability / gamma / clamp / update in place.
//
// Cells larger than CELL_FAST_MAX make the step ineligible for this path (the host-side verdict sends
// such inputs to the general path; if one shows up anyway the step is skipped and the sticky
// bad-data flag is set).
#include "sdm_internal.h"
#include "sdm_pair.cuh"

namespace sdm {

constexpr int CF_BLOCK = 256;
constexpr int CF_WARPS = CF_BLOCK / 32;

__global__ void __launch_bounds__(256)
k_cell_bounds(const int* __restrict__ cell_id, u32 n_sd, int n_cell, u32* __restrict__ cell_start,
              u32* __restrict__ ctl, u32* __restrict__ sticky, int32_t* __restrict__ dbg_cell_start) {
    const u32 i = blockIdx.x * 256u + threadIdx.x;
    if (i >= n_sd) return;
    const int c = __ldg(cell_id + i);
    const int prev = (i == 0) ? -1 : __ldg(cell_id + i - 1);
    if (c < 0 || c >= n_cell || c < prev) {  // out of range, or not sorted after all: skip the step, report
        sticky[STICKY_BAD_DATA] = 1u;
        ctl[CTL_UNSORTED] = 1u;
        return;
    }
    // position i opens cell c and every empty cell between prev and c
    for (int q = prev + 1; q <= c; ++q) {
        cell_start[q] = i;
        if (dbg_cell_start) dbg_cell_start[q] = (int32_t)i;
    }
    if (i == n_sd - 1) {
        for (int q = c + 1; q <= n_cell; ++q) {
            cell_start[q] = n_sd;
            if (dbg_cell_start) dbg_cell_start[q] = (int32_t)n_sd;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Bitonic sort of 32*R 64-bit words held R per lane, element index e = lane*R + r (blocked), ascending.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void cmpx(u64& a, u64& b, bool asc) {  // in-lane compare-exchange
    const u64 lo = a < b ? a : b;
    const u64 hi = a < b ? b : a;
    a = asc ? lo : hi;
    b = asc ? hi : lo;
}

template <int R>
__device__ __forceinline__ void warp_bitonic_sort(u64 (&x)[R], int lane) {
    constexpr int N = 32 * R;
#pragma unroll
    for (int k = 2; k <= N; k <<= 1) {
#pragma unroll
        for (int j = k >> 1; j > 0; j >>= 1) {
            if (j >= R) {  // partner in another lane, same r
                const int lj = j / R;
                const bool lower = (lane & lj) == 0;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const int e_k = (k >= N) ? 0 : ((k >= R) ? (lane & (k / R)) : (r & k));
                    const bool asc = e_k == 0;
                    const u64 y = __shfl_xor_sync(0xffffffffu, x[r], lj);
                    const bool keep_min = (lower == asc);
                    const u64 mn = x[r] < y ? x[r] : y;
                    const u64 mx = x[r] < y ? y : x[r];
                    x[r] = keep_min ? mn : mx;
                }
            } else {  // partner in the same lane: r ^ j
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    if ((r & j) == 0) {
                        const int e_k = (k >= N) ? 0 : ((k >= R) ? (lane & (k / R)) : (r & k));
                        cmpx(x[r], x[r | j], e_k == 0);
                    }
                }
            }
        }
    }
}

struct FusedArgs {
    PairArgs pair;
    int n_cell;
    int32_t* dbg_perm;
    u32* sticky;
    const u32* ctl;
};

template <int R>
__device__ __forceinline__ void warp_cell(const FusedArgs& a, u32 start, u32 n_c, int lane) {
    u64 x[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const u32 e = lane * R + r;
        x[r] = ~0ull;
        if (e < n_c) x[r] = ((u64)philox_perm_key(a.pair.pk, (u64)(start + e)) << 32) | (u64)e;
    }
    warp_bitonic_sort<R>(x, lane);
    if (a.dbg_perm) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const u32 e = lane * R + r;
            if (e < n_c) a.dbg_perm[start + e] = (int32_t)(start + (u32)x[r]);
        }
    }
    if (R >= 2) {
#pragma unroll
        for (int r = 0; r + 1 < R; r += 2) {
            const u32 e = lane * R + r;
            if (e + 1 < n_c) pair_collide(a.pair, start + (u32)x[r], start + (u32)x[r + 1], n_c);
        }
    } else {
        const u64 y = __shfl_down_sync(0xffffffffu, x[0], 1);
        if ((lane & 1) == 0 && (u32)lane + 1 < n_c) pair_collide(a.pair, start + (u32)x[0], start + (u32)y, n_c);
    }
}

__global__ void __launch_bounds__(CF_BLOCK) k_cell_fused(const FusedArgs a) {
    if (a.ctl[CTL_UNSORTED]) return;  // k_cell_bounds found cell_id out of order: the step is skipped
    const int lane = threadIdx.x & 31;
    const int c = blockIdx.x * CF_WARPS + (threadIdx.x >> 5);
    if (c >= a.n_cell) return;
    const u32 start = __ldg(a.pair.cell_start + c);
    const u32 n_c = __ldg(a.pair.cell_start + c + 1) - start;
    if (n_c < 2) {
        if (n_c == 1 && a.dbg_perm && lane == 0) a.dbg_perm[start] = (int32_t)start;
        return;
    }
    if (n_c <= 32) warp_cell<1>(a, start, n_c, lane);
    else if (n_c <= 64) warp_cell<2>(a, start, n_c, lane);
    else if (n_c <= 128) warp_cell<4>(a, start, n_c, lane);
    else if (n_c <= CELL_FAST_MAX) warp_cell<8>(a, start, n_c, lane);
    else if (lane == 0) a.sticky[STICKY_BAD_DATA] = 1u;  // ineligible cell on the fast path
}

cudaError_t launch_cell_fused(sdm_ctx* ctx, int64_t* xi, double* v, const int32_t* cell_id, int64_t n_sd,
                              int32_t n_cell, double dtdV, const KernelParams& kp, const PhiloxKeys& pk) {
    {
        LaunchScope scope(ctx, PROF_CELL_BOUNDS);
        k_cell_bounds<<<(u32)((n_sd + 255) / 256), 256, 0, ctx->stream>>>(
            cell_id, (u32)n_sd, n_cell, ctx->ws.cell_start, ctx->ws.ctl, ctx->ws.sticky, ctx->dbg_cell_start);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    FusedArgs a;
    a.pair.sorted = nullptr;
    a.pair.xi = reinterpret_cast<long long*>(xi);
    a.pair.v = v;
    a.pair.cell_start = ctx->ws.cell_start;
    a.pair.n_sd = (u32)n_sd;
    a.pair.idxbits = 0;
    a.pair.cshift = 0;
    a.pair.single_cell = 0;
    a.pair.dtdV = dtdV;
    a.pair.kp = kp;
    a.pair.pk = pk;
    a.pair.dbg_gamma = reinterpret_cast<long long*>(ctx->dbg_gamma);
    a.pair.dbg_gamma_clamped = reinterpret_cast<long long*>(ctx->dbg_gamma_clamped);
    a.n_cell = n_cell;
    a.dbg_perm = ctx->dbg_perm;
    a.sticky = ctx->ws.sticky;
    a.ctl = ctx->ws.ctl;
    LaunchScope scope(ctx, PROF_CELL_FUSED);
    k_cell_fused<<<(u32)((n_cell + CF_WARPS - 1) / CF_WARPS), CF_BLOCK, 0, ctx->stream>>>(a);
    return cudaGetLastError();
}

}  // namespace sdm
