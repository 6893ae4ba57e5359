// Per-cell shuffle fused with the pair kernel (rows a3 + a4 of SURVEY.md section 8(a) in one launch;
// SURVEY 8(f) NEXT-1).  Once the super-droplets of a cell are known as one contiguous run -- either
// because cell_id itself is non-decreasing (CELL_SORTED path: the run is a slice of the arrays) or
// because an LSD radix sort on the cell_id digits alone has grouped their indices (HYBRID path: the
// run is a slice of the sorted index array) -- the order inside the cell is produced by ONE WARP that
// sorts the cell's (Philox key, position in the run) words in registers and then applies the pair
// rule to neighbours.  The total order is (cell, key, index), exactly what the global LSD sort of
// (cell_id << 32 | key) and the oracle's std::stable_sort produce, so the output is bit-identical,
// at 36-48 B/SD of HBM traffic instead of 148.
//
//   k_cell_bounds<SRC>  reads the cell of every position once: verifies range, order and the cell-size
//                       limit, writes cell_start[0..n_cell].  Any violation sets CTL_SKIP: the fused
//                       kernel then does nothing (the state is never half-updated).
//   k_cell_fused<W>     one warp per cell, n_c <= 32 R, R in {1,2,4,8}.  Sort word = 32 bits:
//                       (top 24 bits of the Philox key) << 8 | position-in-run, sorted by an
//                       all-ascending bitonic network (IMNMX + SHFL, 2 instructions per compare).
//                       Dropping the low 8 key bits is exact unless two neighbours of the sorted run
//                       share their top 24 bits (4.8e-4 per 128-SD cell); the warp detects that and
//                       redoes its cell with full 64-bit (key << 32 | position) words.
#include "sdm_internal.h"
#include "sdm_pair.cuh"

namespace sdm {

constexpr int CF_BLOCK = 256;
constexpr int CF_WARPS = CF_BLOCK / 32;
constexpr int CB_BLOCK = 256;
constexpr int CB_ITEMS = 4;

// ---------------------------------------------------------------------------------------------
// Cell boundaries of an array whose cells are contiguous.  SRC = 0: cell_id int32[n];
// SRC = 1: sorted words u64 (cell << idxbits | index);  SRC = 2: the same in u32 words.
// ---------------------------------------------------------------------------------------------
template <int SRC>
__device__ __forceinline__ int cell_at(const void* src, u32 i, int idxbits) {
    if (SRC == 0) return __ldg(reinterpret_cast<const int*>(src) + i);
    if (SRC == 1) return (int)(__ldg(reinterpret_cast<const u64*>(src) + i) >> idxbits);
    return (int)(__ldg(reinterpret_cast<const u32*>(src) + i) >> idxbits);
}

template <int SRC>
__global__ void __launch_bounds__(CB_BLOCK)
k_cell_bounds(const void* __restrict__ src, u32 n_sd, int n_cell, int idxbits, u32 max_cell,
              u32* __restrict__ cell_start, u32* __restrict__ ctl, u32* __restrict__ sticky,
              int32_t* __restrict__ dbg_cell_start) {
    const u32 i0 = (blockIdx.x * CB_BLOCK + threadIdx.x) * CB_ITEMS;  // lanes past the end stay for the shuffle
    int c[CB_ITEMS];
    const bool full = i0 + CB_ITEMS <= n_sd;
    if (full && SRC == 0) {  // n_sd-independent alignment: the launcher guarantees 16-byte alignment
        const int4 q = __ldg(reinterpret_cast<const int4*>(reinterpret_cast<const int*>(src) + i0));
        c[0] = q.x; c[1] = q.y; c[2] = q.z; c[3] = q.w;
    } else {
#pragma unroll
        for (int k = 0; k < CB_ITEMS; ++k) c[k] = (i0 + k < n_sd) ? cell_at<SRC>(src, i0 + k, idxbits) : 0x7fffffff;
    }
    int prev = __shfl_up_sync(0xffffffffu, c[CB_ITEMS - 1], 1);
    if ((threadIdx.x & 31) == 0) prev = (i0 == 0 || i0 > n_sd) ? -1 : cell_at<SRC>(src, i0 - 1, idxbits);
    bool bad = false;
#pragma unroll
    for (int k = 0; k < CB_ITEMS; ++k) {
        const u32 i = i0 + k;
        if (i < n_sd) {
            const int cc = c[k];
            if (cc < 0 || cc >= n_cell || cc < prev) {
                bad = true;
            } else {
                // a cell larger than the fused kernel's register tile: position i - max_cell is in it too
                if (i >= max_cell && cell_at<SRC>(src, i - max_cell, idxbits) == cc) bad = true;
                for (int q = prev + 1; q <= cc; ++q) {  // i opens cell cc and every empty cell before it
                    cell_start[q] = i;
                    if (dbg_cell_start) dbg_cell_start[q] = (int32_t)i;
                }
                if (i == n_sd - 1) {
                    for (int q = cc + 1; q <= n_cell; ++q) {
                        cell_start[q] = n_sd;
                        if (dbg_cell_start) dbg_cell_start[q] = (int32_t)n_sd;
                    }
                }
            }
            prev = cc;
        }
    }
    if (bad) {  // out of range, out of order or too large: the step is skipped and reported
        sticky[STICKY_BAD_DATA] = 1u;
        ctl[CTL_UNSORTED] = 1u;
    }
}

// ---------------------------------------------------------------------------------------------
// Bitonic sort of 32*R words held R per lane, element e = lane*R + r (blocked), ascending.
// All-ascending formulation: merge of size k = one "flip" stage (partner e ^ (k-1)) followed by
// half-cleaners (partner e ^ j, j = k/4 .. 1); the lower position always keeps the minimum.
// ---------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ void cmpx_asc(T& a, T& b) {
    const T lo = a < b ? a : b;
    const T hi = a < b ? b : a;
    a = lo;
    b = hi;
}

template <typename T>
__device__ __forceinline__ T shfl_xor_any(T x, int m) {
    return __shfl_xor_sync(0xffffffffu, x, m);
}

template <typename T, int R>
__device__ __forceinline__ void warp_bitonic_sort(T (&x)[R], int lane) {
    constexpr int N = 32 * R;
#pragma unroll
    for (int k = 2; k <= N; k <<= 1) {
        if (k <= R) {  // flip inside the lane
#pragma unroll
            for (int r = 0; r < R; ++r)
                if ((r & (k >> 1)) == 0) cmpx_asc(x[r], x[r ^ (k - 1)]);
        } else {  // flip across lanes: lane ^ (k/R - 1), register R-1-r
            const int lm = k / R - 1;
            const bool lower = (lane & (k / (2 * R))) == 0;
            T y[R];
#pragma unroll
            for (int r = 0; r < R; ++r) y[r] = shfl_xor_any(x[R - 1 - r], lm);
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const T mn = x[r] < y[r] ? x[r] : y[r];
                const T mx = x[r] < y[r] ? y[r] : x[r];
                x[r] = lower ? mn : mx;
            }
        }
#pragma unroll
        for (int j = k >> 2; j > 0; j >>= 1) {
            if (j >= R) {
                const int lj = j / R;
                const bool lower = (lane & lj) == 0;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const T y = shfl_xor_any(x[r], lj);
                    const T mn = x[r] < y ? x[r] : y;
                    const T mx = x[r] < y ? y : x[r];
                    x[r] = lower ? mn : mx;
                }
            } else {
#pragma unroll
                for (int r = 0; r < R; ++r)
                    if ((r & j) == 0) cmpx_asc(x[r], x[r | j]);
            }
        }
    }
}

struct FusedArgs {
    PairArgs pair;
    int n_cell;
    int key_bits;         // key bits kept in the 32-bit sort word (24; tests lower it to force the wide redo)
    const void* run_idx;  // HYBRID: sorted words whose low idxbits are the original index; else nullptr
    u64 idx_mask;
    int32_t* dbg_perm;
    u32* sticky;
    const u32* ctl;
};

// Original array index of position e of the run that starts at `start`.
template <int WORD>
__device__ __forceinline__ u32 run_index(const FusedArgs& a, u32 start, u32 e) {
    if (WORD == 0) return start + e;
    if (WORD == 1) return (u32)(__ldg(reinterpret_cast<const u64*>(a.run_idx) + start + e) & a.idx_mask);
    return __ldg(reinterpret_cast<const u32*>(a.run_idx) + start + e) & (u32)a.idx_mask;
}

// Applies the pair rule to the sorted run: sorted slot s = lane*R + r holds run position pos[r].
template <int WORD, int R>
__device__ __forceinline__ void collide_sorted(const FusedArgs& a, u32 start, u32 n_c, int lane, const u32 (&pos)[R]) {
    if (a.dbg_perm) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const u32 s = lane * R + r;
            if (s < n_c) a.dbg_perm[start + s] = (int32_t)run_index<WORD>(a, start, pos[r]);
        }
    }
    if (R >= 2) {
#pragma unroll
        for (int r = 0; r + 1 < R; r += 2) {
            const u32 s = lane * R + r;
            if (s + 1 < n_c)
                pair_collide<false>(a.pair, run_index<WORD>(a, start, pos[r]), run_index<WORD>(a, start, pos[r + 1]), n_c);
        }
    } else {
        const u32 nxt = __shfl_down_sync(0xffffffffu, pos[0], 1);
        if ((lane & 1) == 0 && (u32)lane + 1 < n_c)
            pair_collide<false>(a.pair, run_index<WORD>(a, start, pos[0]), run_index<WORD>(a, start, nxt), n_c);
    }
}

template <int WORD, int R>
__device__ __forceinline__ void warp_cell(const FusedArgs& a, u32 start, u32 n_c, int lane) {
    u32 key[R];
    u32 x[R];
    const int drop = 32 - a.key_bits;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const u32 e = lane * R + r;
        key[r] = 0;
        x[r] = 0xFFFFFFFFu;  // padding sorts to the end (a real word ends in e < n_c <= 255 when its key is all ones)
        if (e < n_c) {
            key[r] = philox_perm_key(a.pair.pk, (u64)run_index<WORD>(a, start, e));
            x[r] = ((key[r] >> drop) << 8) | e;
        }
    }
    warp_bitonic_sort<u32, R>(x, lane);
    // neighbours with equal truncated keys: their order is decided by the dropped bits -> wide redo
    bool tie = false;
#pragma unroll
    for (int r = 0; r + 1 < R; ++r) tie |= (((x[r] ^ x[r + 1]) >> 8) == 0) && ((u32)(lane * R + r + 1) < n_c);
    const u32 nxt = __shfl_down_sync(0xffffffffu, x[0], 1);
    tie |= (lane < 31) && (((x[R - 1] ^ nxt) >> 8) == 0) && ((u32)(lane * R + R) < n_c);
    u32 pos[R];
    if (__any_sync(0xffffffffu, tie)) {
        u64 wide[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const u32 e = lane * R + r;
            wide[r] = (e < n_c) ? (((u64)key[r] << 32) | (u64)e) : ~0ull;
        }
        warp_bitonic_sort<u64, R>(wide, lane);
#pragma unroll
        for (int r = 0; r < R; ++r) pos[r] = (u32)wide[r] & 0xFFu;
    } else {
#pragma unroll
        for (int r = 0; r < R; ++r) pos[r] = x[r] & 0xFFu;
    }
    collide_sorted<WORD, R>(a, start, n_c, lane, pos);
}

template <int WORD>
__global__ void __launch_bounds__(CF_BLOCK) k_cell_fused(const FusedArgs a) {
    if (a.ctl[CTL_UNSORTED]) return;  // k_cell_bounds refused the input: the step is skipped as a whole
    const int lane = threadIdx.x & 31;
    const int c = blockIdx.x * CF_WARPS + (threadIdx.x >> 5);
    if (c >= a.n_cell) return;
    const u32 start = __ldg(a.pair.cell_start + c);
    const u32 n_c = __ldg(a.pair.cell_start + c + 1) - start;
    if (n_c < 2) {
        if (n_c == 1 && a.dbg_perm && lane == 0) a.dbg_perm[start] = (int32_t)run_index<WORD>(a, start, 0);
        return;
    }
    if (n_c <= 32) warp_cell<WORD, 1>(a, start, n_c, lane);
    else if (n_c <= 64) warp_cell<WORD, 2>(a, start, n_c, lane);
    else if (n_c <= 128) warp_cell<WORD, 4>(a, start, n_c, lane);
    else if (n_c <= CELL_FAST_MAX) warp_cell<WORD, 8>(a, start, n_c, lane);
    else if (lane == 0) a.sticky[STICKY_BAD_DATA] = 1u;  // unreachable: k_cell_bounds refuses such cells
}

// src_kind: 0 = cell_id array itself (CELL_SORTED), 1 = u64 sorted words, 2 = u32 sorted words (HYBRID)
cudaError_t launch_cell_bounds(sdm_ctx* ctx, int src_kind, const void* src, int64_t n_sd, int32_t n_cell,
                               int idxbits) {
    const u32 grid = (u32)((n_sd + CB_BLOCK * CB_ITEMS - 1) / (CB_BLOCK * CB_ITEMS));
    LaunchScope scope(ctx, PROF_CELL_BOUNDS);
    Workspace& ws = ctx->ws;
    if (src_kind == 0) {
        if ((reinterpret_cast<uintptr_t>(src) & 15u) == 0)
            k_cell_bounds<0><<<grid, CB_BLOCK, 0, ctx->stream>>>(src, (u32)n_sd, n_cell, 0, (u32)CELL_FAST_MAX,
                                                                ws.cell_start, ws.ctl, ws.sticky, ctx->dbg_cell_start);
        else  // misaligned cell_id: the scalar-load instantiation (SRC = 2 reads 4-byte words, idxbits = 0)
            k_cell_bounds<2><<<grid, CB_BLOCK, 0, ctx->stream>>>(src, (u32)n_sd, n_cell, 0, (u32)CELL_FAST_MAX,
                                                                ws.cell_start, ws.ctl, ws.sticky, ctx->dbg_cell_start);
    } else if (src_kind == 1) {
        k_cell_bounds<1><<<grid, CB_BLOCK, 0, ctx->stream>>>(src, (u32)n_sd, n_cell, idxbits, (u32)CELL_FAST_MAX,
                                                            ws.cell_start, ws.ctl, ws.sticky, ctx->dbg_cell_start);
    } else {
        k_cell_bounds<2><<<grid, CB_BLOCK, 0, ctx->stream>>>(src, (u32)n_sd, n_cell, idxbits, (u32)CELL_FAST_MAX,
                                                            ws.cell_start, ws.ctl, ws.sticky, ctx->dbg_cell_start);
    }
    return cudaGetLastError();
}

cudaError_t launch_cell_fused(sdm_ctx* ctx, int src_kind, const void* run_idx, int idxbits, int64_t* xi, double* v,
                              int64_t n_sd, int32_t n_cell, double dtdV, const KernelParams& kp,
                              const PhiloxKeys& pk) {
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
    a.key_bits = ctx->narrow_key_bits;
    a.run_idx = run_idx;
    a.idx_mask = (idxbits >= 64) ? ~0ull : ((1ull << idxbits) - 1ull);
    a.dbg_perm = ctx->dbg_perm;
    a.sticky = ctx->ws.sticky;
    a.ctl = ctx->ws.ctl;
    const u32 grid = (u32)((n_cell + CF_WARPS - 1) / CF_WARPS);
    LaunchScope scope(ctx, PROF_CELL_FUSED);
    if (src_kind == 0) k_cell_fused<0><<<grid, CF_BLOCK, 0, ctx->stream>>>(a);
    else if (src_kind == 1) k_cell_fused<1><<<grid, CF_BLOCK, 0, ctx->stream>>>(a);
    else k_cell_fused<2><<<grid, CF_BLOCK, 0, ctx->stream>>>(a);
    return cudaGetLastError();
}

}  // namespace sdm
