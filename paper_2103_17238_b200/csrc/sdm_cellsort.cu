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

constexpr int CF_WARPS = 4;
constexpr int CF_BLOCK = CF_WARPS * 32;
constexpr int CF_MIN_BLOCKS = 8;  // measured on B200: 8, 10 and 12 resident blocks give 81, 84, 87 us on cfg3
constexpr int CB_BLOCK = 256;
constexpr int CB_ITEMS = 8;

// ---------------------------------------------------------------------------------------------
// Cell boundaries of an array whose cells are contiguous.  SRC = 0: cell_id int32[n];
// SRC = 1: sorted words u64 (cell << idxbits | index);  SRC = 2: the same in u32 words.
// Eight positions per thread, read with 16-byte loads (VEC; the scalar instantiation serves a
// misaligned cell_id); the cell-size check re-reads position i - max_cell the same way (L2 hits).
// ---------------------------------------------------------------------------------------------
template <int SRC>
__device__ __forceinline__ int cell_at(const void* src, u32 i, int idxbits) {
    if (SRC == 0) return __ldg(reinterpret_cast<const int*>(src) + i);
    if (SRC == 1) return (int)(__ldg(reinterpret_cast<const u64*>(src) + i) >> idxbits);
    return (int)(__ldg(reinterpret_cast<const u32*>(src) + i) >> idxbits);
}

template <int SRC, bool VEC>
__device__ __forceinline__ void cells_at8(const void* src, u32 i0, u32 n_sd, int idxbits, int (&c)[CB_ITEMS]) {
    if (VEC && i0 + CB_ITEMS <= n_sd) {  // i0 is a multiple of 8 and the base is 16-byte aligned
        if (SRC == 1) {
            const ulonglong2* p = reinterpret_cast<const ulonglong2*>(reinterpret_cast<const u64*>(src) + i0);
#pragma unroll
            for (int q = 0; q < CB_ITEMS / 2; ++q) {
                const ulonglong2 w = __ldg(p + q);
                c[2 * q] = (int)(w.x >> idxbits);
                c[2 * q + 1] = (int)(w.y >> idxbits);
            }
        } else {
            const uint4* p = reinterpret_cast<const uint4*>(reinterpret_cast<const u32*>(src) + i0);
#pragma unroll
            for (int q = 0; q < CB_ITEMS / 4; ++q) {
                const uint4 w = __ldg(p + q);
                c[4 * q] = (int)(w.x >> idxbits);      // SRC = 0: idxbits = 0, the word is the cell_id itself
                c[4 * q + 1] = (int)(w.y >> idxbits);
                c[4 * q + 2] = (int)(w.z >> idxbits);
                c[4 * q + 3] = (int)(w.w >> idxbits);
            }
        }
    } else {
#pragma unroll
        for (int k = 0; k < CB_ITEMS; ++k) c[k] = (i0 + k < n_sd) ? cell_at<SRC>(src, i0 + k, idxbits) : 0x7fffffff;
    }
}

// Position i opens cell cc and closes cell prev (opening every empty cell in between).  The closed cell
// [s, i) is larger than max_cell exactly when position i - 1 - max_cell still belongs to it (sorted input),
// so the cell-size limit costs one extra load per cell, not per super-droplet.  Returns "too large".
template <int SRC>
__device__ __forceinline__ bool open_cells(const void* src, int idxbits, int prev, int cc, u32 i, u32 max_cell,
                                           u32* __restrict__ cell_start, int32_t* __restrict__ dbg_cell_start) {
    for (int q = prev + 1; q <= cc; ++q) {
        cell_start[q] = i;
        if (dbg_cell_start) dbg_cell_start[q] = (int32_t)i;
    }
    return prev >= 0 && i > max_cell && cell_at<SRC>(src, i - 1u - max_cell, idxbits) == prev;
}

template <int SRC, bool VEC>
__global__ void __launch_bounds__(CB_BLOCK)
k_cell_bounds(const void* __restrict__ src, u32 n_sd, int n_cell, int idxbits, u32 max_cell, u32 epoch,
              u32* __restrict__ cell_start, u32* __restrict__ ctl, u32* __restrict__ sticky,
              int32_t* __restrict__ dbg_cell_start) {
    // the fused kernel that follows accumulates the zero count; no separate memset of the control block
    if (blockIdx.x == 0 && threadIdx.x == 0) ctl[CTL_ZERO_COUNT] = 0u;
    const u32 i0 = (blockIdx.x * CB_BLOCK + threadIdx.x) * CB_ITEMS;  // lanes past the end stay for the shuffle
    int c[CB_ITEMS];
    cells_at8<SRC, VEC>(src, i0, n_sd, idxbits, c);
    int prev = __shfl_up_sync(0xffffffffu, c[CB_ITEMS - 1], 1);
    if ((threadIdx.x & 31) == 0) prev = (i0 == 0 || i0 > n_sd) ? -1 : cell_at<SRC>(src, i0 - 1, idxbits);
    bool bad = false;
    if (i0 + CB_ITEMS < n_sd) {
        // interior thread, straight-line: every value in range (then the differences cannot overflow);
        // the OR of the differences to the predecessor is negative when the order is broken, zero when the
        // thread holds no cell boundary (the common case), positive otherwise
        bad = (u32)prev + 1u > (u32)n_cell;  // prev is -1 (array start) or a cell_id that must be in range too
        int ored = 0;
        int p = prev;
#pragma unroll
        for (int k = 0; k < CB_ITEMS; ++k) {
            bad |= (u32)c[k] >= (u32)n_cell;
            ored |= c[k] - p;
            p = c[k];
        }
        bad |= ored < 0;
        if (!bad && ored != 0) {
            p = prev;
#pragma unroll
            for (int k = 0; k < CB_ITEMS; ++k) {
                if (c[k] != p) bad |= open_cells<SRC>(src, idxbits, p, c[k], i0 + k, max_cell, cell_start, dbg_cell_start);
                p = c[k];
            }
        }
    } else {
#pragma unroll
        for (int k = 0; k < CB_ITEMS; ++k) {
            const u32 i = i0 + k;
            if (i < n_sd) {
                const int cc = c[k];
                if (cc < 0 || cc >= n_cell || cc < prev) {
                    bad = true;
                } else {
                    if (cc != prev) bad |= open_cells<SRC>(src, idxbits, prev, cc, i, max_cell, cell_start, dbg_cell_start);
                    if (i == n_sd - 1)  // the array end closes cell cc and opens the (empty) rest
                        bad |= open_cells<SRC>(src, idxbits, cc, n_cell, n_sd, max_cell, cell_start, dbg_cell_start);
                }
                prev = cc;
            }
        }
    }
    if (bad) {  // out of range, out of order or too large: the step is skipped and reported
        sticky[STICKY_BAD_DATA] = 1u;
        ctl[CTL_UNSORTED] = epoch;  // tagged with this step's epoch: stale refusals never match
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
    u32* ctl;
    u32 epoch;  // ctl[CTL_UNSORTED] == epoch: k_cell_bounds refused this step's input
};

// Original array index of position e of the run that starts at `start`.
template <int WORD>
__device__ __forceinline__ u32 run_index(const FusedArgs& a, u32 start, u32 e) {
    if (WORD == 0) return start + e;
    if (WORD == 1) return (u32)(__ldg(reinterpret_cast<const u64*>(a.run_idx) + start + e) & a.idx_mask);
    return __ldg(reinterpret_cast<const u32*>(a.run_idx) + start + e) & (u32)a.idx_mask;
}

// Per-warp staging of one cell in shared memory, indexed by the position e in the run: the attributes
// are loaded ONCE, coalesced, before the (ALU-bound) key generation and sort, so the HBM latency hides
// under them; the pair phase then reads its two members by sorted position from shared memory.
template <int WORD, int RMAX>
struct CellStage {
    longlong2 xv[32 * RMAX];  // (multiplicity, volume bits)
    uint2 uw[32 * RMAX];      // Philox words 2, 3 of the SD (its uniform, used if it lands on an even slot)
    u32 key[32 * RMAX];       // full Philox permutation key (wide redo only)
    u32 idx[WORD == 0 ? 1 : 32 * RMAX];  // HYBRID: original index
};

template <int R>
__device__ __forceinline__ u32 select_reg(const u32 (&x)[R], int i) {
    u32 v = x[0];
#pragma unroll
    for (int r = 1; r < R; ++r)
        if (i == r) v = x[r];
    return v;
}

// One warp, one cell of 2 <= n_c <= 32 R super-droplets (n_c = 1 only counts its zero).  Returns this
// lane's share of the number of zero multiplicities the cell holds AFTER the step.
template <int WORD, int RMAX, int R>
__device__ __forceinline__ u32 warp_cell(const FusedArgs& a, CellStage<WORD, RMAX>& st, u32 start, u32 n_c, int lane) {
    static_assert(R <= RMAX, "register tile within the staging tile");
    const PairArgs& pa = a.pair;
    u32 zeros = 0;
    // ---- a1 + load: striped positions e = 32 r + lane (coalesced), everything parked in shared memory ----
    u32 idx[R];
    long long xi[R];
    double vol[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const u32 e = 32u * r + lane;
        idx[r] = 0; xi[r] = 1; vol[r] = 0.0;
        if (e < n_c) {
            idx[r] = run_index<WORD>(a, start, e);
            xi[r] = pa.xi[idx[r]];
            vol[r] = pa.v[idx[r]];
        }
    }
    // keys first: Philox needs only the index, so the attribute loads above stay in flight under it
    u32 x[R];
    const int drop = 32 - a.key_bits;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const u32 e = 32u * r + lane;
        x[r] = 0xFFFFFFFFu;  // padding sorts to the end
        if (e < n_c && n_c >= 2) {
            const PhiloxOut w = philox4x32_10(pa.pk, (u64)idx[r]);
            st.uw[e] = make_uint2(w.w2, w.w3);
            st.key[e] = w.w0;
            if (WORD != 0) st.idx[e] = idx[r];
            x[r] = ((w.w0 >> drop) << 8) | e;
        }
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const u32 e = 32u * r + lane;
        if (e < n_c) {
            zeros += (xi[r] == 0);
            st.xv[e] = make_longlong2(xi[r], __double_as_longlong(vol[r]));
        }
    }
    if (n_c < 2) {
        if (a.dbg_perm && lane == 0) a.dbg_perm[start] = (int32_t)idx[0];
        return zeros;
    }
    // ---- a3: sort (truncated key, position) words; slot s = lane R + r afterwards ----
    warp_bitonic_sort<u32, R>(x, lane);
    // neighbours with equal truncated keys: their order is decided by the dropped bits -> wide redo
    bool tie = false;
#pragma unroll
    for (int r = 0; r + 1 < R; ++r) tie |= (((x[r] ^ x[r + 1]) >> 8) == 0) && ((u32)(lane * R + r + 1) < n_c);
    const u32 nxt = __shfl_down_sync(0xffffffffu, x[0], 1);
    tie |= (lane < 31) && (((x[R - 1] ^ nxt) >> 8) == 0) && ((u32)(lane * R + R) < n_c);
    __syncwarp();  // the staging writes of all lanes are visible from here on
    u32 pos[R];
    if (__any_sync(0xffffffffu, tie)) {
        u64 wide[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {  // the real words occupy the first n_c slots of the narrow result
            const u32 e = x[r] & 0xFFu;
            wide[r] = ((u32)(lane * R + r) < n_c) ? (((u64)st.key[e] << 32) | (u64)e) : ~0ull;
        }
        warp_bitonic_sort<u64, R>(wide, lane);
#pragma unroll
        for (int r = 0; r < R; ++r) pos[r] = (u32)wide[r] & 0xFFu;
    } else {
#pragma unroll
        for (int r = 0; r < R; ++r) pos[r] = x[r] & 0xFFu;
    }
    if (a.dbg_perm) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const u32 s = lane * R + r;
            if (s < n_c) a.dbg_perm[start + s] = (int32_t)(WORD == 0 ? start + pos[r] : st.idx[pos[r]]);
        }
    }
    // ---- a4, phase A: every pair of neighbouring slots -- can its gamma be non-zero? ----
    constexpr int NP = (R >= 2) ? R / 2 : 1;
    u32 first[NP], second[NP];  // run positions of the pair's members, in shuffled order
    u32 need = 0;               // bit q: pair q of this lane must run the full rule
#pragma unroll
    for (int q = 0; q < NP; ++q) {
        bool valid;
        if (R >= 2) {
            first[q] = pos[2 * q];
            second[q] = pos[(2 * q + 1) % R];
            valid = (u32)(lane * R + 2 * q + 1) < n_c;
        } else {
            first[q] = pos[0];
            second[q] = __shfl_down_sync(0xffffffffu, pos[0], 1);
            valid = ((lane & 1) == 0) && ((u32)lane + 1u < n_c);
        }
        if (valid) {
            if (pa.dbg_gamma) {
                need |= 1u << q;
            } else {
                const longlong2 A = st.xv[first[q]], B = st.xv[second[q]];
                if (A.x != 0 && B.x != 0) {  // a dead partner: gamma~ = 0 whatever gamma is (R7)
                    const bool swap = A.x < B.x;
                    const uint2 w = st.uw[first[q]];
                    const double vA = __longlong_as_double(A.y), vB = __longlong_as_double(B.y);
                    if (pair_may_collide(pa, swap ? B.x : A.x, swap ? vB : vA, swap ? vA : vB, w.x, w.y, n_c))
                        need |= 1u << q;
                }
            }
        }
    }
    // ---- phase B: the full fp64 rule, only where needed; lanes take their pending pairs one at a time ----
    while (__any_sync(0xffffffffu, need != 0)) {
        if (need) {
            const int q = __ffs(need) - 1;
            need &= need - 1u;
            const u32 ea = select_reg<NP>(first, q), eb = select_reg<NP>(second, q);
            const longlong2 A = st.xv[ea], B = st.xv[eb];
            const uint2 w = st.uw[ea];
            const u32 ja = (WORD == 0) ? start + ea : st.idx[ea];
            const u32 jb = (WORD == 0) ? start + eb : st.idx[eb];
            zeros += pair_apply(pa, ja, jb, A.x, __longlong_as_double(A.y), B.x, __longlong_as_double(B.y), w.x, w.y, n_c);
        }
    }
    return zeros;
}

template <int WORD, int RMAX>
__global__ void __launch_bounds__(CF_BLOCK, CF_MIN_BLOCKS) k_cell_fused(const FusedArgs a) {
    __shared__ CellStage<WORD, RMAX> s_stage[CF_WARPS];
    if (a.ctl[CTL_UNSORTED] == a.epoch) return;  // k_cell_bounds refused the input: the step is skipped as a whole
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    CellStage<WORD, RMAX>& st = s_stage[warp];
    // one warp per cell, one launch wave after another: the block scheduler balances the (data-dependent)
    // cost of the cells; a persistent strided loop measured 12 % slower on cfg3
    const int c = blockIdx.x * CF_WARPS + warp;
    u32 zeros = 0;
    if (c < a.n_cell) {
        const u32 start = __ldg(a.pair.cell_start + c);
        const u32 n_c = __ldg(a.pair.cell_start + c + 1) - start;
        if (n_c == 0) {
        } else if (n_c <= 32) {
            zeros = warp_cell<WORD, RMAX, 1>(a, st, start, n_c, lane);
        } else if (RMAX >= 2 && n_c <= 64) {
            if constexpr (RMAX >= 2) zeros = warp_cell<WORD, RMAX, 2>(a, st, start, n_c, lane);
        } else if (RMAX >= 4 && n_c <= 128) {
            if constexpr (RMAX >= 4) zeros = warp_cell<WORD, RMAX, 4>(a, st, start, n_c, lane);
        } else if (RMAX >= 8 && n_c <= 256) {
            if constexpr (RMAX >= 8) zeros = warp_cell<WORD, RMAX, 8>(a, st, start, n_c, lane);
        } else if (lane == 0) {
            a.sticky[STICKY_BAD_DATA] = 1u;  // unreachable: k_cell_bounds refuses such cells
        }
    }
    // a5, fused: the number of zero multiplicities after the step (sdm_remove_zero_multiplicity reads it)
    zeros = __reduce_add_sync(0xffffffffu, zeros);
    if (lane == 0 && zeros) atomicAdd(a.ctl + CTL_ZERO_COUNT, zeros);
}

// src_kind: 0 = cell_id array itself (CELL_SORTED), 1 = u64 sorted words, 2 = u32 sorted words (HYBRID).
// max_cell = 32 * rmax: the largest cell the fused kernel launched next can hold.
cudaError_t launch_cell_bounds(sdm_ctx* ctx, int src_kind, const void* src, int64_t n_sd, int32_t n_cell,
                               int idxbits, int rmax) {
    const u32 grid = (u32)((n_sd + CB_BLOCK * CB_ITEMS - 1) / (CB_BLOCK * CB_ITEMS));
    const u32 max_cell = 32u * (u32)rmax;
    LaunchScope scope(ctx, PROF_CELL_BOUNDS);
    Workspace& ws = ctx->ws;
    const bool vec = (reinterpret_cast<uintptr_t>(src) & 15u) == 0;
#define SDM_BOUNDS(SRC, VEC, IDXBITS)                                                                       \
    k_cell_bounds<SRC, VEC><<<grid, CB_BLOCK, 0, ctx->stream>>>(src, (u32)n_sd, n_cell, IDXBITS, max_cell, \
                                                                ctx->epoch, ws.cell_start, ws.ctl, ws.sticky,      \
                                                                ctx->dbg_cell_start)
    if (src_kind == 0) {
        if (vec) SDM_BOUNDS(0, true, 0);
        else SDM_BOUNDS(0, false, 0);
    } else if (src_kind == 1) {
        if (vec) SDM_BOUNDS(1, true, idxbits);
        else SDM_BOUNDS(1, false, idxbits);
    } else {
        if (vec) SDM_BOUNDS(2, true, idxbits);
        else SDM_BOUNDS(2, false, idxbits);
    }
#undef SDM_BOUNDS
    return cudaGetLastError();
}

template <int WORD, int RMAX>
static void prefer_shared_carveout() {  // the staging tiles want the shared-memory end of the L1 split
    static bool done = false;
    if (!done) {
        cudaFuncSetAttribute(k_cell_fused<WORD, RMAX>, cudaFuncAttributePreferredSharedMemoryCarveout,
                             cudaSharedmemCarveoutMaxShared);
        done = true;
    }
}

template <int WORD>
static void launch_fused_word(const FusedArgs& a, int rmax, u32 grid, cudaStream_t st) {
    prefer_shared_carveout<WORD, 2>();
    prefer_shared_carveout<WORD, 4>();
    prefer_shared_carveout<WORD, 8>();
    if (rmax <= 2) k_cell_fused<WORD, 2><<<grid, CF_BLOCK, 0, st>>>(a);
    else if (rmax <= 4) k_cell_fused<WORD, 4><<<grid, CF_BLOCK, 0, st>>>(a);
    else k_cell_fused<WORD, 8><<<grid, CF_BLOCK, 0, st>>>(a);
}

cudaError_t launch_cell_fused(sdm_ctx* ctx, int src_kind, const void* run_idx, int idxbits, int rmax, int64_t* xi,
                              double* v, int64_t n_sd, int32_t n_cell, double dtdV, const KernelParams& kp,
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
    set_bound_constants(a.pair);
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
    a.epoch = ctx->epoch;
    const u32 grid = (u32)((n_cell + CF_WARPS - 1) / CF_WARPS);
    LaunchScope scope(ctx, PROF_CELL_FUSED);
    if (src_kind == 0) launch_fused_word<0>(a, rmax, grid, ctx->stream);
    else if (src_kind == 1) launch_fused_word<1>(a, rmax, grid, ctx->stream);
    else launch_fused_word<2>(a, rmax, grid, ctx->stream);
    return cudaGetLastError();
}

}  // namespace sdm
