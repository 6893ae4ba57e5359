// Per-cell shuffle fused with the pair kernel (rows a3 + a4 of SURVEY.md section 8(a) in one launch;
// SURVEY 8(f) NEXT-1).  Once the super-droplets of a cell are known as one contiguous run -- either
// because cell_id itself is non-decreasing (CELL_SORTED path: the run is a slice of the arrays) or
// because an LSD radix sort on the cell_id digits alone has grouped their indices (HYBRID path: the
// run is a slice of the sorted index array) -- the order inside the cell is produced by a GROUP OF G
// LANES that sorts the cell's (Philox key, position in the run) words in registers, R words per lane,
// and then applies the pair rule to neighbours.  The total order is (cell, key, index), exactly what
// the global LSD sort of (cell_id << 32 | key) and the oracle's std::stable_sort produce, so the output
// is bit-identical, at 32-48 B/SD of HBM traffic instead of 148.
//
//   k_cell_bounds<SRC>  reads the cell of every position once (a pure streaming kernel): verifies range and
//                       order, writes cell_start[0..n_cell].
//   k_cell_classes      one thread per cell: size class (<= 32, 48, 64, 96, 128, 192, 256 entries), the cell ids grouped by
//                       class (so that every warp of the fused kernel works on cells of one class) and the
//                       verdict (device flag for the fused kernel, mapped host words for the path choice and
//                       the launch geometry).  When the input does not fit the fused kernel launched next,
//                       that kernel does nothing (the state is never half-updated).
//   k_cell_fused<R>     size class k = cells of at most P = class_slots(k) entries.  The power-of-two classes are
//                       sorted by G = P / R lanes holding R words each, the classes in between (48, 96, 192: a
//                       quarter fewer slots for the cells that fit them) by P / 6 lanes holding 6 words
//                       (group_sort6); a warp takes 32 / G cells.  With R = 8 a cell of 128 runs 18 of the 28
//                       bitonic stages inside the lanes (1 instruction per element) and 10 across lanes
//                       (SHFL + 2 VIMNMX per element); R = 16 (22 + 6) executes 12 % fewer instructions still but
//                       its straight-line code no longer streams through the instruction caches (30 % of the
//                       stall samples "no instruction": profiles/r2b_README.md), so it is not built.
//                       Sort word = 32 bits: (top 24 bits of the Philox key)
//                       << 8 | position-in-run.  Dropping the low 8 key bits is exact unless two neighbours
//                       of the sorted run share their top 24 bits (4.8e-4 per 128-SD cell); the group detects
//                       that and orders such runs by the regenerated full key.
#include "sdm_internal.h"
#include "sdm_pair.cuh"

namespace sdm {

constexpr int CF_WARPS = 4;       // measured on B200 (profiles/r2b_README.md): 2 warps per block 15 % slower
constexpr int CF_MIN_BLOCKS = 9;  // 56 registers; 8 (64 registers) and 7 measured the same on configs[3]
constexpr int CF_BLOCK = CF_WARPS * 32;
constexpr int CB_BLOCK = 256;
constexpr int CB_K = 4;                         // quads (4 positions, one 16-byte load for int32 sources) per thread and iteration
constexpr int CB_CHUNK = CB_BLOCK * CB_K * 4;   // positions per block and iteration
constexpr u32 CLASS_REFUSED = (u32)CELL_CLASSES;  // a cell of more than 256 entries, or unsorted / out-of-range input

// ---------------------------------------------------------------------------------------------
// Cell boundaries of an array whose cells are contiguous.  SRC = 0: cell_id int32[n];
// SRC = 1: sorted words u64 (cell << idxbits | index);  SRC = 2: the same in u32 words.
// A streaming kernel: a resident grid strides over chunks of 4096 positions; every thread has four
// independent, warp-coalesced 16-byte loads in flight per iteration (VEC; the scalar instantiation serves
// a misaligned cell_id) and in the common case -- no cell boundary among its positions -- writes nothing.
// ---------------------------------------------------------------------------------------------
template <int SRC>
__device__ __forceinline__ int cell_at(const void* src, u32 i, int idxbits) {
    if (SRC == 0) return __ldg(reinterpret_cast<const int*>(src) + i);
    if (SRC == 1) return (int)(__ldg(reinterpret_cast<const u64*>(src) + i) >> idxbits);
    return (int)(__ldg(reinterpret_cast<const u32*>(src) + i) >> idxbits);
}

template <int SRC, bool VEC>
__device__ __forceinline__ void cells_at4(const void* src, u32 i0, u32 n_sd, int idxbits, int (&c)[4]) {
    if (VEC && i0 + 4 <= n_sd) {  // i0 is a multiple of 4 and the base is 16-byte aligned
        if (SRC == 1) {
            const ulonglong2* p = reinterpret_cast<const ulonglong2*>(reinterpret_cast<const u64*>(src) + i0);
            const ulonglong2 w0 = __ldg(p), w1 = __ldg(p + 1);
            c[0] = (int)(w0.x >> idxbits); c[1] = (int)(w0.y >> idxbits);
            c[2] = (int)(w1.x >> idxbits); c[3] = (int)(w1.y >> idxbits);
        } else {
            const uint4 w = __ldg(reinterpret_cast<const uint4*>(reinterpret_cast<const u32*>(src) + i0));
            c[0] = (int)(w.x >> idxbits);  // SRC = 0: idxbits = 0, the word is the cell_id itself
            c[1] = (int)(w.y >> idxbits);
            c[2] = (int)(w.z >> idxbits);
            c[3] = (int)(w.w >> idxbits);
        }
    } else {
#pragma unroll
        for (int k = 0; k < 4; ++k) c[k] = (i0 + k < n_sd) ? cell_at<SRC>(src, i0 + k, idxbits) : 0x7fffffff;
    }
}

// Position i opens cell cc (and every empty cell between prev and cc).
__device__ __forceinline__ void open_cells(int prev, int cc, u32 i, u32* __restrict__ cell_start,
                                           int32_t* __restrict__ dbg_cell_start) {
    for (int q = prev + 1; q <= cc; ++q) {
        cell_start[q] = i;
        if (dbg_cell_start) dbg_cell_start[q] = (int32_t)i;
    }
}

template <int SRC, bool VEC>
__global__ void __launch_bounds__(CB_BLOCK)
k_cell_bounds(const void* __restrict__ src, u32 n_sd, int n_cell, int idxbits, u32* __restrict__ cell_start,
              u32* __restrict__ ctl, u32* __restrict__ run, int32_t* __restrict__ dbg_cell_start) {
    // the fused kernel that follows accumulates the zero count; no separate memset of the control block
    if (blockIdx.x == 0 && threadIdx.x == 0) ctl[CTL_ZERO_COUNT] = 0u;
    const int lane = threadIdx.x & 31;
    bool bad = false;
    const u32 n_chunks = (n_sd + CB_CHUNK - 1) / CB_CHUNK;
    for (u32 ch = blockIdx.x; ch < n_chunks; ch += gridDim.x) {
        const u32 base = ch * (u32)CB_CHUNK;
        int c[CB_K][4];
        int before[CB_K];  // lane 0: the cell of the position before the warp's 128 positions of round k
#pragma unroll
        for (int k = 0; k < CB_K; ++k) {
            const u32 i0 = base + ((u32)k * CB_BLOCK + threadIdx.x) * 4u;
            cells_at4<SRC, VEC>(src, i0, n_sd, idxbits, c[k]);
            before[k] = (lane == 0 && i0 > 0 && i0 <= n_sd) ? cell_at<SRC>(src, i0 - 1, idxbits) : -1;
        }
#pragma unroll
        for (int k = 0; k < CB_K; ++k) {
            const u32 i0 = base + ((u32)k * CB_BLOCK + threadIdx.x) * 4u;  // lanes past the end stay for the shuffle
            int prev = __shfl_up_sync(0xffffffffu, c[k][3], 1);
            if (lane == 0) prev = before[k];
            if (i0 + 4 < n_sd) {
                // interior quad, straight-line: every value in range (then the differences cannot overflow); the
                // OR of the differences to the predecessor is negative when the order is broken, zero when the
                // quad holds no cell boundary (the common case), positive otherwise
                bool b = (u32)prev + 1u > (u32)n_cell;  // prev is -1 (array start) or a cell_id that must be in range too
                int ored = 0;
                int p = prev;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    b |= (u32)c[k][j] >= (u32)n_cell;
                    ored |= c[k][j] - p;
                    p = c[k][j];
                }
                b |= ored < 0;
                if (!b && ored != 0) {
                    p = prev;
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        if (c[k][j] != p) open_cells(p, c[k][j], i0 + j, cell_start, dbg_cell_start);
                        p = c[k][j];
                    }
                }
                bad |= b;
            } else {
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const u32 i = i0 + j;
                    if (i < n_sd) {
                        const int cc = c[k][j];
                        if (cc < 0 || cc >= n_cell || cc < prev) {
                            bad = true;
                        } else {
                            if (cc != prev) open_cells(prev, cc, i, cell_start, dbg_cell_start);
                            if (i == n_sd - 1)  // the array end opens the (empty) rest and closes the array
                                open_cells(cc, n_cell, n_sd, cell_start, dbg_cell_start);
                        }
                        prev = cc;
                    }
                }
            }
        }
    }
    // out of range or out of order: refused like a cell that is too large (k_cell_classes publishes the verdict)
    if (__any_sync(0xffffffffu, bad) && lane == 0) atomicMax(&run[RUN_BOUNDS_CLASS], CLASS_REFUSED);
}

// Second half of the analysis, one thread per cell: the size class of every cell from cell_start (class k: at most
// class_slots(k) = 32, 48, 64, 96, 128, 192, 256 entries; refused: larger), the cell ids grouped by class (list[k * stride ...]: cells of
// fewer than two entries go to class 0 -- the fused kernel still counts a lone zero multiplicity; the order inside a
// class is the (nearly ascending) order in which the warps draw their slots -- cells are independent, so no result
// depends on it), and the verdict: the last block publishes the worst class and the class counts through the mapped
// status words, and raises the device-side refusal flag the fused kernel looks at.
__global__ void __launch_bounds__(256)
k_cell_classes(const u32* __restrict__ cell_start, int n_cell, u32 strict, u32 epoch, u32* __restrict__ ctl,
               u32* __restrict__ sticky, u32* __restrict__ run, volatile u32* __restrict__ mapped,
               u32* __restrict__ list, u32 stride) {
    __shared__ u32 s_cls;
    if (threadIdx.x == 0) s_cls = 0u;
    __syncthreads();
    const int c = blockIdx.x * 256 + threadIdx.x;
    const int lane = threadIdx.x & 31;
    u32 cls = 0xFFu;
    if (c < n_cell) {
        const u32 n = cell_start[c + 1] - cell_start[c];
        cls = CLASS_REFUSED;
#pragma unroll
        for (int k = CELL_CLASSES - 1; k >= 0; --k)
            if (n <= (u32)class_slots(k)) cls = (u32)k;
    }
    const u32 lt = lanemask_lt();
#pragma unroll
    for (u32 k = 0; k < CLASS_REFUSED; ++k) {
        const u32 m = __ballot_sync(0xffffffffu, cls == k);
        if (m == 0u) continue;
        const int leader = __ffs(m) - 1;
        u32 base = 0;
        if (lane == leader) base = atomicAdd(&run[RUN_LIST_CURSOR + k], (u32)__popc(m));
        base = __shfl_sync(0xffffffffu, base, leader);
        if (cls == k) list[(size_t)k * stride + base + __popc(m & lt)] = (u32)c;
    }
    const u32 wcls = __reduce_max_sync(0xffffffffu, cls == 0xFFu ? 0u : cls);
    if (lane == 0 && wcls) atomicMax(&s_cls, wcls);
    __syncthreads();
    if (threadIdx.x == 0) {
        if (s_cls) atomicMax(&run[RUN_BOUNDS_CLASS], s_cls);
        __threadfence();
        const u32 t = atomicAdd(&run[RUN_BOUNDS_TICKET], 1u);
        if (t == gridDim.x - 1) {  // the last block: every other block's class and list entries are visible (fence + ticket)
            __threadfence();
            const u32 worst = atomicExch(&run[RUN_BOUNDS_CLASS], 0u);
            run[RUN_BOUNDS_TICKET] = 0u;
            if (worst >= CLASS_REFUSED) {  // the step is skipped as a whole and reported
                ctl[CTL_UNSORTED] = epoch;  // tagged with this step's epoch: stale refusals never match
                if (strict) sticky[STICKY_BAD_DATA] = 1u;
            }
            for (u32 k = 0; k < CLASS_REFUSED; ++k) mapped[MAPPED_CLASS_COUNT + k] = atomicExch(&run[RUN_LIST_CURSOR + k], 0u);
            mapped[MAPPED_VERDICT_CLASS] = worst;
            __threadfence_system();
            mapped[MAPPED_VERDICT_EPOCH] = epoch;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Bitonic sort of G*R words held R per lane by a group of G lanes (lg = lane within the group), element
// slot = lg*R + r (blocked), ascending.  All-ascending formulation: merge of size k = one "flip" stage
// (partner slot ^ (k-1)) followed by half-cleaners (partner slot ^ j, j = k/4 .. 1); the lower slot always
// keeps the minimum.
// ---------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ void cmpx_asc(T& a, T& b) {
    const T lo = a < b ? a : b;
    const T hi = a < b ? b : a;
    a = lo;
    b = hi;
}

// The same for R = 6 words per lane (cells of up to 48 / 96 / 192 entries: three quarters of the next power of two, a
// quarter fewer slots than that class would spend on them).  The network is the blocked bitonic sort with the lanes'
// runs as its units: an optimal 12-comparator network sorts the six words of a lane; a merge over m lanes is the flip
// across lanes (partner lane ^ (m - 1), registers reversed), the half-cleaners at lane distances m/4 .. 1 -- each works
// on bitonic sequences of the even length 2 lj 6, which is all the half-cleaner theorem needs -- and then every lane
// holds a bitonic sequence of six words: one half-cleaner at distance 3 and a 3-sorter per half put it in order.
__device__ __forceinline__ void lane_sort6(u32 (&x)[6]) {
    cmpx_asc(x[0], x[5]); cmpx_asc(x[1], x[3]); cmpx_asc(x[2], x[4]);
    cmpx_asc(x[1], x[2]); cmpx_asc(x[3], x[4]);
    cmpx_asc(x[0], x[3]); cmpx_asc(x[2], x[5]);
    cmpx_asc(x[0], x[1]); cmpx_asc(x[2], x[3]); cmpx_asc(x[4], x[5]);
    cmpx_asc(x[1], x[2]); cmpx_asc(x[3], x[4]);
}
__device__ __forceinline__ void lane_merge6(u32 (&x)[6]) {  // a bitonic sequence of six words
    cmpx_asc(x[0], x[3]); cmpx_asc(x[1], x[4]); cmpx_asc(x[2], x[5]);
    cmpx_asc(x[0], x[2]); cmpx_asc(x[3], x[5]);
    cmpx_asc(x[0], x[1]); cmpx_asc(x[3], x[4]);
    cmpx_asc(x[1], x[2]); cmpx_asc(x[4], x[5]);
}
template <int G>
__device__ __forceinline__ void group_sort6(u32 (&x)[6], int lg) {
    lane_sort6(x);
#pragma unroll
    for (int m = 2; m <= G; m <<= 1) {
        {
            const bool lower = (lg & (m >> 1)) == 0;
            u32 y[6];
#pragma unroll
            for (int r = 0; r < 6; ++r) y[r] = __shfl_xor_sync(0xffffffffu, x[5 - r], m - 1);
#pragma unroll
            for (int r = 0; r < 6; ++r) {
                const u32 mn = min(x[r], y[r]);
                const u32 mx = max(x[r], y[r]);
                x[r] = lower ? mn : mx;
            }
        }
#pragma unroll
        for (int lj = m >> 2; lj > 0; lj >>= 1) {
            const bool lower = (lg & lj) == 0;
#pragma unroll
            for (int r = 0; r < 6; ++r) {
                const u32 y = __shfl_xor_sync(0xffffffffu, x[r], lj);
                const u32 mn = min(x[r], y);
                const u32 mx = max(x[r], y);
                x[r] = lower ? mn : mx;
            }
        }
        lane_merge6(x);
    }
}

template <int R, int G>
__device__ __forceinline__ void group_bitonic_sort(u32 (&x)[R], int lg) {
    if constexpr (R == 6) {
        group_sort6<G>(x, lg);
        return;
    } else {
    constexpr int N = G * R;
#pragma unroll
    for (int k = 2; k <= N; k <<= 1) {
        if (k <= R) {  // flip inside the lane
#pragma unroll
            for (int r = 0; r < R; ++r)
                if ((r & (k >> 1)) == 0) cmpx_asc(x[r], x[r ^ (k - 1)]);
        } else {  // flip across lanes: lane ^ (k/R - 1), register R-1-r
            const int lm = k / R - 1;
            const bool lower = (lg & (k / (2 * R))) == 0;
            u32 y[R];
#pragma unroll
            for (int r = 0; r < R; ++r) y[r] = __shfl_xor_sync(0xffffffffu, x[R - 1 - r], lm);
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const u32 mn = min(x[r], y[r]);
                const u32 mx = max(x[r], y[r]);
                x[r] = lower ? mn : mx;
            }
        }
#pragma unroll
        for (int j = k >> 2; j > 0; j >>= 1) {
            if (j >= R) {
                const int lj = j / R;
                const bool lower = (lg & lj) == 0;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const u32 y = __shfl_xor_sync(0xffffffffu, x[r], lj);
                    const u32 mn = min(x[r], y);
                    const u32 mx = max(x[r], y);
                    x[r] = lower ? mn : mx;
                }
            } else {
#pragma unroll
                for (int r = 0; r < R; ++r)
                    if ((r & j) == 0) cmpx_asc(x[r], x[r | j]);
            }
        }
    }
    }  // R != 6
}

struct FusedArgs {
    PairArgs pair;
    int n_cell;
    int key_bits;         // key bits kept in the 32-bit sort word (24; tests lower it to force the tie repair)
    const void* run_idx;  // HYBRID: sorted words whose low idxbits are the original index; else nullptr
    int run_u32;          // HYBRID: the words are 32 bits wide
    u64 idx_mask;
    int32_t* dbg_perm;
    u32* sticky;
    u32* ctl;
    u32 epoch;  // ctl[CTL_UNSORTED] == epoch: k_cell_bounds refused this step's input
    // the cells by size class: class k is served by blocks [class_block_end[k-1], class_block_end[k])
    const u32* class_cells[CELL_CLASSES];  // cell ids of the class; nullptr = the cells 0 .. class_count - 1 themselves
    u32 class_count[CELL_CLASSES];
    u32 class_block_end[CELL_CLASSES];
    u32 only_class;       // the one class that has blocks in this launch; CELL_CLASSES: several have
    u32 cell_offset;      // class_cells == nullptr: the first cell of the launch
    u32 n_steps;          // consecutive steps of the launch (pair.pk holds the first); > 1 only without compactions and debug outputs
    // zero bookkeeping (row a5 fused into a4) and the halt protocol of sdm_coalescence_steps (see sdm_api.cu):
    u32* zc_accum;        // += zero multiplicities the array holds after this step
    const u32* zc_check;  // non-null: the previous step's count, after which a compaction was due -- if it is not 0
                          // the run halts here (nothing is updated) until the host has compacted
    u32* zc_clear;        // non-null: the slot the NEXT step accumulates into (zeroed by block 0)
    u32 halt_tag;         // != 0: a step of a multi-step run; written to run[RUN_HALT] and to the mapped status
                          // block when this step halts
    u32* run;             // RUN_* words
    volatile u32* mapped; // pinned host status words (MAPPED_*), written with a system-scope fence
};

// Original array index of position e of the run that starts at `start` (the Philox counter, R1).
// HYB: 0 = the arrays are in run order; 1 = HYBRID, attributes gathered through the index words; 2 = HYBRID with a
// resident copy: pair.xi / pair.v are cell-grouped copies in run order, only the Philox counter comes from the words.
template <int HYB>
__device__ __forceinline__ u32 run_index(const FusedArgs& a, u32 start, u32 e) {
    if (HYB == 0) return start + e;
    if (a.run_u32) return __ldg(reinterpret_cast<const u32*>(a.run_idx) + start + e) & (u32)a.idx_mask;
    return (u32)(__ldg(reinterpret_cast<const u64*>(a.run_idx) + start + e) & a.idx_mask);
}

// Where position e of the run keeps its attributes: HYB = 0 / 2 at the position itself (the arrays, or the
// cell-grouped copy of a resident run, are in run order), HYB = 1 at its original index.
template <int HYB>
__device__ __forceinline__ u32 attr_index(u32 start, u32 e, u32 idx) { return HYB == 1 ? idx : start + e; }

// Per-warp staging of the fp32 side values of the first-level pair test, indexed by cell-in-warp * P + position
// in the run: written once per super-droplet right after the (coalesced) attribute load, read by sorted position.
// The exact attributes are NOT staged: the few pairs that pass the first level read them again (L1 / L2 hits).
template <int R>
struct WarpStage {
    float2 fl[32 * R];  // (multiplicity rounded UP to fp32, volume rounded UP to fp32)
    u32 w3[32 * R];     // Philox word 3 of the super-droplet (the high word of its uniform)
};

template <int R>
__device__ __forceinline__ u32 select_reg(const u32 (&x)[R], int i) {
    u32 v = x[0];
#pragma unroll
    for (int r = 1; r < R; ++r)
        if (i == r) v = x[r];
    return v;
}

// The full Philox permutation key of position e of a run (the rare tie repair only; kept out of line).
template <int HYB>
__device__ __noinline__ u32 tie_full_key(const FusedArgs* a, PhiloxStep ps, u32 start, u32 e) {
    return philox4x32_10(a->pair.pk, ps, (u64)run_index<HYB>(*a, start, e)).w0;
}

// Two neighbouring sort words (wa before wb) that agree on the truncated key: is (full key, position) of wa larger
// than that of wb?  Padding words (position >= n_c) count as key 0xFFFFFFFF: a real word never moves behind them.
template <int HYB>
__device__ __forceinline__ bool tie_out_of_order(const FusedArgs& a, const PhiloxStep& ps, u32 start, u32 n_c, u32 wa, u32 wb) {
    const u32 ea = wa & 0xFFu, eb = wb & 0xFFu;
    const u32 ka = ea < n_c ? tie_full_key<HYB>(&a, ps, start, ea) : 0xFFFFFFFFu;
    const u32 kb = eb < n_c ? tie_full_key<HYB>(&a, ps, start, eb) : 0xFFFFFFFFu;
    return ka > kb || (ka == kb && ea > eb);
}

// Words that agree on the truncated key form runs that the narrow sort left in position order; the low key bits it
// dropped decide their true order.  Odd-even style repair in registers: a bubble pass inside every lane, one
// exchange across each lane boundary of the group, repeated until a pass swaps nothing anywhere in the warp.
template <int HYB, int G, int R>
__device__ __forceinline__ void repair_ties(const FusedArgs& a, const PhiloxStep& ps, u32 (&x)[R], u32 start, u32 n_c, int lg) {
    static_assert(R >= 2, "the two boundary words of a lane are different registers");
    bool again;
    do {
        bool sw = false;
#pragma unroll
        for (int r = 0; r + 1 < R; ++r) {
            if ((x[r] ^ x[r + 1]) < 0x100u && tie_out_of_order<HYB>(a, ps, start, n_c, x[r], x[r + 1])) {
                const u32 t = x[r]; x[r] = x[r + 1]; x[r + 1] = t;
                sw = true;
            }
        }
        // both lanes of a boundary take the same decision from the same two words
        const u32 nx = __shfl_down_sync(0xffffffffu, x[0], 1), pv = __shfl_up_sync(0xffffffffu, x[R - 1], 1);
        const bool swn = lg < G - 1 && (x[R - 1] ^ nx) < 0x100u && tie_out_of_order<HYB>(a, ps, start, n_c, x[R - 1], nx);
        const bool swp = lg > 0 && (pv ^ x[0]) < 0x100u && tie_out_of_order<HYB>(a, ps, start, n_c, pv, x[0]);
        if (swn) x[R - 1] = nx;
        if (swp) x[0] = pv;
        sw |= swn | swp;
        again = __any_sync(0xffffffffu, sw);
    } while (again);
}


// A group of G lanes, one cell of 2 <= n_c <= G R super-droplets per group (n_c = 0: the group idles along).
// Returns this lane's share of the number of zero multiplicities the cell holds AFTER the step.  The hot flow is
// straight-line code: loads, Philox blocks (computed for padding slots too, so the R chains interleave), sort and
// the first-level pair test are predicated, not branched.
// FULL: every group of the warp has n_c == G R (no padding, no guards); the caller branches warp-uniformly.
template <int KIND, int HYB, int G, int R, bool FULL, int RS>
__device__ __forceinline__ u32 group_cells(const FusedArgs& a, const PhiloxStep& ps, WarpStage<RS>& st, const u32 start,
                                           const u32 n_c_in, const int lane) {
    constexpr int P = G * R;
    static_assert(P <= 256, "the position takes 8 bits of the sort word");
    static_assert(R <= RS && R % 2 == 0, "the warp's cells fit the staging tile; pairs never straddle two lanes");
    const u32 n_c = FULL ? (u32)P : n_c_in;
    const PairArgs& pa = a.pair;
    const int lg = lane & (G - 1);
    const u32 cbase = (u32)(lane / G) * (u32)P;  // this cell's slice of the staging arrays
    u32 zeros = 0;
    // ---- a1 + load: striped positions e = G r + lg (coalesced within the cell); the fp32 side values and Philox
    //      word 3 are parked in shared memory, the sort word stays in registers ----
    u32 x[R];
    const int drop = 32 - a.key_bits;
    constexpr int LB = R % 4 == 0 ? 4 : (R % 3 == 0 ? 3 : 2);  // loads in flight per lane and batch (8 measured the same)
#pragma unroll
    for (int b = 0; b < R; b += LB) {
        u32 idx[LB];
        long long xi[LB];
        double vol[LB];
#pragma unroll
        for (int t = 0; t < LB; ++t) {
            const u32 e = (u32)(b + t) * G + lg;
            idx[t] = 0; xi[t] = 1; vol[t] = 0.0;
            if (FULL || e < n_c) {
                idx[t] = run_index<HYB>(a, start, e);
                const u32 at = attr_index<HYB>(start, e, idx[t]);
                xi[t] = pa.xi[at];
                vol[t] = pa.v[at];
            }
        }
#pragma unroll
        for (int t = 0; t < LB; ++t) {
            const u32 e = (u32)(b + t) * G + lg;
            // keys first: Philox needs only the index, so the attribute loads stay in flight under it
            const PhiloxOut w = philox4x32_10(pa.pk, ps, (u64)idx[t]);
            // padding sorts to the end (a real word with the same upper bits has a smaller position) and keeps a
            // position inside the cell's staging slice, so that the unguarded reads of the pair test stay in bounds
            x[b + t] = (FULL || e < n_c) ? (((w.w0 >> drop) << 8) | e) : (0xFFFFFF00u | e);
            const float xf = __ll2float_ru(xi[t]);  // 0 -> 0.0f, xi >= 1 -> >= 1.0f (padding slots hold xi = 1)
            zeros += (xf == 0.0f);
            if (FULL || e < n_c) {
                st.fl[cbase + e] = make_float2(xf, __double2float_ru(vol[t]));
                st.w3[cbase + e] = w.w3;
            }
        }
    }
    // ---- a3: sort (truncated key, position) words; slot s = lg R + r afterwards ----
    group_bitonic_sort<R, G>(x, lg);
    // neighbours with equal truncated keys: their order is decided by the dropped bits -> repair
    u32 ties = 0xFFFFFFFFu;  // smallest XOR of two neighbouring words that are both real
    const u32 nxt = __shfl_down_sync(0xffffffffu, x[0], 1);
#pragma unroll
    for (int r = 0; r + 1 < R; ++r)
        if (FULL || (u32)(lg * R + r + 1) < n_c) ties = min(ties, x[r] ^ x[r + 1]);
    if (lg < G - 1 && (FULL || (u32)(lg * R + R) < n_c)) ties = min(ties, x[R - 1] ^ nxt);
    __syncwarp();  // the staging writes of all lanes are visible from here on
    // (out of line -- one copy per words-per-lane instead of one per size class -- the repair was measured 2 % slower on
    // configs[3] and 2 % faster on configs[4]: the call pins registers around it in the whole kernel)
    if (__any_sync(0xffffffffu, ties < 0x100u)) repair_ties<HYB, G, R>(a, ps, x, start, n_c, lg);
    if (a.dbg_perm) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const u32 s = lg * R + r;
            if (s < n_c) a.dbg_perm[start + s] = (int32_t)run_index<HYB>(a, start, x[r] & 0xFFu);
        }
    }
    // ---- a4, level 1: every pair of neighbouring slots -- a dozen fp32 operations decide "gamma = 0 for sure" ----
    constexpr int NP = R / 2;
    u32 need = 0;  // bit q: pair q of this lane goes on to the exact levels
    const float cscale = pa.cheap_c * (float)pair_scale_int(n_c);
    const bool dbg = pa.dbg_gamma != nullptr;
#pragma unroll
    for (int q = 0; q < NP; ++q) {
        const u32 ea = x[2 * q] & 0xFFu, eb = x[2 * q + 1] & 0xFFu;  // run positions of the pair's members, shuffled order
        const bool valid = FULL || (u32)(lg * R + 2 * q + 1) < n_c;
        // (slots past n_c hold padding positions: the staged values read there are unspecified, `valid` drops them)
        const float2 A = st.fl[cbase + ea], B = st.fl[cbase + eb];
        const u32 w3a = st.w3[cbase + ea];
        // a dead partner (xi = 0 rounds up to 0.0f, xi >= 1 to >= 1.0f): gamma~ = 0 whatever gamma is (R7)
        const bool alive = fminf(A.x, B.x) != 0.0f;
        const bool may = pair_cheap_may_collide<KIND>(cscale, fmaxf(A.x, B.x), A.y, B.y, w3a);
        if (valid && (dbg || (alive && may))) need |= 1u << q;
    }
    // ---- levels 2 and 3: the fp32 interval bound and the full fp64 rule, only where needed; lanes take
    //      their pending pairs one at a time and read the exact attributes again ----
    while (__any_sync(0xffffffffu, need != 0)) {
        if (need) {
            const int q = __ffs(need) - 1;
            need &= need - 1u;
            const u32 ea = select_reg<R>(x, 2 * q) & 0xFFu, eb = select_reg<R>(x, 2 * q + 1) & 0xFFu;
            const u32 ja = run_index<HYB>(a, start, ea), jb = run_index<HYB>(a, start, eb);
            const u32 ta = attr_index<HYB>(start, ea, ja), tb = attr_index<HYB>(start, eb, jb);
            const long long xa = pa.xi[ta], xb = pa.xi[tb];
            const double va = pa.v[ta], vb = pa.v[tb];
            const bool swap = xa < xb;
            // w2 = 0 makes u a lower bound of the true uniform: the test stays conservative
            if (dbg || pair_may_collide(pa, swap ? xb : xa, swap ? vb : va, swap ? va : vb, 0u, st.w3[cbase + ea], n_c)) {
                const PhiloxOut w = philox4x32_10(pa.pk, ps, (u64)ja);  // the exact uniform of the first member (R2)
                // (a resident run has no debug outputs, the only other use of the first index)
                zeros += pair_apply(pa, ta, tb, xa, va, xb, vb, w.w2, w.w3, n_c);
            }
        }
    }
    return zeros;
}

// The warp's 32 / G cells of size class P = G R: cells [wfirst * 32 / G, ...) of the class list.
template <int KIND, int HYB, int G, int R, int RS>
__device__ __forceinline__ u32 class_cells(const FusedArgs& a, const PhiloxStep& ps, WarpStage<RS>& st,
                                           const u32* __restrict__ list, u32 count, u32 wfirst, int lane) {
    constexpr int P = G * R;
    const u32 ci = wfirst * (u32)(32 / G) + (u32)(lane / G);
    u32 start = 0, n_c = 0;
    if (ci < count) {
        const u32 c = list ? __ldg(list + ci) : ci + a.cell_offset;
        start = __ldg(a.pair.cell_start + c);
        n_c = __ldg(a.pair.cell_start + c + 1) - start;
    }
    u32 zeros = 0;
    if (n_c == 1 && (lane & (G - 1)) == 0) {  // nothing to pair; a lone super-droplet still counts as a zero when its multiplicity is 0
        const u32 i = run_index<HYB>(a, start, 0);
        zeros = (a.pair.xi[attr_index<HYB>(start, 0, i)] == 0);
        if (a.dbg_perm) a.dbg_perm[start] = (int32_t)i;
    }
    if (n_c > (u32)P) {  // unreachable: k_cell_bounds refuses such cells and the lists follow its classes
        a.sticky[STICKY_BAD_DATA] = 1u;
        n_c = 0;
    }
    if (n_c < 2) n_c = 0;
    if (!__any_sync(0xffffffffu, n_c != 0)) return zeros;
    // regular grids fill their slots exactly (configs[2], [3]: 32 and 128 per cell): that case runs without guards
    // (the odd classes do without that variant: it is 4 % faster on exactly full tiles and as much code again)
    if constexpr (R != CELL_ODD_WORDS) {
        if (__all_sync(0xffffffffu, n_c == (u32)P)) return zeros + group_cells<KIND, HYB, G, R, true, RS>(a, ps, st, start, n_c, lane);
    }
    return zeros + group_cells<KIND, HYB, G, R, false, RS>(a, ps, st, start, n_c, lane);
}

template <int KIND, int HYB, int R>
__global__ void __launch_bounds__(CF_BLOCK, CF_MIN_BLOCKS) k_cell_fused(const __grid_constant__ FusedArgs a) {
    constexpr int RS = R < CELL_ODD_WORDS ? CELL_ODD_WORDS : R;  // the odd classes hold 6 words per lane
    __shared__ WarpStage<RS> s_stage[CF_WARPS];
    if (a.ctl[CTL_UNSORTED] == a.epoch) return;  // k_cell_bounds refused the input: the step is skipped as a whole
    if (a.halt_tag) {  // a step of sdm_coalescence_steps: a halted run stays halted until the host has compacted
        const u32 halted = a.run[RUN_HALT];
        const u32 due_zeros = a.zc_check ? *a.zc_check : 0u;
        if (halted | due_zeros) {
            if (!halted && blockIdx.x == 0 && threadIdx.x == 0) {
                a.run[RUN_HALT] = a.halt_tag;
                a.mapped[MAPPED_ZEROS] = due_zeros;
                __threadfence_system();
                a.mapped[MAPPED_HALT] = a.halt_tag;
            }
            return;
        }
    }
    if (a.zc_clear && blockIdx.x == 0 && threadIdx.x == 0) *a.zc_clear = 0u;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpStage<RS>& st = s_stage[warp];
    // blocks are dealt out class by class, one launch wave after another: the block scheduler balances the
    // (data-dependent) cost of the cells; a persistent strided loop measured 12 % slower on cfg3
    // (with several classes in the launch the block ranges are taken from the back, the largest cells first: the last
    // wave then consists of the cheapest blocks -- cfg4 85.7 -> 84.3 us)
    const u32 bid = a.only_class == (u32)CELL_CLASSES ? gridDim.x - 1u - blockIdx.x : blockIdx.x;
    // (a warp lives for two cells of configs[3], 1400 instructions: the search over the classes is skipped when the
    // launch holds one class only -- the prologue of a warp is 6 % of the kernel's instructions)
    u32 cls = a.only_class, bfirst = 0;
    if (a.only_class == (u32)CELL_CLASSES) {
        cls = 0;
#pragma unroll
        for (u32 k = 0; k + 1 < (u32)CELL_CLASSES; ++k)
            if (bid >= a.class_block_end[k]) { cls = k + 1; bfirst = a.class_block_end[k]; }
    }
    const u32 wfirst = (bid - bfirst) * CF_WARPS + warp;
    // n_steps > 1 (a run without compactions, sdm_coalescence_steps): cells never interact, so the warp takes its cells
    // through all the steps of the launch by itself -- their attributes come back from L1 / L2, and no kernel boundary
    // (ramp, tail, launch) separates two steps of a small problem
    // (only the R = 4 kernels, the ones small problems run, carry the loop: in the R = 8 kernels its live values cost
    // spills -- configs[4] 93 -> 103 us)
    constexpr bool MULTI = FUSED_MULTI_STEP(R);
    const u64 step0 = ((u64)a.pair.pk.step_hi << 32) | (u64)a.pair.pk.step_lo;
    const u32 n_steps = MULTI ? a.n_steps : 1u;
    u32 zeros = 0;
    for (u32 s = 0; s < n_steps; ++s) {
        PhiloxStep ps;
        if constexpr (MULTI) {
            ps = make_philox_step(step0 + (u64)s);
        } else {
            ps.step_hi = a.pair.pk.step_hi;
            ps.p1_lo = a.pair.pk.p1_lo;
            ps.p1_hi = a.pair.pk.p1_hi;
        }
        // class k: P = class_slots(k) slots per cell; even classes on G = P / R lanes of R words, odd ones on P / 6 lanes of 6
#define SDM_EVEN_CLASS(K)                                                                                              \
    if constexpr (class_lanes(K, R) >= 2 && class_lanes(K, R) <= 32)                                                   \
        zeros = class_cells<KIND, HYB, class_lanes(K, R), R, RS>(a, ps, st, a.class_cells[K], a.class_count[K], wfirst, lane)
#define SDM_ODD_CLASS(K)                                                                                               \
    zeros = class_cells<KIND, HYB, class_lanes(K, R), CELL_ODD_WORDS, RS>(a, ps, st, a.class_cells[K], a.class_count[K], wfirst, lane)
        switch (cls) {
            case 0: SDM_EVEN_CLASS(0); break;
            case 1: SDM_ODD_CLASS(1); break;
            case 2: SDM_EVEN_CLASS(2); break;
            case 3: SDM_ODD_CLASS(3); break;
            case 4: SDM_EVEN_CLASS(4); break;
            case 5: SDM_ODD_CLASS(5); break;
            default: SDM_EVEN_CLASS(6); break;
        }
#undef SDM_EVEN_CLASS
#undef SDM_ODD_CLASS
        __syncwarp();  // the next step's loads (other lanes) see this step's updates; the staging tile is free again
    }
    // a5, fused: the number of zero multiplicities after the (last) step (sdm_remove_zero_multiplicity reads it)
    zeros = __reduce_add_sync(0xffffffffu, zeros);
    if (lane == 0 && zeros) atomicAdd(a.zc_accum, zeros);
}

// src_kind: 0 = cell_id array itself (CELL_SORTED), 1 = u64 sorted words, 2 = u32 sorted words (HYBRID).
// strict: a refusal also raises the sticky SDM_ERR_BAD_DATA.  Two launches: the streaming boundary kernel over the
// super-droplets, then the per-cell class kernel that publishes the verdict.
cudaError_t launch_cell_bounds(sdm_ctx* ctx, int src_kind, const void* src, int64_t n_sd, int32_t n_cell,
                               int idxbits, bool strict) {
    const long long n_chunks = (n_sd + CB_CHUNK - 1) / CB_CHUNK;
    const long long resident = (long long)ctx->sm_count * 8;
    const u32 grid = (u32)(n_chunks < resident ? n_chunks : resident);
    Workspace& ws = ctx->ws;
    const bool vec = (reinterpret_cast<uintptr_t>(src) & 15u) == 0;
    {
        LaunchScope scope(ctx, PROF_CELL_BOUNDS);
#define SDM_BOUNDS(SRC, VEC, IDXBITS)                                                                                   \
    k_cell_bounds<SRC, VEC><<<grid, CB_BLOCK, 0, ctx->stream>>>(src, (u32)n_sd, n_cell, IDXBITS, ws.cell_start, ws.ctl, \
                                                                ws.run, ctx->dbg_cell_start)
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
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    LaunchScope scope(ctx, PROF_CELL_CLASSES);
    k_cell_classes<<<(n_cell + 255) / 256, 256, 0, ctx->stream>>>(ws.cell_start, n_cell, strict ? 1u : 0u, ctx->epoch, ws.ctl,
                                                                  ws.sticky, ws.run, ctx->mapped, ws.class_list,
                                                                  (u32)ctx->max_n_cell);
    return cudaGetLastError();
}

// No shared-memory carve-out preference is set for the fused kernel: it needs 6-12 KB per block, and with the L1
// squeezed to its minimum (the round-1 setting) a warp's scattered gathers on the HYBRID path ran out of lines to
// allocate for pending misses -- 444 us instead of 178 us on interleaved configs[3] (profiles/r2b_README.md).
cudaError_t init_cell_fused(sdm_ctx*) { return cudaSuccess; }

template <int R>
static void launch_fused_r(const FusedArgs& a, int hyb, u32 grid, cudaStream_t st) {
    const bool golovin = a.pair.kp.kind == 0;
    if (golovin && hyb == 0) k_cell_fused<0, 0, R><<<grid, CF_BLOCK, 0, st>>>(a);
    else if (golovin && hyb == 1) k_cell_fused<0, 1, R><<<grid, CF_BLOCK, 0, st>>>(a);
    else if (golovin) k_cell_fused<0, 2, R><<<grid, CF_BLOCK, 0, st>>>(a);
    else if (hyb == 0) k_cell_fused<1, 0, R><<<grid, CF_BLOCK, 0, st>>>(a);
    else if (hyb == 1) k_cell_fused<1, 1, R><<<grid, CF_BLOCK, 0, st>>>(a);
    else k_cell_fused<1, 2, R><<<grid, CF_BLOCK, 0, st>>>(a);
}

// A resident HYBRID run (sdm_coalescence_steps): the attributes are gathered ONCE into cell-grouped copies, every step
// of the run then streams them like the CELL_SORTED path (the gather through the index words costs 180 us per step on
// interleaved configs[3], the coalesced step 70 us), and they are scattered back when the run ends or halts.
template <typename TW, bool BACK>
__global__ void __launch_bounds__(256) k_resident_move(const TW* __restrict__ words, TW idx_mask, u32 n_sd,
                                                        long long* __restrict__ xi, double* __restrict__ v,
                                                        long long* __restrict__ res_xi, double* __restrict__ res_v) {
    constexpr int U = 4;  // independent random accesses in flight per thread
    const u32 stride = gridDim.x * 256u * U;
    for (u32 p0 = blockIdx.x * 256u * U + threadIdx.x; p0 < n_sd; p0 += stride) {
        u32 i[U];
        long long x[U];
        double w[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const u32 p = p0 + (u32)u * 256u;
            i[u] = p < n_sd ? (u32)(words[p] & idx_mask) : 0u;
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const u32 p = p0 + (u32)u * 256u;
            if (p < n_sd) {
                x[u] = BACK ? res_xi[p] : xi[i[u]];
                w[u] = BACK ? res_v[p] : v[i[u]];
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const u32 p = p0 + (u32)u * 256u;
            if (p < n_sd) {
                if (BACK) {
                    xi[i[u]] = x[u];
                    v[i[u]] = w[u];
                } else {
                    res_xi[p] = x[u];
                    res_v[p] = w[u];
                }
            }
        }
    }
}

cudaError_t launch_resident_move(sdm_ctx* ctx, bool back, int src_kind, const void* run_idx, int idxbits, int64_t* xi,
                                 double* v, int64_t n_sd) {
    LaunchScope scope(ctx, PROF_RESIDENT_MOVE);
    const u32 need = (u32)((n_sd + 1023) / 1024);
    const u32 cap = (u32)ctx->sm_count * 8u;
    const u32 grid = need < cap ? need : cap;
    long long* x = reinterpret_cast<long long*>(xi);
    long long* rx = reinterpret_cast<long long*>(ctx->ws.res_xi);
    double* rv = ctx->ws.res_v;
    const u64 mask = (1ull << idxbits) - 1ull;
    if (src_kind == 2) {
        const u32* w = reinterpret_cast<const u32*>(run_idx);
        if (back) k_resident_move<u32, true><<<grid, 256, 0, ctx->stream>>>(w, (u32)mask, (u32)n_sd, x, v, rx, rv);
        else k_resident_move<u32, false><<<grid, 256, 0, ctx->stream>>>(w, (u32)mask, (u32)n_sd, x, v, rx, rv);
    } else {
        const u64* w = reinterpret_cast<const u64*>(run_idx);
        if (back) k_resident_move<u64, true><<<grid, 256, 0, ctx->stream>>>(w, mask, (u32)n_sd, x, v, rx, rv);
        else k_resident_move<u64, false><<<grid, 256, 0, ctx->stream>>>(w, mask, (u32)n_sd, x, v, rx, rv);
    }
    return cudaGetLastError();
}

// Words per lane of the group sort.  8 costs fewer instructions per super-droplet (more of the bitonic stages stay
// inside the lanes); small problems, whose warps would not fill the machine then, take 4 (configs[2]: 10.6 us
// against 11.8 us).  Cells of more than 192 entries need 8 (32 lanes x 8 words).
int fused_words_per_lane(const sdm_ctx* ctx, const CellClasses& cc) {
    if (cc.worst == (u32)CELL_CLASSES - 1 || ctx->fused_r == 8) return 8;
    if (ctx->fused_r == 4) return 4;
    long long slots = 0;
    for (int k = 0; k < CELL_CLASSES; ++k) slots += (long long)cc.count[k] * class_slots(k);
    return slots / (32 * 8) >= (long long)ctx->sm_count * 32 ? 8 : 4;
}

bool fused_multi_step(const sdm_ctx* ctx, const CellClasses& cc) { return FUSED_MULTI_STEP(fused_words_per_lane(ctx, cc)); }

cudaError_t launch_cell_fused(sdm_ctx* ctx, int src_kind, const void* run_idx, int idxbits, const CellClasses& cc,
                              int64_t* xi, double* v, int64_t n_sd, int32_t n_cell, double dtdV, const KernelParams& kp,
                              const PhiloxKeys& pk, const StepLinks& links) {
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
    a.cell_offset = cc.mixed ? 0u : cc.cell_offset;
    a.n_steps = links.n_steps ? links.n_steps : 1u;
    if (a.n_steps > 1u && !fused_multi_step(ctx, cc)) return cudaErrorInvalidValue;
    a.key_bits = ctx->narrow_key_bits;
    a.run_idx = run_idx;
    a.run_u32 = src_kind == 2;
    a.idx_mask = (idxbits >= 64) ? ~0ull : ((1ull << idxbits) - 1ull);
    a.dbg_perm = ctx->dbg_perm;
    a.sticky = ctx->ws.sticky;
    a.ctl = ctx->ws.ctl;
    a.epoch = ctx->epoch;
    a.zc_accum = links.zc_accum ? links.zc_accum : ctx->ws.ctl + CTL_ZERO_COUNT;
    a.zc_check = links.zc_check;
    a.zc_clear = links.zc_clear;
    a.halt_tag = links.halt_tag;
    a.run = ctx->ws.run;
    a.mapped = ctx->mapped;
    const int R = fused_words_per_lane(ctx, cc);
    u32 blocks = 0;
    int n_used = 0;
    a.only_class = (u32)CELL_CLASSES;
    for (int k = 0; k < CELL_CLASSES; ++k) {
        const u32 cells_per_block = (u32)CF_WARPS * 32u / (u32)class_lanes(k, R);  // CF_WARPS * 32 / G
        const u32 before = blocks;
        a.class_count[k] = cc.count[k];
        a.class_cells[k] = cc.mixed ? ctx->ws.class_list + (size_t)k * (size_t)ctx->max_n_cell : nullptr;
        blocks += (cc.count[k] + cells_per_block - 1) / cells_per_block;
        a.class_block_end[k] = blocks;
        if (blocks > before) { a.only_class = n_used ? (u32)CELL_CLASSES : (u32)k; ++n_used; }
    }
    if (blocks == 0) return cudaSuccess;
    LaunchScope scope(ctx, PROF_CELL_FUSED);
    const int hyb = src_kind == 0 ? 0 : (links.resident ? 2 : 1);
    if (R == 4) launch_fused_r<4>(a, hyb, blocks, ctx->stream);
    else launch_fused_r<8>(a, hyb, blocks, ctx->stream);
    return cudaGetLastError();
}

}  // namespace sdm
