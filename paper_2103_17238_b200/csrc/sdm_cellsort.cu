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
//   k_cell_bounds<SRC>  reads the cell of every position once: verifies range and order, finds the largest
//                       cell's size class, writes cell_start[0..n_cell] and publishes the verdict (device flag
//                       for the fused kernel, mapped host word for AUTO's path choice).  When the input does
//                       not fit the fused kernel launched next, that kernel does nothing (the state is never
//                       half-updated).
//   k_cell_fused<W>     one warp per cell, n_c <= 32 R, R in {1,2,4,8}.  Sort word = 32 bits:
//                       (top 24 bits of the Philox key) << 8 | position-in-run, sorted by an
//                       all-ascending bitonic network (IMNMX + SHFL, 2 instructions per compare).
//                       Dropping the low 8 key bits is exact unless two neighbours of the sorted run
//                       share their top 24 bits (4.8e-4 per 128-SD cell); the warp detects that and
//                       redoes its cell with full 64-bit (key << 32 | position) words.
#include "sdm_internal.h"
#include "sdm_pair.cuh"

namespace sdm {

#ifndef SDM_CF_WARPS
#define SDM_CF_WARPS 4
#endif
#ifndef SDM_CF_MIN_BLOCKS
#define SDM_CF_MIN_BLOCKS 9
#endif
constexpr int CF_WARPS = SDM_CF_WARPS;  // tuning constants (profiles/): -DSDM_CF_WARPS / -DSDM_CF_MIN_BLOCKS via SDM_NVCC_EXTRA
constexpr int CF_BLOCK = CF_WARPS * 32;
constexpr int CF_MIN_BLOCKS = SDM_CF_MIN_BLOCKS;
constexpr int CB_BLOCK = 256;
constexpr int CB_K = 4;                         // quads (4 positions, one 16-byte load for int32 sources) per thread and iteration
constexpr int CB_CHUNK = CB_BLOCK * CB_K * 4;   // positions per block and iteration

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

// Position i opens cell cc and closes cell prev (opening every empty cell in between).  The closed cell
// [s, i) holds more than m entries exactly when position i - 1 - m still belongs to it (sorted input), so its
// size class costs up to three extra loads per cell, not per super-droplet.  Returns the size class of the
// closed cell: 0 (<= 64), 1 (<= 128), 2 (<= 256), 3 (larger).
template <int SRC>
__device__ __forceinline__ u32 open_cells(const void* src, int idxbits, int prev, int cc, u32 i,
                                          u32* __restrict__ cell_start, int32_t* __restrict__ dbg_cell_start) {
    for (int q = prev + 1; q <= cc; ++q) {
        cell_start[q] = i;
        if (dbg_cell_start) dbg_cell_start[q] = (int32_t)i;
    }
    if (prev < 0) return 0;
    u32 cls = 0;
    if (i > 64u && cell_at<SRC>(src, i - 65u, idxbits) == prev) {
        cls = 1;
        if (i > 128u && cell_at<SRC>(src, i - 129u, idxbits) == prev) {
            cls = 2;
            if (i > 256u && cell_at<SRC>(src, i - 257u, idxbits) == prev) cls = 3;
        }
    }
    return cls;
}

template <int SRC, bool VEC>
__global__ void __launch_bounds__(CB_BLOCK)
k_cell_bounds(const void* __restrict__ src, u32 n_sd, int n_cell, int idxbits, u32 max_class, u32 strict, u32 epoch,
              u32* __restrict__ cell_start, u32* __restrict__ ctl, u32* __restrict__ sticky, u32* __restrict__ run,
              volatile u32* __restrict__ mapped, int32_t* __restrict__ dbg_cell_start) {
    __shared__ u32 s_cls;
    // the fused kernel that follows accumulates the zero count; no separate memset of the control block
    if (blockIdx.x == 0 && threadIdx.x == 0) ctl[CTL_ZERO_COUNT] = 0u;
    if (threadIdx.x == 0) s_cls = 0u;
    const int lane = threadIdx.x & 31;
    bool bad = false;
    u32 cls = 0;
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
                        if (c[k][j] != p)
                            cls = max(cls, open_cells<SRC>(src, idxbits, p, c[k][j], i0 + j, cell_start, dbg_cell_start));
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
                            if (cc != prev)
                                cls = max(cls, open_cells<SRC>(src, idxbits, prev, cc, i, cell_start, dbg_cell_start));
                            if (i == n_sd - 1)  // the array end closes cell cc and opens the (empty) rest
                                cls = max(cls, open_cells<SRC>(src, idxbits, cc, n_cell, n_sd, cell_start, dbg_cell_start));
                        }
                        prev = cc;
                    }
                }
            }
        }
    }
    if (bad) cls = 3;  // out of range or out of order: refused like a cell that is too large
    cls = __reduce_max_sync(0xffffffffu, cls);
    __syncthreads();
    if (lane == 0 && cls) atomicMax(&s_cls, cls);
    __syncthreads();
    if (threadIdx.x == 0) {
        if (s_cls) atomicMax(&run[RUN_BOUNDS_CLASS], s_cls);
        __threadfence();
        const u32 t = atomicAdd(&run[RUN_BOUNDS_TICKET], 1u);
        if (t == gridDim.x - 1) {  // the last block: every other block's class is visible (fence + ticket)
            __threadfence();
            const u32 worst = atomicExch(&run[RUN_BOUNDS_CLASS], 0u);
            run[RUN_BOUNDS_TICKET] = 0u;
            const bool refuse = worst > max_class;
            if (refuse) {  // the step is skipped as a whole and reported
                ctl[CTL_UNSORTED] = epoch;  // tagged with this step's epoch: stale refusals never match
                if (strict) sticky[STICKY_BAD_DATA] = 1u;
            }
            mapped[MAPPED_VERDICT_CLASS] = worst;
            __threadfence_system();
            mapped[MAPPED_VERDICT_EPOCH] = epoch;
        }
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
// Two 16-byte stores per super-droplet: the exact attributes, and the fp32 side values of the cheap early-out.
template <int WORD, int RMAX>
struct CellStage {
    longlong2 xv[32 * RMAX];  // (multiplicity, volume bits)
    float4 aux[32 * RMAX];    // {xi rounded UP to fp32, v rounded UP to fp32, Philox word 3 (bits), Philox key (bits)}
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

// One warp, one cell of 2 <= n_c <= 32 R super-droplets.  Returns this lane's share of the number of zero
// multiplicities the cell holds AFTER the step.  The hot flow is straight-line code: loads, Philox blocks (computed
// for padding slots too, so the R chains interleave), sort and the first-level pair test are predicated, not branched.
// FULL: n_c == 32 R (every slot holds a super-droplet: no padding, no guards); the caller branches warp-uniformly.
template <int WORD, int RMAX, int R, int KIND, bool FULL>
__device__ __forceinline__ u32 warp_cell(const FusedArgs& a, CellStage<WORD, RMAX>& st, u32 start, u32 n_c_in, int lane) {
    static_assert(R <= RMAX, "register tile within the staging tile");
    const u32 n_c = FULL ? 32u * R : n_c_in;
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
    u32 x[R], w3[R], key[R];
    const int drop = 32 - a.key_bits;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const u32 e = 32u * r + lane;
        const PhiloxOut w = philox4x32_10(pa.pk, (u64)idx[r]);
        w3[r] = w.w3; key[r] = w.w0;
        // padding sorts to the end (a real word with the same upper bits has a smaller position) and keeps a
        // position inside the staging tile, so that the unguarded reads of the pair test stay in bounds
        x[r] = (e < n_c) ? (((w.w0 >> drop) << 8) | e) : (0xFFFFFF00u | e);
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const u32 e = 32u * r + lane;
        const float xf = __ll2float_ru(xi[r]);  // 0 -> 0.0f, xi >= 1 -> >= 1.0f (padding slots hold xi = 1)
        zeros += (xf == 0.0f);
        if (e < n_c) {
            st.xv[e] = make_longlong2(xi[r], __double_as_longlong(vol[r]));
            st.aux[e] = make_float4(xf, __double2float_ru(vol[r]), __uint_as_float(w3[r]), __uint_as_float(key[r]));
            if (WORD != 0) st.idx[e] = idx[r];
        }
    }
    // ---- a3: sort (truncated key, position) words; slot s = lane R + r afterwards ----
    warp_bitonic_sort<u32, R>(x, lane);
    // neighbours with equal truncated keys: their order is decided by the dropped bits -> wide redo
    u32 ties = 0xFFFFFFFFu;  // smallest XOR of two neighbouring words that are both real
    const u32 nxt = __shfl_down_sync(0xffffffffu, x[0], 1);
    if (FULL) {  // a full tile has no padding
#pragma unroll
        for (int r = 0; r + 1 < R; ++r) ties = min(ties, x[r] ^ x[r + 1]);
        if (lane < 31) ties = min(ties, x[R - 1] ^ nxt);
    } else {
#pragma unroll
        for (int r = 0; r + 1 < R; ++r)
            if ((u32)(lane * R + r + 1) < n_c) ties = min(ties, x[r] ^ x[r + 1]);
        if (lane < 31 && (u32)(lane * R + R) < n_c) ties = min(ties, x[R - 1] ^ nxt);
    }
    __syncwarp();  // the staging writes of all lanes are visible from here on
    u32 pos[R];
    if (__any_sync(0xffffffffu, ties < 0x100u)) {
        u64 wide[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {  // the real words occupy the first n_c slots of the narrow result
            const u32 e = x[r] & 0xFFu;
            wide[r] = ((u32)(lane * R + r) < n_c) ? (((u64)__float_as_uint(st.aux[e].w) << 32) | (u64)e) : ~0ull;
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
    // ---- a4, level 1: every pair of neighbouring slots -- a dozen fp32 operations decide "gamma = 0 for sure" ----
    constexpr int NP = (R >= 2) ? R / 2 : 1;
    u32 first[NP], second[NP];  // run positions of the pair's members, in shuffled order
    u32 need = 0;               // bit q: pair q of this lane goes on to the exact levels
    const float cscale = pa.cheap_c * (float)pair_scale_int(n_c);
    const bool dbg = pa.dbg_gamma != nullptr;
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
        // (slots past n_c hold padding positions: the staged values read there are unspecified, `valid` drops them)
        const float4 A = st.aux[first[q]], B = st.aux[second[q]];
        // a dead partner (xi = 0 rounds up to 0.0f, xi >= 1 to >= 1.0f): gamma~ = 0 whatever gamma is (R7)
        const bool alive = fminf(A.x, B.x) != 0.0f;
        const bool may = pair_cheap_may_collide<KIND>(cscale, fmaxf(A.x, B.x), A.y, B.y, __float_as_uint(A.z));
        if (valid && (dbg || (alive && may))) need |= 1u << q;
    }
    // ---- levels 2 and 3: the fp32 interval bound and the full fp64 rule, only where needed; lanes take
    //      their pending pairs one at a time ----
    while (__any_sync(0xffffffffu, need != 0)) {
        if (need) {
            const int q = __ffs(need) - 1;
            need &= need - 1u;
            const u32 ea = select_reg<NP>(first, q), eb = select_reg<NP>(second, q);
            const longlong2 A = st.xv[ea], B = st.xv[eb];
            const double vA = __longlong_as_double(A.y), vB = __longlong_as_double(B.y);
            const bool swap = A.x < B.x;
            const u32 w3a = __float_as_uint(st.aux[ea].z);
            // w2 = 0 makes u a lower bound of the true uniform: the test stays conservative
            if (dbg || pair_may_collide(pa, swap ? B.x : A.x, swap ? vB : vA, swap ? vA : vB, 0u, w3a, n_c)) {
                const u32 ja = (WORD == 0) ? start + ea : st.idx[ea];
                const u32 jb = (WORD == 0) ? start + eb : st.idx[eb];
                const PhiloxOut w = philox4x32_10(pa.pk, (u64)ja);  // the exact uniform of the first member (R2)
                zeros += pair_apply(pa, ja, jb, A.x, vA, B.x, vB, w.w2, w.w3, n_c);
            }
        }
    }
    return zeros;
}

template <int WORD, int RMAX, int R, int KIND>
__device__ __forceinline__ u32 warp_cell_any(const FusedArgs& a, CellStage<WORD, RMAX>& st, u32 start, u32 n_c, int lane) {
    // regular grids fill their tiles exactly (configs[2], [3]: 32 and 128 per cell): that case runs without guards
    if (n_c == 32u * R) return warp_cell<WORD, RMAX, R, KIND, true>(a, st, start, n_c, lane);
    return warp_cell<WORD, RMAX, R, KIND, false>(a, st, start, n_c, lane);
}

template <int WORD, int RMAX, int KIND>
__global__ void __launch_bounds__(CF_BLOCK, CF_MIN_BLOCKS) k_cell_fused(const FusedArgs a) {
    __shared__ CellStage<WORD, RMAX> s_stage[CF_WARPS];
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
    CellStage<WORD, RMAX>& st = s_stage[warp];
    // one warp per cell, one launch wave after another: the block scheduler balances the (data-dependent)
    // cost of the cells; a persistent strided loop measured 12 % slower on cfg3
    const int c = blockIdx.x * CF_WARPS + warp;
    u32 zeros = 0;
    if (c < a.n_cell) {
        const u32 start = __ldg(a.pair.cell_start + c);
        const u32 n_c = __ldg(a.pair.cell_start + c + 1) - start;
        if (n_c < 2) {  // nothing to pair; a lone super-droplet still counts as a zero when its multiplicity is 0
            if (n_c == 1 && lane == 0) {
                const u32 i = run_index<WORD>(a, start, 0);
                zeros = (a.pair.xi[i] == 0);
                if (a.dbg_perm) a.dbg_perm[start] = (int32_t)i;
            }
        } else if (n_c <= 32) {
            zeros = warp_cell_any<WORD, RMAX, 1, KIND>(a, st, start, n_c, lane);
        } else if (RMAX >= 2 && n_c <= 64) {
            if constexpr (RMAX >= 2) zeros = warp_cell_any<WORD, RMAX, 2, KIND>(a, st, start, n_c, lane);
        } else if (RMAX >= 4 && n_c <= 128) {
            if constexpr (RMAX >= 4) zeros = warp_cell_any<WORD, RMAX, 4, KIND>(a, st, start, n_c, lane);
        } else if (RMAX >= 8 && n_c <= 256) {
            if constexpr (RMAX >= 8) zeros = warp_cell_any<WORD, RMAX, 8, KIND>(a, st, start, n_c, lane);
        } else if (lane == 0) {
            a.sticky[STICKY_BAD_DATA] = 1u;  // unreachable: k_cell_bounds refuses such cells
        }
    }
    // a5, fused: the number of zero multiplicities after the step (sdm_remove_zero_multiplicity reads it)
    zeros = __reduce_add_sync(0xffffffffu, zeros);
    if (lane == 0 && zeros) atomicAdd(a.zc_accum, zeros);
}

// src_kind: 0 = cell_id array itself (CELL_SORTED), 1 = u64 sorted words, 2 = u32 sorted words (HYBRID).
// rmax: register tile of the fused kernel launched next; it holds cells of up to 32 * rmax super-droplets.
cudaError_t launch_cell_bounds(sdm_ctx* ctx, int src_kind, const void* src, int64_t n_sd, int32_t n_cell,
                               int idxbits, int rmax, bool strict) {
    const long long n_chunks = (n_sd + CB_CHUNK - 1) / CB_CHUNK;
    const long long resident = (long long)ctx->sm_count * 6;
    const u32 grid = (u32)(n_chunks < resident ? n_chunks : resident);
    const u32 max_class = rmax <= 2 ? 0u : (rmax <= 4 ? 1u : 2u);
    LaunchScope scope(ctx, PROF_CELL_BOUNDS);
    Workspace& ws = ctx->ws;
    const bool vec = (reinterpret_cast<uintptr_t>(src) & 15u) == 0;
#define SDM_BOUNDS(SRC, VEC, IDXBITS)                                                                               \
    k_cell_bounds<SRC, VEC><<<grid, CB_BLOCK, 0, ctx->stream>>>(src, (u32)n_sd, n_cell, IDXBITS, max_class,          \
                                                                strict ? 1u : 0u, ctx->epoch, ws.cell_start, ws.ctl, \
                                                                ws.sticky, ws.run, ctx->mapped, ctx->dbg_cell_start)
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

// The staging tiles want the shared-memory end of the L1 split.  The attribute is per device and per function:
// it is set once per context (contexts live on one device) for every instantiation, and the result is checked.
template <int WORD, int RMAX>
static cudaError_t prefer_shared_carveout() {
    cudaError_t e = cudaFuncSetAttribute(k_cell_fused<WORD, RMAX, 0>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                         cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_cell_fused<WORD, RMAX, 1>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                cudaSharedmemCarveoutMaxShared);
}

cudaError_t init_cell_fused(sdm_ctx*) {
    cudaError_t e;
#define SDM_CARVE(W)                                                         \
    if ((e = prefer_shared_carveout<W, 2>()) != cudaSuccess) return e;       \
    if ((e = prefer_shared_carveout<W, 4>()) != cudaSuccess) return e;       \
    if ((e = prefer_shared_carveout<W, 8>()) != cudaSuccess) return e;
    SDM_CARVE(0) SDM_CARVE(1) SDM_CARVE(2)
#undef SDM_CARVE
    return cudaSuccess;
}

template <int WORD, int KIND>
static void launch_fused_kind(const FusedArgs& a, int rmax, u32 grid, cudaStream_t st) {
    if (rmax <= 2) k_cell_fused<WORD, 2, KIND><<<grid, CF_BLOCK, 0, st>>>(a);
    else if (rmax <= 4) k_cell_fused<WORD, 4, KIND><<<grid, CF_BLOCK, 0, st>>>(a);
    else k_cell_fused<WORD, 8, KIND><<<grid, CF_BLOCK, 0, st>>>(a);
}

template <int WORD>
static void launch_fused_word(const FusedArgs& a, int rmax, u32 grid, cudaStream_t st) {
    if (a.pair.kp.kind == 0) launch_fused_kind<WORD, 0>(a, rmax, grid, st);
    else launch_fused_kind<WORD, 1>(a, rmax, grid, st);
}

cudaError_t launch_cell_fused(sdm_ctx* ctx, int src_kind, const void* run_idx, int idxbits, int rmax, int64_t* xi,
                              double* v, int64_t n_sd, int32_t n_cell, double dtdV, const KernelParams& kp,
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
    a.key_bits = ctx->narrow_key_bits;
    a.run_idx = run_idx;
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
    const u32 grid = (u32)((n_cell + CF_WARPS - 1) / CF_WARPS);
    LaunchScope scope(ctx, PROF_CELL_FUSED);
    if (src_kind == 0) launch_fused_word<0>(a, rmax, grid, ctx->stream);
    else if (src_kind == 1) launch_fused_word<1>(a, rmax, grid, ctx->stream);
    else launch_fused_word<2>(a, rmax, grid, ctx->stream);
    return cudaGetLastError();
}

}  // namespace sdm
