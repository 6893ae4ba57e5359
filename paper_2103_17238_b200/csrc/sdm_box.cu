// The whole coalescence step of a small box (one cell, n_sd <= BOX_MAX super-droplets) in ONE launch of ONE block
// ("includes the single-CTA fused step for tiny N"; configs[0], the paper's own box example,
// PAPER.md:48-53, 73-75).  The GENERAL path needs five dependent launches for such a step and is bound by their
// latencies (44 us per step for 8192 super-droplets); here rows a1, a3 and a4 run back to back out of shared memory:
//
//   a1  every thread generates the Philox keys of its BOX_ITEMS super-droplets (kept in registers);
//   a3  the keys are uniform 32-bit numbers, so a counting placement replaces the comparison network: bucket = the top
//       key bits (about 4 super-droplets per bucket), one shared-memory atomic per super-droplet gives its slot
//       inside the bucket, an exclusive scan of the bucket counts gives the bucket starts, the 46-bit words
//       (key << 14 | index) are scattered to start + slot, and every word then finds its exact place by counting the
//       smaller words of its own bucket.  The result is the ascending order of (key, index): the oracle's
//       std::stable_sort order (ties between equal keys by index), for any key distribution -- a skewed one only
//       makes the buckets longer;
//   a4  thread t takes the pairs (2p, 2p + 1), p = t, t + 1024, ...: the same pair rule as every other path
//       (pair_collide: exact early-out, Philox block of the first member regenerated).
//
// A single block cannot beat many SMs on bandwidth, but at this size nothing is bandwidth: the step is the sum of a
// few shared-memory round trips.  An earlier attempt with a bitonic network over the 8192 words in shared memory (91
// stages x 16 B per word) took 95-114 us (profiles/r1c_README.md); the counting placement touches every word a
// handful of times.
#include "sdm_internal.h"
#include "sdm_pair.cuh"

namespace sdm {

constexpr int BOX_THREADS = 1024;
constexpr int BOX_ITEMS = BOX_MAX / BOX_THREADS;  // super-droplets per thread
constexpr int BOX_IDX_BITS = 14;
constexpr int BOX_MAX_BUCKETS = 4096;
static_assert(BOX_MAX <= (1 << BOX_IDX_BITS) && BOX_ITEMS * BOX_THREADS == BOX_MAX, "box tile");

struct BoxArgs {
    PairArgs pair;
    int bucket_shift;  // bucket = key >> bucket_shift
    int n_bucket;      // 1 << (32 - bucket_shift), a multiple of 32, <= BOX_MAX_BUCKETS
    int32_t* dbg_perm;
    int32_t* dbg_cell_start;
};

__global__ void __launch_bounds__(BOX_THREADS, 1) k_box_step(const __grid_constant__ BoxArgs a) {
    extern __shared__ u64 s_words[];                  // [n_sd] (key << 14 | index), bucket by bucket
    __shared__ u32 s_count[BOX_MAX_BUCKETS];          // bucket counts, then bucket starts
    __shared__ u32 s_warp[BOX_THREADS / 32];
    const u32 n = a.pair.n_sd;
    unsigned short* s_idx = reinterpret_cast<unsigned short*>(s_words + n);  // [n_sd] indices in shuffled order
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int b = tid; b < a.n_bucket; b += BOX_THREADS) s_count[b] = 0u;
    __syncthreads();
    // ---- a1 + bucket histogram ----
    u32 key[BOX_ITEMS], slot[BOX_ITEMS];
#pragma unroll
    for (int k = 0; k < BOX_ITEMS; ++k) {
        const u32 i = (u32)tid + (u32)k * BOX_THREADS;
        key[k] = philox_perm_key(a.pair.pk, (u64)i);  // computed for every slot: the chains of a thread interleave
        slot[k] = 0;
        if (i < n) slot[k] = atomicAdd(&s_count[key[k] >> a.bucket_shift], 1u);
    }
    __syncthreads();
    // ---- exclusive scan of the bucket counts (n_bucket / 1024 consecutive buckets per thread, at most 4) ----
    {
        const int per = a.n_bucket / BOX_THREADS;  // 0 when there are fewer buckets than threads
        u32 c[BOX_MAX_BUCKETS / BOX_THREADS];
        u32 sum = 0;
        if (per == 0) {
            c[0] = tid < a.n_bucket ? s_count[tid] : 0u;
            sum = c[0];
        } else {
#pragma unroll
            for (int j = 0; j < BOX_MAX_BUCKETS / BOX_THREADS; ++j) {
                c[j] = j < per ? s_count[tid * per + j] : 0u;
                sum += c[j];
            }
        }
        u32 incl = sum;
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
            s_warp[lane] = wi - w;
        }
        __syncthreads();
        u32 run = s_warp[warp] + incl - sum;
        if (per == 0) {
            if (tid < a.n_bucket) s_count[tid] = run;
        } else {
#pragma unroll
            for (int j = 0; j < BOX_MAX_BUCKETS / BOX_THREADS; ++j) {
                if (j < per) s_count[tid * per + j] = run;
                run += c[j];
            }
        }
    }
    __syncthreads();
    // ---- scatter into the buckets (arrival order inside a bucket) ----
#pragma unroll
    for (int k = 0; k < BOX_ITEMS; ++k) {
        const u32 i = (u32)tid + (u32)k * BOX_THREADS;
        if (i < n) s_words[s_count[key[k] >> a.bucket_shift] + slot[k]] = ((u64)key[k] << BOX_IDX_BITS) | (u64)i;
    }
    __syncthreads();
    // ---- exact place inside the bucket: the number of smaller words among its members ----
    // (a thread takes the words at positions tid, tid + 1024, ...: neighbouring lanes sit in the same or in
    //  neighbouring buckets, so a warp's loops are about equally long)
    for (u32 p = tid; p < n; p += BOX_THREADS) {
        const u64 mine = s_words[p];
        const u32 b = (u32)(mine >> (BOX_IDX_BITS + a.bucket_shift));
        const u32 lo = s_count[b], hi = (b + 1 < (u32)a.n_bucket) ? s_count[b + 1] : n;
        u32 smaller = 0;
        for (u32 q = lo; q < hi; ++q) smaller += (s_words[q] < mine);
        s_idx[lo + smaller] = (unsigned short)(mine & ((1u << BOX_IDX_BITS) - 1u));
    }
    __syncthreads();
    if (a.dbg_perm)
        for (u32 p = tid; p < n; p += BOX_THREADS) a.dbg_perm[p] = (int32_t)s_idx[p];
    if (a.dbg_cell_start && tid == 0) {
        a.dbg_cell_start[0] = 0;
        a.dbg_cell_start[1] = (int32_t)n;
    }
    // ---- a4: pairs of neighbours in the shuffled order ----
    for (u32 p = tid; 2u * p + 1u < n; p += BOX_THREADS) pair_collide(a.pair, (u32)s_idx[2u * p], (u32)s_idx[2u * p + 1u], n);
}

cudaError_t init_box_step(sdm_ctx*) {
    return cudaFuncSetAttribute(k_box_step, cudaFuncAttributeMaxDynamicSharedMemorySize, BOX_MAX * 10);
}

cudaError_t launch_box_step(sdm_ctx* ctx, int64_t* xi, double* v, int64_t n_sd, double dtdV, const KernelParams& kp,
                            const PhiloxKeys& pk) {
    BoxArgs a;
    a.pair.sorted = nullptr;
    a.pair.xi = reinterpret_cast<long long*>(xi);
    a.pair.v = v;
    a.pair.cell_start = nullptr;
    a.pair.n_sd = (u32)n_sd;
    a.pair.idxbits = 0;
    a.pair.cshift = 0;
    a.pair.single_cell = 1;
    a.pair.dtdV = dtdV;
    a.pair.kp = kp;
    set_bound_constants(a.pair);
    a.pair.pk = pk;
    a.pair.dbg_gamma = reinterpret_cast<long long*>(ctx->dbg_gamma);
    a.pair.dbg_gamma_clamped = reinterpret_cast<long long*>(ctx->dbg_gamma_clamped);
    // about four super-droplets per bucket; at least one warp's worth of buckets
    int bits = 5;
    while ((1 << bits) * 4 < n_sd && (1 << bits) < BOX_MAX_BUCKETS) ++bits;
    a.bucket_shift = 32 - bits;
    a.n_bucket = 1 << bits;
    a.dbg_perm = ctx->dbg_perm;
    a.dbg_cell_start = ctx->dbg_cell_start;
    LaunchScope scope(ctx, PROF_BOX_STEP);
    k_box_step<<<1, BOX_THREADS, (size_t)n_sd * 10, ctx->stream>>>(a);
    return cudaGetLastError();
}

}  // namespace sdm
