// The coalescence steps of a small box (one cell, n_sd <= BOX_MAX super-droplets) in ONE launch: of one block
// (k_box_steps, described first) or of a cluster of eight blocks (k_box_cluster, further down: the default)
// ("includes the single-CTA fused step for tiny N"; configs[0], the paper's own box example,
// PAPER.md:48-53, 73-75).  The GENERAL path needs five dependent launches for such a step and is bound by their
// latencies (44 us per step for 8192 super-droplets).  Here the state (multiplicities and volumes, 128 KB) is loaded
// into shared memory once, any number of consecutive steps run out of shared memory, and the state is written back:
//
//   a1  every thread generates the Philox keys of its BOX_ITEMS super-droplets (kept in registers);
//   a3  the keys are uniform 32-bit numbers, so a counting placement replaces the comparison network: bucket = the top
//       13 key bits (8192 buckets: about one super-droplet per bucket), one shared-memory atomic per super-droplet
//       gives its slot inside the bucket, an exclusive scan of the bucket counts gives the bucket starts, the 32-bit
//       words (low 19 key bits << 13 | index) are scattered to start + slot, and every word then finds its exact
//       place by counting the smaller words of its own bucket.  The result is the ascending order of (key, index):
//       the oracle's std::stable_sort order (ties between equal keys by index), for any key distribution -- a skewed
//       one only makes the buckets longer;
//   a4  thread t takes the pairs (2p, 2p + 1), p = t, t + 1024, ...: the same pair rule as every other path
//       (pair_may_collide: exact early-out; pair_apply_to: the rule in fp64), the Philox block of the first member
//       regenerated, the attributes read and written in shared memory.
//
// A single block cannot beat many SMs on bandwidth, but at this size nothing is bandwidth: the step is the sum of a
// few shared-memory round trips, and inside a run not even a kernel launch separates two steps (3.3 us each on this
// host).  An earlier attempt with a bitonic network over the 8192 words in shared memory (91 stages x 16 B per word)
// took 95-114 us (profiles/r1c_README.md); the counting placement touches every word a handful of times.
#include <cooperative_groups.h>

#include "sdm_internal.h"
#include "sdm_pair.cuh"

namespace sdm {

constexpr int BOX_THREADS = 1024;
constexpr int BOX_ITEMS = BOX_MAX / BOX_THREADS;  // super-droplets per thread
constexpr int BOX_IDX_BITS = 13;
constexpr int BOX_BUCKET_BITS = 13;               // one bucket per super-droplet of a full box: runs of 1-5 words
constexpr int BOX_BUCKETS = 1 << BOX_BUCKET_BITS;
constexpr int BOX_PER_THREAD = BOX_BUCKETS / BOX_THREADS;
// inside a bucket the top 13 key bits agree, so the low 19 key bits above the 13-bit index order its members: the
// words are 32 bits wide
static_assert(BOX_MAX <= (1 << BOX_IDX_BITS) && BOX_ITEMS * BOX_THREADS == BOX_MAX, "box tile");
static_assert(32 - BOX_BUCKET_BITS + BOX_IDX_BITS == 32, "bucket-local sort word fills 32 bits");

struct BoxArgs {
    PairArgs pair;    // pair.pk holds the first step; pair.xi / pair.v are the caller's arrays
    u32 n_steps;      // consecutive steps of this launch (debug outputs: 1)
    int32_t* dbg_perm;
    int32_t* dbg_cell_start;
};

__global__ void __launch_bounds__(BOX_THREADS, 1) k_box_steps(const __grid_constant__ BoxArgs a) {
    extern __shared__ long long s_xi[];               // [n_sd] the multiplicities for the whole launch
    __shared__ u32 s_count[BOX_BUCKETS];              // bucket counts, then bucket starts
    __shared__ u32 s_warp[BOX_THREADS / 32];
    const u32 n = a.pair.n_sd;
    double* s_v = reinterpret_cast<double*>(s_xi + n);                       // [n_sd] the volumes
    u32* s_words = reinterpret_cast<u32*>(s_v + n);                          // [n_sd] (low key bits << 13 | index), bucket by bucket
    unsigned short* s_idx = reinterpret_cast<unsigned short*>(s_words + n);  // [n_sd] indices in shuffled order
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (u32 i = tid; i < n; i += BOX_THREADS) {
        s_xi[i] = a.pair.xi[i];
        s_v[i] = a.pair.v[i];
    }
    const u64 step0 = ((u64)a.pair.pk.step_hi << 32) | (u64)a.pair.pk.step_lo;
    const bool dbg = a.pair.dbg_gamma != nullptr;
    for (u32 s = 0; s < a.n_steps; ++s) {
        const PhiloxStep ps = make_philox_step(step0 + (u64)s);
        {
            uint4* z = reinterpret_cast<uint4*>(s_count);
            for (int b = tid; b < BOX_BUCKETS / 4; b += BOX_THREADS) z[b] = make_uint4(0u, 0u, 0u, 0u);
        }
        __syncthreads();  // also: the previous step's pair phase (or the initial load) is complete
        // ---- a1 + bucket histogram ----
        u32 key[BOX_ITEMS], slot[BOX_ITEMS];
#pragma unroll
        for (int k = 0; k < BOX_ITEMS; ++k) {
            const u32 i = (u32)tid + (u32)k * BOX_THREADS;
            key[k] = philox4x32_10(a.pair.pk, ps, (u64)i).w0;  // computed for every slot: the chains of a thread interleave
            slot[k] = 0;
            if (i < n) slot[k] = atomicAdd(&s_count[key[k] >> (32 - BOX_BUCKET_BITS)], 1u);
        }
        __syncthreads();
        // ---- exclusive scan of the bucket counts (BOX_PER_THREAD consecutive buckets per thread) ----
        {
            u32 c[BOX_PER_THREAD];
            u32 sum = 0;
            const uint4* src = reinterpret_cast<const uint4*>(s_count + tid * BOX_PER_THREAD);
#pragma unroll
            for (int j = 0; j < BOX_PER_THREAD / 4; ++j) {
                const uint4 q = src[j];
                c[4 * j] = q.x; c[4 * j + 1] = q.y; c[4 * j + 2] = q.z; c[4 * j + 3] = q.w;
                sum += q.x + q.y + q.z + q.w;
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
            uint4* dst = reinterpret_cast<uint4*>(s_count + tid * BOX_PER_THREAD);
#pragma unroll
            for (int j = 0; j < BOX_PER_THREAD / 4; ++j) {
                uint4 q;
                q.x = run; run += c[4 * j];
                q.y = run; run += c[4 * j + 1];
                q.z = run; run += c[4 * j + 2];
                q.w = run; run += c[4 * j + 3];
                dst[j] = q;
            }
        }
        __syncthreads();
        // ---- scatter into the buckets (arrival order inside a bucket) ----
#pragma unroll
        for (int k = 0; k < BOX_ITEMS; ++k) {
            const u32 i = (u32)tid + (u32)k * BOX_THREADS;
            if (i < n) s_words[s_count[key[k] >> (32 - BOX_BUCKET_BITS)] + slot[k]] = (key[k] << BOX_IDX_BITS) | i;
        }
        __syncthreads();
        // ---- exact place inside the bucket: the number of smaller words among its members ----
#pragma unroll
        for (int k = 0; k < BOX_ITEMS; ++k) {
            const u32 i = (u32)tid + (u32)k * BOX_THREADS;
            if (i < n) {
                const u32 b = key[k] >> (32 - BOX_BUCKET_BITS);
                const u32 mine = (key[k] << BOX_IDX_BITS) | i;
                const u32 lo = s_count[b], hi = (b + 1 < (u32)BOX_BUCKETS) ? s_count[b + 1] : n;
                u32 smaller = 0;
                for (u32 q = lo; q < hi; ++q) smaller += (s_words[q] < mine);
                s_idx[lo + smaller] = (unsigned short)i;
            }
        }
        __syncthreads();
        if (a.dbg_perm)
            for (u32 p = tid; p < n; p += BOX_THREADS) a.dbg_perm[p] = (int32_t)s_idx[p];
        // ---- a4: pairs of neighbours in the shuffled order, on the shared-memory copy of the state ----
        for (u32 p = tid; 2u * p + 1u < n; p += BOX_THREADS) {
            const u32 j0 = s_idx[2u * p], k0 = s_idx[2u * p + 1u];
            const long long x0 = s_xi[j0], x1 = s_xi[k0];
            const double v0 = s_v[j0], v1 = s_v[k0];
            // a dead partner: gamma~ = 0 whatever gamma is (R7); only the debug gamma output needs the probability
            if ((x0 == 0 || x1 == 0) && !dbg) continue;
            const PhiloxOut w = philox4x32_10(a.pair.pk, ps, (u64)j0);  // uniform of the first-shuffled member (R2)
            const bool swap = x0 < x1;
            if (dbg || pair_may_collide(a.pair, swap ? x1 : x0, swap ? v1 : v0, swap ? v0 : v1, w.w2, w.w3, n))
                pair_apply_to(a.pair, s_xi, s_v, j0, k0, x0, v0, x1, v1, w.w2, w.w3, n);
        }
        // (the next step's first barrier orders these writes before its reads)
    }
    __syncthreads();
    for (u32 i = tid; i < n; i += BOX_THREADS) {
        a.pair.xi[i] = s_xi[i];
        a.pair.v[i] = s_v[i];
    }
    if (a.dbg_cell_start && tid == 0) {
        a.dbg_cell_start[0] = 0;
        a.dbg_cell_start[1] = (int32_t)n;
    }
}

// ---------------------------------------------------------------------------------------------------------------
// The same steps on a thread-block CLUSTER of 8 blocks (8 SMs, distributed shared memory): one block's issue rate was
// the limit of k_box_steps (12 us per step, 40 % of it the Philox blocks).  Block r of the cluster owns the
// super-droplets [1024 r, 1024 r + 1024) -- their multiplicities and volumes live in ITS shared memory for the whole
// launch -- and the 1024 buckets whose top three key bits are r, i.e. a contiguous eighth of the shuffled order.
// Scattered accesses to another block's shared memory are slow (8192 4-byte remote atomics cost 2.6 us, 8192 remote
// stores 1.2 us, the 8192 16-byte remote loads of the pair phase about 4 us: measured by truncating the kernel), so
// the placement is organised like a radix-sort pass, with one scattered remote store per super-droplet:
//   thread (r, t) generates the Philox key of super-droplet i = 1024 r + t and counts it in the block's OWN histogram
//   of all 8192 buckets (the old value is its rank among the block's entries of that bucket);            cluster barrier
//   thread t of block r gathers the eight blocks' counts of bucket 1024 r + t (coalesced remote rows), the block scans
//   the totals, and the thread writes back to every source block where its entries of the bucket start;   cluster barrier
//   the thread writes its word (low key bits above the index) to start + rank in the owner's array;       cluster barrier
//   thread t orders the words of bucket t (about one) exactly and writes the indices in shuffled order;   cluster barrier
//   thread (r, t) takes the pair whose first member is the block's shuffled position t (even global position), reads
//   both members' (multiplicity, volume) from their owners' shared memory (one 16-byte access each), applies the
//   rule there;                                                                                          cluster barrier
// ---------------------------------------------------------------------------------------------------------------
constexpr int BC_CLUSTER = 8;
constexpr int BC_THREADS = BOX_MAX / BC_CLUSTER;      // super-droplets (and owned buckets) per block
constexpr int BC_CAP = 2 * BC_THREADS;                // words a block's buckets can take (Poisson(1024) never gets there)
static_assert(BC_THREADS == 1024 && (BOX_BUCKETS / BC_CLUSTER) == BC_THREADS, "one owned bucket per thread");

struct __align__(16) BoxState {
    long long xi;
    double v;
};

// GOLOVIN: the kernel kind as a compile-time constant -- the pair rule of a Golovin box then carries none of the
// geometric kernel's code (cube roots, fall speeds, efficiency table); with ONE pair per thread and step the fetch of
// that straight-line code, not its execution, was most of the pair phase.
// Cluster barrier with release / acquire at cluster scope (the phases only exchange data through the cluster's
// shared memory): cooperative_groups' cluster.sync() adds a GPU-scope fence and an L1 invalidation to every barrier.
__device__ __forceinline__ void cluster_barrier() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

template <bool GOLOVIN>
__global__ void __cluster_dims__(BC_CLUSTER, 1, 1) __launch_bounds__(BC_THREADS, 1)
k_box_cluster(const __grid_constant__ BoxArgs a, u32* __restrict__ sticky) {
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    extern __shared__ u32 s_hist2[];                  // 2 x [8192] the block's counts of every bucket -> where its entries
                                                      // start; steps alternate between the halves (see the end of the loop)
    __shared__ BoxState s_state[BC_THREADS];          // the block's super-droplets, for the whole launch
    __shared__ u32 s_start[BC_THREADS];               // starts of the owned buckets in s_words
    __shared__ u32 s_words[BC_CAP];                   // (low 19 key bits << 13 | index), bucket by bucket
    __shared__ unsigned short s_idx[BC_CAP];          // indices in shuffled order
    __shared__ u32 s_warp[BC_THREADS / 32];
    __shared__ u32 s_total;                           // entries in this block's buckets
    __shared__ u32 s_tot[BC_CLUSTER];                 // every block's total (copied after the scan)
    __shared__ u32 s_head;                            // (step + 1) << 16 | first shuffled index: published after the ranking
                                                      // (a launch runs at most 4096 steps, BOX_RUN_MAX in sdm_api.cu)
    const u32 n = a.pair.n_sd;
    const u32 rank = cluster.block_rank();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const u32 i = rank * BC_THREADS + (u32)tid;       // my super-droplet
    if (i < n) {
        s_state[tid].xi = a.pair.xi[i];
        s_state[tid].v = a.pair.v[i];
    }
    {
        uint4* z = reinterpret_cast<uint4*>(s_hist2);
        for (int q = tid; q < BOX_BUCKETS / 4; q += BC_THREADS) z[q] = make_uint4(0u, 0u, 0u, 0u);
    }
    if (tid == 0) s_head = 0u;
    const u64 step0 = ((u64)a.pair.pk.step_hi << 32) | (u64)a.pair.pk.step_lo;
    const bool dbg = a.pair.dbg_gamma != nullptr;
    PairArgs pa = a.pair;  // (only the fields the pair rule reads are materialised)
    if (GOLOVIN) pa.kp.kind = 0;
    cluster_barrier();
    for (u32 s = 0; s < a.n_steps; ++s) {
        const PhiloxStep ps = make_philox_step(step0 + (u64)s);
        u32* s_hist = s_hist2 + (s & 1u) * (u32)BOX_BUCKETS;
        // ---- a1 + rank among the block's entries of the bucket ----
        const u32 key = philox4x32_10(a.pair.pk, ps, (u64)i).w0;
        const u32 gb = key >> (32 - BOX_BUCKET_BITS);  // bucket 0 .. 8191; its owner is gb >> 10
        u32 slot = 0;
        if (i < n) slot = atomicAdd(&s_hist[gb], 1u);
        cluster_barrier();
        // ---- owner side: the eight blocks' counts of my bucket, scan of the totals, starts back to the sources ----
        {
            const u32 g = rank * BC_THREADS + (u32)tid;
            u32 c[BC_CLUSTER];
            u32 sum = 0;
#pragma unroll
            for (int b = 0; b < BC_CLUSTER; ++b) {
                c[b] = cluster.map_shared_rank(s_hist, b)[g];
                sum += c[b];
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
                if (lane == 31) s_total = wi;
            }
            __syncthreads();
            u32 run = s_warp[warp] + incl - sum;  // start of my bucket
            s_start[tid] = run;
#pragma unroll
            for (int b = 0; b < BC_CLUSTER; ++b) {
                cluster.map_shared_rank(s_hist, b)[g] = run;  // where block b's entries of this bucket start
                run += c[b];
            }
        }
        cluster_barrier();
        // ---- scatter into the owner's buckets; everybody learns every block's total ----
        if (tid < BC_CLUSTER) s_tot[tid] = *cluster.map_shared_rank(&s_total, tid);
        if (i < n) {
            const u32 pos = s_hist[gb] + slot;
            if (pos < (u32)BC_CAP) cluster.map_shared_rank(s_words, gb / BC_THREADS)[pos] = (key << BOX_IDX_BITS) | i;
            else sticky[STICKY_BAD_DATA] = 1u;  // cannot happen: twice the average in one eighth of the key range
        }
        cluster_barrier();
        // ---- exact order inside my bucket (about one word): place = number of smaller words ----
        const u32 total = min(s_tot[rank], (u32)BC_CAP);
        {
            const u32 lo = s_start[tid], hi = (tid + 1 < BC_THREADS) ? s_start[tid + 1] : total;
            for (u32 p = lo; p < hi && p < (u32)BC_CAP; ++p) {
                const u32 mine = s_words[p];
                u32 smaller = 0;
                for (u32 q = lo; q < hi; ++q) smaller += (s_words[q] < mine);
                s_idx[lo + smaller] = (unsigned short)(mine & ((1u << BOX_IDX_BITS) - 1u));
            }
        }
        // No cluster barrier here: the pairs work on state that no block touches during the ranking, and the one word a
        // block needs from a neighbour's ranking -- the partner of its last word, the neighbour's first shuffled index
        // -- is published with the step's tag and polled by the one thread that needs it.
        __syncthreads();
        if (tid == 0) {
            __threadfence_block();
            *reinterpret_cast<volatile u32*>(&s_head) = ((s + 1u) << 16) | (u32)s_idx[0];
        }
        // ---- a4: the pairs whose first member is one of this block's shuffled positions ----
        u32 first = 0;  // global shuffled position of the block's first word
        for (u32 r = 0; r < rank; ++r) first += s_tot[r];
        if (a.dbg_perm)
            for (u32 p = tid; p < total; p += BC_THREADS) a.dbg_perm[first + p] = (int32_t)s_idx[p];
        for (u32 p = tid; p < total; p += BC_THREADS) {
            const u32 g = first + p;
            if ((g & 1u) != 0u || g + 1u >= n) continue;
            const u32 j0 = s_idx[p];
            u32 k0;
            if (p + 1u < total) {
                k0 = s_idx[p + 1u];
            } else {  // the partner opens the next non-empty block
                u32 r = rank + 1u;
                while (s_tot[r] == 0u) ++r;  // g + 1 < n: there is one
                const volatile u32* head = cluster.map_shared_rank(&s_head, r);
                u32 h;
                do h = *head; while ((h >> 16) != s + 1u);  // that block's ranking of this step is complete
                k0 = h & 0xFFFFu;
            }
            BoxState* p0 = cluster.map_shared_rank(s_state, j0 / BC_THREADS) + (j0 % BC_THREADS);
            BoxState* p1 = cluster.map_shared_rank(s_state, k0 / BC_THREADS) + (k0 % BC_THREADS);
            const longlong2 r0 = *reinterpret_cast<const longlong2*>(p0), r1 = *reinterpret_cast<const longlong2*>(p1);
            const PhiloxOut w = philox4x32_10(a.pair.pk, ps, (u64)j0);  // uniform of the first-shuffled member (R2); runs under the remote loads
            const long long x0 = r0.x, x1 = r1.x;
            const double v0 = __longlong_as_double(r0.y), v1 = __longlong_as_double(r1.y);
            // a dead partner: gamma~ = 0 whatever gamma is (R7); only the debug gamma output needs the probability
            if ((x0 == 0 || x1 == 0) && !dbg) continue;
            const bool swap = x0 < x1;
            if (dbg || pair_may_collide(pa, swap ? x1 : x0, swap ? v1 : v0, swap ? v0 : v1, w.w2, w.w3, n))
                pair_apply_at(pa, &p0->xi, &p0->v, &p1->xi, &p1->v, j0, x0, v0, x1, v1, w.w2, w.w3, n);
        }
        {   // the next step's histogram: the other half, which nobody has touched since the scatter of the step before
            // this one.  No cluster barrier closes the step: the next one starts with block-local work (keys, local
            // histogram), and what the others may still be doing here -- pairs on this block's state, a look at its
            // first shuffled index -- is not touched again before the barriers of the next step's exchange.
            uint4* z = reinterpret_cast<uint4*>(s_hist2 + ((s + 1u) & 1u) * (u32)BOX_BUCKETS);
            for (int q = tid; q < BOX_BUCKETS / 4; q += BC_THREADS) z[q] = make_uint4(0u, 0u, 0u, 0u);
        }
        __syncthreads();
    }
    cluster_barrier();  // the last step's pairs have written this block's state
    if (i < n) {
        a.pair.xi[i] = s_state[tid].xi;
        a.pair.v[i] = s_state[tid].v;
    }
    if (a.dbg_cell_start && rank == 0 && tid == 0) {
        a.dbg_cell_start[0] = 0;
        a.dbg_cell_start[1] = (int32_t)n;
    }
}

constexpr size_t BOX_SMEM_PER_SD = 8 + 8 + 4 + 2;  // xi, v, sort word, shuffled index

cudaError_t init_box_step(sdm_ctx*) {
    cudaError_t e = cudaFuncSetAttribute(k_box_cluster<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * BOX_BUCKETS * 4);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k_box_cluster<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * BOX_BUCKETS * 4);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_box_steps, cudaFuncAttributeMaxDynamicSharedMemorySize, BOX_MAX * BOX_SMEM_PER_SD);
}

// `pk` carries the first step; steps step .. step + n_steps - 1 run back to back inside the launch.
cudaError_t launch_box_steps(sdm_ctx* ctx, int64_t* xi, double* v, int64_t n_sd, double dtdV, const KernelParams& kp,
                             const PhiloxKeys& pk, int64_t n_steps) {
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
    a.n_steps = (u32)n_steps;
    a.dbg_perm = ctx->dbg_perm;
    a.dbg_cell_start = ctx->dbg_cell_start;
    LaunchScope scope(ctx, PROF_BOX_STEP);
    if (ctx->box_cluster && kp.kind == 0)  // one cluster of eight blocks
        k_box_cluster<true><<<BC_CLUSTER, BC_THREADS, 2 * BOX_BUCKETS * 4, ctx->stream>>>(a, ctx->ws.sticky);
    else if (ctx->box_cluster)
        k_box_cluster<false><<<BC_CLUSTER, BC_THREADS, 2 * BOX_BUCKETS * 4, ctx->stream>>>(a, ctx->ws.sticky);
    else
        k_box_steps<<<1, BOX_THREADS, (size_t)n_sd * BOX_SMEM_PER_SD, ctx->stream>>>(a);
    return cudaGetLastError();
}

}  // namespace sdm
