// The per-cell shuffle of ONE big cell (a box model above the one-block size: configs[1], 2^20 super-droplets) without
// LSD passes: a two-level counting placement by the bits of the Philox key, then the pair kernel of the GENERAL path
// (SDM_PATH_BUCKET; SURVEY.md 8(f) NEXT-1 carried over to single-cell inputs).
//
// The keys are uniform 32-bit numbers.  Level 1 cuts the cell into 2^cb COARSE buckets by the top cb key bits, 1024-2048
// entries each on average; a Poisson count never reaches twice such an average, so every bucket gets a fixed slab of
// `cap` = 2 x average + 64 words and no histogram pass is needed:
//   k_bucket_scatter   a block counts its chunk's entries per bucket in shared memory, reserves their range of the
//                      bucket's slab with ONE global atomic per bucket and writes the index words there (arrival order)
// Level 2, k_bucket_sort: one block per coarse bucket.  Its first shuffled position is the sum of the counts of the
// buckets before it (buckets are contiguous ranges of the shuffled order); it puts its entries in exact (key, index)
// order the way the box step does -- fine bucket = the next 11-13 key bits (about one entry each), one shared atomic per
// entry, scan, scatter of 32-bit words (remaining key bits above the index), exact place by counting the smaller words
// of the fine bucket -- and writes the indices to their shuffled positions.  k_pair then pairs neighbours exactly as
// on the GENERAL path.  Against that path's four chained radix passes (each a wave of tiles waiting on its
// predecessors: 15 us apiece at 2^20 entries) nothing here waits on a neighbour.  Same total order (key, index) =>
// same bits.  Level 1 depends on nothing but the step number: the time loop (sdm_coalescence_steps) runs the next
// step's k_bucket_scatter on a side stream beside this step's pair kernel (enqueue_bucket_step, sdm_api.cu).
#include "sdm_internal.h"

namespace sdm {

constexpr int BK_BLOCK = 512;                   // k_bucket_scatter (256 x 8: 16.4 us instead of 14.5): both kernels are single waves of
                                                // short blocks, a thread's serial chain is what they wait for
constexpr int BK_ITEMS = 4;
constexpr int BK_CHUNK = BK_BLOCK * BK_ITEMS;
constexpr int BS_BLOCK = 512;                   // k_bucket_sort (256 x 16 entries per thread: 21.4 us instead of 17.5 on configs[1])
constexpr int BS_ITEMS = 8;
constexpr int BS_CAP = BS_BLOCK * BS_ITEMS;     // largest coarse bucket the level-2 block takes
constexpr int BS_MAX_FINE_BITS = 13;

__global__ void __launch_bounds__(BK_BLOCK)
k_bucket_scatter(u32 n_sd, int cb, u32 cap, const __grid_constant__ PhiloxKeys pk, u32* __restrict__ cursor,
                 u32* __restrict__ words, u32* __restrict__ sticky, int32_t* __restrict__ dbg_cell_start) {
    extern __shared__ u32 s_mem[];  // cnt[2^cb] | base[2^cb]
    const u32 n_bucket = 1u << cb;
    u32* s_cnt = s_mem;
    u32* s_base = s_mem + n_bucket;
    for (u32 b = threadIdx.x; b < n_bucket; b += BK_BLOCK) s_cnt[b] = 0u;
    if (dbg_cell_start && blockIdx.x == 0 && threadIdx.x == 0) { dbg_cell_start[0] = 0; dbg_cell_start[1] = (int32_t)n_sd; }
    __syncthreads();
    const u32 stride = gridDim.x * BK_CHUNK;
    for (u32 base = blockIdx.x * BK_CHUNK; base < n_sd; base += stride) {
        u32 key[BK_ITEMS], rank[BK_ITEMS];
#pragma unroll
        for (int k = 0; k < BK_ITEMS; ++k) key[k] = philox_perm_key(pk, (u64)(base + k * BK_BLOCK + threadIdx.x));
#pragma unroll
        for (int k = 0; k < BK_ITEMS; ++k) {
            rank[k] = 0;
            if (base + k * BK_BLOCK + threadIdx.x < n_sd) rank[k] = atomicAdd(&s_cnt[key[k] >> (32 - cb)], 1u);
        }
        __syncthreads();
        for (u32 b = threadIdx.x; b < n_bucket; b += BK_BLOCK) {  // one global atomic per bucket this chunk touches
            const u32 c = s_cnt[b];
            if (c) {
                s_base[b] = atomicAdd(&cursor[b], c);
                s_cnt[b] = 0u;
            }
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < BK_ITEMS; ++k) {
            const u32 i = base + k * BK_BLOCK + threadIdx.x;
            if (i < n_sd) {
                const u32 b = key[k] >> (32 - cb);
                const u32 pos = s_base[b] + rank[k];
                if (pos < cap) words[(size_t)b * cap + pos] = i;
                else sticky[STICKY_BAD_DATA] = 1u;  // cannot happen: a bucket of twice the average
            }
        }
        __syncthreads();  // s_base is rewritten by the next chunk
    }
}

// One block per coarse bucket: its entries (at most min(cap, BS_CAP)) in exact (key, index) order.  fb fine-bucket bits
// follow the cb coarse bits; the 32-bit bucket-local word is (remaining 32 - cb - fb key bits) << idxbits | index, which
// fits because fb >= idxbits - cb (launcher).
__global__ void __launch_bounds__(BS_BLOCK)
k_bucket_sort(const u32* __restrict__ words, const u32* __restrict__ count, int cb, u32 cap, int fb, int idxbits,
              const __grid_constant__ PhiloxKeys pk, u64* __restrict__ sorted, u32* __restrict__ sticky) {
    extern __shared__ u32 s_mem[];  // fine counts / ends [2^fb] | bucket-ordered words [n_b]
    __shared__ u32 s_warp[BS_BLOCK / 32];
    __shared__ u32 s_lo;
    const u32 n_fine = 1u << fb;
    u32* s_fine = s_mem;
    u32* s_w = s_mem + n_fine;
    const u32 b = blockIdx.x;
    const u32 n_b = __ldg(count + b);
    if (n_b == 0) return;
    if (n_b > cap || n_b > (u32)BS_CAP) {  // cannot happen: twice the largest average bucket
        if (threadIdx.x == 0) sticky[STICKY_BAD_DATA] = 1u;
        return;
    }
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // first shuffled position of the bucket: the counts of all buckets before it
    {
        u32 part = 0;
        for (u32 q = tid; q < b; q += BS_BLOCK) part += __ldg(count + q);
        part = __reduce_add_sync(0xffffffffu, part);
        if (lane == 0) s_warp[warp] = part;
    }
    for (u32 f = tid; f < n_fine; f += BS_BLOCK) s_fine[f] = 0u;
    __syncthreads();
    if (tid == 0) {
        u32 t = 0;
        for (int w = 0; w < BS_BLOCK / 32; ++w) t += s_warp[w];
        s_lo = t;
    }
    const u32* __restrict__ my_words = words + (size_t)b * cap;
    u32 key[BS_ITEMS];
    const int fshift = 32 - cb - fb;
#pragma unroll
    for (int k = 0; k < BS_ITEMS; ++k) {
        const u32 e = (u32)tid + (u32)k * BS_BLOCK;
        key[k] = 0;
        if ((u32)k * BS_BLOCK < n_b) {  // block-uniform: rounds past the bucket's end cost nothing
            key[k] = philox_perm_key(pk, (u64)(e < n_b ? __ldg(my_words + e) : 0u));
            if (e < n_b) atomicAdd(&s_fine[(key[k] >> fshift) & (n_fine - 1u)], 1u);
        }
    }
    __syncthreads();
    const u32 lo_b = s_lo;
    {  // exclusive scan of the fine counts: n_fine / BS_BLOCK consecutive values per thread
        const u32 per = n_fine / BS_BLOCK;
        u32 sum = 0;
        for (u32 j = 0; j < per; ++j) sum += s_fine[tid * per + j];
        u32 incl = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const u32 y = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += y;
        }
        __syncthreads();  // s_warp: the bucket-start partial sums have been consumed
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        u32 woff = 0;
        for (int w = 0; w < warp; ++w) woff += s_warp[w];
        u32 run = woff + incl - sum;
        for (u32 j = 0; j < per; ++j) {
            const u32 c = s_fine[tid * per + j];
            s_fine[tid * per + j] = run;
            run += c;
        }
    }
    __syncthreads();
    // scatter into the fine buckets: a second atomic on the starts hands out the slots and leaves s_fine[f] = the END of
    // fine bucket f (= the start of f + 1)
    const u32 low_mask = fshift > 0 ? ((1u << fshift) - 1u) : 0u;
#pragma unroll
    for (int k = 0; k < BS_ITEMS; ++k) {
        const u32 e = (u32)tid + (u32)k * BS_BLOCK;
        if (e < n_b) {
            const u32 pos = atomicAdd(&s_fine[(key[k] >> fshift) & (n_fine - 1u)], 1u);
            s_w[pos] = ((key[k] & low_mask) << idxbits) | __ldg(my_words + e);
        }
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < BS_ITEMS; ++k) {
        const u32 e = (u32)tid + (u32)k * BS_BLOCK;
        if (e < n_b) {
            const u32 f = (key[k] >> fshift) & (n_fine - 1u);
            const u32 i = __ldg(my_words + e);
            const u32 mine = ((key[k] & low_mask) << idxbits) | i;
            const u32 lo = f ? s_fine[f - 1u] : 0u, hi = s_fine[f];
            u32 smaller = 0;
            for (u32 q = lo; q < hi; ++q) smaller += (s_w[q] < mine);
            sorted[lo_b + lo + smaller] = (u64)i;  // the pair kernel's word: the index in the low bits
        }
    }
}

// Coarse key bits of the placement: the fewest that leave at most 2048 entries per bucket on average (at least one
// bit).  `bits_override` > 0 (tests): that many.
int bucket_bits(int64_t n_sd, int bits_override) {
    if (bits_override > 0) return bits_override < BUCKET_MAX_BITS ? bits_override : BUCKET_MAX_BITS;
    int bits = 1;
    while (bits < BUCKET_MAX_BITS && ((int64_t)2048 << bits) < n_sd) ++bits;
    return bits;
}

// Fine-bucket bits of level 2 for cb coarse bits: the 32-bit bucket-local word holds (32 - cb - fb) key bits above the
// index, so fb >= idxbits - cb; 0 when no legal value exists (a forced, too small cb on a large array).
int bucket_fine_bits(int64_t n_sd, int cb) {
    int idxbits = 1;
    while (((int64_t)1 << idxbits) < n_sd) ++idxbits;
    int fb = idxbits - cb > 11 ? idxbits - cb : 11;
    if (fb > 32 - cb) fb = 32 - cb;
    return (fb > BS_MAX_FINE_BITS || fb < 9 || fb < idxbits - cb) ? 0 : fb;
}

// One block per chunk of 2048 entries while that fits eight resident blocks per SM (configs[1]: 512 blocks, each a
// short chain Philox -> shared atomics -> one round of global atomics -> stores; more blocks in flight hide it), a
// strided loop above that.
static u32 resident_grid(const sdm_ctx* ctx, int64_t n_sd) {
    const long long chunks = (n_sd + BK_CHUNK - 1) / BK_CHUNK;
    const long long resident = (long long)ctx->sm_count * 8;
    return (u32)(chunks < resident ? (chunks > 0 ? chunks : 1) : resident);
}

cudaError_t init_bucket_path(sdm_ctx*) {
    return cudaFuncSetAttribute(k_bucket_sort, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                ((1 << BS_MAX_FINE_BITS) + BS_CAP) * 4);
}

// Words per coarse-bucket slab: twice the average count plus slack, at most what a level-2 block takes.
u32 bucket_slab_words(int64_t n_sd, int cb) {
    const int64_t avg = (n_sd + ((int64_t)1 << cb) - 1) >> cb;
    int64_t cap = 2 * avg + 64;
    if (cap > n_sd) cap = n_sd;  // a bucket cannot hold more than everything
    return (u32)cap;
}

// Level 1 of the placement on stream `st` (ctx->stream, or the context's side stream when the time loop runs it beside
// the previous step's pair kernel): the slabs live in buf_b (carved with room for 2^cb x cap words), the counts in
// ws.bucket_count (zeroed by the caller on the same stream).
cudaError_t launch_bucket_scatter(sdm_ctx* ctx, int64_t n_sd, int cb, const PhiloxKeys& pk, cudaStream_t st) {
    Workspace& ws = ctx->ws;
    const u32 n_bucket = 1u << cb;
    const u32 cap = bucket_slab_words(n_sd, cb);
    if (bucket_fine_bits(n_sd, cb) == 0) return cudaErrorInvalidValue;  // bucket_fits() keeps such shapes away
    LaunchScope scope(ctx, PROF_BUCKET);
    k_bucket_scatter<<<resident_grid(ctx, n_sd), BK_BLOCK, 2 * n_bucket * 4, st>>>(
        (u32)n_sd, cb, cap, pk, ws.bucket_count, reinterpret_cast<u32*>(ws.buf_b), ws.sticky, ctx->dbg_cell_start);
    return cudaGetLastError();
}

// Level 2 on ctx->stream; `sorted` (u64[n_sd]) receives the index of every shuffled position.
cudaError_t launch_bucket_sort(sdm_ctx* ctx, int64_t n_sd, int cb, const PhiloxKeys& pk, u64* sorted) {
    Workspace& ws = ctx->ws;
    const u32 n_bucket = 1u << cb;
    const u32 cap = bucket_slab_words(n_sd, cb);
    int idxbits = 1;
    while (((int64_t)1 << idxbits) < n_sd) ++idxbits;
    const int fb = bucket_fine_bits(n_sd, cb);
    if (fb == 0) return cudaErrorInvalidValue;
    LaunchScope scope(ctx, PROF_BUCKET);
    k_bucket_sort<<<n_bucket, BS_BLOCK, ((size_t)(1u << fb) + BS_CAP) * 4, ctx->stream>>>(
        reinterpret_cast<const u32*>(ws.buf_b), ws.bucket_count, cb, cap, fb, idxbits, pk, sorted, ws.sticky);
    return cudaGetLastError();
}

}  // namespace sdm
