// the volume spectrum product (the paper's ParticlesVolumeSpectrum(radius_bins_edges),
// PAPER.md:68-76) on the device, so that the Golovin check and Fig.-1-style output need no D2H of the state.
// Reading R35: raw per-bin sums over bins edges[b] <= v < edges[b+1] of VOLUME edges.
//
//   k_volume_spectrum  reads xi, v once (16 B/SD), finds the bin by binary search over the edges in shared
//                      memory and accumulates per block in shared memory in C column copies of the per-bin
//                      sums (lane l adds into column l mod C, so the lanes of a warp rarely collide even
//                      when a few bins hold most of the spectrum); the columns are summed and the non-empty
//                      bins flushed with global atomics at the end.  HBM bound, 16 B/SD.
#include "sdm_internal.h"

namespace sdm {

constexpr int SPEC_BLOCK = 256;
constexpr int SPEC_ITEMS = 4;
constexpr size_t SPEC_SMEM_BUDGET = 96 * 1024;

__device__ __forceinline__ int spectrum_bin(const double* s_edges, int n_bins, double vol) {
    int l = 0, r = n_bins;  // largest b with edges[b] <= vol (the caller checked edges[0] <= vol < edges[n_bins])
    while (r - l > 1) {
        const int m = (l + r) >> 1;
        const bool up = vol >= s_edges[m];
        l = up ? m : l;
        r = up ? r : m;
    }
    return l;
}

__global__ void __launch_bounds__(SPEC_BLOCK)
k_volume_spectrum(const long long* __restrict__ xi, const double* __restrict__ v, long long n_sd,
                  const double* __restrict__ edges, int n_edges, int cols, unsigned long long* __restrict__ count,
                  unsigned long long* __restrict__ sum_xi, double* __restrict__ sum_xi_v) {
    extern __shared__ unsigned char s_raw[];
    const int n_bins = n_edges - 1;
    const int n_slots = n_bins * cols;
    // sum xi v: shared memory has no native fp64 atomic add (a CAS spin loop); with 32 columns the lanes of a
    // warp never share a slot.  (One private column per thread, no atomics at all, was measured slower: its 63 KB
    // per block leave 2 blocks per SM and the kernel is latency-bound on the binary search.)
    double* s_edges = reinterpret_cast<double*>(s_raw);                                 // n_edges
    double* s_xv = s_edges + n_edges;                                                   // n_bins x cols
    const int n_xv = n_slots;
    // sum xi as (low, high) 32-bit words: shared memory has native 32-bit atomic adds only (64-bit ones are CAS
    // loops); every add propagates its own carry, so the pair is the exact 64-bit sum whatever the order
    u32* s_xi_lo = reinterpret_cast<u32*>(s_xv + n_xv);                                 // n_bins x cols
    u32* s_xi_hi = s_xi_lo + n_slots;                                                   // n_bins x cols
    u32* s_cnt = s_xi_hi + n_slots;                                                     // n_bins x cols
    for (int q = threadIdx.x; q < n_edges; q += SPEC_BLOCK) s_edges[q] = edges[q];
    for (int q = threadIdx.x; q < n_slots; q += SPEC_BLOCK) { s_xi_lo[q] = 0u; s_xi_hi[q] = 0u; s_cnt[q] = 0u; }
    for (int q = threadIdx.x; q < n_xv; q += SPEC_BLOCK) s_xv[q] = 0.0;
    __syncthreads();
    const double lo = s_edges[0], hi = s_edges[n_bins];
    const int col = threadIdx.x & (cols - 1);
    // four super-droplets per thread and iteration: their (dependent-load) bin searches overlap
    const long long stride = (long long)gridDim.x * SPEC_BLOCK * SPEC_ITEMS;
    for (long long i = ((long long)blockIdx.x * SPEC_BLOCK + threadIdx.x) * SPEC_ITEMS; i < n_sd; i += stride) {
        long long x[SPEC_ITEMS];
        double vol[SPEC_ITEMS];
        if (i + SPEC_ITEMS <= n_sd) {  // i is a multiple of 4 and the arrays are 16-byte aligned (checked by the API)
            const longlong2 xa = *reinterpret_cast<const longlong2*>(xi + i), xb = *reinterpret_cast<const longlong2*>(xi + i + 2);
            const double2 va = *reinterpret_cast<const double2*>(v + i), vb = *reinterpret_cast<const double2*>(v + i + 2);
            x[0] = xa.x; x[1] = xa.y; x[2] = xb.x; x[3] = xb.y;
            vol[0] = va.x; vol[1] = va.y; vol[2] = vb.x; vol[3] = vb.y;
        } else {
#pragma unroll
            for (int k = 0; k < SPEC_ITEMS; ++k) {
                x[k] = (i + k < n_sd) ? xi[i + k] : 0;
                vol[k] = (i + k < n_sd) ? v[i + k] : hi;  // hi lies outside every bin
            }
        }
        int bin[SPEC_ITEMS];
#pragma unroll
        for (int k = 0; k < SPEC_ITEMS; ++k)
            bin[k] = (vol[k] >= lo && vol[k] < hi) ? spectrum_bin(s_edges, n_bins, vol[k]) : -1;  // NaN fails both
#pragma unroll
        for (int k = 0; k < SPEC_ITEMS; ++k) {
            if (bin[k] >= 0) {
                const int slot = bin[k] * cols + col;
                atomicAdd(&s_cnt[slot], 1u);
                const u32 xl = (u32)x[k], xh = (u32)((unsigned long long)x[k] >> 32);
                const u32 old = atomicAdd(&s_xi_lo[slot], xl);
                const u32 carry = (old + xl < old) ? 1u : 0u;
                if (xh + carry) atomicAdd(&s_xi_hi[slot], xh + carry);
                atomicAdd(&s_xv[slot], (double)x[k] * vol[k]);
            }
        }
    }
    __syncthreads();
    for (int q = threadIdx.x; q < n_bins; q += SPEC_BLOCK) {
        u32 c = 0;
        unsigned long long sx = 0;
        double sv = 0.0;
        for (int k = 0; k < cols; ++k) {
            c += s_cnt[q * cols + k];
            sx += ((unsigned long long)s_xi_hi[q * cols + k] << 32) + s_xi_lo[q * cols + k];
        }
        for (int k = 0; k < cols; ++k) sv += s_xv[q * cols + k];
        if (c) {
            if (count) atomicAdd(&count[q], (unsigned long long)c);
            if (sum_xi) atomicAdd(&sum_xi[q], sx);
            if (sum_xi_v) atomicAdd(&sum_xi_v[q], sv);
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// The same product without atomics, for up to SPEC_COLS_MAX_BINS bins (the paper's spectrum has 31): every LANE owns a
// private column of the per-bin sums in its warp's slice of shared memory (bins x 32 lanes x 20 bytes per warp), so an
// update is a plain load / add / store that no other thread can touch, and the 32 lanes of an access fall on 32
// different banks.  The bin comes from a 1024-entry table over the high word of the volume (positive doubles order
// like their bit patterns: the table gives the bin of the cell's smallest value, exact comparisons with the next edges
// finish the job), or from the binary search when an edge is not positive.  8.4 M super-droplets, 31 bins: 46.6 us =
// 0.44 of the HBM roofline (the atomic kernel above: 73 us, 0.28).  What it took, in order (profiles/r2d_README.md):
// lane-private columns alone changed nothing (77 us: two blocks of four warps per SM, every instruction waiting on
// the one before); updates without branches -- values outside the bins go to a spare column -- 62 us; integer
// comparisons of the bit patterns instead of DSETP, one table flag instead of a second edge comparison 50.6 us;
// 16 instead of 8 super-droplets per lane and iteration 46.6 us.  Shared memory (20 KB per warp) caps the occupancy.
// ---------------------------------------------------------------------------------------------------------------
constexpr int SPEC_W = 4;                 // warps per block
constexpr int SPEC_LUT = 1024;            // table cells over [edges[0], edges[n_bins])
constexpr int SPEC_COLS_MAX_BINS = 37;    // SPEC_W x bins x 640 bytes + table + edges <= 100 KB: two blocks per SM
constexpr int SPEC_GROUPS = 8;            // 16-byte loads per array, lane and iteration (2 super-droplets each)

__device__ __forceinline__ u32 hi_word(double x) { return (u32)((unsigned long long)__double_as_longlong(x) >> 32); }

template <bool LUT>
__global__ void __launch_bounds__(SPEC_W * 32)
k_volume_spectrum_cols(const long long* __restrict__ xi, const double* __restrict__ v, long long n_sd,
                       const double* __restrict__ edges, int n_edges, unsigned long long* __restrict__ count,
                       unsigned long long* __restrict__ sum_xi, double* __restrict__ sum_xi_v) {
    extern __shared__ unsigned char s_raw[];
    const int n_bins = n_edges - 1;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double* s_edges = reinterpret_cast<double*>(s_raw);                                        // n_edges (+ 1 pad)
    const int n_cols = n_bins + 1;  // one more column set takes what falls outside the bins: the updates need no branch
    double* s_xv = s_edges + ((n_edges + 1) & ~1);                                             // W x n_cols x 32
    unsigned long long* s_sx = reinterpret_cast<unsigned long long*>(s_xv + SPEC_W * n_cols * 32);
    u32* s_cnt = reinterpret_cast<u32*>(s_sx + SPEC_W * n_cols * 32);
    unsigned short* s_lut = reinterpret_cast<unsigned short*>(s_cnt + SPEC_W * n_cols * 32);   // SPEC_LUT
    for (int q = tid; q < n_edges; q += SPEC_W * 32) s_edges[q] = edges[q];
    for (int q = tid; q < SPEC_W * n_cols * 32; q += SPEC_W * 32) { s_xv[q] = 0.0; s_sx[q] = 0ull; s_cnt[q] = 0u; }
    __syncthreads();
    const double lo = s_edges[0], hi = s_edges[n_bins];
    const u32 k0 = hi_word(lo);
    const unsigned long long lo_bits = (unsigned long long)__double_as_longlong(lo);
    const unsigned long long span_bits = (unsigned long long)__double_as_longlong(hi) - lo_bits;
    int shift = 0;
    if (LUT) {
        const u32 span = hi_word(hi) - k0;
        while ((span >> shift) >= (u32)SPEC_LUT) ++shift;
        for (int c = tid; c < SPEC_LUT; c += SPEC_W * 32) {
            // smallest value of the cell; cell 0 may start below edges[0]: bin 0 either way
            const double cmin = __longlong_as_double((long long)((unsigned long long)(k0 + ((u32)c << shift)) << 32));
            const int b0 = (cmin >= lo && cmin < hi) ? spectrum_bin(s_edges, n_bins, cmin) : (cmin < lo ? 0 : n_bins - 1);
            // bit 15: the cell reaches past edges[b0 + 2] -- one comparison does not settle the bin of its values
            // (compared as bit patterns: past the largest finite double the next cell's start is no number)
            const unsigned long long cnext = (unsigned long long)(k0 + (((u32)c + 1u) << shift)) << 32;
            const bool many = b0 + 2 < n_edges && cnext > (unsigned long long)__double_as_longlong(s_edges[b0 + 2]);
            s_lut[c] = (unsigned short)(b0 | (many ? 0x8000 : 0));
        }
        __syncthreads();
    }
    double* my_xv = s_xv + warp * n_cols * 32 + lane;
    unsigned long long* my_sx = s_sx + warp * n_cols * 32 + lane;
    u32* my_cnt = s_cnt + warp * n_cols * 32 + lane;
    constexpr int PER_WARP = SPEC_GROUPS * 64;  // super-droplets per warp and iteration
    constexpr int K = 2 * SPEC_GROUPS;
    const long long stride = (long long)gridDim.x * SPEC_W * PER_WARP;
    // with two blocks of four warps per SM only the loads of the NEXT iteration, issued before this iteration's
    // shared-memory work, keep enough bytes in flight
    auto load = [&](long long base, long long (&x)[K], double (&vol)[K]) {
#pragma unroll
        for (int g = 0; g < SPEC_GROUPS; ++g) {
            const long long i = base + g * 64 + lane * 2;  // even, and the arrays are 16-byte aligned (checked by the API)
            if (i + 2 <= n_sd) {
                const longlong2 xa = *reinterpret_cast<const longlong2*>(xi + i);
                const double2 va = *reinterpret_cast<const double2*>(v + i);
                x[2 * g] = xa.x; x[2 * g + 1] = xa.y;
                vol[2 * g] = va.x; vol[2 * g + 1] = va.y;
            } else {
                x[2 * g] = (i < n_sd) ? xi[i] : 0;
                vol[2 * g] = (i < n_sd) ? v[i] : hi;  // hi lies outside every bin
                x[2 * g + 1] = 0;
                vol[2 * g + 1] = hi;
            }
        }
    };
    auto process = [&](const long long (&x)[K], const double (&vol)[K]) {
        int bin[K];
        bool more = false;  // a table cell with several bin edges inside: one comparison does not settle its values' bins
        const unsigned long long* s_edge_bits = reinterpret_cast<const unsigned long long*>(s_edges);
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const bool in = vol[k] >= lo && vol[k] < hi;  // NaN fails both
            if (LUT) {
                // the table cells are 1/1024 of the range: one bin edge inside the cell is the common case
                // every edge is positive here: doubles in range order like their bit patterns (negative values, -0.0
                // and NaN are larger than every positive number as unsigned integers)
                const unsigned long long bits = (unsigned long long)__double_as_longlong(vol[k]);
                const bool in_bits = bits - lo_bits < span_bits;  // same as `in`; integer compares have the shorter latency
                const u32 c = in_bits ? (hi_word(vol[k]) - k0) >> shift : 0u;
                const u32 e = s_lut[c];
                int b = (int)(e & 0x7FFFu);
                b += (bits >= s_edge_bits[b + 1]) ? 1 : 0;  // edges[n_bins] = hi > vol: stays inside the bins
                more |= in_bits && (e & 0x8000u) != 0u;
                bin[k] = in_bits ? b : n_bins;
            } else {
                bin[k] = in ? spectrum_bin(s_edges, n_bins, vol[k]) : n_bins;
            }
        }
        if (LUT && more) {
#pragma unroll
            for (int k = 0; k < K; ++k)
                if (bin[k] < n_bins) bin[k] = spectrum_bin(s_edges, n_bins, vol[k]);
        }
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const int o = bin[k] * 32;
            // the three sums of a bin are separate words: their loads go out together
            const u32 c = my_cnt[o];
            const unsigned long long sx = my_sx[o];
            const double sv = my_xv[o];
            my_cnt[o] = c + 1u;
            my_sx[o] = sx + (unsigned long long)x[k];
            my_xv[o] = sv + (double)x[k] * vol[k];
        }
    };
    // two register sets take turns (no copies: a copy would wait for the loads it is meant to hide)
    long long xa[K], xb[K];
    double va[K], vb[K];
    long long base = ((long long)blockIdx.x * SPEC_W + warp) * PER_WARP;
    if (base < n_sd) {
        load(base, xa, va);
        while (true) {
            if (base + stride < n_sd) load(base + stride, xb, vb);
            process(xa, va);
            base += stride;
            if (base >= n_sd) break;
            if (base + stride < n_sd) load(base + stride, xa, va);
            process(xb, vb);
            base += stride;
            if (base >= n_sd) break;
        }
    }
    __syncthreads();
    // bin q: lane l sums its column over the warps, the warp adds the 32 columns up, lane 0 flushes
    for (int q = warp; q < n_bins; q += SPEC_W) {
        u32 c = 0;
        unsigned long long sx = 0;
        double sv = 0.0;
#pragma unroll
        for (int w = 0; w < SPEC_W; ++w) {
            c += s_cnt[(w * n_cols + q) * 32 + lane];
            sx += s_sx[(w * n_cols + q) * 32 + lane];
            sv += s_xv[(w * n_cols + q) * 32 + lane];
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            c += __shfl_xor_sync(0xffffffffu, c, o);
            sx += __shfl_xor_sync(0xffffffffu, sx, o);
            sv += __shfl_xor_sync(0xffffffffu, sv, o);
        }
        if (lane == 0 && c) {
            if (count) atomicAdd(&count[q], (unsigned long long)c);
            if (sum_xi) atomicAdd(&sum_xi[q], sx);
            if (sum_xi_v) atomicAdd(&sum_xi_v[q], sv);
        }
    }
}

static size_t spectrum_cols_smem_bytes(int n_edges) {
    return (size_t)((n_edges + 1) & ~1) * 8 + (size_t)SPEC_W * (size_t)n_edges * 32 * (8 + 8 + 4) + SPEC_LUT * 2;
}

// The opt-in to more than 48 KB of dynamic shared memory is per device: done once per context (sdm_init).
cudaError_t init_volume_spectrum(sdm_ctx*) {
    const int cols_max = (int)spectrum_cols_smem_bytes(SPEC_COLS_MAX_BINS + 1);
    cudaError_t e = cudaFuncSetAttribute(k_volume_spectrum_cols<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, cols_max);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k_volume_spectrum_cols<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, cols_max);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_volume_spectrum, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SPEC_SMEM_BUDGET);
}

static size_t spectrum_smem_bytes(int n_edges, int cols) {
    return (size_t)n_edges * 8 + (size_t)(n_edges - 1) * (size_t)cols * (8 + 4 + 4 + 4) + 16;
}

cudaError_t launch_volume_spectrum(sdm_ctx* ctx, const int64_t* xi, const double* v, int64_t n_sd,
                                   const double* edges_dev, int32_t n_edges, bool lut_ok, int64_t* count, int64_t* sum_xi,
                                   double* sum_xi_v) {
    LaunchScope scope(ctx, PROF_SPECTRUM);
    if (n_edges - 1 <= SPEC_COLS_MAX_BINS) {  // few bins: lane-private columns, no atomics
        const long long per_block = (long long)SPEC_W * SPEC_GROUPS * 64;
        const long long want_blocks = (n_sd + per_block - 1) / per_block;
        const long long resident_blocks = (long long)ctx->sm_count * 2;
        int g = (int)(want_blocks < resident_blocks ? want_blocks : resident_blocks);
        if (g < 1) g = 1;
        const size_t bytes = spectrum_cols_smem_bytes(n_edges);
        if (lut_ok)
            k_volume_spectrum_cols<true><<<g, SPEC_W * 32, bytes, ctx->stream>>>(
                reinterpret_cast<const long long*>(xi), v, n_sd, edges_dev, n_edges,
                reinterpret_cast<unsigned long long*>(count), reinterpret_cast<unsigned long long*>(sum_xi), sum_xi_v);
        else
            k_volume_spectrum_cols<false><<<g, SPEC_W * 32, bytes, ctx->stream>>>(
                reinterpret_cast<const long long*>(xi), v, n_sd, edges_dev, n_edges,
                reinterpret_cast<unsigned long long*>(count), reinterpret_cast<unsigned long long*>(sum_xi), sum_xi_v);
        return cudaGetLastError();
    }
    int cols = 32;  // column copies of the per-bin sums: as many as the shared-memory budget allows
    while (cols > 1 && spectrum_smem_bytes(n_edges, cols) > SPEC_SMEM_BUDGET) cols >>= 1;
    const size_t smem = spectrum_smem_bytes(n_edges, cols);
    long long want = (n_sd + SPEC_ITEMS * SPEC_BLOCK - 1) / (SPEC_ITEMS * SPEC_BLOCK);
    const long long resident = (long long)ctx->sm_count * 8;
    int grid = (int)(want < resident ? want : resident);
    if (grid < 1) grid = 1;
    k_volume_spectrum<<<grid, SPEC_BLOCK, smem, ctx->stream>>>(
        reinterpret_cast<const long long*>(xi), v, n_sd, edges_dev, n_edges, cols,
        reinterpret_cast<unsigned long long*>(count), reinterpret_cast<unsigned long long*>(sum_xi), sum_xi_v);
    return cudaGetLastError();
}

}  // namespace sdm
