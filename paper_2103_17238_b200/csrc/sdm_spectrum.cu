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

// The opt-in to more than 48 KB of dynamic shared memory is per device: done once per context (sdm_init).
cudaError_t init_volume_spectrum(sdm_ctx*) {
    return cudaFuncSetAttribute(k_volume_spectrum, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SPEC_SMEM_BUDGET);
}

static size_t spectrum_smem_bytes(int n_edges, int cols) {
    return (size_t)n_edges * 8 + (size_t)(n_edges - 1) * (size_t)cols * (8 + 4 + 4 + 4) + 16;
}

cudaError_t launch_volume_spectrum(sdm_ctx* ctx, const int64_t* xi, const double* v, int64_t n_sd,
                                   const double* edges_dev, int32_t n_edges, int64_t* count, int64_t* sum_xi,
                                   double* sum_xi_v) {
    int cols = 32;  // column copies of the per-bin sums: as many as the shared-memory budget allows
    while (cols > 1 && spectrum_smem_bytes(n_edges, cols) > SPEC_SMEM_BUDGET) cols >>= 1;
    const size_t smem = spectrum_smem_bytes(n_edges, cols);
    long long want = (n_sd + SPEC_ITEMS * SPEC_BLOCK - 1) / (SPEC_ITEMS * SPEC_BLOCK);
    const long long resident = (long long)ctx->sm_count * 8;
    int grid = (int)(want < resident ? want : resident);
    if (grid < 1) grid = 1;
    LaunchScope scope(ctx, PROF_SPECTRUM);
    k_volume_spectrum<<<grid, SPEC_BLOCK, smem, ctx->stream>>>(
        reinterpret_cast<const long long*>(xi), v, n_sd, edges_dev, n_edges, cols,
        reinterpret_cast<unsigned long long*>(count), reinterpret_cast<unsigned long long*>(sum_xi), sum_xi_v);
    return cudaGetLastError();
}

}  // namespace sdm
