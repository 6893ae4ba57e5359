// An entry point that allocates NOTHING, for callers that cannot call cudaMalloc (code under CUDA graph capture,
// tight serving loops, harnesses that forbid allocation): sdm_remove_zero_multiplicity_static, the stable in-place
// removal of zero-multiplicity super-droplets (north_star (d)) without a context and
// without a workspace.  Every other entry point works on the caller's workspace through an sdm_ctx, and sdm_init
// creates streams, events and pinned host memory; this one needs none of that.
//
// The scratch memory of the compaction -- the ticket counter and one look-back word per tile of 2048 entries -- lives
// in the file-scope device array g_static_scratch below: (64 + 32768) x 4 bytes = 128.25 KB, enough for
// SDM_STATIC_MAX_N_SD = 2^26 super-droplets.  Every GPU that loads the library holds the array until the process
// exits.  In host code the NAME of the array is only a host-side stand-in: its device address comes from
// cudaGetSymbolAddress, asked once per device with that device current (static_scratch_of), and that pointer is what
// the memset and the kernel get.
//
// All calls on a device share the array, and it keeps the last call's contents: every call clears the words it is
// going to use on its stream before the kernel.  Calls that overlap on the GPU (two streams, two host threads) RACE
// on it -- the caller serialises them.
//
// The kernel is k_compact's algorithm (sdm_compact.cu: single pass, ticketed tiles, decoupled look-back by one warp
// over a window of 32 predecessors, in place) as a variant that also delivers the result on the device: the last tile
// writes the number of survivors to the caller's *n_sd_out_dev, so the call never synchronises and nothing comes back
// through host memory.  The existing path (k_count_zero + k_compact through the context) is untouched.
#include <mutex>

#include "sdm_internal.h"

namespace sdm {

constexpr long long STATIC_MAX_N_SD = 1ll << 26;
constexpr u32 STATIC_HEADER_WORDS = 64;  // word 0: the ticket counter; the tile states follow the 256-byte header
constexpr u32 STATIC_MAX_TILES = (u32)(STATIC_MAX_N_SD / CMP_TILE);
constexpr u32 STATIC_FLAG_AGG = 1u << 30;
constexpr u32 STATIC_FLAG_PREFIX = 2u << 30;
constexpr u32 STATIC_VALUE_MASK = (1u << 30) - 1u;
static_assert(STATIC_MAX_N_SD % CMP_TILE == 0 && STATIC_MAX_N_SD <= (1ll << 30), "tile states hold 30-bit counts");

static __device__ __align__(256) u32 g_static_scratch[STATIC_HEADER_WORDS + STATIC_MAX_TILES];

__global__ void __launch_bounds__(CMP_BLOCK)
k_compact_static(long long* __restrict__ xi, double* __restrict__ v, int* __restrict__ cell_id, u32 n_sd,
                 u32* __restrict__ scratch, long long* __restrict__ n_sd_out) {
    __shared__ u32 s_tile;
    __shared__ u32 s_wcount[CMP_BLOCK / 32];
    __shared__ u32 s_prefix;
    u32* const ticket = scratch;
    u32* const state = scratch + STATIC_HEADER_WORDS;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    __syncthreads();
    const u32 tile = s_tile;
    const u32 base = tile * (u32)CMP_TILE;

    long long x[CMP_ITEMS];
    double vv[CMP_ITEMS];
    int cc[CMP_ITEMS];
    u32 rank[CMP_ITEMS];
    u32 keepmask = 0;
    const u32 wbase = base + warp * 32u * CMP_ITEMS + lane;
#pragma unroll
    for (int k = 0; k < CMP_ITEMS; ++k) {
        const u32 i = wbase + k * 32u;
        x[k] = 0; vv[k] = 0.0; cc[k] = 0;
        if (i < n_sd) { x[k] = xi[i]; vv[k] = v[i]; cc[k] = cell_id[i]; }
    }
    u32 wrun = 0;  // survivors of this warp so far (rounds in memory order)
#pragma unroll
    for (int k = 0; k < CMP_ITEMS; ++k) {
        const bool keep = x[k] != 0;  // out-of-range entries were loaded as 0
        const u32 b = __ballot_sync(0xffffffffu, keep);
        rank[k] = wrun + __popc(b & lanemask_lt());
        wrun += __popc(b);
        keepmask |= (keep ? 1u : 0u) << k;
    }
    if (lane == 0) s_wcount[warp] = wrun;
    __syncthreads();  // every load of this block has completed: only now may a successor learn this tile's count
    u32 woff = 0, total = 0;
#pragma unroll
    for (int w = 0; w < CMP_BLOCK / 32; ++w) {
        const u32 cnt = s_wcount[w];
        if (w < warp) woff += cnt;
        total += cnt;
    }
    if (warp == 0) {
        u32 excl = 0;
        if (tile == 0) {
            if (lane == 0) st_release_u32(state + tile, STATIC_FLAG_PREFIX | total);
        } else {
            if (lane == 0) st_release_u32(state + tile, STATIC_FLAG_AGG | total);
            for (int j = (int)tile - 1; j >= 0; j -= 32) {  // lane l looks at tile j - l
                const int q = j - lane;
                u32 sv = STATIC_FLAG_PREFIX;  // before tile 0: prefix 0
                if (q >= 0) {
                    do sv = ld_relaxed_u32(state + q);
                    while ((sv & ~STATIC_VALUE_MASK) == 0u);
                }
                const u32 pm = __ballot_sync(0xffffffffu, (sv & ~STATIC_VALUE_MASK) == STATIC_FLAG_PREFIX);
                const int first = pm ? __ffs(pm) - 1 : 32;  // nearest predecessor that already knows its prefix
                excl += __reduce_add_sync(0xffffffffu, lane <= first ? (sv & STATIC_VALUE_MASK) : 0u);
                if (pm) break;
            }
            __threadfence();  // acquire side of the predecessors' releases
            if (lane == 0) st_release_u32(state + tile, STATIC_FLAG_PREFIX | (excl + total));
        }
        if (lane == 0) {
            s_prefix = excl;
            if (base + (u32)CMP_TILE >= n_sd) *n_sd_out = (long long)(excl + total);  // the last tile: the survivors
        }
    }
    __syncthreads();
    const u32 dst0 = s_prefix + woff;
    // nothing was removed before or inside this tile: every survivor is already in place
    if (s_prefix == base && total == min((u32)CMP_TILE, n_sd - base)) return;
#pragma unroll
    for (int k = 0; k < CMP_ITEMS; ++k) {
        if ((keepmask >> k) & 1u) {
            const u32 dst = dst0 + rank[k];
            xi[dst] = x[k];
            v[dst] = vv[k];
            cell_id[dst] = cc[k];
        }
    }
}

namespace {

constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mutex;
u32* g_static_ptr[STATIC_MAX_DEVICES] = {};  // device address of g_static_scratch on device d (nullptr: not asked yet)

// Set-up, once per device: the device address of the scratch array ON THE CURRENT DEVICE.
int static_scratch_of(int device, u32** out) {
    if (device < 0 || device >= STATIC_MAX_DEVICES) return SDM_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[device]) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_static_scratch) != cudaSuccess || !p) {
            cudaGetLastError();
            return SDM_ERR_CUDA;
        }
        g_static_ptr[device] = reinterpret_cast<u32*>(p);
    }
    *out = g_static_ptr[device];
    return SDM_OK;
}

}  // namespace
}  // namespace sdm

extern "C" {

int64_t sdm_static_max_n_sd(void) { return (int64_t)sdm::STATIC_MAX_N_SD; }

int sdm_static_setup(void) {
    int device = -1;
    if (cudaGetDevice(&device) != cudaSuccess) return SDM_ERR_CUDA;
    sdm::u32* scratch = nullptr;
    return sdm::static_scratch_of(device, &scratch);
}

int sdm_remove_zero_multiplicity_static(int64_t* multiplicity, double* volume, int32_t* cell_id, int64_t n_sd,
                                        int64_t* n_sd_out_dev, void* cuda_stream) {
    using namespace sdm;
    if (n_sd < 0 || !n_sd_out_dev) return SDM_ERR_INVALID_ARG;
    if (n_sd > STATIC_MAX_N_SD) return SDM_ERR_STATIC_LIMIT;  // before anything is touched
    if (n_sd > 0 && (!multiplicity || !volume || !cell_id)) return SDM_ERR_INVALID_ARG;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    if (n_sd == 0) return cudaMemsetAsync(n_sd_out_dev, 0, 8, st) == cudaSuccess ? SDM_OK : SDM_ERR_CUDA;
    int device = -1;
    if (cudaGetDevice(&device) != cudaSuccess) return SDM_ERR_CUDA;
    u32* scratch = nullptr;
    const int rc = static_scratch_of(device, &scratch);
    if (rc != SDM_OK) return rc;
    const u32 n_tiles = (u32)((n_sd + CMP_TILE - 1) / CMP_TILE);
    // the array keeps the last call's ticket and tile states: clear the words this call uses
    if (cudaMemsetAsync(scratch, 0, ((size_t)STATIC_HEADER_WORDS + n_tiles) * 4, st) != cudaSuccess) return SDM_ERR_CUDA;
    k_compact_static<<<n_tiles, CMP_BLOCK, 0, st>>>(reinterpret_cast<long long*>(multiplicity), volume, cell_id, (u32)n_sd,
                                                    scratch, reinterpret_cast<long long*>(n_sd_out_dev));
    return cudaGetLastError() == cudaSuccess ? SDM_OK : SDM_ERR_CUDA;
}

}  // extern "C"
