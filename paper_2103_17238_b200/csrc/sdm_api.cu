// The C ABI of libsdm_b200.so (include/sdm.h): argument validation, workspace carving and the
// launch sequence of one coalescence step.  No device memory is allocated here; everything is
// enqueued on the caller's stream.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>

#include "sdm_internal.h"

namespace sdm {

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

static inline int bits_for(uint64_t max_value) {  // bits needed to represent max_value
    int b = 0;
    while (max_value) { ++b; max_value >>= 1; }
    return b;
}

// Key digits the LSD passes sort: with m super-droplets per cell on average, the top kb = log2(m) + 8 key bits
// (rounded up to whole digits) already separate all but ~m / 2^kb <= 2^-8 of the neighbours inside a cell; the
// remaining ties are put in exact (key, index) order by k_tie_repair, so the result does not depend on `skip`.
Plan make_plan(int64_t n_sd, int32_t n_cell, int skip_key_digits) {
    Plan p;
    p.cbits = bits_for((uint64_t)(n_cell - 1));
    p.idxbits = bits_for((uint64_t)(n_sd > 1 ? n_sd - 1 : 1));
    if (skip_key_digits < 0) {
        const uint64_t m = (uint64_t)((n_sd + n_cell - 1) / n_cell);
        int kb = ((bits_for(m > 1 ? m : 1) + 8 + 7) / 8) * 8;
        if (kb > 32) kb = 32;
        skip_key_digits = (32 - kb) / 8;
    }
    p.skip = skip_key_digits > 3 ? 3 : skip_key_digits;
    p.n_cpass = (p.cbits + 7) / 8;
    p.n_pass = (4 - p.skip) + p.n_cpass;
    p.n_tiles = (int)((n_sd + SORT_TILE - 1) / SORT_TILE);
    return p;
}

// packed = (sortkey >> 8) << idxbits | idx must fit 64 bits, and pass 1 carries a 12-bit tile-local
// index below the (32 + cbits)-bit sort key.
static bool plan_fits(const Plan& p) {
    return (24 + p.cbits + p.idxbits <= 64) && (32 + p.cbits + SORT_TILE_BITS <= 64);
}

Workspace carve_workspace(void* base, int64_t max_n_sd, int32_t max_n_cell) {
    Workspace w;
    char* p = reinterpret_cast<char*>(base);
    size_t off = 0;
    const size_t max_tiles = (size_t)((max_n_sd + SORT_TILE - 1) / SORT_TILE) + 1;
    const size_t cmp_tiles = (size_t)((max_n_sd + CMP_TILE - 1) / CMP_TILE) + 1;
    auto take = [&](size_t bytes) {
        char* q = p ? p + off : nullptr;
        off = align_up(off + bytes, 256);
        return q;
    };
    // sticky | ctl are adjacent (256 B each) so that one small D2H copy reports both (STATUS_WORDS)
    static_assert(STICKY_WORDS * 4 == 256 && CTL_WORDS * 4 == 256, "status block layout");
    w.sticky = reinterpret_cast<u32*>(take(STICKY_WORDS * 4));
    const size_t ctl_off = off;
    w.ctl = reinterpret_cast<u32*>(take(CTL_WORDS * 4));
    w.digit_hist = reinterpret_cast<u32*>(take((size_t)MAX_PASSES * RADIX * 4));
    w.zero_bytes_fixed = off - ctl_off;
    w.cell_count = reinterpret_cast<u32*>(take(((size_t)max_n_cell + 1) * 4));
    w.tile_state = reinterpret_cast<u32*>(take((size_t)MAX_PASSES * max_tiles * RADIX * 4));
    w.cell_start = reinterpret_cast<u32*>(take(((size_t)max_n_cell + 2) * 4));
    w.class_list = reinterpret_cast<u32*>(take((size_t)CELL_CLASSES * (size_t)max_n_cell * 4));
    w.bucket_count = reinterpret_cast<u32*>(take(((size_t)1 << BUCKET_MAX_BITS) * 4));
    w.buf_a = reinterpret_cast<u64*>(take((size_t)max_n_sd * 8 + 16));
    // also the bucket slabs of the BUCKET path: 2^cb x (2 x average + 64) 4-byte words <= 8 n + 2^BUCKET_MAX_BITS x 264 bytes
    w.buf_b = reinterpret_cast<u64*>(take((size_t)max_n_sd * 8 + 16 + ((size_t)512 << BUCKET_MAX_BITS)));
    w.cmp_state = reinterpret_cast<u32*>(take(cmp_tiles * 4));
    w.spec_edges = reinterpret_cast<double*>(take((size_t)SPECTRUM_MAX_EDGES * 8));
    w.eff_radius = reinterpret_cast<double*>(take((size_t)EFF_MAX_R * 8));
    w.eff_table = reinterpret_cast<double*>(take((size_t)EFF_MAX_R * EFF_MAX_P * 8));
    w.scan_state_bytes = ((size_t)max_n_cell / 4096 + 2) * 8;
    w.scan_state = reinterpret_cast<u64*>(take(w.scan_state_bytes));
    w.run = reinterpret_cast<u32*>(take(RUN_WORDS * 4));
    w.res_xi = reinterpret_cast<int64_t*>(take((size_t)max_n_sd * 8 + 16));
    w.res_v = reinterpret_cast<double*>(take((size_t)max_n_sd * 8 + 16));
    w.total_bytes = off;
    return w;
}

// hybrid words: (cell_id << idxbits | index) in 64 bits, and pass 0 stages (cell_id << 12 | tile-local index)
static bool hybrid_fits(const Plan& p) { return p.cbits >= 1 && p.cbits + p.idxbits <= 64 && p.cbits + SORT_TILE_BITS <= 64; }

static bool sizes_ok(int64_t max_n_sd, int32_t max_n_cell) {
    return max_n_sd >= 0 && max_n_sd < (1LL << 30) && max_n_cell >= 1;
}

static int note_cuda(sdm_ctx* ctx, cudaError_t e) {
    if (e == cudaSuccess) return SDM_OK;
    ctx->cuda_error = (int)e;
    return SDM_ERR_CUDA;
}

// The fused kernels leave the post-step number of zero multiplicities in ctl[CTL_ZERO_COUNT].
static void note_zero_hint(sdm_ctx* ctx, const void* xi, int64_t n_sd) {
    ctx->zero_hint_valid = ctx->track_zeros;
    ctx->zero_hint_xi = xi;
    ctx->zero_hint_n_sd = n_sd;
}

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

constexpr int HOST_CHUNKS = 8;                 // pieces of sdm_coalescence_step_host's pipeline
constexpr int64_t HOST_PIPE_MIN = 1 << 18;     // smaller problems are not worth the extra stream traffic

}  // namespace sdm

using namespace sdm;

static void free_ctx(sdm_ctx* ctx) {
    if (!ctx) return;
    if (ctx->prof_events) {
        for (ProfEvent& e : *ctx->prof_events) { cudaEventDestroy(e.start); cudaEventDestroy(e.stop); }
        delete ctx->prof_events;
    }
    if (ctx->verdict_host) cudaFreeHost(ctx->verdict_host);
    if (ctx->status_host) cudaFreeHost(ctx->status_host);
    if (ctx->mapped) cudaFreeHost(const_cast<u32*>(ctx->mapped));
    if (ctx->verdict_event) cudaEventDestroy(ctx->verdict_event);
    for (cudaEvent_t e : ctx->chunk_event)
        if (e) cudaEventDestroy(e);
    for (cudaEvent_t e : ctx->host_in)
        if (e) cudaEventDestroy(e);
    for (cudaEvent_t e : ctx->host_done)
        if (e) cudaEventDestroy(e);
    if (ctx->side_go) cudaEventDestroy(ctx->side_go);
    if (ctx->side_done) cudaEventDestroy(ctx->side_done);
    if (ctx->side) cudaStreamDestroy(ctx->side);
    if (ctx->copy_in) cudaStreamDestroy(ctx->copy_in);
    if (ctx->copy_out) cudaStreamDestroy(ctx->copy_out);
    delete ctx;
}

extern "C" {

size_t sdm_workspace_bytes(int64_t max_n_sd, int32_t max_n_cell) {
    if (!sizes_ok(max_n_sd, max_n_cell)) return 0;
    return carve_workspace(nullptr, max_n_sd, max_n_cell).total_bytes;
}

int sdm_init(sdm_ctx** out, int device, int64_t max_n_sd, int32_t max_n_cell, void* workspace_dev,
             size_t workspace_bytes, void* cuda_stream) {
    if (!out) return SDM_ERR_INVALID_ARG;
    *out = nullptr;
    if (!workspace_dev || !sizes_ok(max_n_sd, max_n_cell)) return SDM_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(workspace_dev) & 255u) != 0) return SDM_ERR_INVALID_ARG;
    if (workspace_bytes < sdm_workspace_bytes(max_n_sd, max_n_cell)) return SDM_ERR_CAPACITY;
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || device < 0 || device >= n_dev) return SDM_ERR_CUDA;
    if (cudaSetDevice(device) != cudaSuccess) return SDM_ERR_CUDA;
    sdm_ctx* ctx = new (std::nothrow) sdm_ctx();
    if (!ctx) return SDM_ERR_CUDA;
    std::memset(ctx, 0, sizeof(*ctx));
    ctx->prof_events = new (std::nothrow) std::vector<ProfEvent>();
    if (!ctx->prof_events) { delete ctx; return SDM_ERR_CUDA; }
    ctx->device = device;
    ctx->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    ctx->max_n_sd = max_n_sd;
    ctx->max_n_cell = max_n_cell;
    ctx->ws = carve_workspace(workspace_dev, max_n_sd, max_n_cell);
    ctx->path = SDM_PATH_AUTO;
    ctx->narrow_key_bits = 24;
    ctx->box_cluster = 1;
    ctx->skip_key_digits = -1;
    ctx->epoch = 2;
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess || sms <= 0) {
        free_ctx(ctx);
        return SDM_ERR_CUDA;
    }
    ctx->sm_count = sms;
    if (cudaHostAlloc(reinterpret_cast<void**>(&ctx->verdict_host), sizeof(Verdict), cudaHostAllocDefault) != cudaSuccess ||
        cudaHostAlloc(reinterpret_cast<void**>(&ctx->status_host), (STICKY_WORDS + CTL_WORDS) * 4, cudaHostAllocDefault) !=
            cudaSuccess ||
        cudaHostAlloc(reinterpret_cast<void**>(const_cast<u32**>(&ctx->mapped)), MAPPED_WORDS * 4,
                      cudaHostAllocMapped | cudaHostAllocPortable) != cudaSuccess ||
        cudaEventCreateWithFlags(&ctx->verdict_event, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&ctx->chunk_event[0], cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&ctx->chunk_event[1], cudaEventDisableTiming) != cudaSuccess ||
        init_cell_fused(ctx) != cudaSuccess || init_box_step(ctx) != cudaSuccess || init_bucket_path(ctx) != cudaSuccess ||
        init_volume_spectrum(ctx) != cudaSuccess) {
        free_ctx(ctx);
        return SDM_ERR_CUDA;
    }
    for (int q = 0; q < MAPPED_WORDS; ++q) ctx->mapped[q] = 0u;
    if (cudaMemsetAsync(ctx->ws.sticky, 0, STICKY_WORDS * 4, ctx->stream) != cudaSuccess ||
        cudaMemsetAsync(ctx->ws.run, 0, RUN_WORDS * 4, ctx->stream) != cudaSuccess ||
        cudaMemsetAsync(ctx->ws.ctl, 0, CTL_WORDS * 4, ctx->stream) != cudaSuccess ||
        cudaMemsetAsync(ctx->ws.scan_state, 0, ctx->ws.scan_state_bytes, ctx->stream) != cudaSuccess) {
        free_ctx(ctx);
        return SDM_ERR_CUDA;
    }
    *out = ctx;
    return SDM_OK;
}

void sdm_destroy(sdm_ctx* ctx) { free_ctx(ctx); }

int sdm_profile_enable(sdm_ctx* ctx, int on) {
    if (!ctx) return SDM_ERR_INVALID_ARG;
    ctx->profiling = on ? 1 : 0;
    return SDM_OK;
}

int sdm_profile_read(sdm_ctx* ctx, double* ms_out, int64_t* launches_out) {
    if (!ctx || !ms_out || !launches_out) return SDM_ERR_INVALID_ARG;
    for (int c = 0; c < PROF_CLASSES; ++c) { ms_out[c] = 0.0; launches_out[c] = 0; }
    if (cudaSetDevice(ctx->device) != cudaSuccess) return SDM_ERR_CUDA;
    int rc;
    if ((rc = note_cuda(ctx, cudaStreamSynchronize(ctx->stream)))) return rc;
    for (size_t i = 0; i < ctx->prof_used; ++i) {
        ProfEvent& e = (*ctx->prof_events)[i];
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, e.start, e.stop) == cudaSuccess) {
            ms_out[e.cls] += (double)ms;
            launches_out[e.cls] += 1;
        }
    }
    ctx->prof_used = 0;
    return SDM_OK;
}

const char* sdm_strerror(int status) {
    switch (status) {
        case SDM_OK: return "ok";
        case SDM_ERR_INVALID_ARG: return "invalid argument";
        case SDM_ERR_CAPACITY: return "problem larger than the context capacity (or workspace too small)";
        case SDM_ERR_CUDA: return "CUDA error";
        case SDM_ERR_BAD_DATA: return "bad data on device (cell_id out of range, or an input the explicitly chosen path cannot take)";
        case SDM_ERR_STATIC_LIMIT:
            return "size beyond the fixed scratch array of the allocation-free entry point (sdm_static_max_n_sd: 2^26 super-droplets)";
        default: return "unknown status";
    }
}

int sdm_set_path(sdm_ctx* ctx, int path) {
    if (!ctx || path < SDM_PATH_AUTO || path > SDM_PATH_BUCKET) return SDM_ERR_INVALID_ARG;
    ctx->path = path;
    ctx->verdict_valid = 0;  // AUTO re-learns the cell order on its next step
    return SDM_OK;
}

int sdm_set_option(sdm_ctx* ctx, int option, int64_t value) {
    if (!ctx) return SDM_ERR_INVALID_ARG;
    if (option == SDM_OPT_NARROW_KEY_BITS && value >= 1 && value <= 24) {
        ctx->narrow_key_bits = (int)value;
        return SDM_OK;
    }
    if (option == SDM_OPT_SKIP_KEY_DIGITS && value >= -1 && value <= 3) {
        ctx->skip_key_digits = (int)value;
        return SDM_OK;
    }
    if (option == SDM_OPT_INDEX_BASE && value >= 0) {
        ctx->index_base = (u64)value;
        return SDM_OK;
    }
    if (option == SDM_OPT_FUSED_WORDS_PER_LANE && (value == 0 || value == 4 || value == 8)) {
        ctx->fused_r = (int)value;
        return SDM_OK;
    }
    if (option == SDM_OPT_BOX_CLUSTER && (value == 0 || value == 1)) {
        ctx->box_cluster = (int)value;
        return SDM_OK;
    }
    if (option == SDM_OPT_BUCKET_BITS && value >= 0 && value <= BUCKET_MAX_BITS) {
        ctx->bucket_bits_opt = (int)value;
        return SDM_OK;
    }
    if (option == SDM_OPT_TRACK_ZEROS && (value == 0 || value == 1)) {
        ctx->track_zeros = (int)value;
        ctx->zero_hint_valid = 0;
        return SDM_OK;
    }
    return SDM_ERR_INVALID_ARG;
}

int sdm_last_path(sdm_ctx* ctx) { return ctx ? ctx->last_path : 0; }

int64_t sdm_launch_count(sdm_ctx* ctx) { return ctx ? ctx->launches : 0; }

int sdm_volume_spectrum(sdm_ctx* ctx, const int64_t* multiplicity, const double* volume, int64_t n_sd,
                        const double* volume_edges, int32_t n_edges, int64_t* count, int64_t* sum_xi,
                        double* sum_xi_v) {
    if (!ctx || !volume_edges || n_sd < 0 || n_edges < 2 || n_edges > SPECTRUM_MAX_EDGES) return SDM_ERR_INVALID_ARG;
    if (n_sd > 0 && (!multiplicity || !volume)) return SDM_ERR_INVALID_ARG;
    if (n_sd > 0 && (!aligned16(multiplicity) || !aligned16(volume))) return SDM_ERR_INVALID_ARG;
    for (int32_t e = 0; e < n_edges; ++e) {
        if (!std::isfinite(volume_edges[e])) return SDM_ERR_INVALID_ARG;
        if (e > 0 && !(volume_edges[e] > volume_edges[e - 1])) return SDM_ERR_INVALID_ARG;
    }
    if (ctx->cuda_error) return SDM_ERR_CUDA;
    if (cudaSetDevice(ctx->device) != cudaSuccess) return SDM_ERR_CUDA;
    cudaStream_t st = ctx->stream;
    const size_t nb = (size_t)(n_edges - 1);
    int rc;
    if (count && (rc = note_cuda(ctx, cudaMemsetAsync(count, 0, nb * 8, st)))) return rc;
    if (sum_xi && (rc = note_cuda(ctx, cudaMemsetAsync(sum_xi, 0, nb * 8, st)))) return rc;
    if (sum_xi_v && (rc = note_cuda(ctx, cudaMemsetAsync(sum_xi_v, 0, nb * 8, st)))) return rc;
    if (n_sd == 0) return SDM_OK;
    // the edges are pageable host memory: this copy is staged before the call returns
    if ((rc = note_cuda(ctx, cudaMemcpyAsync(ctx->ws.spec_edges, volume_edges, (size_t)n_edges * 8,
                                             cudaMemcpyHostToDevice, st))))
        return rc;
    return note_cuda(ctx, launch_volume_spectrum(ctx, multiplicity, volume, n_sd, ctx->ws.spec_edges, n_edges, volume_edges[0] > 0.0, count,
                                                 sum_xi, sum_xi_v));
}

int sdm_debug_outputs(sdm_ctx* ctx, int32_t* perm_out, int64_t* gamma_out, int64_t* gamma_clamped_out,
                      int32_t* cell_start_out) {
    if (!ctx) return SDM_ERR_INVALID_ARG;
    ctx->dbg_perm = perm_out;
    ctx->dbg_gamma = gamma_out;
    ctx->dbg_gamma_clamped = gamma_clamped_out;
    ctx->dbg_cell_start = cell_start_out;
    return SDM_OK;
}

static int validate_step(sdm_ctx* ctx, const void* xi, const void* v, const void* cell_id, int64_t n_sd,
                         int32_t n_cell, double dt, double dV, const sdm_kernel_params* kp) {
    if (!ctx || !kp) return SDM_ERR_INVALID_ARG;
    if (n_sd < 0 || n_cell < 1) return SDM_ERR_INVALID_ARG;
    if (n_sd > 0 && (!xi || !v || !cell_id)) return SDM_ERR_INVALID_ARG;
    if (!(dt > 0.0) || !(dV > 0.0) || !std::isfinite(dt) || !std::isfinite(dV)) return SDM_ERR_INVALID_ARG;
    const double dtdV = dt / dV;
    if (!std::isfinite(dtdV) || !(dtdV > 0.0)) return SDM_ERR_INVALID_ARG;
    if (kp->kind != SDM_KERNEL_GOLOVIN && kp->kind != SDM_KERNEL_GEOMETRIC && kp->kind != SDM_KERNEL_GEOMETRIC_TABLE)
        return SDM_ERR_INVALID_ARG;
    if (kp->kind == SDM_KERNEL_GOLOVIN && !(kp->b >= 0.0 && std::isfinite(kp->b))) return SDM_ERR_INVALID_ARG;
    if (kp->kind == SDM_KERNEL_GEOMETRIC && !(kp->E >= 0.0 && std::isfinite(kp->E))) return SDM_ERR_INVALID_ARG;
    if (kp->kind == SDM_KERNEL_GEOMETRIC_TABLE && ctx->eff_n_r == 0) return SDM_ERR_INVALID_ARG;  // no table installed
    if (n_sd > ctx->max_n_sd || n_cell > ctx->max_n_cell) return SDM_ERR_CAPACITY;
    return SDM_OK;
}

namespace {

// What one step works on: the caller's arrays and the per-call constants (everything but the step index).
struct StepArgs {
    int64_t* xi;
    double* v;
    const int32_t* cell_id;
    int64_t n_sd;
    int32_t n_cell;
    double dtdV;
    KernelParams dkp;
    uint64_t seed;
};

KernelParams device_kernel_params(const sdm_ctx* ctx, const sdm_kernel_params* kp) {
    KernelParams d;
    d.kind = kp->kind;
    d.b = kp->b;
    d.Epi = kp->E * 3.141592653589793;
    d.n_r = d.n_p = 0;
    d.eff_radius = d.eff_table = nullptr;
    if (kp->kind == SDM_KERNEL_GEOMETRIC_TABLE) {  // the bounds of the early-out use the table's maximum
        d.Epi = ctx->eff_max * 3.141592653589793;
        d.n_r = ctx->eff_n_r;
        d.n_p = ctx->eff_n_p;
        d.eff_radius = ctx->ws.eff_radius;
        d.eff_table = ctx->ws.eff_table;
    }
    return d;
}

StepArgs make_step_args(const sdm_ctx* ctx, int64_t* xi, double* v, const int32_t* cell_id, int64_t n_sd,
                        int32_t n_cell, double dt, double dV, const sdm_kernel_params* kp, uint64_t seed) {
    StepArgs A;
    A.xi = xi; A.v = v; A.cell_id = cell_id; A.n_sd = n_sd; A.n_cell = n_cell;
    A.dtdV = dt / dV;
    A.dkp = device_kernel_params(ctx, kp);
    A.seed = seed;
    return A;
}

// one epoch per step (and per analysis) tags the device-side flags and scan states (no per-step memsets of them)
int next_epoch(sdm_ctx* ctx) {
    if (++ctx->epoch >= (1u << 30)) {
        ctx->epoch = 2;
        return note_cuda(ctx, cudaMemsetAsync(ctx->ws.scan_state, 0, ctx->ws.scan_state_bytes, ctx->stream));
    }
    return SDM_OK;
}

int clear_debug_gammas(sdm_ctx* ctx, int64_t n_sd) {
    int rc;
    if (ctx->dbg_gamma)
        if ((rc = note_cuda(ctx, cudaMemsetAsync(ctx->dbg_gamma, 0, (size_t)n_sd * 8, ctx->stream)))) return rc;
    if (ctx->dbg_gamma_clamped)
        if ((rc = note_cuda(ctx, cudaMemsetAsync(ctx->dbg_gamma_clamped, 0, (size_t)n_sd * 8, ctx->stream)))) return rc;
    return SDM_OK;
}

// GENERAL path, north_star (b) literally: keys + histograms, cell scan, LSD radix passes, tie repair, pairs.
int enqueue_general_step(sdm_ctx* ctx, const StepArgs& A, uint64_t step) {
    int rc;
    const Plan plan = make_plan(A.n_sd, A.n_cell, ctx->skip_key_digits);
    if (!plan_fits(plan)) return SDM_ERR_CAPACITY;
    cudaStream_t st = ctx->stream;
    Workspace& ws = ctx->ws;
    if ((rc = clear_debug_gammas(ctx, A.n_sd))) return rc;
    if ((rc = next_epoch(ctx))) return rc;
    const PhiloxKeys pk = make_philox_keys(A.seed, step, ctx->index_base);
    ctx->zero_hint_valid = 0;
    // zero the per-step control block, the digit histograms, the cell counts and the look-back states
    if ((rc = note_cuda(ctx, cudaMemsetAsync(ws.ctl, 0, ws.zero_bytes_fixed, st)))) return rc;
    if (A.n_cell > 1)
        if ((rc = note_cuda(ctx, cudaMemsetAsync(ws.cell_count, 0, ((size_t)A.n_cell + 1) * 4, st)))) return rc;
    if ((rc = note_cuda(ctx, cudaMemsetAsync(ws.tile_state, 0, (size_t)plan.n_pass * plan.n_tiles * RADIX * 4, st))))
        return rc;
    // a1 + a2: keys, digit histograms, cell histogram; then the cell scan
    if ((rc = note_cuda(ctx, launch_keys_hist(ctx, A.cell_id, A.n_sd, A.n_cell, plan, pk, ws.buf_b)))) return rc;
    if ((rc = note_cuda(ctx, launch_cell_scan(ctx, A.n_cell, A.n_sd)))) return rc;
    // a3: LSD radix passes, ping-pong between buf_b and buf_a
    u64* in = ws.buf_b;
    u64* out = ws.buf_a;
    for (int pass = 0; pass < plan.n_pass; ++pass) {
        if ((rc = note_cuda(ctx, launch_sort_pass(ctx, pass, in, out, A.n_sd, plan)))) return rc;
        u64* t = in; in = out; out = t;
    }
    if (plan.skip > 0)  // exact (key, index) order inside the runs the skipped digits left tied
        if ((rc = note_cuda(ctx, launch_tie_repair(ctx, in, A.n_sd, plan, pk)))) return rc;
    const u64* sorted = in;
    if (ctx->dbg_perm)
        if ((rc = note_cuda(ctx, launch_debug_perm(ctx, sorted, A.n_sd, plan)))) return rc;
    // a4: pairs
    if ((rc = note_cuda(ctx, launch_pair(ctx, sorted, A.xi, A.v, A.n_sd, A.n_cell, plan, A.dtdV, A.dkp, pk)))) return rc;
    ctx->last_path = SDM_PATH_GENERAL;
    // what this step learned about cell_id is AUTO's hint for the next one (asynchronous copy)
    ctx->verdict_valid = 0;
    if (A.n_cell > 1) {
        if ((rc = note_cuda(ctx, cudaMemcpyAsync(ctx->verdict_host, ws.ctl + CTL_UNSORTED, sizeof(Verdict),
                                                 cudaMemcpyDeviceToHost, st))))
            return rc;
        if ((rc = note_cuda(ctx, cudaEventRecord(ctx->verdict_event, st)))) return rc;
        ctx->verdict_cell_ptr = A.cell_id;
        ctx->verdict_n_sd = A.n_sd;
        ctx->verdict_n_cell = A.n_cell;
        ctx->verdict_valid = 1;
    }
    return SDM_OK;
}

// BOX path: a single cell of at most BOX_MAX super-droplets, whole steps inside one launch (one cluster or one block).
bool box_fits(const sdm_ctx* ctx, const StepArgs& A) {
    return A.n_cell == 1 && A.n_sd <= BOX_MAX && (ctx->path == SDM_PATH_AUTO || ctx->path == SDM_PATH_BOX);
}

constexpr int64_t BOX_RUN_MAX = 4096;  // steps of one box launch (a few tens of milliseconds)

// Steps step .. step + *n_steps - 1 of the box in one launch; with debug outputs bound (they describe ONE step) a
// single step.  *n_steps returns the number of steps enqueued.
int enqueue_box_steps(sdm_ctx* ctx, const StepArgs& A, uint64_t step, int64_t* n_steps) {
    int rc;
    if ((rc = clear_debug_gammas(ctx, A.n_sd))) return rc;
    int64_t k = *n_steps < BOX_RUN_MAX ? *n_steps : BOX_RUN_MAX;
    if (ctx->dbg_perm || ctx->dbg_gamma || ctx->dbg_gamma_clamped || ctx->dbg_cell_start) k = 1;
    const PhiloxKeys pk = make_philox_keys(A.seed, step, ctx->index_base);
    ctx->zero_hint_valid = 0;
    ctx->verdict_valid = 0;
    if ((rc = note_cuda(ctx, launch_box_steps(ctx, A.xi, A.v, A.n_sd, A.dtdV, A.dkp, pk, k)))) return rc;
    ctx->last_path = SDM_PATH_BOX;
    *n_steps = k;
    return SDM_OK;
}

// BUCKET path: one cell too large for the box step -- two-level counting placement by the key bits, then the pair
// kernel (sdm_bucket.cu).  AUTO takes it for every single cell above BOX_MAX that the placement can hold (at most 2048
// entries per coarse bucket on average: 2^23 super-droplets).
bool bucket_fits(const sdm_ctx* ctx, const StepArgs& A) {
    if (A.n_cell != 1 || A.n_sd < 1 || A.n_sd > ((int64_t)2048 << BUCKET_MAX_BITS)) return false;
    if (bucket_fine_bits(A.n_sd, bucket_bits(A.n_sd, ctx->bucket_bits_opt)) == 0) return false;
    return ctx->path == SDM_PATH_BUCKET || (ctx->path == SDM_PATH_AUTO && A.n_sd > BOX_MAX);
}

// `ahead`: the caller (the time loop) guarantees that its next action is this very call for step + 1 on the same arrays
// and sizes: level 1 of that step's placement -- which needs nothing but the step number -- is then started on the side
// stream as soon as level 2 of this step has released the counts and slabs, and runs beside this step's pair kernel
// (configs[1]: 46 -> 35 us per step).  Not with debug outputs or kernel profiling (the events bracket ctx->stream).
int enqueue_bucket_step(sdm_ctx* ctx, const StepArgs& A, uint64_t step, bool ahead) {
    int rc;
    cudaStream_t st = ctx->stream;
    Workspace& ws = ctx->ws;
    const Plan plan = make_plan(A.n_sd, 1, ctx->skip_key_digits);  // idxbits of the pair kernel's words
    const int cb = bucket_bits(A.n_sd, ctx->bucket_bits_opt);
    if ((rc = clear_debug_gammas(ctx, A.n_sd))) return rc;
    const PhiloxKeys pk = make_philox_keys(A.seed, step, ctx->index_base);
    ctx->verdict_valid = 0;
    ctx->zero_hint_valid = 0;
    const bool have = ctx->side_valid && ctx->side_step == step && ctx->side_n_sd == A.n_sd;
    if (ctx->side_valid)  // started ahead: level 2 waits for it (a placement nobody asked for any more is redone below)
        if ((rc = note_cuda(ctx, cudaStreamWaitEvent(st, ctx->side_done, 0)))) return rc;
    ctx->side_valid = 0;
    if (!have) {
        if ((rc = note_cuda(ctx, cudaMemsetAsync(ws.bucket_count, 0, ((size_t)1 << cb) * 4, st)))) return rc;
        if ((rc = note_cuda(ctx, launch_bucket_scatter(ctx, A.n_sd, cb, pk, st)))) return rc;
    }
    if ((rc = note_cuda(ctx, launch_bucket_sort(ctx, A.n_sd, cb, pk, ws.buf_a)))) return rc;
    if (ahead && !ctx->profiling && !(ctx->dbg_perm || ctx->dbg_gamma || ctx->dbg_gamma_clamped || ctx->dbg_cell_start)) {
        if (!ctx->side) {
            if (cudaStreamCreateWithFlags(&ctx->side, cudaStreamNonBlocking) != cudaSuccess ||
                cudaEventCreateWithFlags(&ctx->side_go, cudaEventDisableTiming) != cudaSuccess ||
                cudaEventCreateWithFlags(&ctx->side_done, cudaEventDisableTiming) != cudaSuccess)
                return note_cuda(ctx, cudaErrorUnknown);
        }
        const PhiloxKeys pk_next = make_philox_keys(A.seed, step + 1, ctx->index_base);
        if ((rc = note_cuda(ctx, cudaEventRecord(ctx->side_go, st)))) return rc;
        if ((rc = note_cuda(ctx, cudaStreamWaitEvent(ctx->side, ctx->side_go, 0)))) return rc;
        if ((rc = note_cuda(ctx, cudaMemsetAsync(ws.bucket_count, 0, ((size_t)1 << cb) * 4, ctx->side)))) return rc;
        if ((rc = note_cuda(ctx, launch_bucket_scatter(ctx, A.n_sd, cb, pk_next, ctx->side)))) return rc;
        if ((rc = note_cuda(ctx, cudaEventRecord(ctx->side_done, ctx->side)))) return rc;
        ctx->side_valid = 1;
        ctx->side_step = step + 1;
        ctx->side_n_sd = A.n_sd;
    }
    if (ctx->dbg_perm)
        if ((rc = note_cuda(ctx, launch_debug_perm(ctx, ws.buf_a, A.n_sd, plan)))) return rc;
    if ((rc = note_cuda(ctx, launch_pair(ctx, ws.buf_a, A.xi, A.v, A.n_sd, 1, plan, A.dtdV, A.dkp, pk)))) return rc;
    ctx->last_path = SDM_PATH_BUCKET;
    return SDM_OK;
}

// One step without the per-cell analysis: the box step or the bucket path when they fit, else GENERAL.
int enqueue_unfused_step(sdm_ctx* ctx, const StepArgs& A, uint64_t step, bool next_is_step_plus_1 = false) {
    int64_t one = 1;
    if (box_fits(ctx, A)) return enqueue_box_steps(ctx, A, step, &one);
    if (bucket_fits(ctx, A)) return enqueue_bucket_step(ctx, A, step, next_is_step_plus_1);
    return enqueue_general_step(ctx, A, step);
}

// The index runs of the fused kernel: CELL_SORTED reads the arrays directly (kind 0); HYBRID gathers through the
// words `run_idx` (kind 1: u64, kind 2: u32) that LSD passes over the cell_id digits alone have grouped by cell.
struct FusedSource {
    int kind;
    const void* run_idx;
    int idxbits;
    CellClasses cc;  // filled in by wait_verdict
    bool resident;   // the steps work on ws.res_xi / ws.res_v (run_fused_steps)
};

// cell boundaries straight from cell_id (CELL_SORTED)
int enqueue_sorted_prepare(sdm_ctx* ctx, const StepArgs& A, bool strict, FusedSource* src) {
    int rc;
    if ((rc = next_epoch(ctx))) return rc;
    src->kind = 0; src->run_idx = nullptr; src->idxbits = 0; src->resident = false;
    return note_cuda(ctx, launch_cell_bounds(ctx, 0, A.cell_id, A.n_sd, A.n_cell, 0, strict));
}

// cell-digit LSD passes + cell boundaries of the grouped words (HYBRID)
int enqueue_hybrid_prepare(sdm_ctx* ctx, const StepArgs& A, const Plan& plan, bool strict, FusedSource* src) {
    int rc;
    cudaStream_t st = ctx->stream;
    Workspace& ws = ctx->ws;
    if ((rc = next_epoch(ctx))) return rc;
    const int n_cpass = plan.n_cpass;
    const bool narrow = plan.cbits + plan.idxbits <= 32 && plan.cbits + SORT_TILE_BITS <= 32;
    if ((rc = note_cuda(ctx, cudaMemsetAsync(ws.ctl, 0, ws.zero_bytes_fixed, st)))) return rc;
    if ((rc = note_cuda(ctx, cudaMemsetAsync(ws.tile_state, 0, (size_t)n_cpass * plan.n_tiles * RADIX * 4, st))))
        return rc;
    if ((rc = note_cuda(ctx, launch_cell_digit_hist(ctx, A.cell_id, A.n_sd, A.n_cell, plan)))) return rc;
    void* in = nullptr;
    void* out = ws.buf_a;
    for (int pass = 0; pass < n_cpass; ++pass) {
        if ((rc = note_cuda(ctx, launch_cell_sort_pass(ctx, pass, narrow, A.cell_id, in, out, A.n_sd, A.n_cell, plan))))
            return rc;
        in = out;
        out = (out == (void*)ws.buf_a) ? (void*)ws.buf_b : (void*)ws.buf_a;
    }
    src->kind = narrow ? 2 : 1;
    src->resident = false;
    src->run_idx = in;
    src->idxbits = plan.idxbits;
    return note_cuda(ctx, launch_cell_bounds(ctx, src->kind, in, A.n_sd, A.n_cell, plan.idxbits, strict));
}

int enqueue_fused_step(sdm_ctx* ctx, const StepArgs& A, const FusedSource& src, uint64_t step,
                       const StepLinks& links, bool bump_epoch) {
    int rc;
    if ((rc = clear_debug_gammas(ctx, A.n_sd))) return rc;
    if (bump_epoch && (rc = next_epoch(ctx))) return rc;
    const PhiloxKeys pk = make_philox_keys(A.seed, step, ctx->index_base);
    StepLinks l = links;
    l.resident = src.resident;
    if ((rc = note_cuda(ctx, launch_cell_fused(ctx, src.kind, src.run_idx, src.idxbits, src.cc,
                                               src.resident ? ctx->ws.res_xi : A.xi, src.resident ? ctx->ws.res_v : A.v,
                                               A.n_sd, A.n_cell, A.dtdV, A.dkp, pk, l))))
        return rc;
    ctx->last_path = src.kind == 0 ? SDM_PATH_CELL_SORTED : SDM_PATH_HYBRID;
    return SDM_OK;
}

// Waits, WITHOUT draining the stream behind it, until k_cell_bounds of `epoch` has published its verdict in the
// mapped status block: the worst cell-size class (CELL_CLASSES = the fused kernel cannot take this input) and the
// number of cells per class.  Cells of nearly one size are all served as the worst class (no indirection); mixed
// sizes go through the class lists k_cell_classes has written.
int wait_verdict(sdm_ctx* ctx, u32 epoch, int32_t n_cell, CellClasses* cc) {
    volatile u32* m = ctx->mapped;
    for (unsigned long spin = 1;; ++spin) {
        if (m[MAPPED_VERDICT_EPOCH] == epoch) break;
        if ((spin & 0xFFFu) == 0) {  // the stream ran dry without a verdict: a launch failed
            const cudaError_t q = cudaStreamQuery(ctx->stream);
            if (q == cudaErrorNotReady) { (void)cudaGetLastError(); continue; }
            if (q != cudaSuccess) return note_cuda(ctx, q);
            if (m[MAPPED_VERDICT_EPOCH] == epoch) break;
            return note_cuda(ctx, cudaErrorUnknown);
        }
    }
    std::atomic_thread_fence(std::memory_order_acquire);
    cc->worst = m[MAPPED_VERDICT_CLASS];
    cc->mixed = false;
    cc->cell_offset = 0;
    for (int k = 0; k < CELL_CLASSES; ++k) cc->count[k] = 0;
    if (cc->worst >= (u32)CELL_CLASSES) return SDM_OK;
    uint64_t total = 0;
    for (int k = 0; k < CELL_CLASSES; ++k) total += (cc->count[k] = m[MAPPED_CLASS_COUNT + k]);
    if (total != (uint64_t)n_cell) return note_cuda(ctx, cudaErrorUnknown);  // cannot happen: every cell is listed once
    if ((uint64_t)cc->count[cc->worst] * 4u >= (uint64_t)n_cell * 3u) {
        for (int k = 0; k < CELL_CLASSES; ++k) cc->count[k] = (u32)k == cc->worst ? (u32)n_cell : 0u;
        return SDM_OK;
    }
    cc->mixed = true;
    return SDM_OK;
}

// AUTO's hint: what the last GENERAL step on this very (cell_id pointer, n_sd, n_cell) saw.  Waits for its
// asynchronous copy (AUTO waits for the analysis enqueued behind it anyway).  Returns false when there is none.
bool auto_hint(sdm_ctx* ctx, const StepArgs& A, Verdict* hint) {
    if (!(ctx->verdict_valid && ctx->verdict_cell_ptr == A.cell_id && ctx->verdict_n_sd == A.n_sd &&
          ctx->verdict_n_cell == A.n_cell))
        return false;
    if (note_cuda(ctx, cudaEventSynchronize(ctx->verdict_event)) != SDM_OK) return false;
    *hint = *ctx->verdict_host;
    return true;
}

// AUTO: analyses cell_id on the device, waits for the verdict and prepares the fused kernel's input when it fits.
// *fits = false: take the GENERAL path (nothing was updated).  The analysis never raises SDM_ERR_BAD_DATA by itself.
int auto_prepare(sdm_ctx* ctx, const StepArgs& A, const Plan& plan, bool* fits, FusedSource* src) {
    *fits = false;
    if (A.n_cell <= 1) return SDM_OK;
    Verdict hint;
    const bool have_hint = auto_hint(ctx, A, &hint);
    if (have_hint && hint.max_count > (u32)CELL_FAST_MAX) return SDM_OK;
    int rc;
    src->cc.worst = (u32)CELL_CLASSES;
    if (!have_hint || !hint.unsorted) {
        if ((rc = enqueue_sorted_prepare(ctx, A, false, src))) return rc;
        if ((rc = wait_verdict(ctx, ctx->epoch, A.n_cell, &src->cc))) return rc;
    } else if (hybrid_fits(plan)) {
        if ((rc = enqueue_hybrid_prepare(ctx, A, plan, false, src))) return rc;
        if ((rc = wait_verdict(ctx, ctx->epoch, A.n_cell, &src->cc))) return rc;
    }
    *fits = src->cc.worst < (u32)CELL_CLASSES;
    return SDM_OK;
}

// An explicitly chosen CELL_SORTED / HYBRID path: the same analysis, but an input that does not fit is the caller's
// error -- k_cell_bounds (strict) has then raised the sticky SDM_ERR_BAD_DATA and nothing is updated.
int explicit_prepare(sdm_ctx* ctx, const StepArgs& A, const Plan& plan, bool hybrid, bool* fits, FusedSource* src) {
    int rc;
    if ((rc = hybrid ? enqueue_hybrid_prepare(ctx, A, plan, true, src) : enqueue_sorted_prepare(ctx, A, true, src))) return rc;
    if ((rc = wait_verdict(ctx, ctx->epoch, A.n_cell, &src->cc))) return rc;
    *fits = src->cc.worst < (u32)CELL_CLASSES;
    return SDM_OK;
}

}  // namespace

int sdm_coalescence_step(sdm_ctx* ctx, int64_t* multiplicity, double* volume, const int32_t* cell_id,
                         int64_t n_sd, int32_t n_cell, double dt, double dV, const sdm_kernel_params* kp,
                         uint64_t seed, uint64_t step) {
    int rc = validate_step(ctx, multiplicity, volume, cell_id, n_sd, n_cell, dt, dV, kp);
    if (rc != SDM_OK) return rc;
    if (n_sd > 0 && (!aligned16(multiplicity) || !aligned16(volume))) return SDM_ERR_INVALID_ARG;
    if (ctx->cuda_error) return SDM_ERR_CUDA;
    if (cudaSetDevice(ctx->device) != cudaSuccess) return SDM_ERR_CUDA;
    const Plan plan = make_plan(n_sd, n_cell, ctx->skip_key_digits);
    if (!plan_fits(plan)) return SDM_ERR_CAPACITY;
    if (n_sd == 0) {  // legal no-op; the debug cell_start is still defined (all zeros)
        if (ctx->dbg_cell_start)
            if ((rc = note_cuda(ctx, cudaMemsetAsync(ctx->dbg_cell_start, 0, ((size_t)n_cell + 1) * 4, ctx->stream))))
                return rc;
        return SDM_OK;
    }
    const StepArgs A = make_step_args(ctx, multiplicity, volume, cell_id, n_sd, n_cell, dt, dV, kp, seed);
    const StepLinks no_links = {nullptr, nullptr, nullptr, 0u, 1u, false};
    ctx->zero_hint_valid = 0;
    // ---- path selection (include/sdm.h, sdm_path) ----
    FusedSource src;
    bool fused = false;
    if (n_cell > 1 && (ctx->path == SDM_PATH_CELL_SORTED || (ctx->path == SDM_PATH_HYBRID && hybrid_fits(plan)))) {
        if ((rc = explicit_prepare(ctx, A, plan, ctx->path == SDM_PATH_HYBRID, &fused, &src))) return rc;
        if (!fused) {  // refused: the step is skipped as a whole, the sticky flag reports it
            ctx->last_path = ctx->path;
            return SDM_OK;
        }
    } else if (ctx->path == SDM_PATH_AUTO) {
        if ((rc = auto_prepare(ctx, A, plan, &fused, &src))) return rc;
    }
    if (!fused) return enqueue_unfused_step(ctx, A, step);
    if ((rc = enqueue_fused_step(ctx, A, src, step, no_links, false))) return rc;
    note_zero_hint(ctx, multiplicity, n_sd);
    return SDM_OK;
}

// ---- sdm_remove_zero_multiplicity and its parts ----
namespace {

// Enqueues the in-place compaction of a known number of zeros (> 0).
int enqueue_compact(sdm_ctx* ctx, int64_t* xi, double* v, int32_t* cell_id, int64_t n_sd) {
    int rc;
    cudaStream_t st = ctx->stream;
    const size_t n_tiles = (size_t)((n_sd + CMP_TILE - 1) / CMP_TILE);
    if ((rc = note_cuda(ctx, cudaMemsetAsync(ctx->ws.ctl + CTL_CMP_TICKET, 0, 4, st)))) return rc;
    if ((rc = note_cuda(ctx, cudaMemsetAsync(ctx->ws.cmp_state, 0, n_tiles * 4, st)))) return rc;
    return note_cuda(ctx, launch_compact(ctx, xi, v, cell_id, n_sd));
}

}  // namespace

int sdm_remove_zero_multiplicity(sdm_ctx* ctx, int64_t* multiplicity, double* volume, int32_t* cell_id,
                                 int64_t n_sd, int64_t* n_sd_out) {
    if (!ctx || !n_sd_out || n_sd < 0) return SDM_ERR_INVALID_ARG;
    if (n_sd > 0 && (!multiplicity || !volume || !cell_id)) return SDM_ERR_INVALID_ARG;
    if (n_sd > 0 && !aligned16(multiplicity)) return SDM_ERR_INVALID_ARG;
    if (n_sd > ctx->max_n_sd) return SDM_ERR_CAPACITY;
    if (ctx->cuda_error) return SDM_ERR_CUDA;
    if (cudaSetDevice(ctx->device) != cudaSuccess) return SDM_ERR_CUDA;
    *n_sd_out = n_sd;
    int rc;
    cudaStream_t st = ctx->stream;
    // one 512-byte copy into pinned memory reports the sticky words [0, 64) and the control block [64, 128)
    u32* hs = ctx->status_host;
    // SDM_OPT_TRACK_ZEROS: the fused step kernel that just updated this very array counted its zeros
    bool hinted = ctx->zero_hint_valid && ctx->zero_hint_xi == multiplicity && ctx->zero_hint_n_sd == n_sd && n_sd > 0;
    ctx->zero_hint_valid = 0;
    for (int attempt = 0; attempt < 2; ++attempt) {
        if (n_sd > 0 && !hinted) {
            if ((rc = note_cuda(ctx, cudaMemsetAsync(ctx->ws.ctl + CTL_ZERO_COUNT, 0, 4, st)))) return rc;
            if ((rc = note_cuda(ctx, launch_count_zero(ctx, multiplicity, n_sd)))) return rc;
        }
        if ((rc = note_cuda(ctx, cudaMemcpyAsync(hs, ctx->ws.sticky, (STICKY_WORDS + CTL_WORDS) * 4,
                                                 cudaMemcpyDeviceToHost, st))))
            return rc;
        if ((rc = note_cuda(ctx, cudaStreamSynchronize(st)))) return rc;
        if (!(hinted && hs[STICKY_WORDS + CTL_UNSORTED] == ctx->epoch)) break;
        hinted = false;  // the step refused its input and counted nothing: count now
    }
    const int64_t zeros = n_sd > 0 ? (int64_t)hs[STICKY_WORDS + CTL_ZERO_COUNT] : 0;
    const u32 bad_data = hs[STICKY_BAD_DATA];
    if (zeros > 0)
        if ((rc = enqueue_compact(ctx, multiplicity, volume, cell_id, n_sd))) return rc;
    *n_sd_out = n_sd - zeros;
    // stable compaction keeps a sorted cell_id sorted and cannot grow a cell: AUTO's hint carries over
    if (ctx->verdict_valid && ctx->verdict_cell_ptr == cell_id && ctx->verdict_n_sd == n_sd)
        ctx->verdict_n_sd = n_sd - zeros;
    if (bad_data) {
        cudaMemsetAsync(ctx->ws.sticky, 0, STICKY_WORDS * 4, st);
        ctx->verdict_valid = 0;
        return SDM_ERR_BAD_DATA;
    }
    return SDM_OK;
}

// ---- sdm_coalescence_steps: the time loop on the device ----
namespace {

constexpr int64_t RUN_CHUNK = 64;  // fused steps enqueued between two looks at the halt word
constexpr int64_t RUN_STEPS_PER_LAUNCH = 64;  // at most this many steps inside one launch of the fused kernel (= one chunk)
// HYBRID runs at least this long keep cell-grouped copies of the attributes (interleaved configs[3]: the two moves cost
// 670 us together, every step saves 110 us)
constexpr int64_t RUN_RESIDENT_MIN_STEPS = 8;
constexpr int64_t RUN_MULTI_STEP_MAX_SD = 1 << 21;  // ... for problems up to this size (configs[2]: 7.6 -> 3.4 us per step)

// Reads and clears the sticky data-error flag after the stream has been drained.
int finish_run(sdm_ctx* ctx) {
    int rc;
    u32 bad = 0;
    if (ctx->side_valid) {  // a placement started ahead that no step consumed (a run cut short): nothing stays in flight
        if ((rc = note_cuda(ctx, cudaStreamWaitEvent(ctx->stream, ctx->side_done, 0)))) return rc;
        ctx->side_valid = 0;
    }
    if ((rc = note_cuda(ctx, cudaMemcpyAsync(&bad, ctx->ws.sticky + STICKY_BAD_DATA, 4, cudaMemcpyDeviceToHost,
                                             ctx->stream))))
        return rc;
    if ((rc = note_cuda(ctx, cudaStreamSynchronize(ctx->stream)))) return rc;
    if (bad) {
        cudaMemsetAsync(ctx->ws.sticky, 0, STICKY_WORDS * 4, ctx->stream);
        ctx->verdict_valid = 0;
        return SDM_ERR_BAD_DATA;
    }
    return SDM_OK;
}

// Fused steps [*s, n_steps) of the run, enqueued chunk by chunk with no host synchronisation in between.  Each step
// counts the zero multiplicities it leaves behind (slot s mod 3 of the run block); the step after a due
// compaction looks at that count first and, when it is not 0, HALTS the run: it and every later step already
// enqueued exit without touching the state, and the host -- which watches the mapped halt word from one chunk
// behind -- compacts and resumes from the halted step.  Returns with *s = first step not yet applied,
// *halt_zeros > 0 when a compaction of that many zeros is due before step *s (stream drained), else 0.
int run_fused_steps(sdm_ctx* ctx, const StepArgs& A, const FusedSource& src_in, uint64_t step0, int64_t* s,
                    int64_t n_steps, int64_t compact_every, bool allow_resident, int64_t* halt_zeros) {
    int rc;
    FusedSource src = src_in;
    cudaStream_t st = ctx->stream;
    u32* run = ctx->ws.run;
    *halt_zeros = 0;
    const int64_t s_begin = *s;
    ctx->mapped[MAPPED_HALT] = 0u;
    if ((rc = note_cuda(ctx, cudaMemsetAsync(run + RUN_HALT, 0, 4 * 4, st)))) return rc;  // halt word + three zero slots
    int64_t enq = s_begin;  // steps enqueued so far
    int64_t launch = 0;     // launches so far: launch L counts its zeros into slot L mod 3
    int n_chunks = 0;
    bool halted = false;
    // cells never interact, so one launch can take its cells through several steps (k_cell_fused, n_steps) as long as no
    // compaction falls between them; debug outputs describe one step
    // (large problems gain nothing -- configs[4]: 93 us per step either way -- and keep the shorter launches)
    const bool debug_out = ctx->dbg_perm || ctx->dbg_gamma || ctx->dbg_gamma_clamped || ctx->dbg_cell_start;
    const bool one_by_one = debug_out || A.n_sd > RUN_MULTI_STEP_MAX_SD || !fused_multi_step(ctx, src.cc);
    // HYBRID: a long enough run works on cell-grouped copies of the attributes (gathered once here,
    // scattered back below) instead of gathering them through the index words in every step
    src.resident = src.kind != 0 && !debug_out && allow_resident && n_steps - s_begin >= RUN_RESIDENT_MIN_STEPS;
    if (src.resident &&
        (rc = note_cuda(ctx, launch_resident_move(ctx, false, src.kind, src.run_idx, src.idxbits, A.xi, A.v, A.n_sd))))
        return rc;
    while (enq < n_steps && !halted) {
        const int64_t c_end = (n_steps - enq > RUN_CHUNK) ? enq + RUN_CHUNK : n_steps;
        while (enq < c_end) {
            int64_t k = c_end - enq < RUN_STEPS_PER_LAUNCH ? c_end - enq : RUN_STEPS_PER_LAUNCH;
            if (compact_every > 0 && compact_every - (enq % compact_every) < k) k = compact_every - (enq % compact_every);
            if (one_by_one) k = 1;
            StepLinks links;
            links.zc_accum = run + RUN_ZC0 + (launch % 3);
            links.zc_clear = run + RUN_ZC0 + ((launch + 1) % 3);
            const bool due_before = compact_every > 0 && enq > s_begin && (enq % compact_every) == 0;
            links.zc_check = due_before ? run + RUN_ZC0 + ((launch + 2) % 3) : nullptr;  // the previous launch's slot
            links.halt_tag = (u32)(enq - s_begin) + 1u;
            links.n_steps = (u32)k;
            if ((rc = enqueue_fused_step(ctx, A, src, step0 + (uint64_t)enq, links, true))) return rc;
            enq += k;
            ++launch;
        }
        if ((rc = note_cuda(ctx, cudaEventRecord(ctx->chunk_event[n_chunks & 1], st)))) return rc;
        ++n_chunks;
        if (n_chunks >= 2) {  // one chunk stays queued behind the one that is running
            if ((rc = note_cuda(ctx, cudaEventSynchronize(ctx->chunk_event[n_chunks & 1])))) return rc;
            halted = ctx->mapped[MAPPED_HALT] != 0u;
        }
    }
    // (a halted run left the copies as the last applied step wrote them)
    if (src.resident &&
        (rc = note_cuda(ctx, launch_resident_move(ctx, true, src.kind, src.run_idx, src.idxbits, A.xi, A.v, A.n_sd))))
        return rc;
    if ((rc = note_cuda(ctx, cudaStreamSynchronize(st)))) return rc;
    std::atomic_thread_fence(std::memory_order_acquire);
    const u32 tag = ctx->mapped[MAPPED_HALT];
    if (tag != 0u) {  // steps before s_begin + tag - 1 were applied; that one and all later ones were not
        *s = s_begin + (int64_t)tag - 1;
        *halt_zeros = (int64_t)ctx->mapped[MAPPED_ZEROS];
        return SDM_OK;
    }
    *s = n_steps;
    // a compaction due after the last step: its count sits in that step's slot
    if (compact_every > 0 && n_steps > s_begin && (n_steps % compact_every) == 0) {
        u32 z = 0;
        if ((rc = note_cuda(ctx, cudaMemcpy(&z, run + RUN_ZC0 + ((launch + 2) % 3), 4, cudaMemcpyDeviceToHost)))) return rc;
        *halt_zeros = (int64_t)z;
    }
    return SDM_OK;
}

}  // namespace

int sdm_coalescence_steps(sdm_ctx* ctx, int64_t* multiplicity, double* volume, int32_t* cell_id, int64_t n_sd,
                          int32_t n_cell, double dt, double dV, const sdm_kernel_params* kp, uint64_t seed,
                          uint64_t step0, int64_t n_steps, int64_t compact_every, int64_t* n_sd_out) {
    int rc = validate_step(ctx, multiplicity, volume, cell_id, n_sd, n_cell, dt, dV, kp);
    if (rc != SDM_OK) return rc;
    if (!n_sd_out || n_steps < 0 || compact_every < 0) return SDM_ERR_INVALID_ARG;
    if (n_sd > 0 && (!aligned16(multiplicity) || !aligned16(volume))) return SDM_ERR_INVALID_ARG;
    if (ctx->cuda_error) return SDM_ERR_CUDA;
    if (cudaSetDevice(ctx->device) != cudaSuccess) return SDM_ERR_CUDA;
    *n_sd_out = n_sd;
    ctx->zero_hint_valid = 0;
    int64_t n = n_sd;
    int64_t s = 0;
    bool general_only = (n_cell <= 1) || ctx->path == SDM_PATH_GENERAL || ctx->path == SDM_PATH_BOX || ctx->path == SDM_PATH_BUCKET;
    bool allow_resident = true;
    while (s < n_steps && n > 0) {
        const StepArgs A = make_step_args(ctx, multiplicity, volume, cell_id, n, n_cell, dt, dV, kp, seed);
        const Plan plan = make_plan(n, n_cell, ctx->skip_key_digits);
        if (!plan_fits(plan)) return SDM_ERR_CAPACITY;
        FusedSource src;
        bool fused = false;
        if (!general_only) {
            if (ctx->path == SDM_PATH_AUTO) {
                if ((rc = auto_prepare(ctx, A, plan, &fused, &src))) return rc;
            } else {  // explicit CELL_SORTED / HYBRID: an input that does not fit is the caller's error
                const bool hybrid = ctx->path == SDM_PATH_HYBRID;
                if (hybrid && !hybrid_fits(plan)) {
                    general_only = true;
                    continue;
                }
                if ((rc = explicit_prepare(ctx, A, plan, hybrid, &fused, &src))) return rc;
                if (!fused) {
                    *n_sd_out = n;
                    rc = finish_run(ctx);
                    return rc != SDM_OK ? rc : SDM_ERR_BAD_DATA;
                }
            }
        }
        int64_t zeros = 0;
        if (fused) {
            const int64_t s_before = s;
            if ((rc = run_fused_steps(ctx, A, src, step0, &s, n_steps, compact_every, allow_resident, &zeros))) return rc;
            // compactions that keep finding zeros after a few steps: the next runs gather in every step instead
            if (zeros > 0 && s - s_before < RUN_RESIDENT_MIN_STEPS) allow_resident = false;
            if (zeros > 0) {
                if ((rc = enqueue_compact(ctx, multiplicity, volume, cell_id, n))) return rc;
                n -= zeros;
            }
        } else {
            // GENERAL steps; under AUTO the first one also tells whether the fused kernel could take this array
            // (cells of at most 256 super-droplets), and the loop comes back to try
            bool retry_fused = false;
            while (s < n_steps && !retry_fused) {
                if (box_fits(ctx, A)) {  // every step up to the next due compaction in one launch
                    int64_t k = n_steps - s;
                    if (compact_every > 0 && compact_every - (s % compact_every) < k) k = compact_every - (s % compact_every);
                    if ((rc = enqueue_box_steps(ctx, A, step0 + (uint64_t)s, &k))) return rc;
                    s += k;
                } else {
                    // the next iteration runs step s + 1 on the same arrays unless the run ends or a compaction is due
                    const bool next_follows = general_only && s + 1 < n_steps && !(compact_every > 0 && ((s + 1) % compact_every) == 0);
                    if ((rc = enqueue_unfused_step(ctx, A, step0 + (uint64_t)s, next_follows))) return rc;
                    ++s;
                }
                if (!general_only) {
                    Verdict hint;
                    if (auto_hint(ctx, A, &hint) && hint.max_count <= (u32)CELL_FAST_MAX && hint.unsorted &&
                        hybrid_fits(plan))
                        retry_fused = true;
                    else
                        general_only = true;
                }
                if (compact_every > 0 && (s % compact_every) == 0) {
                    int64_t n_new = n;
                    if ((rc = sdm_remove_zero_multiplicity(ctx, multiplicity, volume, cell_id, n, &n_new))) return rc;
                    if (n_new != n) {
                        n = n_new;
                        break;  // the arrays shrank: new plan
                    }
                }
            }
        }
    }
    *n_sd_out = n;
    return finish_run(ctx);
}

int sdm_cell_stats(sdm_ctx* ctx, const int64_t* multiplicity, const double* volume, const int32_t* cell_id,
                   int64_t n_sd, int32_t n_cell, int32_t* count, int64_t* sum_xi, double* sum_xi_v,
                   double* sum_xi_v2) {
    if (!ctx || n_sd < 0 || n_cell < 1) return SDM_ERR_INVALID_ARG;
    if (n_sd > 0 && (!multiplicity || !volume || !cell_id)) return SDM_ERR_INVALID_ARG;
    if (ctx->cuda_error) return SDM_ERR_CUDA;
    if (cudaSetDevice(ctx->device) != cudaSuccess) return SDM_ERR_CUDA;
    int rc;
    cudaStream_t st = ctx->stream;
    if (count && (rc = note_cuda(ctx, cudaMemsetAsync(count, 0, (size_t)n_cell * 4, st)))) return rc;
    if (sum_xi && (rc = note_cuda(ctx, cudaMemsetAsync(sum_xi, 0, (size_t)n_cell * 8, st)))) return rc;
    if (sum_xi_v && (rc = note_cuda(ctx, cudaMemsetAsync(sum_xi_v, 0, (size_t)n_cell * 8, st)))) return rc;
    if (sum_xi_v2 && (rc = note_cuda(ctx, cudaMemsetAsync(sum_xi_v2, 0, (size_t)n_cell * 8, st)))) return rc;
    if (n_sd == 0) return SDM_OK;
    return note_cuda(ctx, launch_cell_stats(ctx, multiplicity, volume, cell_id, n_sd, n_cell, count, sum_xi,
                                            sum_xi_v, sum_xi_v2));
}

int sdm_cell_id_from_positions(sdm_ctx* ctx, const double* x, const double* z, int64_t n_sd, int32_t nx, int32_t nz,
                               int32_t* cell_id) {
    if (!ctx || n_sd < 0 || nx < 1 || nz < 1 || (int64_t)nx * nz > 2147483647LL) return SDM_ERR_INVALID_ARG;
    if (n_sd > 0 && (!x || !z || !cell_id)) return SDM_ERR_INVALID_ARG;
    if (ctx->cuda_error) return SDM_ERR_CUDA;
    if (n_sd == 0) return SDM_OK;
    if (cudaSetDevice(ctx->device) != cudaSuccess) return SDM_ERR_CUDA;
    return note_cuda(ctx, launch_displace(ctx, false, const_cast<double*>(x), const_cast<double*>(z), cell_id, n_sd, nx,
                                          nz, nullptr, nullptr, 0.0));
}

int sdm_displace(sdm_ctx* ctx, double* x, double* z, int32_t* cell_id, int64_t n_sd, int32_t nx, int32_t nz,
                 const double* u_cell, const double* w_cell, double dt) {
    if (!ctx || n_sd < 0 || nx < 1 || nz < 1 || (int64_t)nx * nz > 2147483647LL) return SDM_ERR_INVALID_ARG;
    if (!(dt > 0.0) || !std::isfinite(dt) || !u_cell || !w_cell) return SDM_ERR_INVALID_ARG;
    if (n_sd > 0 && (!x || !z || !cell_id)) return SDM_ERR_INVALID_ARG;
    if (ctx->cuda_error) return SDM_ERR_CUDA;
    if (n_sd == 0) return SDM_OK;
    if (cudaSetDevice(ctx->device) != cudaSuccess) return SDM_ERR_CUDA;
    return note_cuda(ctx, launch_displace(ctx, true, x, z, cell_id, n_sd, nx, nz, u_cell, w_cell, dt));
}

int sdm_set_collision_efficiency(sdm_ctx* ctx, const double* radius, int32_t n_r, int32_t n_p, const double* table) {
    if (!ctx) return SDM_ERR_INVALID_ARG;
    if (!radius && !table && n_r == 0 && n_p == 0) {  // remove the table
        ctx->eff_n_r = ctx->eff_n_p = 0;
        return SDM_OK;
    }
    if (!radius || !table || n_r < 2 || n_p < 2) return SDM_ERR_INVALID_ARG;
    if (n_r > EFF_MAX_R || n_p > EFF_MAX_P) return SDM_ERR_CAPACITY;
    double e_max = 0.0;
    for (int32_t i = 0; i < n_r; ++i) {
        if (!std::isfinite(radius[i]) || (i > 0 && !(radius[i] > radius[i - 1]))) return SDM_ERR_INVALID_ARG;
        for (int32_t j = 0; j < n_p; ++j) {
            const double e = table[(size_t)i * n_p + j];
            if (!std::isfinite(e) || e < 0.0) return SDM_ERR_INVALID_ARG;
            if (e > e_max) e_max = e;
        }
    }
    if (ctx->cuda_error) return SDM_ERR_CUDA;
    if (cudaSetDevice(ctx->device) != cudaSuccess) return SDM_ERR_CUDA;
    int rc;
    // pageable host memory: both copies are staged before the call returns
    if ((rc = note_cuda(ctx, cudaMemcpyAsync(ctx->ws.eff_radius, radius, (size_t)n_r * 8, cudaMemcpyHostToDevice,
                                             ctx->stream))))
        return rc;
    if ((rc = note_cuda(ctx, cudaMemcpyAsync(ctx->ws.eff_table, table, (size_t)n_r * n_p * 8, cudaMemcpyHostToDevice,
                                             ctx->stream))))
        return rc;
    ctx->eff_n_r = n_r;
    ctx->eff_n_p = n_p;
    ctx->eff_max = e_max;
    return SDM_OK;
}

int sdm_poll_error(sdm_ctx* ctx) {
    if (!ctx) return SDM_ERR_INVALID_ARG;
    if (ctx->cuda_error) return SDM_ERR_CUDA;
    if (cudaSetDevice(ctx->device) != cudaSuccess) return SDM_ERR_CUDA;
    u32 bad = 0;
    int rc;
    if ((rc = note_cuda(ctx, cudaMemcpyAsync(&bad, ctx->ws.sticky + STICKY_BAD_DATA, 4, cudaMemcpyDeviceToHost,
                                             ctx->stream))))
        return rc;
    if ((rc = note_cuda(ctx, cudaStreamSynchronize(ctx->stream)))) return rc;
    if (bad) {
        cudaMemsetAsync(ctx->ws.sticky, 0, STICKY_WORDS * 4, ctx->stream);
        ctx->verdict_valid = 0;  // AUTO re-learns the cell order on the next step
        return SDM_ERR_BAD_DATA;
    }
    return SDM_OK;
}

size_t sdm_host_staging_bytes(int64_t max_n_sd) {
    if (max_n_sd < 0 || max_n_sd >= (1LL << 30)) return 0;
    const size_t n = (size_t)max_n_sd;
    return align_up(n * 8 + 16, 256) * 2 + align_up(n * 4 + 16, 256);
}

int sdm_bind_host_staging(sdm_ctx* ctx, void* staging_dev, size_t staging_bytes) {
    if (!ctx || !staging_dev) return SDM_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(staging_dev) & 255u) != 0) return SDM_ERR_INVALID_ARG;
    if (staging_bytes < sdm_host_staging_bytes(ctx->max_n_sd)) return SDM_ERR_CAPACITY;
    ctx->staging = staging_dev;
    ctx->staging_bytes = staging_bytes;
    if (!ctx->copy_in) {  // the host entry point overlaps uploads, step and downloads on streams of its own
        if (cudaSetDevice(ctx->device) != cudaSuccess) return SDM_ERR_CUDA;
        if (cudaStreamCreateWithFlags(&ctx->copy_in, cudaStreamNonBlocking) != cudaSuccess ||
            cudaStreamCreateWithFlags(&ctx->copy_out, cudaStreamNonBlocking) != cudaSuccess)
            return SDM_ERR_CUDA;
        for (int k = 0; k < HOST_CHUNKS; ++k)
            if (cudaEventCreateWithFlags(&ctx->host_in[k], cudaEventDisableTiming) != cudaSuccess ||
                cudaEventCreateWithFlags(&ctx->host_done[k], cudaEventDisableTiming) != cudaSuccess)
                return SDM_ERR_CUDA;
    }
    return SDM_OK;
}

namespace {

// The host entry point as a pipeline (cell-major arrays of many small cells: configs[2..4]).  cell_id goes up first and is
// analysed as a whole; the attributes go up in HOST_CHUNKS pieces cut at cell boundaries on a stream of their own, the
// fused kernel runs on the cells of a piece as soon as it has arrived, and the piece goes back on a third stream while
// the next one is still arriving -- PCIe carries both directions at once, so the call costs about the larger of upload
// and download instead of their sum.  Returns SDM_OK with *done = false when the input does not qualify (nothing has
// been applied; cell_id and the attributes are on the device by then, on ctx->stream's side of an event): the caller
// runs the plain sequence.
int host_step_pipelined(sdm_ctx* ctx, int64_t* xi_h, double* v_h, int32_t* c_h, int64_t* d_xi, double* d_v, int32_t* d_c,
                        int64_t n_sd, int32_t n_cell, double dt, double dV, const sdm_kernel_params* kp, uint64_t seed,
                        uint64_t step, int compact, int64_t* n_sd_out, bool* done) {
    int rc;
    *done = false;
    cudaStream_t st = ctx->stream;
    // piece boundaries: whole cells (the lower bound of a cell id in the -- presumably sorted -- host array)
    int64_t cut[HOST_CHUNKS + 1];
    int32_t cell_cut[HOST_CHUNKS + 1];
    for (int k = 0; k <= HOST_CHUNKS; ++k) {
        cell_cut[k] = (int32_t)(((int64_t)n_cell * k) / HOST_CHUNKS);
        cut[k] = k == HOST_CHUNKS ? n_sd : (int64_t)(std::lower_bound(c_h, c_h + n_sd, cell_cut[k]) - c_h);
    }
    cut[0] = 0;
    for (int k = 1; k <= HOST_CHUNKS; ++k)  // an unsorted array gives arbitrary bounds: keep the pieces a partition of [0, n_sd)
        if (cut[k] < cut[k - 1]) cut[k] = cut[k - 1];
    if ((rc = note_cuda(ctx, cudaMemcpyAsync(d_c, c_h, (size_t)n_sd * 4, cudaMemcpyHostToDevice, st)))) return rc;
    for (int k = 0; k < HOST_CHUNKS; ++k) {
        const size_t off = (size_t)cut[k], len = (size_t)(cut[k + 1] - cut[k]);
        if (len) {
            if ((rc = note_cuda(ctx, cudaMemcpyAsync(d_xi + off, xi_h + off, len * 8, cudaMemcpyHostToDevice, ctx->copy_in)))) return rc;
            if ((rc = note_cuda(ctx, cudaMemcpyAsync(d_v + off, v_h + off, len * 8, cudaMemcpyHostToDevice, ctx->copy_in)))) return rc;
        }
        if ((rc = note_cuda(ctx, cudaEventRecord(ctx->host_in[k], ctx->copy_in)))) return rc;
    }
    // the analysis of the whole array: sorted, small cells of nearly one size?
    const StepArgs A = make_step_args(ctx, d_xi, d_v, d_c, n_sd, n_cell, dt, dV, kp, seed);
    FusedSource src;
    if ((rc = enqueue_sorted_prepare(ctx, A, false, &src))) return rc;
    if ((rc = wait_verdict(ctx, ctx->epoch, n_cell, &src.cc))) return rc;
    if (src.cc.worst >= (u32)CELL_CLASSES || src.cc.mixed) {
        // not this path's input: hand the (uploaded) arrays to the plain sequence
        if ((rc = note_cuda(ctx, cudaStreamWaitEvent(st, ctx->host_in[HOST_CHUNKS - 1], 0)))) return rc;
        return SDM_OK;
    }
    // sorted (verified on the device), so the lower bounds above are the cells' true first entries
    if ((rc = clear_debug_gammas(ctx, n_sd))) return rc;
    const PhiloxKeys pk = make_philox_keys(seed, step, ctx->index_base);
    const StepLinks no_links = {nullptr, nullptr, nullptr, 0u, 1u, false};
    for (int k = 0; k < HOST_CHUNKS; ++k) {
        const size_t off = (size_t)cut[k], len = (size_t)(cut[k + 1] - cut[k]);
        const u32 cells = (u32)(cell_cut[k + 1] - cell_cut[k]);
        if ((rc = note_cuda(ctx, cudaStreamWaitEvent(st, ctx->host_in[k], 0)))) return rc;
        if (cells) {
            CellClasses cc = src.cc;
            cc.count[cc.worst] = cells;
            cc.cell_offset = (u32)cell_cut[k];
            if ((rc = note_cuda(ctx, launch_cell_fused(ctx, 0, nullptr, 0, cc, d_xi, d_v, n_sd, n_cell, A.dtdV, A.dkp, pk, no_links))))
                return rc;
        }
        if ((rc = note_cuda(ctx, cudaEventRecord(ctx->host_done[k], st)))) return rc;
        if ((rc = note_cuda(ctx, cudaStreamWaitEvent(ctx->copy_out, ctx->host_done[k], 0)))) return rc;
        if (len) {
            if ((rc = note_cuda(ctx, cudaMemcpyAsync(xi_h + off, d_xi + off, len * 8, cudaMemcpyDeviceToHost, ctx->copy_out)))) return rc;
            if ((rc = note_cuda(ctx, cudaMemcpyAsync(v_h + off, d_v + off, len * 8, cudaMemcpyDeviceToHost, ctx->copy_out)))) return rc;
        }
    }
    ctx->last_path = SDM_PATH_CELL_SORTED;
    *done = true;
    int64_t n_out = n_sd;
    if (compact) {
        // the fused launches have counted the zeros (k_cell_bounds cleared the count): no counting pass
        ctx->zero_hint_valid = 1;
        ctx->zero_hint_xi = d_xi;
        ctx->zero_hint_n_sd = n_sd;
        if ((rc = sdm_remove_zero_multiplicity(ctx, d_xi, d_v, d_c, n_sd, &n_out))) return rc;
        *n_sd_out = n_out;
        if (n_out != n_sd) {  // entries moved: what is on its way to the host is stale -- fetch the compacted arrays
            if ((rc = note_cuda(ctx, cudaStreamSynchronize(ctx->copy_out)))) return rc;
            if ((rc = note_cuda(ctx, cudaMemcpyAsync(c_h, d_c, (size_t)n_out * 4, cudaMemcpyDeviceToHost, st)))) return rc;
            if ((rc = note_cuda(ctx, cudaMemcpyAsync(xi_h, d_xi, (size_t)n_out * 8, cudaMemcpyDeviceToHost, st)))) return rc;
            if ((rc = note_cuda(ctx, cudaMemcpyAsync(v_h, d_v, (size_t)n_out * 8, cudaMemcpyDeviceToHost, st)))) return rc;
        }
    }
    if ((rc = note_cuda(ctx, cudaStreamSynchronize(ctx->copy_out)))) return rc;
    return finish_run(ctx);
}

}  // namespace

int sdm_coalescence_step_host(sdm_ctx* ctx, int64_t* multiplicity_host, double* volume_host,
                              int32_t* cell_id_host, int64_t n_sd, int32_t n_cell, double dt, double dV,
                              const sdm_kernel_params* kp, uint64_t seed, uint64_t step, int compact,
                              int64_t* n_sd_out) {
    int rc = validate_step(ctx, multiplicity_host, volume_host, cell_id_host, n_sd, n_cell, dt, dV, kp);
    if (rc != SDM_OK) return rc;
    if (!ctx->staging || (compact && !n_sd_out)) return SDM_ERR_INVALID_ARG;
    if (n_sd_out) *n_sd_out = n_sd;
    if (n_sd == 0) return SDM_OK;
    if (cudaSetDevice(ctx->device) != cudaSuccess) return SDM_ERR_CUDA;
    const size_t n = (size_t)ctx->max_n_sd;
    char* base = reinterpret_cast<char*>(ctx->staging);
    int64_t* d_xi = reinterpret_cast<int64_t*>(base);
    double* d_v = reinterpret_cast<double*>(base + align_up(n * 8 + 16, 256));
    int32_t* d_c = reinterpret_cast<int32_t*>(base + 2 * align_up(n * 8 + 16, 256));
    cudaStream_t st = ctx->stream;
    // the staging area is refilled by every call: what AUTO learned about the previous contents does not carry over
    ctx->verdict_valid = 0;
    const bool no_debug = !ctx->dbg_perm && !ctx->dbg_cell_start;
    if (ctx->path == SDM_PATH_AUTO && n_cell > 1 && n_sd >= HOST_PIPE_MIN && no_debug && aligned16(d_xi) && aligned16(d_v)) {
        bool done = false;
        rc = host_step_pipelined(ctx, multiplicity_host, volume_host, cell_id_host, d_xi, d_v, d_c, n_sd, n_cell, dt, dV, kp, seed,
                                 step, compact, n_sd_out, &done);
        if (rc != SDM_OK || done) return rc;
    } else {
        if ((rc = note_cuda(ctx, cudaMemcpyAsync(d_xi, multiplicity_host, (size_t)n_sd * 8, cudaMemcpyHostToDevice, st)))) return rc;
        if ((rc = note_cuda(ctx, cudaMemcpyAsync(d_v, volume_host, (size_t)n_sd * 8, cudaMemcpyHostToDevice, st)))) return rc;
        if ((rc = note_cuda(ctx, cudaMemcpyAsync(d_c, cell_id_host, (size_t)n_sd * 4, cudaMemcpyHostToDevice, st)))) return rc;
    }
    rc = sdm_coalescence_step(ctx, d_xi, d_v, d_c, n_sd, n_cell, dt, dV, kp, seed, step);
    if (rc != SDM_OK) return rc;
    int64_t n_out = n_sd;
    if (compact) {
        rc = sdm_remove_zero_multiplicity(ctx, d_xi, d_v, d_c, n_sd, &n_out);
        if (rc != SDM_OK) return rc;
        *n_sd_out = n_out;
        if (n_out != n_sd)
            if ((rc = note_cuda(ctx, cudaMemcpyAsync(cell_id_host, d_c, (size_t)n_out * 4, cudaMemcpyDeviceToHost, st)))) return rc;
    }
    if ((rc = note_cuda(ctx, cudaMemcpyAsync(multiplicity_host, d_xi, (size_t)n_out * 8, cudaMemcpyDeviceToHost, st)))) return rc;
    if ((rc = note_cuda(ctx, cudaMemcpyAsync(volume_host, d_v, (size_t)n_out * 8, cudaMemcpyDeviceToHost, st)))) return rc;
    // this call synchronises anyway: report a data error of its own step now, not at some later poll
    return finish_run(ctx);
}

int sdm_philox_fill(sdm_ctx* ctx, uint64_t seed, uint64_t step, uint64_t i0, int64_t n, uint32_t* key_out,
                    double* u_out) {
    if (!ctx || n < 0) return SDM_ERR_INVALID_ARG;
    if (n == 0) return SDM_OK;
    if (cudaSetDevice(ctx->device) != cudaSuccess) return SDM_ERR_CUDA;
    return note_cuda(ctx, launch_philox_fill(ctx, make_philox_keys(seed, step), i0, n, key_out, u_out));
}

int sdm_kernel_eval(sdm_ctx* ctx, const sdm_kernel_params* kp, const double* vj, const double* vk, int64_t n,
                    double* K_out) {
    if (!ctx || !kp || n < 0 || (n > 0 && (!vj || !vk || !K_out))) return SDM_ERR_INVALID_ARG;
    if (n == 0) return SDM_OK;
    if (cudaSetDevice(ctx->device) != cudaSuccess) return SDM_ERR_CUDA;
    if (kp->kind == SDM_KERNEL_GEOMETRIC_TABLE && ctx->eff_n_r == 0) return SDM_ERR_INVALID_ARG;
    return note_cuda(ctx, launch_kernel_eval(ctx, device_kernel_params(ctx, kp), vj, vk, n, K_out));
}

}  // extern "C"
