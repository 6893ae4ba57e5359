// The C ABI of libsdm_b200.so (include/sdm.h): argument validation, workspace carving and the
// launch sequence of one coalescence step.  No device memory is allocated here; everything is
// enqueued on the caller's stream.
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
    return (24 + p.cbits + p.idxbits <= 64) && (32 + p.cbits + 12 <= 64);
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
    w.buf_a = reinterpret_cast<u64*>(take((size_t)max_n_sd * 8 + 16));
    w.buf_b = reinterpret_cast<u64*>(take((size_t)max_n_sd * 8 + 16));
    w.cmp_state = reinterpret_cast<u32*>(take(cmp_tiles * 4));
    w.spec_edges = reinterpret_cast<double*>(take((size_t)SPECTRUM_MAX_EDGES * 8));
    w.scan_state_bytes = ((size_t)max_n_cell / 4096 + 2) * 8;
    w.scan_state = reinterpret_cast<u64*>(take(w.scan_state_bytes));
    w.total_bytes = off;
    return w;
}

// hybrid words: (cell_id << idxbits | index) in 64 bits, and pass 0 stages (cell_id << 12 | tile-local index)
static bool hybrid_fits(const Plan& p) { return p.cbits >= 1 && p.cbits + p.idxbits <= 64 && p.cbits + 12 <= 64; }

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
    if (ctx->verdict_event) cudaEventDestroy(ctx->verdict_event);
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
        cudaEventCreateWithFlags(&ctx->verdict_event, cudaEventDisableTiming) != cudaSuccess) {
        free_ctx(ctx);
        return SDM_ERR_CUDA;
    }
    if (cudaMemsetAsync(ctx->ws.sticky, 0, STICKY_WORDS * 4, ctx->stream) != cudaSuccess ||
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
        case SDM_ERR_BAD_DATA: return "bad data on device (cell_id out of range or negative multiplicity)";
        default: return "unknown status";
    }
}

int sdm_set_path(sdm_ctx* ctx, int path) {
    if (!ctx || path < SDM_PATH_AUTO || path > SDM_PATH_HYBRID) return SDM_ERR_INVALID_ARG;
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
    return note_cuda(ctx, launch_volume_spectrum(ctx, multiplicity, volume, n_sd, ctx->ws.spec_edges, n_edges, count,
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
    if (kp->kind != SDM_KERNEL_GOLOVIN && kp->kind != SDM_KERNEL_GEOMETRIC) return SDM_ERR_INVALID_ARG;
    if (kp->kind == SDM_KERNEL_GOLOVIN && !(kp->b >= 0.0 && std::isfinite(kp->b))) return SDM_ERR_INVALID_ARG;
    if (kp->kind == SDM_KERNEL_GEOMETRIC && !(kp->E >= 0.0 && std::isfinite(kp->E))) return SDM_ERR_INVALID_ARG;
    if (n_sd > ctx->max_n_sd || n_cell > ctx->max_n_cell) return SDM_ERR_CAPACITY;
    return SDM_OK;
}

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
    cudaStream_t st = ctx->stream;
    Workspace& ws = ctx->ws;

    if (n_sd == 0) {  // legal no-op; the debug cell_start is still defined (all zeros)
        if (ctx->dbg_cell_start)
            if ((rc = note_cuda(ctx, cudaMemsetAsync(ctx->dbg_cell_start, 0, ((size_t)n_cell + 1) * 4, st)))) return rc;
        return SDM_OK;
    }

    if (ctx->dbg_gamma)
        if ((rc = note_cuda(ctx, cudaMemsetAsync(ctx->dbg_gamma, 0, (size_t)n_sd * 8, st)))) return rc;
    if (ctx->dbg_gamma_clamped)
        if ((rc = note_cuda(ctx, cudaMemsetAsync(ctx->dbg_gamma_clamped, 0, (size_t)n_sd * 8, st)))) return rc;
    const PhiloxKeys pk = make_philox_keys(seed, step, ctx->index_base);
    KernelParams dkp;
    dkp.kind = kp->kind;
    dkp.b = kp->b;
    dkp.Epi = kp->E * 3.141592653589793;
    const double dtdV = dt / dV;

    // one epoch per step tags the device-side flags and scan states of this step (no per-step memsets of them)
    if (++ctx->epoch >= (1u << 30)) {
        ctx->epoch = 2;
        if ((rc = note_cuda(ctx, cudaMemsetAsync(ws.scan_state, 0, ws.scan_state_bytes, st)))) return rc;
    }
    // ---- path selection (include/sdm.h, sdm_path) ----
    int path = SDM_PATH_GENERAL;
    if (n_cell > 1) {
        if (ctx->path == SDM_PATH_CELL_SORTED || ctx->path == SDM_PATH_HYBRID) {
            path = ctx->path;
        } else if (ctx->path == SDM_PATH_AUTO && ctx->verdict_valid && ctx->verdict_cell_ptr == cell_id &&
                   ctx->verdict_n_sd == n_sd && ctx->verdict_n_cell == n_cell &&
                   cudaEventQuery(ctx->verdict_event) == cudaSuccess) {
            if (ctx->verdict_host->max_count <= (u32)CELL_FAST_MAX)
                path = ctx->verdict_host->unsorted ? SDM_PATH_HYBRID : SDM_PATH_CELL_SORTED;
        }
    }
    if (path == SDM_PATH_HYBRID && !hybrid_fits(plan)) path = SDM_PATH_GENERAL;
    // register tile of the fused kernel: 32 * rmax >= the largest cell (known from the verdict under AUTO)
    int rmax = CELL_FAST_MAX / 32;
    if (ctx->path == SDM_PATH_AUTO && path != SDM_PATH_GENERAL) {
        const u32 mc = ctx->verdict_host->max_count;
        rmax = mc <= 64 ? 2 : (mc <= 128 ? 4 : 8);
    }
    ctx->zero_hint_valid = 0;
    if (path == SDM_PATH_CELL_SORTED) {
        if ((rc = note_cuda(ctx, launch_cell_bounds(ctx, 0, cell_id, n_sd, n_cell, 0, rmax)))) return rc;
        if ((rc = note_cuda(ctx, launch_cell_fused(ctx, 0, nullptr, 0, rmax, multiplicity, volume, n_sd, n_cell, dtdV, dkp,
                                                   pk))))
            return rc;
        ctx->last_path = SDM_PATH_CELL_SORTED;
        note_zero_hint(ctx, multiplicity, n_sd);
        return SDM_OK;
    }
    if (path == SDM_PATH_HYBRID) {
        const int n_cpass = plan.n_cpass;
        const bool narrow = plan.cbits + plan.idxbits <= 32 && plan.cbits + 12 <= 32;
        if ((rc = note_cuda(ctx, cudaMemsetAsync(ws.ctl, 0, ws.zero_bytes_fixed, st)))) return rc;
        if ((rc = note_cuda(ctx, cudaMemsetAsync(ws.tile_state, 0, (size_t)n_cpass * plan.n_tiles * RADIX * 4, st))))
            return rc;
        if ((rc = note_cuda(ctx, launch_cell_digit_hist(ctx, cell_id, n_sd, n_cell, plan)))) return rc;
        void* in = nullptr;
        void* out = ws.buf_a;
        for (int pass = 0; pass < n_cpass; ++pass) {
            if ((rc = note_cuda(ctx, launch_cell_sort_pass(ctx, pass, narrow, cell_id, in, out, n_sd, n_cell, plan))))
                return rc;
            in = out;
            out = (out == (void*)ws.buf_a) ? (void*)ws.buf_b : (void*)ws.buf_a;
        }
        const int kind = narrow ? 2 : 1;
        if ((rc = note_cuda(ctx, launch_cell_bounds(ctx, kind, in, n_sd, n_cell, plan.idxbits, rmax)))) return rc;
        if ((rc = note_cuda(ctx, launch_cell_fused(ctx, kind, in, plan.idxbits, rmax, multiplicity, volume, n_sd, n_cell,
                                                   dtdV, dkp, pk))))
            return rc;
        ctx->last_path = SDM_PATH_HYBRID;
        note_zero_hint(ctx, multiplicity, n_sd);
        return SDM_OK;
    }

    // zero the per-step control block, the digit histograms, the cell counts and the look-back states
    if ((rc = note_cuda(ctx, cudaMemsetAsync(ws.ctl, 0, ws.zero_bytes_fixed, st)))) return rc;
    if (n_cell > 1)
        if ((rc = note_cuda(ctx, cudaMemsetAsync(ws.cell_count, 0, ((size_t)n_cell + 1) * 4, st)))) return rc;
    if ((rc = note_cuda(ctx, cudaMemsetAsync(ws.tile_state, 0, (size_t)plan.n_pass * plan.n_tiles * RADIX * 4, st))))
        return rc;

    // a1 + a2: keys, digit histograms, cell histogram; then the cell scan
    if ((rc = note_cuda(ctx, launch_keys_hist(ctx, cell_id, n_sd, n_cell, plan, pk, ws.buf_b)))) return rc;
    if ((rc = note_cuda(ctx, launch_cell_scan(ctx, n_cell, n_sd)))) return rc;
    // a3: LSD radix passes, ping-pong between buf_b and buf_a
    u64* in = ws.buf_b;
    u64* out = ws.buf_a;
    for (int pass = 0; pass < plan.n_pass; ++pass) {
        if ((rc = note_cuda(ctx, launch_sort_pass(ctx, pass, in, out, n_sd, plan)))) return rc;
        u64* t = in; in = out; out = t;
    }
    if (plan.skip > 0)  // exact (key, index) order inside the runs the skipped digits left tied
        if ((rc = note_cuda(ctx, launch_tie_repair(ctx, in, n_sd, plan, pk)))) return rc;
    const u64* sorted = in;
    if (ctx->dbg_perm)
        if ((rc = note_cuda(ctx, launch_debug_perm(ctx, sorted, n_sd, plan)))) return rc;
    // a4: pairs
    if ((rc = note_cuda(ctx, launch_pair(ctx, sorted, multiplicity, volume, n_sd, n_cell, plan, dtdV, dkp, pk))))
        return rc;
    ctx->last_path = SDM_PATH_GENERAL;
    // what this step learned about cell_id feeds AUTO's choice for the next one (asynchronous copy)
    ctx->verdict_valid = 0;
    if (n_cell > 1 && ctx->path == SDM_PATH_AUTO) {
        if ((rc = note_cuda(ctx, cudaMemcpyAsync(ctx->verdict_host, ws.ctl + CTL_UNSORTED, sizeof(Verdict),
                                                 cudaMemcpyDeviceToHost, st))))
            return rc;
        if ((rc = note_cuda(ctx, cudaEventRecord(ctx->verdict_event, st)))) return rc;
        ctx->verdict_cell_ptr = cell_id;
        ctx->verdict_n_sd = n_sd;
        ctx->verdict_n_cell = n_cell;
        ctx->verdict_valid = 1;
    }
    return SDM_OK;
}

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
    if (zeros > 0) {
        const size_t n_tiles = (size_t)((n_sd + CMP_TILE - 1) / CMP_TILE);
        if ((rc = note_cuda(ctx, cudaMemsetAsync(ctx->ws.ctl + CTL_CMP_TICKET, 0, 4, st)))) return rc;
        if ((rc = note_cuda(ctx, cudaMemsetAsync(ctx->ws.cmp_state, 0, n_tiles * 4, st)))) return rc;
        if ((rc = note_cuda(ctx, launch_compact(ctx, multiplicity, volume, cell_id, n_sd)))) return rc;
    }
    *n_sd_out = n_sd - zeros;
    // stable compaction keeps a sorted cell_id sorted and cannot grow a cell: the verdict carries over
    if (ctx->verdict_valid && ctx->verdict_cell_ptr == cell_id && ctx->verdict_n_sd == n_sd)
        ctx->verdict_n_sd = n_sd - zeros;
    if (bad_data) {
        cudaMemsetAsync(ctx->ws.sticky, 0, STICKY_WORDS * 4, st);
        ctx->verdict_valid = 0;
        return SDM_ERR_BAD_DATA;
    }
    return SDM_OK;
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
    return SDM_OK;
}

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
    if ((rc = note_cuda(ctx, cudaMemcpyAsync(d_xi, multiplicity_host, (size_t)n_sd * 8, cudaMemcpyHostToDevice, st)))) return rc;
    if ((rc = note_cuda(ctx, cudaMemcpyAsync(d_v, volume_host, (size_t)n_sd * 8, cudaMemcpyHostToDevice, st)))) return rc;
    if ((rc = note_cuda(ctx, cudaMemcpyAsync(d_c, cell_id_host, (size_t)n_sd * 4, cudaMemcpyHostToDevice, st)))) return rc;
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
    return note_cuda(ctx, cudaStreamSynchronize(st));
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
    KernelParams dkp;
    dkp.kind = kp->kind;
    dkp.b = kp->b;
    dkp.Epi = kp->E * 3.141592653589793;
    return note_cuda(ctx, launch_kernel_eval(ctx, dkp, vj, vk, n, K_out));
}

}  // extern "C"
