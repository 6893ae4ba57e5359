// Host-side internals shared by the translation units of libsdm_b200.so: the context, the
// workspace map and the launcher prototypes.  See DESIGN.md "Data layout in HBM".
#pragma once
#include <cstddef>
#include <cstdint>
#include <vector>
#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>  // header-only; a no-op unless a profiler is attached

#include "../../include/sdm.h"
#include "sdm_device.cuh"

namespace sdm {

constexpr int RADIX_BITS = 8;
constexpr int RADIX = 1 << RADIX_BITS;
constexpr int MAX_PASSES = 8;  // 4 key digits + up to 4 cell-id digits (n_cell <= 2^31)

// Onesweep pass tile: SORT_BLOCK threads x SORT_ITEMS keys.
#ifndef SORT_BLOCK_THREADS
#define SORT_BLOCK_THREADS 256
#endif
#ifndef SORT_ITEMS_PER_THREAD
#define SORT_ITEMS_PER_THREAD 16
#endif
constexpr int SORT_BLOCK = SORT_BLOCK_THREADS;
constexpr int SORT_ITEMS = SORT_ITEMS_PER_THREAD;
constexpr int SORT_TILE = SORT_BLOCK * SORT_ITEMS;
constexpr int SORT_TILE_BITS = SORT_TILE == 4096 ? 12 : SORT_TILE == 8192 ? 13 : SORT_TILE == 2048 ? 11 : -1;

// Largest cell the register-resident per-cell sort of the fast path handles (16 lanes x 16 or 32 lanes x 8 words).
constexpr int CELL_FAST_MAX = 256;
// Most coarse key bits of the BUCKET path's placement (sdm_bucket.cu): 4096 buckets of at most 2048 entries on average.
constexpr int BUCKET_MAX_BITS = 12;
// Largest single-cell problem the box step takes (sdm_box.cu).
constexpr int BOX_MAX = 8192;
// Cell-size classes of the fused kernel: class k = cells of at most class_slots(k) = 32, 48, 64, 96, 128, 192, 256
// entries.  Even classes are sorted by P / R lanes holding R = 8 (or 4) words each, odd ones by P / 6 lanes holding 6.
constexpr int CELL_CLASSES = 7;
constexpr int CELL_ODD_WORDS = 6;
__host__ __device__ constexpr int class_slots(int k) { return (k & 1) ? (48 << (k >> 1)) : (32 << (k >> 1)); }
__host__ __device__ constexpr int class_lanes(int k, int r_even) { return (k & 1) ? (8 << (k >> 1)) : class_slots(k) / r_even; }
static_assert(class_slots(CELL_CLASSES - 1) == CELL_FAST_MAX, "the largest class is the largest cell of the fast path");

// Largest collision-efficiency table sdm_set_collision_efficiency accepts (radii x ratios).
constexpr int EFF_MAX_R = 128;
constexpr int EFF_MAX_P = 128;

// Largest number of bin edges sdm_volume_spectrum accepts (edges + per-bin sums live in shared memory).
constexpr int SPECTRUM_MAX_EDGES = 1025;

// Compaction tile.
constexpr int CMP_BLOCK = 256;
constexpr int CMP_ITEMS = 8;
constexpr int CMP_TILE = CMP_BLOCK * CMP_ITEMS;

// Words of the per-step control block (zeroed by one memset at the start of every step).
enum CtlWord {
    CTL_UNSORTED = 0,     // general path: 1 when cell_id is not non-decreasing; fused paths: the step's
                          // epoch when k_cell_bounds refused the input (the step is then skipped)
    CTL_MAX_COUNT = 1,    // general path: largest per-cell count (feeds the host-side path verdict)
    CTL_TICKET0 = 8,      // CTL_TICKET0 + pass: dynamic tile tickets of the sort passes
    CTL_CMP_TICKET = 24,  // compaction ticket
    CTL_ZERO_COUNT = 25,  // compaction: number of zero-multiplicity entries (low word)
    CTL_WORDS = 64
};
// Words of the run block (NOT zeroed per step; zeroed at init and managed by sdm_coalescence_steps).
enum RunWord {
    RUN_HALT = 0,  // != 0: the multi-step run is halted (a due compaction found zeros); fused steps exit at once
    RUN_ZC0 = 1,   // RUN_ZC0 + (s mod 3): zero multiplicities the array holds after step s of the run
    RUN_BOUNDS_TICKET = 4,  // k_cell_bounds: blocks finished (the last one publishes the verdict and resets it)
    RUN_BOUNDS_CLASS = 5,   // k_cell_bounds: worst cell-size class seen so far (reset by the last block)
    RUN_LIST_CURSOR = 12,   // RUN_LIST_CURSOR + k, k = 0..CELL_CLASSES-1: k_cell_classes' fill level of class k's list (reset by its last block)
    RUN_WORDS = 64
};
// Words of the pinned, device-mapped host status block: what the host must learn WITHOUT draining the stream.
enum MappedWord {
    MAPPED_HALT = 0,     // RUN_HALT's tag
    MAPPED_ZEROS = 1,    // the zero count that caused the halt
    MAPPED_VERDICT_EPOCH = 2,  // k_cell_bounds: epoch of the last published verdict
    MAPPED_VERDICT_CLASS = 3,  //   its worst cell-size class: 0 (<= 32 entries) .. 6 (<= 256), see class_slots; CELL_CLASSES (larger,
                               //   or the array is not non-decreasing / holds an out-of-range cell_id)
    MAPPED_CLASS_COUNT = 4,    //   MAPPED_CLASS_COUNT + k, k = 0..CELL_CLASSES-1: number of cells of size class k
    MAPPED_WORDS = 16
};
// Sticky words (zeroed at init and by sdm_poll_error only).
enum StickyWord { STICKY_BAD_DATA = 0, STICKY_WORDS = 64 };

struct Workspace {
    // [zeroed per step] ------------------------------------------------
    u32* ctl;         // CTL_WORDS
    u32* digit_hist;  // MAX_PASSES * RADIX
    u32* cell_count;  // max_n_cell + 1
    u32* tile_state;  // MAX_PASSES * max_tiles * RADIX   (decoupled look-back)
    size_t zero_bytes_fixed;  // ctl + digit_hist (contiguous from ctl)
    // [not zeroed] -----------------------------------------------------
    u32* sticky;      // STICKY_WORDS
    u32* run;         // RUN_WORDS
    u32* cell_start;  // max_n_cell + 1
    u32* class_list;  // CELL_CLASSES x max_n_cell: cell ids grouped by size class (k_cell_classes)
    int64_t* res_xi;  // max_n_sd each: the cell-grouped copies of a resident HYBRID run (launch_resident_move)
    double* res_v;
    u32* bucket_count;  // BUCKET path: 2^BUCKET_MAX_BITS coarse-bucket fill counts (zeroed per step)
    u64* buf_a;       // max_n_sd
    u64* buf_b;       // max_n_sd
    u32* cmp_state;   // max compaction tiles
    double* spec_edges;  // SPECTRUM_MAX_EDGES volume edges of sdm_volume_spectrum
    double* eff_radius;  // EFF_MAX_R radii of the collision-efficiency table
    double* eff_table;   // EFF_MAX_R x EFF_MAX_P entries
    u64* scan_state;  // k_cell_scan slab states (epoch-tagged; zeroed at init)
    size_t scan_state_bytes;
    size_t total_bytes;
};

struct Plan {  // per-step derived quantities
    int cbits;     // bits of (n_cell - 1)
    int idxbits;   // bits of (n_sd - 1), at least 1
    int skip;      // low key digits NOT sorted by the LSD passes (0..3); ties on them are repaired exactly afterwards
    int n_cpass;   // ceil(cbits / 8) cell-id digits
    int n_pass;    // (4 - skip) + n_cpass
    int n_tiles;   // ceil(n_sd / SORT_TILE)
};

}  // namespace sdm

namespace sdm {
// Kernel classes for sdm_profile_read (same order as SDM_PROF_* in include/sdm.h).
enum ProfClass { PROF_KEYS_HIST = 0, PROF_CELL_SCAN, PROF_RADIX_PASS, PROF_PAIR, PROF_COUNT_ZERO, PROF_COMPACT,
                 PROF_CELL_STATS, PROF_OTHER, PROF_CELL_BOUNDS, PROF_CELL_FUSED, PROF_CELL_DIGIT_HIST, PROF_TIE_REPAIR, PROF_SPECTRUM, PROF_DISPLACE, PROF_CELL_CLASSES, PROF_BOX_STEP, PROF_BUCKET, PROF_RESIDENT_MOVE, PROF_CLASSES };
// What the last general-path step learned about the cell_id array (pinned host memory, written by an
// asynchronous copy; valid once `verdict_event` has completed).
struct Verdict { u32 unsorted; u32 max_count; };
struct ProfEvent { cudaEvent_t start, stop; int cls; };
// What k_cell_bounds found out about the cell sizes, as the fused kernel's launch geometry needs it.
struct CellClasses {
    u32 worst;                 // largest class present (CELL_CLASSES: the fused kernel cannot take the input)
    u32 count[CELL_CLASSES];   // cells served as class k (not mixed: every cell as class `worst`)
    bool mixed;                // the cells are dealt out class by class through ws.class_list
    u32 cell_offset;           // not mixed: the launch serves the cells cell_offset .. cell_offset + count[worst] - 1
};
}  // namespace sdm

struct sdm_ctx {
    int device;
    cudaStream_t stream;
    int64_t max_n_sd;
    int32_t max_n_cell;
    int64_t max_tiles;
    sdm::Workspace ws;
    int path;
    int last_path;
    int cuda_error;  // sticky cudaError_t
    int64_t launches;
    // debug outputs
    int32_t* dbg_perm;
    int64_t* dbg_gamma;
    int64_t* dbg_gamma_clamped;
    int32_t* dbg_cell_start;
    // host staging
    void* staging;
    size_t staging_bytes;
    cudaStream_t copy_in, copy_out;          // sdm_coalescence_step_host: uploads / downloads beside the step's stream
    cudaEvent_t host_in[8], host_done[8];    // per chunk: attributes uploaded / step applied
    int sm_count;
    int skip_key_digits;  // SDM_OPT_SKIP_KEY_DIGITS (-1 = automatic)
    int narrow_key_bits;  // key bits kept in the fused kernel's 32-bit sort word (SDM_OPT_NARROW_KEY_BITS)
    int fused_r;          // words per lane of the fused kernel's group sort (SDM_OPT_FUSED_WORDS_PER_LANE; 0 = automatic)
    int bucket_bits_opt;  // key bits of the BUCKET path's placement (SDM_OPT_BUCKET_BITS; 0 = automatic)
    int box_cluster;      // BOX path on a cluster of eight blocks (SDM_OPT_BOX_CLUSTER; default 1) or on one block
    // optional per-launch CUDA-event timing (sdm_profile_enable)
    int profiling;
    std::vector<sdm::ProfEvent>* prof_events;
    size_t prof_used;
    // AUTO path selection: verdict of the last general-path step about (cell_id pointer, n_sd, n_cell)
    sdm::Verdict* verdict_host;  // pinned
    sdm::u32* status_host;       // pinned: sticky words then control block, one D2H copy
    volatile sdm::u32* mapped;   // pinned + mapped: MAPPED_* words written by kernels (same address on the device: UVA)
    cudaEvent_t verdict_event;
    cudaEvent_t chunk_event[2];  // sdm_coalescence_steps: completion of the two chunks of steps in flight
    // BUCKET path inside sdm_coalescence_steps: level 1 of the NEXT step's placement runs on a side stream beside this
    // step's pair kernel (they share nothing: keys depend on the step number only)
    cudaStream_t side;
    cudaEvent_t side_go, side_done;  // level 2 of this step done (the counts and slabs are free) / level 1 of the next step done
    int side_valid;                  // a placement has been started ahead ...
    uint64_t side_step;              // ... for this step
    int64_t side_n_sd;               // ... of this many super-droplets
    // zero-multiplicity count left in ctl[CTL_ZERO_COUNT] by the last fused step (SDM_OPT_TRACK_ZEROS)
    sdm::u32 epoch;  // tag of the current fused-path step (>= 2; see k_cell_bounds)
    sdm::u64 index_base;  // SDM_OPT_INDEX_BASE
    int eff_n_r, eff_n_p;  // collision-efficiency table installed by sdm_set_collision_efficiency (0 = none)
    double eff_max;        // its largest entry: the E of the conservative early-out bounds
    int track_zeros;
    int zero_hint_valid;
    const void* zero_hint_xi;
    int64_t zero_hint_n_sd;
    const void* verdict_cell_ptr;
    int64_t verdict_n_sd;
    int32_t verdict_n_cell;
    int verdict_valid;
};

namespace sdm {

// NVTX range names of the kernel classes (tracing): same order as ProfClass.
inline const char* prof_class_name(int cls) {
    static const char* const names[PROF_CLASSES] = {
        "sdm:keys_hist", "sdm:cell_scan", "sdm:radix_pass", "sdm:pair", "sdm:count_zero", "sdm:compact", "sdm:cell_stats",
        "sdm:other", "sdm:cell_bounds", "sdm:cell_fused", "sdm:cell_digit_hist", "sdm:tie_repair", "sdm:volume_spectrum",
        "sdm:displace", "sdm:cell_classes", "sdm:box_steps", "sdm:bucket", "sdm:resident_move"};
    return (cls >= 0 && cls < PROF_CLASSES) ? names[cls] : "sdm:?";
}

// RAII bracket around one kernel launch: counts it, opens an NVTX range named after the kernel class (visible in
// Nsight Systems / Compute timelines) and, when profiling is on, records a CUDA-event pair on the launching stream.
struct LaunchScope {
    sdm_ctx* ctx;
    cudaEvent_t stop;
    LaunchScope(sdm_ctx* c, int cls) : ctx(c), stop(nullptr) {
        ctx->launches++;
        nvtxRangePushA(prof_class_name(cls));
        if (!ctx->profiling) return;
        if (ctx->prof_used == ctx->prof_events->size()) {
            ProfEvent e;
            if (cudaEventCreate(&e.start) != cudaSuccess || cudaEventCreate(&e.stop) != cudaSuccess) return;
            ctx->prof_events->push_back(e);
        }
        ProfEvent& e = (*ctx->prof_events)[ctx->prof_used++];
        e.cls = cls;
        cudaEventRecord(e.start, ctx->stream);
        stop = e.stop;
    }
    ~LaunchScope() {
        if (stop) cudaEventRecord(stop, ctx->stream);
        nvtxRangePop();
    }
};

Workspace carve_workspace(void* base, int64_t max_n_sd, int32_t max_n_cell);
Plan make_plan(int64_t n_sd, int32_t n_cell, int skip_key_digits /* -1 = choose from n_sd / n_cell */);

// Launchers (each enqueues on ctx->stream and bumps ctx->launches).  Return cudaError_t.
cudaError_t launch_keys_hist(sdm_ctx* ctx, const int32_t* cell_id, int64_t n_sd, int32_t n_cell,
                             const Plan& plan, const PhiloxKeys& pk, u64* sortkey_out);
cudaError_t launch_cell_scan(sdm_ctx* ctx, int32_t n_cell, int64_t n_sd);
int bucket_bits(int64_t n_sd, int bits_override);
int bucket_fine_bits(int64_t n_sd, int cb);
cudaError_t init_bucket_path(sdm_ctx* ctx);
cudaError_t launch_bucket_scatter(sdm_ctx* ctx, int64_t n_sd, int cb, const PhiloxKeys& pk, cudaStream_t st);
cudaError_t launch_bucket_sort(sdm_ctx* ctx, int64_t n_sd, int cb, const PhiloxKeys& pk, u64* sorted);
cudaError_t launch_sort_pass(sdm_ctx* ctx, int pass, const u64* in, u64* out, int64_t n_sd,
                             const Plan& plan);
cudaError_t launch_pair(sdm_ctx* ctx, const u64* sorted, int64_t* xi, double* v, int64_t n_sd,
                        int32_t n_cell, const Plan& plan, double dtdV, const KernelParams& kp,
                        const PhiloxKeys& pk);
cudaError_t launch_cell_sort_pass(sdm_ctx* ctx, int pass, bool narrow, const int32_t* cell_id, const void* in,
                                  void* out, int64_t n_sd, int32_t n_cell, const Plan& plan);
cudaError_t launch_cell_digit_hist(sdm_ctx* ctx, const int32_t* cell_id, int64_t n_sd, int32_t n_cell,
                                   const Plan& plan);
// strict: a refusal (a cell of more than CELL_FAST_MAX entries, unsorted or out-of-range input) also raises the
// sticky SDM_ERR_BAD_DATA (explicit paths); AUTO's analysis passes strict = false and falls back instead.
cudaError_t launch_cell_bounds(sdm_ctx* ctx, int src_kind, const void* src, int64_t n_sd, int32_t n_cell,
                               int idxbits, bool strict);
// Zero bookkeeping / halt protocol of one fused step (all nullable / 0: see FusedArgs in sdm_cellsort.cu).
struct StepLinks {
    u32* zc_accum;
    const u32* zc_check;
    u32* zc_clear;
    u32 halt_tag;
    u32 n_steps;  // 0 / 1: one step; more: that many consecutive steps inside the launch (no compaction in between)
    bool resident;  // HYBRID: xi / v are the cell-grouped resident copies (launch_resident_move), not the caller's arrays
};
// HYBRID runs of sdm_coalescence_steps: gather the attributes into ws.res_xi / ws.res_v in run order (back = false),
// scatter them back to the caller's arrays (back = true)
cudaError_t launch_resident_move(sdm_ctx* ctx, bool back, int src_kind, const void* run_idx, int idxbits, int64_t* xi,
                                 double* v, int64_t n_sd);
// whether the fused kernel this input gets can take several steps per launch (StepLinks.n_steps > 1)
#define FUSED_MULTI_STEP(R) ((R) == 4)
bool fused_multi_step(const sdm_ctx* ctx, const CellClasses& cc);
cudaError_t launch_cell_fused(sdm_ctx* ctx, int src_kind, const void* run_idx, int idxbits, const CellClasses& cc,
                              int64_t* xi, double* v, int64_t n_sd, int32_t n_cell, double dtdV, const KernelParams& kp,
                              const PhiloxKeys& pk, const StepLinks& links);
cudaError_t launch_tie_repair(sdm_ctx* ctx, u64* sorted, int64_t n_sd, const Plan& plan, const PhiloxKeys& pk);
cudaError_t launch_debug_perm(sdm_ctx* ctx, const u64* sorted, int64_t n_sd, const Plan& plan);
cudaError_t launch_count_zero(sdm_ctx* ctx, const int64_t* xi, int64_t n_sd);
cudaError_t launch_compact(sdm_ctx* ctx, int64_t* xi, double* v, int32_t* cell_id, int64_t n_sd);
cudaError_t launch_cell_stats(sdm_ctx* ctx, const int64_t* xi, const double* v, const int32_t* cell_id,
                              int64_t n_sd, int32_t n_cell, int32_t* count, int64_t* sum_xi,
                              double* sum_xi_v, double* sum_xi_v2);
cudaError_t init_cell_fused(sdm_ctx* ctx);       // per-device function attributes, once per context
cudaError_t init_box_step(sdm_ctx* ctx);
cudaError_t launch_box_steps(sdm_ctx* ctx, int64_t* xi, double* v, int64_t n_sd, double dtdV, const KernelParams& kp,
                             const PhiloxKeys& pk, int64_t n_steps);
cudaError_t init_volume_spectrum(sdm_ctx* ctx);
cudaError_t launch_volume_spectrum(sdm_ctx* ctx, const int64_t* xi, const double* v, int64_t n_sd,
                                   const double* edges_dev, int32_t n_edges, bool lut_ok /* edges[0] > 0 */, int64_t* count, int64_t* sum_xi,
                                   double* sum_xi_v);
cudaError_t launch_displace(sdm_ctx* ctx, bool move, double* x, double* z, int32_t* cell_id, int64_t n_sd, int32_t nx,
                            int32_t nz, const double* u_cell, const double* w_cell, double dt);
cudaError_t launch_philox_fill(sdm_ctx* ctx, const PhiloxKeys& pk, u64 i0, int64_t n, u32* key_out,
                               double* u_out);
cudaError_t launch_kernel_eval(sdm_ctx* ctx, const KernelParams& kp, const double* vj, const double* vk,
                               int64_t n, double* K_out);

}  // namespace sdm
