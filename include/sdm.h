/* sdm.h -- C ABI of the B200-native Super-Droplet Method (SDM) coalescence step.
 *
 * What it computes: one Monte-Carlo collisional-growth step of the Super-Droplet Method
 * ("SDM Monte-Carlo algorithm for representing collisional growth (Shima et al., 2009)",
 * /root/reference/PAPER.md:15 Introduction; reference entry PAPER.md:188) on super-droplets
 * carrying the attributes `volume` and `n` = multiplicity, in an environment
 * that supplies the time step `dt` and the cell volume `dv`, with a coalescence
 * kernel object (PAPER.md:66, 75 Golovin; PAPER.md:96 geometric sweep-out).  The statement of
 * each operation is BASELINE.json `north_star` (a)-(d) as read in SURVEY.md section 8(c) and
 * DESIGN.md "Readings".
 *
 * Conventions (apply to every call unless stated otherwise)
 *  - Array arguments are DEVICE pointers owned by the caller; scalars are passed by value.
 *    Pointers marked "host" are host pointers.  The library never allocates device memory: the
 *    caller hands it a workspace of sdm_workspace_bytes() bytes at sdm_init().
 *  - Structure-of-arrays state: multiplicity int64[n_sd], volume fp64[n_sd] (m^3), cell_id
 *    int32[n_sd] in [0, n_cell).  8-byte arrays must be 16-byte aligned (cudaMalloc / torch are).
 *  - All work is enqueued on the cudaStream_t given to sdm_init(); calls are asynchronous unless
 *    they return a value to the host (documented per call).
 *  - Errors: every entry point returns an sdm_status (0 = SDM_OK, negative = error).  Nothing is
 *    printed, nothing throws.  Misuse visible on the host -> SDM_ERR_INVALID_ARG / SDM_ERR_CAPACITY
 *    before any kernel is launched.  Data errors only visible on the device (cell_id outside
 *    [0, n_cell); an input that an explicitly chosen CELL_SORTED / HYBRID path cannot take) set a sticky
 *    flag reported by sdm_poll_error() and by the next synchronising call as SDM_ERR_BAD_DATA; the step
 *    stays memory-safe but its output is then unspecified.  Multiplicities are NOT range-checked: a
 *    negative multiplicity or a negative / non-finite volume is the caller's responsibility (the oracle does
 *    not define them either).
 *  - There is no CPU fallback: without a CUDA device sdm_init() returns SDM_ERR_CUDA.
 */
#ifndef SDM_B200_H_
#define SDM_B200_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sdm_ctx sdm_ctx; /* opaque, host memory, freed by sdm_destroy() */

typedef enum {
    SDM_OK = 0,
    SDM_ERR_INVALID_ARG = -1,
    SDM_ERR_CAPACITY = -2,
    SDM_ERR_CUDA = -3,
    SDM_ERR_BAD_DATA = -4,
    SDM_ERR_STATIC_LIMIT = -5 /* sdm_remove_zero_multiplicity_static: n_sd beyond sdm_static_max_n_sd() */
} sdm_status;

typedef enum { SDM_KERNEL_GOLOVIN = 0, SDM_KERNEL_GEOMETRIC = 1, SDM_KERNEL_GEOMETRIC_TABLE = 2 } sdm_kernel_kind;

/* Coalescence kernel K(v_j, v_k) [m^3 s^-1] (north_star (c)):
 *   Golovin:  K = b (v_j + v_k), b in s^-1, volumes in m^3.
 *   geometric:     K = E pi (r_j + r_k)^2 |v_t(r_j) - v_t(r_k)|, r = cbrt(3 v / 4 pi),
 *                                v_t a three-regime power law (R16).
 *   geometric + table ("more sophisticated collision kernels ... the influence of electric field";
 *                                SURVEY 8(f) NEXT-3): the same with E = E(r_big, r_small / r_big) interpolated
 *                                in the table installed by sdm_set_collision_efficiency(); the field E is ignored. */
typedef struct {
    int32_t kind; /* sdm_kernel_kind */
    int32_t _pad;
    double b; /* Golovin coefficient, >= 0 */
    double E; /* geometric collision efficiency, >= 0 (configs use 1.0) */
} sdm_kernel_params;

/* Collision-efficiency table of SDM_KERNEL_GEOMETRIC_TABLE (reading R39; the paper names the kernels of the Berry
 * 1966 example -- hydrodynamic and electric-field efficiencies -- but prints no numbers, and none are in this
 * repository: the caller supplies them, one table per variant).
 *   radius  HOST fp64[n_r], strictly ascending, metres: the grid of the LARGER radius of the pair
 *   table   HOST fp64[n_r][n_p], row-major, finite and >= 0: E at (radius[i], p_j = j / (n_p - 1)), p = r_small / r_big
 * Bilinear interpolation in a fixed, FMA-free order:  i = last interval with radius[i] <= r_big (clamped),
 * t_r = (r_big - radius[i]) / (radius[i+1] - radius[i]) clamped to [0, 1] (outside the grid: the value on its
 * edge);  f = p (n_p - 1), j = min(floor(f), n_p - 2), t_p = f - j;  e0 = T[i][j] + t_p (T[i][j+1] - T[i][j]),
 * e1 likewise in row i + 1;  E = e0 + t_r (e1 - e0).  A constant table reproduces SDM_KERNEL_GEOMETRIC bit for bit.
 * The table is copied into the context's workspace (2 <= n_r, n_p <= 128); all-NULL / 0 arguments remove it.
 * Errors: INVALID_ARG (bad sizes, radius not ascending, entries negative or not finite), CAPACITY (too large). */
int sdm_set_collision_efficiency(sdm_ctx* ctx, const double* radius /* host */, int32_t n_r, int32_t n_p,
                                 const double* table /* host */);

/* Path selection for sdm_coalescence_step / sdm_coalescence_steps (sdm_set_path).  Every path produces the same bits.
 *   GENERAL      global stable LSD radix sort of (cell_id, Philox key): north_star (b).  Any input.
 *   CELL_SORTED  per-cell register-resident sort fused with the pair kernel.  Legal
 *                only when cell_id is non-decreasing and no cell holds more than 256 super-droplets.
 *   HYBRID       LSD radix passes over the cell_id digits only (grouping the indices by cell), then the same
 *                fused per-cell sort + pair kernel, gathering through the sorted indices.  Any order of
 *                cell_id; legal when n_cell > 1 and no cell holds more than 256 super-droplets.
 *                An explicitly chosen CELL_SORTED or HYBRID verifies its precondition on the device BEFORE anything
 *                is updated: on a violation (the caller's error) the step is NOT applied and the sticky
 *                SDM_ERR_BAD_DATA flag is set.  Like AUTO they wait for the device's verdict on the cell sizes
 *                (it fixes the launch geometry) without draining the stream.
 *   BOX          one cell of at most 8192 super-droplets (the paper's box example; SURVEY 8(f)
 *                NEXT-1 "single-CTA fused step for tiny N"): the whole step -- keys, shuffle by counting placement of
 *                the uniform keys, pair rule -- for any number of consecutive steps in one launch of a cluster of eight
 *                blocks (or of one block, SDM_OPT_BOX_CLUSTER) out of (distributed) shared memory.  Chosen explicitly
 *                on an input that does not fit, the step takes the GENERAL path.
 *   BUCKET       one cell of up to 2^23 super-droplets (configs[1]: a box of 2^20): the Philox keys are uniform, so a
 *                two-level counting placement by their bits replaces the LSD passes -- coarse buckets of 1024-2048
 *                entries by the top bits (histogram and scatter with block-local counting), then one block per
 *                coarse bucket orders it exactly by (key, index) in shared memory the way the BOX step does -- and
 *                the GENERAL path's pair kernel follows.  A coarse bucket of more than 4096 entries (twice the
 *                largest average: it does not happen) would raise the sticky SDM_ERR_BAD_DATA.  Chosen explicitly on
 *                an input that does not fit (several cells, more than 2^23 entries), the step takes the GENERAL path.
 *   AUTO         (default) never refuses valid input.  Every step first analyses cell_id on the device (one
 *                streaming read: range, order, largest cell) and the host waits for that verdict -- a few
 *                microseconds, through a mapped status word, without draining work enqueued behind it -- before
 *                it enqueues either the fused kernel (CELL_SORTED when the array is non-decreasing, HYBRID when the
 *                previous GENERAL step on the same array saw small cells in any order), the BOX step (one small
 *                cell), the BUCKET path (one large cell) or the GENERAL path.  So
 *                cell_id may be rewritten in place between steps (a displacement step does exactly that): the
 *                next step simply takes the path that fits.  sdm_coalescence_steps pays the analysis once per
 *                call instead of once per step.  sdm_set_path() forgets what was learned. */
typedef enum { SDM_PATH_AUTO = 0, SDM_PATH_GENERAL = 1, SDM_PATH_CELL_SORTED = 2, SDM_PATH_HYBRID = 3, SDM_PATH_BOX = 4,
               SDM_PATH_BUCKET = 5 } sdm_path;

/* Bytes of device workspace sdm_init() needs for problems up to (max_n_sd, max_n_cell).
 * Returns 0 when the arguments are invalid (max_n_sd < 0, max_n_sd >= 2^30, max_n_cell < 1). */
size_t sdm_workspace_bytes(int64_t max_n_sd, int32_t max_n_cell);

/* Create a context bound to `device`, the caller's workspace and the caller's stream.
 *   out            host: receives the context
 *   workspace_dev  device memory, >= sdm_workspace_bytes(max_n_sd, max_n_cell), 256-byte aligned,
 *                  owned by the caller and kept alive until sdm_destroy()
 *   cuda_stream    a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); 0 = default stream
 * Launches no kernel except one memset of the workspace header.
 * Errors: INVALID_ARG (null out/workspace, bad sizes), CAPACITY (workspace too small), CUDA. */
int sdm_init(sdm_ctx** out, int device, int64_t max_n_sd, int32_t max_n_cell, void* workspace_dev,
             size_t workspace_bytes, void* cuda_stream);

/* One SDM coalescence step (north_star (a)-(c)):
 *   a1  per super-droplet i one Philox-4x32-10 block, counter {lo(i),hi(i),lo(step),hi(step)},
 *       key {lo(seed),hi(seed)}: word 0 = permutation key, words 3:2 -> 53-bit uniform;
 *   a2  per-cell counts and their exclusive scan;
 *   a3  stable ascending sort of indices by (cell_id << 32 | key): the per-cell random shuffle;
 *   a4  neighbours (2a, 2a+1) of each cell's shuffled run form pairs; for a pair with xi_j >= xi_k
 *       p = K(v_j,v_k) xi_j (dt/dV) (n_c(n_c-1)/2)/floor(n_c/2); gamma = floor(p) + [u < p - floor(p)];
 *       gamma~ = min(gamma, floor(xi_j/xi_k)); xi_j -= gamma~ xi_k, v_k += gamma~ v_j, and when xi_j
 *       reaches 0 the pair splits: xi_j = floor(xi_k/2), xi_k -= floor(xi_k/2), both get the new volume.
 * multiplicity and volume are updated IN PLACE at the original indices; cell_id is read-only; super-
 * droplets are never reordered.  Asynchronous.  (seed, step, array index) fully determine the random
 * numbers, so a run can be resumed bit-exactly.  n_sd == 0 is a no-op.
 * Errors: INVALID_ARG (null pointers, n_sd < 0, n_cell < 1, dt <= 0, dV <= 0, non-finite dt/dV,
 * unknown kernel kind, b < 0 or E < 0, SDM_KERNEL_GEOMETRIC_TABLE without a table), CAPACITY (n_sd > max_n_sd,
 * n_cell > max_n_cell), CUDA. */
int sdm_coalescence_step(sdm_ctx* ctx, int64_t* multiplicity, double* volume, const int32_t* cell_id,
                         int64_t n_sd, int32_t n_cell, double dt, double dV,
                         const sdm_kernel_params* kp, uint64_t seed, uint64_t step);

/* The time loop on the device ("API in brief": the Particulator "control[s] time-stepping"; the
 * loop itself is in the snippet that PAPER.md:80-84 announces and omits, so its statement is SURVEY 8(c)
 * `oracle_run`): exactly
 *     for s in 0 .. n_steps-1:
 *         sdm_coalescence_step(..., n_sd, ..., seed, step0 + s)
 *         if compact_every > 0 and (s + 1) % compact_every == 0:
 *             sdm_remove_zero_multiplicity(..., n_sd, &n_sd)
 * with the same bits as that sequence of calls, but enqueued without a host round trip per step: the path is chosen
 * once per call (see sdm_path), cell boundaries -- cell_id cannot change during the call -- are computed once, and a
 * due compaction costs nothing while no multiplicity is 0: every fused step counts the zeros it leaves behind, and
 * only a non-zero count at a due step halts the run on the device until the host has compacted.  On the cell-sorted
 * paths small inputs (n_sd <= 2^21) take up to 64 consecutive steps inside one kernel launch when no compaction is
 * due in between (a candidate pair lies inside one cell, so cells never interact), and a HYBRID run of
 * eight steps or more works on cell-grouped copies of the attributes in the workspace (gathered once, scattered back
 * before the call returns or compacts); the bits are those of the step-by-step loop.  cell_id is written
 * only by a compaction.  *n_sd_out (host) receives the final number of super-droplets; the call synchronises the
 * stream once, at its end, and then also reports a pending SDM_ERR_BAD_DATA.  n_steps == 0 and n_sd == 0 are no-ops.
 * Errors: as sdm_coalescence_step, plus INVALID_ARG for n_steps < 0, compact_every < 0 or a null n_sd_out. */
int sdm_coalescence_steps(sdm_ctx* ctx, int64_t* multiplicity, double* volume, int32_t* cell_id, int64_t n_sd,
                          int32_t n_cell, double dt, double dV, const sdm_kernel_params* kp, uint64_t seed,
                          uint64_t step0, int64_t n_steps, int64_t compact_every, int64_t* n_sd_out /* host */);

/* Stable stream compaction (north_star (d)): removes every entry whose
 * multiplicity is 0 from (multiplicity, volume, cell_id), in place; survivors keep their relative
 * order (required: the Philox counter is the array index).  The prefix [0, *n_sd_out) is the result,
 * the tail is unspecified.  Writes *n_sd_out on the HOST and therefore synchronises the stream; also
 * reports a pending SDM_ERR_BAD_DATA. */
int sdm_remove_zero_multiplicity(sdm_ctx* ctx, int64_t* multiplicity, double* volume, int32_t* cell_id,
                                 int64_t n_sd, int64_t* n_sd_out /* host */);

/* Per-cell statistics: count[c], sum xi, sum xi*v, sum xi*v*v over the
 * super-droplets of each cell.  Each output is a device array of length n_cell, or NULL to skip it.
 * Integer outputs are exact; the fp64 sums are accumulated in an unspecified order (compare at
 * 1e-12 relative).  Asynchronous. */
int sdm_cell_stats(sdm_ctx* ctx, const int64_t* multiplicity, const double* volume,
                   const int32_t* cell_id, int64_t n_sd, int32_t n_cell, int32_t* count,
                   int64_t* sum_xi, double* sum_xi_v, double* sum_xi_v2);

/* Volume spectrum (the paper's ParticlesVolumeSpectrum(radius_bins_edges) product,
 * PAPER.md:68-76; the normalisation is not in the paper -- reading R35: the raw per-bin sums).  Bin b holds the
 * array entries with volume_edges[b] <= volume < volume_edges[b+1]; entries outside [edges[0], edges[n-1]) are
 * not counted.  volume_edges: HOST array of n_edges (2..1025) finite, strictly ascending VOLUMES [m^3] -- the
 * caller converts its radius edges once (4/3 pi r^3), so no cube root enters the bin decision.  Outputs: DEVICE
 * arrays of n_edges - 1 entries, each nullable: count (entries in the bin, whatever their multiplicity), sum_xi
 * (exact), sum_xi_v (fp64, accumulated in an unspecified order: compare at 1e-12 relative).  Asynchronous.
 * INVALID_ARG for bad edges or sizes. */
int sdm_volume_spectrum(sdm_ctx* ctx, const int64_t* multiplicity, const double* volume, int64_t n_sd,
                        const double* volume_edges /* host */, int32_t n_edges, int64_t* count, int64_t* sum_xi,
                        double* sum_xi_v);

/* Particle displacement on the 2-D kinematic grid and the recomputation of cell_id (the step
 * BEFORE the coalescence path; PAPER.md:80 lists "particle displacement" among the dynamics
 * describe the kinematic_2d slab with its prescribed flow; the paper states no scheme -- readings R36-R38):
 *   positions x, z: DEVICE fp64[n_sd] in GRID UNITS, x in [0, nx), z in [0, nz); both directions periodic;
 *   cell_id = floor(z) * nx + floor(x)  (row-major, x fastest; a position ON a cell edge belongs to the upper cell);
 *   sdm_displace: one explicit-Euler step with the velocity of the cell the super-droplet is in BEFORE the move,
 *       c = cell_id(x, z);  x <- wrap(x + (u_cell[c] * dt), nx);  z <- wrap(z + (w_cell[c] * dt), nz)
 *     u_cell, w_cell: DEVICE fp64[nx * nz], grid units per second, caller-supplied (|u dt| < nx, |w dt| < nz: at most
 *     one period per step); wrap(q, n): q >= n -> q - n; q < 0 -> q + n; a result still outside [0, n) (a tiny negative
 *     q whose q + n rounds to n) -> 0.  One multiplication and one addition per coordinate, no FMA.
 * Both calls (re)write cell_id[n_sd] (DEVICE int32) and are asynchronous; sdm_displace updates x, z in place.  The
 * coalescence step that follows sees a cell_id that is in general no longer sorted: AUTO takes the path that fits.
 * Errors: INVALID_ARG (null pointers, n_sd < 0, nx or nz < 1, nx * nz >= 2^31, dt <= 0 or not finite), CUDA. */
int sdm_cell_id_from_positions(sdm_ctx* ctx, const double* x, const double* z, int64_t n_sd, int32_t nx, int32_t nz,
                               int32_t* cell_id);
int sdm_displace(sdm_ctx* ctx, double* x, double* z, int32_t* cell_id, int64_t n_sd, int32_t nx, int32_t nz,
                 const double* u_cell, const double* w_cell, double dt);

/* Parity instrumentation (off by default; never on in timed runs).  Registers device arrays that
 * every later sdm_coalescence_step fills; pass NULL to switch an output off again.
 *   perm_out[s]           int32[n_sd]  original index at shuffled position s
 *   gamma_out[i]          int64[n_sd]  gamma of the pair whose first-shuffled member is i, else 0
 *   gamma_clamped_out[i]  int64[n_sd]  gamma~ likewise
 *   cell_start_out[c]     int32[n_cell+1] exclusive scan of the per-cell counts */
int sdm_debug_outputs(sdm_ctx* ctx, int32_t* perm_out, int64_t* gamma_out, int64_t* gamma_clamped_out,
                      int32_t* cell_start_out);

/* Selects the implementation path of sdm_coalescence_step (see sdm_path).  Returns INVALID_ARG for an
 * unknown value. */
int sdm_set_path(sdm_ctx* ctx, int path);

/* Test / tuning knobs.  SDM_OPT_NARROW_KEY_BITS: number of Philox-key bits (1..24, default 24) kept in the
 * 32-bit sort word of the fused per-cell kernel; fewer bits make its exact tie repair frequent (tests).
 * The result never depends on it.
 * SDM_OPT_TRACK_ZEROS (0 / 1, default 0): row a5 fused into row a4.  When 1, the fused per-cell kernel
 * (CELL_SORTED and HYBRID paths) also counts, exactly, the zero multiplicities the array holds after the
 * step (it reads every multiplicity anyway), and a sdm_remove_zero_multiplicity call on the same
 * (multiplicity pointer, n_sd) that DIRECTLY follows that step on this context reads the count instead
 * of scanning the array again.  Contract: between the two calls the caller does not write the
 * multiplicity array (if it does, it sets the option again, which drops the stored count).  The GENERAL
 * path, a refused step and any other call order fall back to the counting kernel; results are identical.
 * SDM_OPT_INDEX_BASE (>= 0, default 0): the Philox counter of array entry i becomes index_base + i.  A rank
 * that holds entries [index_base, index_base + n_sd) of a larger array (whole cells only: cells are
 * independent within a step) then produces exactly the bits the unsharded step produces
 * for them -- multi-GPU runs shard by contiguous cell ranges with no collective.  Applies to
 * sdm_coalescence_step and sdm_coalescence_step_host; the caller updates it after a compaction.
 * SDM_OPT_SKIP_KEY_DIGITS (-1 = automatic (default), 0..3): number of low 8-bit digits of the Philox key the
 * GENERAL path's LSD passes leave unsorted.  With few super-droplets per cell the top key digits already
 * order almost every neighbour; the runs that still tie are then put in exact (key, index) order by a
 * repair kernel, so the permutation -- and every result -- is the same for every value (tests force 3).
 * Automatic: sorted key bits = log2(n_sd / n_cell) + 8, rounded up to whole digits.
 * SDM_OPT_FUSED_WORDS_PER_LANE (0 = automatic (default), 4, 8): sort words per lane of the fused per-cell
 * kernel's group sort (a cell of at most 32 << k entries is sorted by (32 << k) / R lanes).  A tuning / test knob:
 * every value gives the same bits; 4 cannot serve cells of more than 128 entries and then falls back to 8.
 * SDM_OPT_BUCKET_BITS (0 = automatic (default), 1..12): coarse key bits of the BUCKET path's placement (2^bits
 * buckets; automatic: the fewest bits that leave at most 2048 entries per bucket on average).  A test knob: every
 * value whose buckets stay within 4096 entries gives the same bits.
 * SDM_OPT_BOX_CLUSTER (0 / 1, default 1): the BOX path on a thread-block cluster of eight blocks (distributed shared
 * memory) or on one block.  Same bits either way.
 * Returns INVALID_ARG for an unknown option or value. */
enum { SDM_OPT_NARROW_KEY_BITS = 0, SDM_OPT_TRACK_ZEROS = 1, SDM_OPT_INDEX_BASE = 2, SDM_OPT_SKIP_KEY_DIGITS = 3,
       SDM_OPT_FUSED_WORDS_PER_LANE = 4, SDM_OPT_BUCKET_BITS = 5, SDM_OPT_BOX_CLUSTER = 6 };
int sdm_set_option(sdm_ctx* ctx, int option, int64_t value);

/* Which path the most recent step took (an sdm_path value other than AUTO), or 0 if none ran yet.  Host-side
 * bookkeeping: does not touch the stream. */
int sdm_last_path(sdm_ctx* ctx);

/* End-to-end variant with HOST buffers (bench.py `e2e`): copies multiplicity, volume and cell_id to the
 * device staging area bound with sdm_bind_host_staging(), runs sdm_coalescence_step there, copies
 * multiplicity and volume back, and synchronises.  Host buffers should be pinned for full PCIe speed.
 * Cell-major arrays of at least 2^18 entries whose cells are small and of nearly one size (configs[2], [3]) go through
 * a pipeline under AUTO: cell_id is uploaded and analysed as a whole, the attributes travel in eight pieces cut at cell
 * boundaries on a stream of their own, the fused kernel runs on the cells of a piece as soon as it has arrived, and
 * the piece returns on a third stream while the next one is arriving -- PCIe carries both directions at once.  Same
 * bits; every other input takes the plain sequence upload, step, download. */
size_t sdm_host_staging_bytes(int64_t max_n_sd);
int sdm_bind_host_staging(sdm_ctx* ctx, void* staging_dev, size_t staging_bytes);
/* With compact != 0 the step is followed by sdm_remove_zero_multiplicity on the staged arrays; the
 * surviving prefix of all three arrays is copied back and *n_sd_out (host, may be NULL when
 * compact == 0) receives the new count; cell_id_host is then written too. */
int sdm_coalescence_step_host(sdm_ctx* ctx, int64_t* multiplicity_host, double* volume_host,
                              int32_t* cell_id_host, int64_t n_sd, int32_t n_cell, double dt, double dV,
                              const sdm_kernel_params* kp, uint64_t seed, uint64_t step, int compact,
                              int64_t* n_sd_out /* host */);

/* Synchronises the stream and returns the sticky status (SDM_OK, SDM_ERR_BAD_DATA, SDM_ERR_CUDA),
 * clearing SDM_ERR_BAD_DATA. */
int sdm_poll_error(sdm_ctx* ctx);

/* Number of kernel launches (memsets excluded) the library has enqueued on this context so far. */
int64_t sdm_launch_count(sdm_ctx* ctx);

/* Per-kernel timing for bench.py's roofline line.  While enabled, every kernel launch is bracketed by
 * a CUDA-event pair on the context's stream.  sdm_profile_read synchronises the stream, adds up the
 * elapsed milliseconds and the launch counts per kernel class (arrays of SDM_PROF_CLASSES entries,
 * host) since the last read, and resets the accumulation. */
enum { SDM_PROF_KEYS_HIST = 0, SDM_PROF_CELL_SCAN, SDM_PROF_RADIX_PASS, SDM_PROF_PAIR, SDM_PROF_COUNT_ZERO,
       SDM_PROF_COMPACT, SDM_PROF_CELL_STATS, SDM_PROF_OTHER, SDM_PROF_CELL_BOUNDS, SDM_PROF_CELL_FUSED,
       SDM_PROF_CELL_DIGIT_HIST, SDM_PROF_TIE_REPAIR, SDM_PROF_SPECTRUM, SDM_PROF_DISPLACE, SDM_PROF_CELL_CLASSES,
       SDM_PROF_BOX_STEP, SDM_PROF_BUCKET, SDM_PROF_CLASSES };
int sdm_profile_enable(sdm_ctx* ctx, int on);
int sdm_profile_read(sdm_ctx* ctx, double* ms_out /* host */, int64_t* launches_out /* host */);

/* Test hooks for the a1 row alone: fills key[i] (uint32) and u[i] (fp64) for i in [i0, i0+n) --
 * device arrays -- with the same device code the step uses.  Asynchronous. */
int sdm_philox_fill(sdm_ctx* ctx, uint64_t seed, uint64_t step, uint64_t i0, int64_t n,
                    uint32_t* key_out, double* u_out);

/* Test hook for the kernel function alone: K_out[i] = K(vj[i], vk[i]) on device arrays. */
int sdm_kernel_eval(sdm_ctx* ctx, const sdm_kernel_params* kp, const double* vj, const double* vk,
                    int64_t n, double* K_out);

/* ---- the entry point that allocates nothing (csrc/sdm_noalloc.cu) ----
 * For callers that cannot call cudaMalloc -- code under CUDA graph capture, tight serving loops, harnesses that forbid
 * allocation.  The same operation as sdm_remove_zero_multiplicity (north_star (d); stable
 * in-place removal of the entries whose multiplicity is 0; the prefix [0, n_out) is the result, the tail is
 * unspecified), but WITHOUT a context and WITHOUT a workspace: its scratch memory (a ticket counter and one word per
 * tile of 2048 entries) is a fixed device array inside the library, 128.25 KB, which every GPU that loads the
 * library holds until the process exits.  The call makes no cudaMalloc / cudaFree / allocating library call, creates
 * no stream or event, and never synchronises:
 *   multiplicity, volume, cell_id   device arrays of n_sd entries, compacted in place
 *   n_sd                            0 <= n_sd <= sdm_static_max_n_sd() = 2^26; larger -> SDM_ERR_STATIC_LIMIT, nothing touched
 *   n_sd_out_dev                    DEVICE int64: receives the number of survivors (written by the kernel)
 *   cuda_stream                     the stream everything is enqueued on (a memset of the scratch words + one kernel)
 * It runs on the CURRENT device.  The first call on a device looks the array's device address up (the set-up step;
 * sdm_static_setup() does only that, for callers who want it done before a graph capture starts).
 * The scratch array is SHARED by all calls on a device and keeps the last call's contents; every call clears what it
 * uses on its own stream.  Two calls that overlap on the GPU (different streams or host threads) race on it: the
 * caller orders them.  Errors: INVALID_ARG (null pointers, n_sd < 0), STATIC_LIMIT, CUDA. */
int64_t sdm_static_max_n_sd(void);
int sdm_static_setup(void);
int sdm_remove_zero_multiplicity_static(int64_t* multiplicity, double* volume, int32_t* cell_id, int64_t n_sd,
                                        int64_t* n_sd_out_dev /* device */, void* cuda_stream);

const char* sdm_strerror(int status);
void sdm_destroy(sdm_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* SDM_B200_H_ */
