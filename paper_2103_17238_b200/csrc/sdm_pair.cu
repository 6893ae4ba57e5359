// Row a4 of SURVEY.md section 8(a): the fused pair kernel (north_star (c)).
// One thread per two consecutive shuffled positions (2t, 2t+1); exactly one of them can be the first
// member of a pair (even offset inside its cell, partner inside the same cell), so every lane that
// owns a pair does the whole probability / gamma / clamp / update chain, and all pairs are covered
// once whatever the parity of the cell starts.
//
// Reads: sorted packed words (8 B/SD, coalesced), cell_start (L2-resident), xi and v gathered at the
// original indices (16 B/SD); writes xi, v in place only where they change.  The uniform of the
// first-shuffled member is regenerated from Philox (never stored).
//
// fp64 discipline: the pair probability and the volume update use __dmul_rn/__dadd_rn in the order
// ((K * xi_j) * dtdV) * scale and gamma~ * v_j + v_k (R10, R13) -- no FMA contraction.
#include "sdm_internal.h"
#include "sdm_pair.cuh"

namespace sdm {

constexpr int PAIR_BLOCK = 128;

__global__ void __launch_bounds__(PAIR_BLOCK) k_pair(const PairArgs a) {
    const u32 t = blockIdx.x * PAIR_BLOCK + threadIdx.x;
    const u32 s0 = 2u * t;
    if (s0 >= a.n_sd) return;
    const u64 idx_mask = (1ull << a.idxbits) - 1ull;
    u64 P0, P1 = 0;
    const bool has1 = s0 + 1u < a.n_sd;
    if (has1) {
        const ulonglong2 pp = *reinterpret_cast<const ulonglong2*>(a.sorted + s0);
        P0 = pp.x; P1 = pp.y;
    } else {
        P0 = a.sorted[s0];
    }
    // cell of position s0
    u32 c0 = a.single_cell ? 0u : (u32)(P0 >> a.cshift);
    u32 start = a.single_cell ? 0u : __ldg(a.cell_start + c0);
    u32 end = a.single_cell ? a.n_sd : __ldg(a.cell_start + c0 + 1);
    u64 Pf, Pg;  // packed words of the pair this thread owns (first, second)
    if (((s0 - start) & 1u) == 0u) {
        if (s0 + 1u >= end) {
            // s0 is the unpaired last SD of its cell; s0+1 (if any) opens the next cell at offset 0
            if (!has1) return;
            const u32 c1 = (u32)(P1 >> a.cshift);
            start = s0 + 1u;
            end = __ldg(a.cell_start + c1 + 1);
            if (s0 + 2u >= end) return;
            Pf = P1; Pg = a.sorted[s0 + 2u];
        } else {
            Pf = P0; Pg = P1;
        }
    } else {
        // s0 is the second member of the previous thread's pair; s0+1 has even offset if in the same cell
        if (!has1) return;
        if (s0 + 1u >= end) {  // s0+1 starts the next cell
            const u32 c1 = (u32)(P1 >> a.cshift);
            start = s0 + 1u;
            end = __ldg(a.cell_start + c1 + 1);
        }
        if (s0 + 2u >= end) return;
        Pf = P1; Pg = a.sorted[s0 + 2u];
    }
    pair_collide(a, (u32)(Pf & idx_mask), (u32)(Pg & idx_mask), end - start);
}

__global__ void __launch_bounds__(256) k_debug_perm(const u64* __restrict__ sorted, u32 n_sd, int idxbits,
                                                    int32_t* __restrict__ perm_out) {
    const u32 s = blockIdx.x * 256u + threadIdx.x;
    if (s < n_sd) perm_out[s] = (int32_t)(sorted[s] & ((1ull << idxbits) - 1ull));
}

cudaError_t launch_pair(sdm_ctx* ctx, const u64* sorted, int64_t* xi, double* v, int64_t n_sd,
                        int32_t n_cell, const Plan& plan, double dtdV, const KernelParams& kp,
                        const PhiloxKeys& pk) {
    PairArgs a;
    a.sorted = sorted;
    a.xi = reinterpret_cast<long long*>(xi);
    a.v = v;
    a.cell_start = ctx->ws.cell_start;
    a.n_sd = (u32)n_sd;
    a.idxbits = plan.idxbits;
    a.cshift = plan.idxbits + 24;
    a.single_cell = (n_cell == 1);
    a.dtdV = dtdV;
    a.kp = kp;
    set_bound_constants(a);
    a.pk = pk;
    a.dbg_gamma = reinterpret_cast<long long*>(ctx->dbg_gamma);
    a.dbg_gamma_clamped = reinterpret_cast<long long*>(ctx->dbg_gamma_clamped);
    const u32 n_threads = (u32)((n_sd + 1) / 2);
    const u32 grid = (n_threads + PAIR_BLOCK - 1) / PAIR_BLOCK;
    LaunchScope scope(ctx, PROF_PAIR);
    k_pair<<<grid, PAIR_BLOCK, 0, ctx->stream>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_debug_perm(sdm_ctx* ctx, const u64* sorted, int64_t n_sd, const Plan& plan) {
    const u32 grid = (u32)((n_sd + 255) / 256);
    LaunchScope scope(ctx, PROF_OTHER);
    k_debug_perm<<<grid, 256, 0, ctx->stream>>>(sorted, (u32)n_sd, plan.idxbits, ctx->dbg_perm);
    return cudaGetLastError();
}

}  // namespace sdm
