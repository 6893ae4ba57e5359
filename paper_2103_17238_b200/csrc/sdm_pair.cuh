// The per-pair rule of the SDM step (north_star (c); SURVEY.md 8(c) O4 body), shared by the general
// pair kernel (sdm_pair.cu) and the fused per-cell kernel (sdm_cellsort.cu).
//
// fp64 discipline: the pair probability and the volume update use __dmul_rn/__dadd_rn in the order
// ((K * xi_j) * dtdV) * scale and gamma~ * v_j + v_k (R10, R13) -- no FMA contraction.
//
// The rule is split in two phases so that a warp can run the cheap one for all of its pairs and the
// expensive one only where it is needed:
//   pair_may_collide  exact-or-conservative test "can gamma be non-zero?" (never a false negative)
//   pair_apply        the whole rule in fp64, exactly as the oracle orders it
#pragma once
#include <cmath>
#include "sdm_internal.h"

namespace sdm {

struct PairArgs {
    const u64* sorted;
    long long* xi;
    double* v;
    const u32* cell_start;
    u32 n_sd;
    int idxbits;
    int cshift;  // packed >> cshift = cell_id
    int single_cell;
    double dtdV;
    float dtdV_up;  // dtdV rounded up to fp32 (bound arithmetic)
    float Epi_up;   // E * pi rounded up to fp32
    float cheap_c;  // constant of pair_cheap_may_collide, rounded up on the host (set_bound_constants)
    KernelParams kp;
    PhiloxKeys pk;
    long long* dbg_gamma;
    long long* dbg_gamma_clamped;
};

// fp32 constants of the geometric bound, rounded UP on the host (after dtdV and kp are set).
inline float float_round_up(double x) {
    float f = (float)x;
    if ((double)f < x) f = nextafterf(f, INFINITY);
    return f;
}
// Relative slack of the cheap bound: covers the approximate cube root (3e-5 on r, fourth power at most),
// the fp32 roundings of the half-dozen multiplications and the 1e-8 of det_cbrt and of the fp64 products.
constexpr double CHEAP_SLACK = 1.0 + 3e-4;
inline void set_bound_constants(PairArgs& a) {
    a.dtdV_up = float_round_up(a.dtdV);
    a.Epi_up = float_round_up(a.kp.Epi);
    // Golovin: p = b (v_j + v_k) xi_j dtdV scale.  Geometric: p <= E pi (2 r_M)^2 vt_ub(r_M) xi_j dtdV scale.
    a.cheap_c = float_round_up((a.kp.kind == 0 ? a.kp.b : 4.0 * a.kp.Epi) * a.dtdV * CHEAP_SLACK);
}

// (n_c (n_c - 1) / 2) / floor(n_c / 2) == n_c if odd else n_c - 1   (R9)
__device__ __forceinline__ u32 pair_scale_int(u32 n_c) { return (n_c & 1u) ? n_c : n_c - 1u; }

// fp32 helpers of the geometric bound.  BOUND_EPS covers every rounding of the fp32 evaluation: the
// approximate cube root 2^(log2(x)/3) from MUFU.LG2/EX2 (|log2 x| <= 100 inside the guarded range ->
// relative error < 6e-6), the fp64 -> fp32 conversions, r sqrt^-1(r) (2 ulp) and a dozen fp32 roundings
// (6e-8 each).  The fall speed goes like r^2 at most, so its relative error is below 2 BOUND_EPS.
constexpr float BOUND_EPS = 3e-5f;

__device__ __forceinline__ float bound_radius(float v) {  // ~ (3 v / 4 pi)^(1/3), relative error < 1e-5
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(__log2f(v * 0.2387324f) * 0.33333334f));  // MUFU.EX2, 2 ulp
    return y;
}
// R16 in fp32.  `near_edge` is set when r is within BOUND_EPS of a regime boundary, where the fp64 radius
// may fall in the other regime (the law jumps there: 0.19 -> 0.32 m/s at 40 um, 4.8 -> 4.92 m/s at 600 um).
__device__ __forceinline__ float bound_fall_speed(float r, bool& near_edge) {
    near_edge |= (fabsf(r - 40e-6f) <= 40e-6f * BOUND_EPS) | (fabsf(r - 600e-6f) <= 600e-6f * BOUND_EPS);
    const float quad = 1.19e8f * (r * r), lin = 8e3f * r, root = 2.01e2f * (r * rsqrtf(r));
    return r < 40e-6f ? quad : (r < 600e-6f ? lin : root);
}

// First level of the early-out, a dozen fp32 operations per pair and no fp64 at all: an upper bound of p from the
// per-droplet fp32 values staged by the fused kernel -- xm >= xi_j = max(xi_0, xi_1) and the volumes, both rounded
// UP to fp32 -- compared with a lower bound of u.  Returns false only when gamma = 0 is certain (u >= p_ub implies
// p < 1 and not (u < p - floor(p))); pairs that pass go on to pair_may_collide / pair_apply.
//   Golovin:   K = b (v_j + v_k) <= b (vf_0 + vf_1).
//   geometric: with r_M the larger radius, (r_j + r_k)^2 <= 4 r_M^2 and |vt_j - vt_k| <= vt(r_M) (vt >= 0 and
//              non-decreasing, jumps included: 0.19 -> 0.32 m/s at 40 um, 4.80 -> 4.92 m/s at 600 um);
//              vt(r) <= 1.19e8 r^2 below 40 um and <= 8.3e3 r everywhere (201 sqrt(r) <= 8.3e3 r from 587 um on),
//              so K <= E pi 4 r_up^2 vt_ub(r_up) for any r_up >= r_M.  r_up = 2^(log2(c vf_M) / 3) (1 + 3e-5).
// cscale = cheap_c * scale(n_c), one product per cell.  A volume below 1e-30 m^3 (flushed logarithm) or a NaN is
// never skipped; an overflowing product gives +inf and is not skipped either.
template <int KIND>
__device__ __forceinline__ bool pair_cheap_may_collide(float cscale, float xm, float vf0, float vf1, u32 w3) {
    const float u_lo = (float)(w3 >> 8) * 0x1.0p-24f;  // exact in fp32, <= u
    float p_ub;
    bool unsure = false;
    if (KIND == 0) {
        p_ub = (vf0 + vf1) * xm * cscale;
    } else {
        const float vM = fmaxf(vf0, vf1);
        unsure = !(vM >= 1e-30f);
        float lg, r;
        asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(lg) : "f"(vM * 0.2387324f));
        asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(lg * 0.33333334f));
        r *= 1.00003f;
        const float r2 = r * r;
        const float t = r < 40e-6f ? 1.19e8f * r2 : 8.3e3f * r;
        p_ub = r2 * t * xm * cscale;
    }
    return unsure || !(u_lo >= p_ub + 1e-30f);
}

// Conservative test: returns false only when gamma = 0 is certain (then the pair changes nothing and,
// without debug outputs, needs no further work).  xj >= xk, (vj, vk) follow that order.
//   Golovin: the exact fp64 probability is five operations, so the test is exact:
//            gamma != 0  <=>  p >= 1  or  u < p            (p < 1 => floor(p) = 0, p - 0 = p)
//   geometric: an upper bound p_ub >= p from ~30 fp32 operations: with relative errors eps on the radii
//            and 2 eps on the fall speeds, K <= E pi ((r_j + r_k)(1 + eps))^2 (|vt_j - vt_k| + 2 eps (vt_j + vt_k)).
//            u >= p_ub (compared through a lower bound of u) => p < 1 and not (u < p) => gamma = 0.
__device__ __forceinline__ bool pair_may_collide(const PairArgs& a, long long xj, double vj, double vk, u32 w2, u32 w3,
                                                 u32 n_c) {
    if (a.kp.kind == 0) {
        const double K = __dmul_rn(a.kp.b, __dadd_rn(vj, vk));
        const double p = __dmul_rn(__dmul_rn(__dmul_rn(K, (double)xj), a.dtdV), (double)pair_scale_int(n_c));
        return (p >= 1.0) || (uniform_from_words(w2, w3) < p) || !(p == p);
    }
    const float fj = (float)vj, fk = (float)vk;
    bool unsure = !(fj > 1e-30f && fj < 1e30f && fk > 1e-30f && fk < 1e30f);  // outside the bound's validity
    const float rj = bound_radius(fj), rk = bound_radius(fk);
    const float tj = bound_fall_speed(rj, unsure), tk = bound_fall_speed(rk, unsure);
    const float up = 1.0f + 4.0f * BOUND_EPS;
    const float dvt = (fabsf(tj - tk) + (2.0f * BOUND_EPS) * (tj + tk)) * up;
    const float s = (rj + rk) * up;
    const float K_ub = a.Epi_up * (s * s) * dvt;
    const float p_ub = K_ub * __ll2float_ru(xj) * a.dtdV_up * (float)pair_scale_int(n_c) * up + 1e-30f;
    const float u_lo = (float)(w3 >> 8) * 0x1.0p-24f;  // exact in fp32, <= u (the low 29 bits are dropped)
    return unsure || !(u_lo >= p_ub);
}

// The whole rule for one pair, exactly.  (j0, k0) = original indices in shuffled order, (x0, v0) / (x1, v1) their pre-step
// attributes, (w2, w3) the Philox words of j0's uniform (R2).  (px0, pv0) / (px1, pv1): where the attributes of j0 / k0
// live (the caller's arrays, a shared-memory copy, or another block's shared memory).  Returns the number of
// super-droplets whose multiplicity became 0 (the split of xi_k = 1, R14).
__device__ __forceinline__ u32 pair_apply_at(const PairArgs& a, long long* px0, double* pv0, long long* px1, double* pv1,
                                             u32 j0, long long x0, double v0, long long x1, double v1, u32 w2, u32 w3,
                                             u32 n_c) {
    long long xj = x0, xk = x1;
    double vj = v0, vk = v1;
    long long *pxj = px0, *pxk = px1;
    double *pvj = pv0, *pvk = pv1;
    if (xj < xk) {  // order so that xi_j >= xi_k; ties keep the shuffled order (R8)
        xj = x1; xk = x0;
        vj = v1; vk = v0;
        pxj = px1; pxk = px0;
        pvj = pv1; pvk = pv0;
    }
    const double u = uniform_from_words(w2, w3);
    const double K = coalescence_kernel(a.kp, vj, vk);
    const double p = __dmul_rn(__dmul_rn(__dmul_rn(K, (double)xj), a.dtdV), (double)pair_scale_int(n_c));
    long long g = 0;
    if (p > 0.0) {
        if (p >= 0x1.0p63) {
            g = 0x7FFFFFFFFFFFFFFFLL;  // R11
        } else {
            const double fl = floor(p);
            g = (long long)fl + ((u < __dsub_rn(p, fl)) ? 1 : 0);
        }
    }
    long long gt = 0;
    u32 new_zeros = 0;
    if (g != 0 && xk != 0) {
        // gamma~ = min(gamma, floor(xi_j / xi_k)); the quotient is >= 1, so gamma == 1 needs no division (R12)
        gt = (g == 1) ? 1 : min(g, xj / xk);
        const double vnew = __dadd_rn(__dmul_rn((double)gt, vj), vk);
        const long long rem = xj - gt * xk;
        if (rem > 0) {
            *pxj = rem;
            *pvk = vnew;
        } else {  // equal-multiplicity split (R14)
            const long long h = xk / 2;
            *pxj = h;
            *pxk = xk - h;
            *pvj = vnew;
            *pvk = vnew;
            new_zeros = (h == 0);
        }
    }
    if (a.dbg_gamma) a.dbg_gamma[j0] = g;
    if (a.dbg_gamma_clamped) a.dbg_gamma_clamped[j0] = gt;
    return new_zeros;
}

// `xi`, `v`: arrays indexed by the original index (the caller's arrays, or a shared-memory copy of them).
__device__ __forceinline__ u32 pair_apply_to(const PairArgs& a, long long* __restrict__ xi, double* __restrict__ v, u32 j0,
                                             u32 k0, long long x0, double v0, long long x1, double v1, u32 w2, u32 w3,
                                             u32 n_c) {
    return pair_apply_at(a, xi + j0, v + j0, xi + k0, v + k0, j0, x0, v0, x1, v1, w2, w3, n_c);
}

__device__ __forceinline__ u32 pair_apply(const PairArgs& a, u32 j0, u32 k0, long long x0, double v0, long long x1,
                                          double v1, u32 w2, u32 w3, u32 n_c) {
    return pair_apply_to(a, a.xi, a.v, j0, k0, x0, v0, x1, v1, w2, w3, n_c);
}

// General pair kernel: gathers the attributes, regenerates j0's Philox block, runs both phases.
__device__ __forceinline__ void pair_collide(const PairArgs& a, u32 j0, u32 k0, u32 n_c) {
    const long long x0 = a.xi[j0], x1 = a.xi[k0];
    const double v0 = a.v[j0], v1 = a.v[k0];
    // a dead partner: gamma~ = 0 whatever gamma is (R7); only the debug gamma output needs the probability
    if ((x0 == 0 || x1 == 0) && !a.dbg_gamma) return;
    const PhiloxOut w = philox4x32_10(a.pk, (u64)j0);  // uniform of the first-shuffled member (R2)
    const bool swap = x0 < x1;
    if (!a.dbg_gamma &&
        !pair_may_collide(a, swap ? x1 : x0, swap ? v1 : v0, swap ? v0 : v1, w.w2, w.w3, n_c))
        return;
    pair_apply(a, j0, k0, x0, v0, x1, v1, w.w2, w.w3, n_c);
}

}  // namespace sdm
