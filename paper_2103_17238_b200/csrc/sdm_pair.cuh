// The per-pair rule of the SDM step (north_star (c); SURVEY.md 8(c) O4 body), shared by the general
// pair kernel (sdm_pair.cu) and the fused per-cell kernel (sdm_cellsort.cu).
//
// fp64 discipline: the pair probability and the volume update use __dmul_rn/__dadd_rn in the order
// ((K * xi_j) * dtdV) * scale and gamma~ * v_j + v_k (R10, R13) -- no FMA contraction.
#pragma once
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
    KernelParams kp;
    PhiloxKeys pk;
    long long* dbg_gamma;
    long long* dbg_gamma_clamped;
};

// Exact early-out for the geometric kernel: an upper bound of the pair probability from a handful of
// fp32 operations, p_ub >= p (every factor rounded up by far more than its error: K <= E pi (2 r_max)^2
// max_regime v_t(r_max), since each regime of the fall-speed law is increasing).  When u >= p_ub then
// p < 1 and not (u < p - floor(p)), i.e. gamma = 0 and nothing changes -- the same result the full fp64
// evaluation gives, without the two cube roots.  Returns +inf when no bound is available.
__device__ __forceinline__ double pair_probability_bound(const PairArgs& a, double v_max, long long xj, double scale) {
    if (a.kp.kind != 1) return __longlong_as_double(0x7FF0000000000000LL);
    const float vm = __double2float_ru(v_max);
    if (!(vm > 1e-30f) || !(vm < 1e30f)) return __longlong_as_double(0x7FF0000000000000LL);
    const float r = __fmul_ru(cbrtf(__fmul_ru(vm, 0.2387325f)), 1.00001f);
    const float vt = fmaxf(fmaxf(__fmul_ru(1.19e8f, __fmul_ru(r, r)), __fmul_ru(8e3f, r)),
                           __fmul_ru(2.01e2f, __fsqrt_ru(r)));
    const float K = __fmul_ru(__fmul_ru(__fmul_ru(4.00001f, __fmul_ru(r, r)), vt), __double2float_ru(a.kp.Epi));
    return __dmul_ru(__dmul_ru(__dmul_ru(__dmul_ru((double)K, (double)xj), a.dtdV), scale), 1.0001);
}

// HAS_U: the caller already holds the uniform of the first-shuffled member (fused kernel: taken from the
// Philox block that also gave its permutation key); otherwise it is regenerated here.
template <bool HAS_U>
__device__ __forceinline__ void pair_collide(const PairArgs& a, u32 j0, u32 k0, u32 n_c, double u_in = 0.0) {
    long long xj = a.xi[j0], xk = a.xi[k0];
    double vj = a.v[j0], vk = a.v[k0];
    u32 j = j0, k = k0;
    if (xj < xk) {  // order so that xi_j >= xi_k; ties keep the shuffled order (R8)
        const long long tx = xj; xj = xk; xk = tx;
        const double tv = vj; vj = vk; vk = tv;
        j = k0; k = j0;
    }
    // a dead partner: gamma~ = 0 whatever gamma is (R7); only the debug gamma output needs the probability
    if (xk == 0 && !a.dbg_gamma) return;
    double u;
    if (HAS_U) {
        u = u_in;
    } else {
        const PhiloxOut w = philox4x32_10(a.pk, (u64)j0);  // uniform of the first-shuffled member (R2)
        u = uniform_from_words(w.w2, w.w3);
    }
    // (n_c (n_c - 1) / 2) / floor(n_c / 2) == n_c if odd else n_c - 1   (R9)
    const double scale = (double)((n_c & 1u) ? n_c : n_c - 1u);
    if (u >= pair_probability_bound(a, fmax(vj, vk), xj, scale)) return;  // gamma = 0, exactly
    const double K = coalescence_kernel(a.kp, vj, vk);
    const double p = __dmul_rn(__dmul_rn(__dmul_rn(K, (double)xj), a.dtdV), scale);
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
    if (g != 0 && xk != 0) {
        // gamma~ = min(gamma, floor(xi_j / xi_k)); the quotient is >= 1, so gamma == 1 needs no division (R12)
        gt = (g == 1) ? 1 : min(g, xj / xk);
        const double vnew = __dadd_rn(__dmul_rn((double)gt, vj), vk);
        const long long rem = xj - gt * xk;
        if (rem > 0) {
            a.xi[j] = rem;
            a.v[k] = vnew;
        } else {  // equal-multiplicity split (R14)
            const long long h = xk / 2;
            a.xi[j] = h;
            a.xi[k] = xk - h;
            a.v[j] = vnew;
            a.v[k] = vnew;
        }
    }
    if (a.dbg_gamma) a.dbg_gamma[j0] = g;
    if (a.dbg_gamma_clamped) a.dbg_gamma_clamped[j0] = gt;
}

}  // namespace sdm
