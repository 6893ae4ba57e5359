// Device-side building blocks of the B200 SDM coalescence step (sm_100a).
// Nothing here is shared with oracle/: the arithmetic is restated from BASELINE.json north_star
// (a)-(c) and the readings in DESIGN.md.  Every fp64 expression that decides an integer uses
// explicit round-to-nearest intrinsics (__dmul_rn/__dadd_rn/__dsub_rn) so no FMA can be formed,
// in the operation order DESIGN.md R10/R13/R17 fixes.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace sdm {

typedef unsigned long long u64;
typedef unsigned int u32;

// ------------------------------------------------------------------------------------------
// a1: Philox-4x32-10 (north_star (a); Salmon et al. 2011).  The ten round keys depend only on
// (seed) and are the same for every super-droplet, so the host precomputes them once per step.
// ------------------------------------------------------------------------------------------
struct PhiloxKeys {
    u32 k0[10];
    u32 k1[10];
    u32 step_lo, step_hi;
    u32 p1_lo, p1_hi;  // 0xCD9E8D57 * step_lo: the first round's second product is the same for every super-droplet
    u64 index_base;  // counter of array entry i is index_base + i (SDM_OPT_INDEX_BASE; R34)
};

__host__ __device__ inline PhiloxKeys make_philox_keys(u64 seed, u64 step, u64 index_base = 0) {
    PhiloxKeys pk;
    u32 a = (u32)seed, b = (u32)(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        pk.k0[r] = a;
        pk.k1[r] = b;
        a += 0x9E3779B9u;
        b += 0xBB67AE85u;
    }
    pk.step_lo = (u32)step;
    pk.step_hi = (u32)(step >> 32);
    const u64 p1 = (u64)0xCD9E8D57u * (u64)pk.step_lo;
    pk.p1_lo = (u32)p1;
    pk.p1_hi = (u32)(p1 >> 32);
    pk.index_base = index_base;
    return pk;
}

struct PhiloxOut {
    u32 w0, w1, w2, w3;
};

// The step-dependent words of the block: counter words 2, 3 = the step, and 0xCD9E8D57 * lo32(step), the first
// round's second product, which is the same for every super-droplet.
struct PhiloxStep {
    u32 step_hi, p1_lo, p1_hi;
};
__host__ __device__ inline PhiloxStep make_philox_step(u64 step) {
    const u64 p1 = (u64)0xCD9E8D57u * (u64)(u32)step;
    PhiloxStep s;
    s.step_hi = (u32)(step >> 32);
    s.p1_lo = (u32)p1;
    s.p1_hi = (u32)(p1 >> 32);
    return s;
}

// `ps` overrides the step stored in `pk` (kernels that loop over steps themselves); the round keys come from `pk`.
__device__ __forceinline__ PhiloxOut philox4x32_10(const PhiloxKeys& pk, const PhiloxStep& ps, u64 i) {
    i += pk.index_base;
    u32 c0 = (u32)i, c1 = (u32)(i >> 32), c2, c3 = ps.step_hi;
    {  // round 0: the counter words 2, 3 are the step, so 0xCD9E8D57 * c2 comes precomputed
        const u64 p0 = (u64)0xD2511F53u * (u64)c0;
        const u32 n0 = ps.p1_hi ^ c1 ^ pk.k0[0];
        c2 = (u32)(p0 >> 32) ^ c3 ^ pk.k1[0];
        c1 = ps.p1_lo;
        c3 = (u32)p0;
        c0 = n0;
    }
#pragma unroll
    for (int r = 1; r < 10; ++r) {
        const u64 p0 = (u64)0xD2511F53u * (u64)c0;  // IMAD.WIDE.U32
        const u64 p1 = (u64)0xCD9E8D57u * (u64)c2;
        const u32 n0 = (u32)(p1 >> 32) ^ c1 ^ pk.k0[r];
        const u32 n2 = (u32)(p0 >> 32) ^ c3 ^ pk.k1[r];
        c1 = (u32)p1;
        c3 = (u32)p0;
        c0 = n0;
        c2 = n2;
    }
    PhiloxOut o;
    o.w0 = c0; o.w1 = c1; o.w2 = c2; o.w3 = c3;
    return o;
}

__device__ __forceinline__ PhiloxOut philox4x32_10(const PhiloxKeys& pk, u64 i) {
    PhiloxStep ps;
    ps.step_hi = pk.step_hi;
    ps.p1_lo = pk.p1_lo;
    ps.p1_hi = pk.p1_hi;
    return philox4x32_10(pk, ps, i);
}

// Permutation key only (word 0).
__device__ __forceinline__ u32 philox_perm_key(const PhiloxKeys& pk, u64 i) { return philox4x32_10(pk, i).w0; }

// 53-bit uniform in [0,1) from words 3:2 (R3).
__device__ __forceinline__ double uniform_from_words(u32 w2, u32 w3) {
    const u64 bits = (((u64)w3 << 32) | (u64)w2) >> 11;
    return __dmul_rn((double)bits, 0x1.0p-53);
}

// ------------------------------------------------------------------------------------------
// Relaxed / release / acquire accesses at gpu scope for the decoupled look-back tile states.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ u32 ld_relaxed_u32(const u32* p) {
    u32 v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed_u32(u32* p, u32 v) {
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ u32 ld_acquire_u32(const u32* p) {
    u32 v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_u32(u32* p, u32 v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

__device__ __forceinline__ u32 lanemask_lt() {
    u32 m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// Streaming (read-once / write-once) global accesses: keep L1 for the gathers that reuse lines.
__device__ __forceinline__ u64 ld_stream_u64(const u64* p) {
    u64 v;
    asm volatile("ld.global.L1::no_allocate.u64 %0, [%1];" : "=l"(v) : "l"(p));
    return v;
}

// ------------------------------------------------------------------------------------------
// Coalescence kernels (north_star (c); R15-R17).  No FMA anywhere.
// ------------------------------------------------------------------------------------------
struct KernelParams {
    int kind;  // 0 Golovin, 1 geometric, 2 geometric with a tabulated collision efficiency (R39)
    double b;
    double Epi;  // E * pi, one host-side product (E * 3.141592653589793); kind 2: E = the table's maximum (bounds only)
    // kind 2: E(r_big, r_small / r_big) on n_r radii (ascending) x n_p ratios j / (n_p - 1); device pointers
    int n_r, n_p;
    const double* eff_radius;
    const double* eff_table;
};

// R39: bilinear interpolation in a fixed order (every product rounded before its sum); outside the radius grid the
// value on its edge.  The interval is the last one whose lower edge is <= r_big (binary search: same interval as the
// linear scan of the definition).
__device__ __forceinline__ double collision_efficiency(const KernelParams& kp, double r_big, double p) {
    int lo = 0, hi = kp.n_r - 1;  // invariant: R[lo] <= r_big (or lo = 0), R[hi] > r_big (or hi = n_r - 1)
    while (hi - lo > 1) {
        const int m = (lo + hi) >> 1;
        if (__ldg(kp.eff_radius + m) <= r_big) lo = m;
        else hi = m;
    }
    const double r0 = __ldg(kp.eff_radius + lo), r1 = __ldg(kp.eff_radius + lo + 1);
    double t_r = __ddiv_rn(__dsub_rn(r_big, r0), __dsub_rn(r1, r0));
    if (!(t_r > 0.0)) t_r = 0.0;
    if (t_r > 1.0) t_r = 1.0;
    const double f = __dmul_rn(p, (double)(kp.n_p - 1));
    int j = (int)floor(f);
    j = j < 0 ? 0 : (j > kp.n_p - 2 ? kp.n_p - 2 : j);
    const double t_p = __dsub_rn(f, (double)j);
    const double* T0 = kp.eff_table + (size_t)lo * kp.n_p + j;
    const double* T1 = T0 + kp.n_p;
    const double a0 = __ldg(T0), a1 = __ldg(T0 + 1), b0 = __ldg(T1), b1 = __ldg(T1 + 1);
    const double e0 = __dadd_rn(a0, __dmul_rn(t_p, __dsub_rn(a1, a0)));
    const double e1 = __dadd_rn(b0, __dmul_rn(t_p, __dsub_rn(b1, b0)));
    return __dadd_rn(e0, __dmul_rn(t_r, __dsub_rn(e1, e0)));
}

// R17: libm-free cube root: integer seed for x^(-1/3), four Newton steps, r = x z^2, one polish.
__device__ __forceinline__ double det_cbrt(double x) {
    if (x == 0.0) return 0.0;
    const long long xb = __double_as_longlong(x);
    const long long zb = 0x553F0A3D70A3D70BLL - xb / 3;
    double z = __longlong_as_double(zb);
    const double four_thirds = 0x1.5555555555555p+0;
    const double one_third = 0x1.5555555555555p-2;
#pragma unroll
    for (int it = 0; it < 4; ++it) {
        const double z3 = __dmul_rn(__dmul_rn(z, z), z);
        z = __dmul_rn(z, __dsub_rn(four_thirds, __dmul_rn(one_third, __dmul_rn(x, z3))));
    }
    double r = __dmul_rn(__dmul_rn(x, z), z);
    const double r3 = __dmul_rn(__dmul_rn(r, r), r);
    r = __dsub_rn(r, __dmul_rn(__dsub_rn(r3, x), __dmul_rn(__dmul_rn(z, z), one_third)));
    return r;
}

// R16: three-regime power-law fall speed (exponents 2, 1, 1/2), SI.
__device__ __forceinline__ double terminal_velocity(double r) {
    if (r < 40e-6) return __dmul_rn(1.19e8, __dmul_rn(r, r));
    if (r < 600e-6) return __dmul_rn(8e3, r);
    return __dmul_rn(2.01e2, __dsqrt_rn(r));
}

__device__ __forceinline__ double coalescence_kernel(const KernelParams& kp, double vj, double vk) {
    if (kp.kind == 0) return __dmul_rn(kp.b, __dadd_rn(vj, vk));
    const double rj = det_cbrt(__dmul_rn(vj, 0.238732414637843));
    const double rk = det_cbrt(__dmul_rn(vk, 0.238732414637843));
    const double s = __dadd_rn(rj, rk);
    const double dv = fabs(__dsub_rn(terminal_velocity(rj), terminal_velocity(rk)));
    double Epi = kp.Epi;
    if (kp.kind == 2) {
        const double r_big = rj > rk ? rj : rk, r_small = rj > rk ? rk : rj;
        const double E = collision_efficiency(kp, r_big, r_big > 0.0 ? __ddiv_rn(r_small, r_big) : 0.0);
        Epi = __dmul_rn(E, 3.141592653589793);
    }
    return __dmul_rn(__dmul_rn(Epi, __dmul_rn(s, s)), dv);
}

}  // namespace sdm
