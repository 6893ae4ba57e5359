// SDM coalescence-step ORACLE -- test infrastructure, NOT the product.
//
// A plain, serial, obviously-correct CPU statement of the Super-Droplet Method
// Monte-Carlo collisional-growth step (Shima et al. 2009), in
// the order and notation of SURVEY.md section 8(c) O1..O6 and BASELINE.json
// north_star (a)..(d).  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may call it.  It shares no code, header,
// table or helper with the CUDA path under paper_2103_17238_b200/csrc/.
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -fno-fast-math -shared -fPIC
// (no FMA contraction, so every fp64 expression below rounds once per operator,
// in the written order -- readings R10, R13, R17 in DESIGN.md).
//
// Pins (tests/test_oracle_*.py, all "-m 'not gpu'"):
//   philox4x32_10 ....... C++26 [rand.predef] 10000th-value requirement, Salmon et
//                         al. 2011 known-answer vectors, curand header cross-check
//   uniform conversion .. extremes + moments
//   shuffle ............. permutation invariants, 3-SD chi-square
//   pair/p/gamma ........ brute-force 2- and 3-SD cells, binomial frequencies
//   update/clamp/split .. hand cases, exact integer-volume conservation
//   whole box run ....... Golovin analytic Smoluchowski solution
//   volume spectrum ..... hand case with values on the edges, numpy.histogram on random data,
//                         closed-form bin masses of the exponential spectrum
//   geometric kernel .... hand values; det_cbrt vs libm cbrt.  Whole-run statistics
//                         with the geometric kernel: PARITY UNPINNED beyond invariants.
//   efficiency table .... a constant table reproduces the geometric kernel bit for bit; a 2 x 2 table by hand;
//                         scipy's RegularGridInterpolator on random tables; clamping outside the grid
//   displacement (O8) ... hand cases on cell edges and at the periodic seam, numpy floor/mod, and a
//                         divergence-free shear field with whole-cell Courant numbers (closed form:
//                         every row shifts by its own number of cells, occupancy permutes)
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <numeric>
#include <vector>

extern "C" {

// ---------------------------------------------------------------------------
// O1  Philox-4x32-10 (Salmon et al. 2011), north_star (a), reading R1.
// ---------------------------------------------------------------------------
void oracle_philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
    uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
    uint32_t k0 = key_in[0], k1 = key_in[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) {  // Weyl key schedule: bump before every round but the first
            k0 += 0x9E3779B9u;
            k1 += 0xBB67AE85u;
        }
        const uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n1 = lo1;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        const uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Words -> (permutation key, uniform).  Readings R1, R3: key = w0; u is the 53-bit
// dyadic fraction ((w3:w2) >> 11) * 2^-53 in [0, 1).
double oracle_uniform_from_words(uint32_t w2, uint32_t w3) {
    const uint64_t bits = (((uint64_t)w3 << 32) | (uint64_t)w2) >> 11;
    return (double)bits * 0x1.0p-53;
}

// One block per super-droplet per step: ctr = {lo32(i), hi32(i), lo32(step), hi32(step)},
// key = {lo32(seed), hi32(seed)}.
void oracle_sd_random(uint64_t seed, uint64_t step, uint64_t i, uint32_t* perm_key, double* u) {
    const uint32_t ctr[4] = {(uint32_t)i, (uint32_t)(i >> 32), (uint32_t)step, (uint32_t)(step >> 32)};
    const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    uint32_t w[4];
    oracle_philox4x32_10(ctr, key, w);
    *perm_key = w[0];
    *u = oracle_uniform_from_words(w[2], w[3]);
}

void oracle_sd_random_batch(uint64_t seed, uint64_t step, uint64_t i0, int64_t n, uint32_t* perm_key,
                            double* u) {
    for (int64_t t = 0; t < n; ++t) oracle_sd_random(seed, step, i0 + (uint64_t)t, &perm_key[t], &u[t]);
}

// ---------------------------------------------------------------------------
// Coalescence kernels K(v_j, v_k)  (north_star (c); PAPER.md:66,75 Golovin,
// PAPER.md:96 "geometric sweep-out"; readings R15, R16, R17).
// ---------------------------------------------------------------------------
struct oracle_kernel_params {
    int32_t kind;  // 0 = Golovin, 1 = geometric, 2 = geometric with a tabulated collision efficiency
    int32_t _pad;
    double b;      // Golovin: K = b (v_j + v_k), b in 1/s, volumes in m^3
    double E;      // geometric: collision efficiency
    // kind 2 ("more sophisticated collision kernels"; reading R39): E(r_big, p)
    int32_t n_r, n_p;        // grid: n_r radii (strictly ascending, m), n_p ratios p_j = j / (n_p - 1)
    const double* radius;    // [n_r]
    const double* table;     // [n_r][n_p], row-major, >= 0
};

// R17: libm-free cube root: integer seed for x^(-1/3), four Newton steps on z,
// r = x z^2, one polishing step on r.  Only + - * and integer ops.
double oracle_det_cbrt(double x) {
    if (x == 0.0) return 0.0;
    int64_t xb;
    std::memcpy(&xb, &x, 8);
    const int64_t zb = (int64_t)0x553F0A3D70A3D70BLL - xb / 3;
    double z;
    std::memcpy(&z, &zb, 8);
    const double four_thirds = 0x1.5555555555555p+0;
    const double one_third = 0x1.5555555555555p-2;
    for (int it = 0; it < 4; ++it) {
        z = z * (four_thirds - one_third * (x * ((z * z) * z)));
    }
    double r = (x * z) * z;
    r = r - (((r * r) * r - x) * ((z * z) * one_third));
    return r;
}

// R16: three-regime power law (exponents 2, 1, 1/2), SI units.
double oracle_terminal_velocity(double r) {
    if (r < 40e-6) return 1.19e8 * (r * r);
    if (r < 600e-6) return 8e3 * r;
    return 2.01e2 * std::sqrt(r);
}

double oracle_radius(double v) { return oracle_det_cbrt(v * 0.238732414637843); }

// R39: tabulated collision efficiency E(r_big, p), p = r_small / r_big in [0, 1], bilinear in a fixed order:
//   i   = the interval of the radius grid that holds r_big (largest i with R[i] <= r_big, clamped to [0, n_r - 2]),
//   t_r = (r_big - R[i]) / (R[i+1] - R[i]) clamped to [0, 1]            (outside the grid: the value on its edge)
//   f   = p * (n_p - 1);  j = min(floor(f), n_p - 2);  t_p = f - j
//   e0  = T[i][j]   + t_p * (T[i][j+1]   - T[i][j])
//   e1  = T[i+1][j] + t_p * (T[i+1][j+1] - T[i+1][j])
//   E   = e0 + t_r * (e1 - e0)                                            (every product rounded before its sum: no FMA)
double oracle_efficiency(const oracle_kernel_params* kp, double r_big, double p) {
    const int32_t n_r = kp->n_r, n_p = kp->n_p;
    int32_t i = 0;
    while (i + 2 < n_r && kp->radius[i + 1] <= r_big) ++i;  // linear scan: the last interval whose lower edge is <= r_big
    double t_r = (r_big - kp->radius[i]) / (kp->radius[i + 1] - kp->radius[i]);
    if (!(t_r > 0.0)) t_r = 0.0;
    if (t_r > 1.0) t_r = 1.0;
    const double f = p * (double)(n_p - 1);
    int32_t j = (int32_t)std::floor(f);
    if (j < 0) j = 0;
    if (j > n_p - 2) j = n_p - 2;
    const double t_p = f - (double)j;
    const double* T0 = kp->table + (size_t)i * n_p;
    const double* T1 = T0 + n_p;
    const double e0 = T0[j] + t_p * (T0[j + 1] - T0[j]);
    const double e1 = T1[j] + t_p * (T1[j + 1] - T1[j]);
    return e0 + t_r * (e1 - e0);
}

double oracle_kernel(const oracle_kernel_params* kp, double vj, double vk) {
    if (kp->kind == 0) {
        return kp->b * (vj + vk);
    }
    const double rj = oracle_radius(vj);
    const double rk = oracle_radius(vk);
    const double s = rj + rk;
    double E = kp->E;
    if (kp->kind == 2) {
        const double r_big = rj > rk ? rj : rk, r_small = rj > rk ? rk : rj;
        E = oracle_efficiency(kp, r_big, r_big > 0.0 ? r_small / r_big : 0.0);
    }
    return ((E * 3.141592653589793) * (s * s)) *
           std::fabs(oracle_terminal_velocity(rj) - oracle_terminal_velocity(rk));
}

// ---------------------------------------------------------------------------
// The per-pair rule (O4 body).  gamma from p and u; clamp; Shima's update with
// the equal-multiplicity split.  xi_j >= xi_k on entry.  Returns gamma-tilde.
// ---------------------------------------------------------------------------
int64_t oracle_gamma_from_p(double p, double u) {
    if (!(p > 0.0)) return 0;
    if (p >= 0x1.0p63) return std::numeric_limits<int64_t>::max();  // R11
    const double fl = std::floor(p);
    return (int64_t)fl + ((u < p - fl) ? 1 : 0);
}

int64_t oracle_pair_update(int64_t* xi_j, int64_t* xi_k, double* v_j, double* v_k, int64_t g) {
    if (g == 0 || *xi_k == 0) return 0;
    const int64_t ratio = *xi_j / *xi_k;
    const int64_t gt = std::min(g, ratio);
    const double vnew = (double)gt * (*v_j) + (*v_k);  // R13 (no FMA: -ffp-contract=off)
    const int64_t rem = *xi_j - gt * (*xi_k);
    if (rem > 0) {
        *xi_j = rem;
        *v_k = vnew;
    } else {  // equal-multiplicity split (R14: h may be 0 when xi_k == 1)
        const int64_t h = *xi_k / 2;
        *xi_j = h;
        *xi_k = *xi_k - h;
        *v_j = vnew;
        *v_k = vnew;
    }
    return gt;
}

// ---------------------------------------------------------------------------
// O1..O4: one coalescence step.  All pointers are HOST pointers.  xi, v updated in
// place at the original indices; cell_id read-only.  Optional outputs (nullable):
//   perm_out[s]           = idx[s] (the shuffled order, cells contiguous)
//   gamma_out[i], gamma_clamped_out[i] at i = idx[start+2a] (first-sorted member), 0 elsewhere
//   cell_start_out[c]     = exclusive scan of per-cell counts, length n_cell+1
// Returns 0, or -1 (invalid argument), -4 (bad data: cell_id out of range).
// ---------------------------------------------------------------------------
//
// index_base (reading R34): the Philox counter of array entry i is index_base + i, so a
// shard that holds entries [index_base, index_base + n_sd) of a larger array (whole cells only) draws
// the numbers the unsharded step draws for them.  oracle_coalescence_step is index_base = 0.
int oracle_coalescence_step_shard(int64_t* xi, double* v, const int32_t* cell_id, int64_t n_sd,
                                  int32_t n_cell, double dt, double dV, const oracle_kernel_params* kp,
                                  uint64_t seed, uint64_t step, uint64_t index_base, int32_t* perm_out,
                                  int64_t* gamma_out, int64_t* gamma_clamped_out, int32_t* cell_start_out) {
    if (n_sd < 0 || n_cell < 1 || !(dt > 0.0) || !(dV > 0.0) || kp == nullptr) return -1;
    const int64_t N = n_sd;
    for (int64_t i = 0; i < N; ++i)
        if (cell_id[i] < 0 || cell_id[i] >= n_cell) return -4;

    // O1: one Philox block per super-droplet
    std::vector<uint32_t> key(N);
    std::vector<double> u(N);
    for (int64_t i = 0; i < N; ++i) oracle_sd_random(seed, step, index_base + (uint64_t)i, &key[i], &u[i]);

    // O2: stable sort of indices by (cell_id << 32) | key, ascending (R4, R5)
    std::vector<uint64_t> sortkey(N);
    for (int64_t i = 0; i < N; ++i) sortkey[i] = ((uint64_t)(uint32_t)cell_id[i] << 32) | key[i];
    std::vector<int32_t> idx(N);
    std::iota(idx.begin(), idx.end(), 0);
    std::stable_sort(idx.begin(), idx.end(),
                     [&](int32_t a, int32_t b) { return sortkey[a] < sortkey[b]; });

    // O3: per-cell counts and exclusive scan
    std::vector<int64_t> count(n_cell, 0), start((size_t)n_cell + 1, 0);
    for (int64_t i = 0; i < N; ++i) count[cell_id[i]] += 1;
    for (int32_t c = 0; c < n_cell; ++c) start[c + 1] = start[c] + count[c];

    if (perm_out) std::copy(idx.begin(), idx.end(), perm_out);
    if (cell_start_out)
        for (int32_t c = 0; c <= n_cell; ++c) cell_start_out[c] = (int32_t)start[c];
    if (gamma_out) std::fill(gamma_out, gamma_out + N, (int64_t)0);
    if (gamma_clamped_out) std::fill(gamma_clamped_out, gamma_clamped_out + N, (int64_t)0);

    const double dtdV = dt / dV;  // R10: one division, then left-to-right products

    // O4: pairs of neighbours in the shuffled order, cell by cell
    for (int32_t c = 0; c < n_cell; ++c) {
        const int64_t n = count[c];
        if (n < 2) continue;  // R6
        const int64_t n_pairs = n / 2;
        // north_star (c): (n_c (n_c - 1) / 2) / floor(n_c / 2), exact in integers (R9)
        const double scale = (double)(((n * (n - 1)) / 2) / n_pairs);
        for (int64_t a = 0; a < n_pairs; ++a) {
            const int32_t j0 = idx[start[c] + 2 * a];
            const int32_t k0 = idx[start[c] + 2 * a + 1];
            int32_t j = j0, k = k0;
            if (xi[j0] < xi[k0]) { j = k0; k = j0; }  // xi_j >= xi_k; tie keeps sorted order (R8)
            const double K = oracle_kernel(kp, v[j], v[k]);
            const double p = ((K * (double)xi[j]) * dtdV) * scale;
            const int64_t g = oracle_gamma_from_p(p, u[j0]);  // R2: uniform of the first-sorted member
            const int64_t gt = oracle_pair_update(&xi[j], &xi[k], &v[j], &v[k], g);
            if (gamma_out) gamma_out[j0] = g;
            if (gamma_clamped_out) gamma_clamped_out[j0] = gt;
        }
    }
    return 0;
}

// O5: stable erase of entries with xi == 0 from (xi, v, cell_id); returns the new n_sd.
int64_t oracle_remove_zero_multiplicity(int64_t* xi, double* v, int32_t* cell_id, int64_t n_sd) {
    int64_t out = 0;
    for (int64_t i = 0; i < n_sd; ++i) {
        if (xi[i] != 0) {
            xi[out] = xi[i];
            v[out] = v[i];
            cell_id[out] = cell_id[i];
            ++out;
        }
    }
    return out;
}

// O6: per-cell count, sum xi, sum xi*v, sum xi*v*v, summed in index order. Outputs nullable.
int oracle_cell_stats(const int64_t* xi, const double* v, const int32_t* cell_id, int64_t n_sd,
                      int32_t n_cell, int32_t* count, int64_t* sum_xi, double* sum_xi_v,
                      double* sum_xi_v2) {
    if (n_sd < 0 || n_cell < 1) return -1;
    for (int32_t c = 0; c < n_cell; ++c) {
        if (count) count[c] = 0;
        if (sum_xi) sum_xi[c] = 0;
        if (sum_xi_v) sum_xi_v[c] = 0.0;
        if (sum_xi_v2) sum_xi_v2[c] = 0.0;
    }
    for (int64_t i = 0; i < n_sd; ++i) {
        const int32_t c = cell_id[i];
        if (c < 0 || c >= n_cell) return -4;
        const double x = (double)xi[i];
        if (count) count[c] += 1;
        if (sum_xi) sum_xi[c] += xi[i];
        if (sum_xi_v) sum_xi_v[c] += x * v[i];
        if (sum_xi_v2) sum_xi_v2[c] += (x * v[i]) * v[i];
    }
    return 0;
}

int oracle_coalescence_step(int64_t* xi, double* v, const int32_t* cell_id, int64_t n_sd,
                            int32_t n_cell, double dt, double dV, const oracle_kernel_params* kp,
                            uint64_t seed, uint64_t step, int32_t* perm_out, int64_t* gamma_out,
                            int64_t* gamma_clamped_out, int32_t* cell_start_out) {
    return oracle_coalescence_step_shard(xi, v, cell_id, n_sd, n_cell, dt, dV, kp, seed, step, 0, perm_out,
                                         gamma_out, gamma_clamped_out, cell_start_out);
}

// ---------------------------------------------------------------------------
// O7  Volume spectrum (the paper's ParticlesVolumeSpectrum(radius_bins_edges)
// product).  The paper is silent on the product's normalisation; reading R35: the raw
// per-bin sums.  Bin b holds the entries with edges[b] <= v < edges[b+1] (edges strictly ascending
// VOLUMES: the caller converts its radius edges once, so no cube root enters the bin decision);
// entries outside [edges[0], edges[n_edges-1]) are not counted.
//   count[b]    number of array entries in the bin (whatever their multiplicity)
//   sum_xi[b]   sum of multiplicities            (exact)
//   sum_xi_v[b] sum of double(xi) * v, in index order
// Returns 0, or -1 (invalid argument: fewer than 2 edges, edges not strictly ascending / not finite).
// ---------------------------------------------------------------------------
int oracle_volume_spectrum(const int64_t* xi, const double* v, int64_t n_sd, const double* edges,
                           int32_t n_edges, int64_t* count, int64_t* sum_xi, double* sum_xi_v) {
    if (n_sd < 0 || n_edges < 2) return -1;
    for (int32_t e = 0; e < n_edges; ++e) {
        if (!std::isfinite(edges[e])) return -1;
        if (e > 0 && !(edges[e] > edges[e - 1])) return -1;
    }
    const int32_t n_bins = n_edges - 1;
    for (int32_t b = 0; b < n_bins; ++b) {
        if (count) count[b] = 0;
        if (sum_xi) sum_xi[b] = 0;
        if (sum_xi_v) sum_xi_v[b] = 0.0;
    }
    for (int64_t i = 0; i < n_sd; ++i) {
        const double x = v[i];
        if (!(x >= edges[0]) || !(x < edges[n_bins])) continue;  // outside (NaN included)
        int32_t b = 0;
        while (!(x < edges[b + 1])) ++b;  // linear scan: the first bin whose upper edge exceeds v
        if (count) count[b] += 1;
        if (sum_xi) sum_xi[b] += xi[i];
        if (sum_xi_v) sum_xi_v[b] += (double)xi[i] * x;
    }
    return 0;
}

// ---------------------------------------------------------------------------
// O8  Displacement + cell_id recomputation (the step BEFORE the coalescence path; the paper's
// "particle displacement" dynamic, on the kinematic_2d grid of PAPER.md:112-118).  The paper gives no
// scheme; readings R36-R38: positions in GRID UNITS, x in [0, nx), z in [0, nz), both directions
// periodic; cell_id = floor(z) * nx + floor(x) (row-major, x fastest); one explicit-Euler step with the velocity
// (grid units per second, caller-supplied per cell) of the cell the super-droplet is in BEFORE the move:
//     c  = cell_of(x, z)
//     x1 = x + (u[c] * dt)          (one multiplication, one addition, no FMA)
//     x1 = wrap(x1, nx)             (at most one period: |u dt| < nx is the caller's contract)
// and the same for z with w[c], nz.  wrap(q, n): q >= n -> q - n;  q < 0 -> q + n;  and if the result is still
// outside [0, n) -- only possible when a tiny negative q rounds q + n up to n -- it is 0.
// ---------------------------------------------------------------------------
double oracle_wrap_periodic(double q, int32_t n) {
    const double dn = (double)n;
    if (q >= dn) q = q - dn;
    else if (q < 0.0) q = q + dn;
    if (!(q >= 0.0 && q < dn)) q = 0.0;
    return q;
}

int32_t oracle_cell_of(double x, double z, int32_t nx, int32_t nz) {
    int64_t ix = (int64_t)std::floor(x), iz = (int64_t)std::floor(z);
    if (ix < 0) ix = 0;  // positions are inside the domain by contract; clamp keeps bad data memory-safe
    if (ix >= nx) ix = nx - 1;
    if (iz < 0) iz = 0;
    if (iz >= nz) iz = nz - 1;
    return (int32_t)(iz * (int64_t)nx + ix);
}

int oracle_cell_id_from_positions(const double* x, const double* z, int64_t n_sd, int32_t nx, int32_t nz,
                                  int32_t* cell_id) {
    if (n_sd < 0 || nx < 1 || nz < 1 || (int64_t)nx * nz > 2147483647LL) return -1;
    for (int64_t i = 0; i < n_sd; ++i) cell_id[i] = oracle_cell_of(x[i], z[i], nx, nz);
    return 0;
}

int oracle_displace(double* x, double* z, int32_t* cell_id, int64_t n_sd, int32_t nx, int32_t nz,
                    const double* u_cell, const double* w_cell, double dt) {
    if (n_sd < 0 || nx < 1 || nz < 1 || (int64_t)nx * nz > 2147483647LL || !(dt > 0.0)) return -1;
    for (int64_t i = 0; i < n_sd; ++i) {
        const int32_t c = oracle_cell_of(x[i], z[i], nx, nz);
        const double x1 = oracle_wrap_periodic(x[i] + (u_cell[c] * dt), nx);
        const double z1 = oracle_wrap_periodic(z[i] + (w_cell[c] * dt), nz);
        x[i] = x1;
        z[i] = z1;
        cell_id[i] = oracle_cell_of(x1, z1, nx, nz);
    }
    return 0;
}

// Exact total of xi*v for integer-valued volumes (R22), in 128-bit integers; returned as hi/lo.
void oracle_total_xi_v_int128(const int64_t* xi, const double* v, int64_t n_sd, int64_t* hi,
                              uint64_t* lo) {
    __int128 acc = 0;
    for (int64_t i = 0; i < n_sd; ++i) acc += (__int128)xi[i] * (__int128)(int64_t)v[i];
    *hi = (int64_t)(acc >> 64);
    *lo = (uint64_t)acc;
}

// Convenience for the whole-run checks and the CPU baseline: `n_steps` consecutive steps
// step0, step0+1, ... with optional compaction every `compact_every` steps (0 = never).
// Returns the final n_sd (>= 0) or a negative error.
int64_t oracle_run(int64_t* xi, double* v, int32_t* cell_id, int64_t n_sd, int32_t n_cell, double dt,
                   double dV, const oracle_kernel_params* kp, uint64_t seed, uint64_t step0,
                   int64_t n_steps, int64_t compact_every) {
    for (int64_t s = 0; s < n_steps; ++s) {
        const int rc = oracle_coalescence_step(xi, v, cell_id, n_sd, n_cell, dt, dV, kp, seed,
                                               step0 + (uint64_t)s, nullptr, nullptr, nullptr, nullptr);
        if (rc != 0) return rc;
        if (compact_every > 0 && ((s + 1) % compact_every) == 0)
            n_sd = oracle_remove_zero_multiplicity(xi, v, cell_id, n_sd);
    }
    return n_sd;
}

}  // extern "C"
