// the step BEFORE the coalescence path -- particle displacement on the 2-D kinematic grid
// ("particle displacement"; PAPER.md:112-118 the kinematic_2d slab) and the recomputation of cell_id,
// which is what produces the scattered cell_id order the GENERAL and HYBRID paths exist for.
// Readings R36-R38: positions in grid units, periodic in both directions, cell_id = floor(z) nx +
// floor(x); one explicit-Euler step with the velocity of the cell the super-droplet is in before the move.
//
//   k_displace          reads x, z (16 B/SD), gathers two velocities (the nx*nz fields stay in L2), writes x, z and
//                       cell_id (20 B/SD): a streaming kernel, HBM bound at 36 B/SD.  Two super-droplets per thread,
//                       16-byte loads and stores.
//   k_cell_of_positions reads x, z, writes cell_id: 20 B/SD.
// fp64 discipline: x + (u * dt) as __dmul_rn / __dadd_rn (no FMA), the wrap as written in the header.
#include "sdm_internal.h"

namespace sdm {

__device__ __forceinline__ double wrap_periodic(double q, double dn) {
    if (q >= dn) q = __dsub_rn(q, dn);
    else if (q < 0.0) q = __dadd_rn(q, dn);
    if (!(q >= 0.0 && q < dn)) q = 0.0;  // a tiny negative q: q + n rounds up to n
    return q;
}

__device__ __forceinline__ int cell_of(double x, double z, int nx, int nz) {
    long long ix = __double2ll_rd(x), iz = __double2ll_rd(z);
    ix = ix < 0 ? 0 : (ix >= nx ? nx - 1 : ix);  // inside the domain by contract; the clamp keeps bad data memory-safe
    iz = iz < 0 ? 0 : (iz >= nz ? nz - 1 : iz);
    return (int)(iz * (long long)nx + ix);
}

template <bool MOVE>
__device__ __forceinline__ int displace_one(double& x, double& z, int nx, int nz, const double* __restrict__ u,
                                            const double* __restrict__ w, double dt) {
    if (MOVE) {
        const int c = cell_of(x, z, nx, nz);
        x = wrap_periodic(__dadd_rn(x, __dmul_rn(__ldg(u + c), dt)), (double)nx);
        z = wrap_periodic(__dadd_rn(z, __dmul_rn(__ldg(w + c), dt)), (double)nz);
    }
    return cell_of(x, z, nx, nz);
}

template <bool MOVE>
__global__ void __launch_bounds__(256)
k_displace(double* __restrict__ x, double* __restrict__ z, int* __restrict__ cell_id, long long n_sd, int nx, int nz,
           const double* __restrict__ u, const double* __restrict__ w, double dt, int vec_ok) {
    const long long stride = (long long)gridDim.x * 256 * 2;
    for (long long i = ((long long)blockIdx.x * 256 + threadIdx.x) * 2; i < n_sd; i += stride) {
        if (vec_ok && i + 1 < n_sd) {
            double2 xx = *reinterpret_cast<const double2*>(x + i);
            double2 zz = *reinterpret_cast<const double2*>(z + i);
            int2 c;
            c.x = displace_one<MOVE>(xx.x, zz.x, nx, nz, u, w, dt);
            c.y = displace_one<MOVE>(xx.y, zz.y, nx, nz, u, w, dt);
            if (MOVE) {
                *reinterpret_cast<double2*>(x + i) = xx;
                *reinterpret_cast<double2*>(z + i) = zz;
            }
            *reinterpret_cast<int2*>(cell_id + i) = c;
        } else {
            for (long long j = i; j < n_sd && j < i + 2; ++j) {
                double xs = x[j], zs = z[j];
                cell_id[j] = displace_one<MOVE>(xs, zs, nx, nz, u, w, dt);
                if (MOVE) { x[j] = xs; z[j] = zs; }
            }
        }
    }
}

cudaError_t launch_displace(sdm_ctx* ctx, bool move, double* x, double* z, int32_t* cell_id, int64_t n_sd, int32_t nx,
                            int32_t nz, const double* u_cell, const double* w_cell, double dt) {
    long long want = (n_sd / 2 + 255) / 256;
    int grid = (int)(want < (long long)ctx->sm_count * 8 ? want : (long long)ctx->sm_count * 8);
    if (grid < 1) grid = 1;
    const int vec_ok = ((reinterpret_cast<uintptr_t>(x) | reinterpret_cast<uintptr_t>(z)) & 15u) == 0 &&
                       (reinterpret_cast<uintptr_t>(cell_id) & 7u) == 0;
    LaunchScope scope(ctx, PROF_DISPLACE);
    if (move)
        k_displace<true><<<grid, 256, 0, ctx->stream>>>(x, z, cell_id, n_sd, nx, nz, u_cell, w_cell, dt, vec_ok);
    else
        k_displace<false><<<grid, 256, 0, ctx->stream>>>(x, z, cell_id, n_sd, nx, nz, u_cell, w_cell, dt, vec_ok);
    return cudaGetLastError();
}

}  // namespace sdm
