// update.cu - moment update (a6), coefficient pack (a1) and convergence residual (a7) of the DVM iteration.
//   convert : raw[13] -> rho, u, T, q, sigma (exact central-moment conversion of Eq.(3)/(5))
//             + per-block partial sums of the total mass
//   finish  : global mass rescale of closed domains, residual partial sums,
//             the per-cell pack (1/tau, A, 1/T, U, Q) the next sweep rebuilds f^S from (Eq.(2), Eq.(10))
//   faces   : rho_w^{n+1} = Phi / Phi_unit (Eq.(9)), rescaled with the field
// All reductions are two-level and fixed-order (deterministic).
#include "dvm_dev.cuh"
#include "update.cuh"

namespace dvm {

constexpr int UB = 256;

__device__ __forceinline__ double block_sum(double v, double *sh)
{
    v = warp_sum(v);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) sh[wid] = v;
    __syncthreads();
    double r = 0.0;
    if (wid == 0) {
        r = lane < (blockDim.x >> 5) ? sh[lane] : 0.0;
        r = warp_sum(r);
    }
    return r;  // valid in warp 0
}

__device__ __forceinline__ void pack_cell(const UpdateParams &U, long long c, double rho, double ux, double uy,
                                          double uz, double T, double qx, double qy, double qz)
{
    const long long n = U.ncell;
    // 1/tau = rho T^{1-omega} / (C_omega Kn)
    U.coef[0 * n + c] = rho * pow(T, 1.0 - U.omega) * U.inv_cw_kn;
    const double pt = 3.14159265358979323846 * T;
    U.coef[1 * n + c] = rho / (pt * sqrt(pt));
    U.coef[2 * n + c] = 1.0 / T;
    U.coef[3 * n + c] = ux;
    U.coef[4 * n + c] = uy;
    U.coef[5 * n + c] = uz;
    const double s = U.shk / (rho * T * T);  // (1 - Pr) * 4/5 / (rho T^2)
    U.coef[6 * n + c] = s * qx;
    U.coef[7 * n + c] = s * qy;
    U.coef[8 * n + c] = s * qz;
}

__global__ void __launch_bounds__(UB) pack_kernel(const UpdateParams U)
{
    const long long c = (long long)blockIdx.x * UB + threadIdx.x;
    if (c >= U.ncell) return;
    const long long n = U.ncell;
    if (U.flags[c] & FLAG_SOLID) {
        for (int m = 0; m < NCOEF; ++m) U.coef[m * n + c] = 0.0;
        return;
    }
    pack_cell(U, c, U.prim[c], U.prim[n + c], U.prim[2 * n + c], U.prim[3 * n + c], U.prim[4 * n + c],
              U.prim[5 * n + c], U.prim[6 * n + c], U.prim[7 * n + c]);
}

__global__ void __launch_bounds__(UB) convert_kernel(const UpdateParams U)
{
    __shared__ double sh[UB / 32];
    const long long c = (long long)blockIdx.x * UB + threadIdx.x;
    const long long n = U.ncell;
    double mass = 0.0;
    if (c < n) {
        if (U.flags[c] & FLAG_SOLID) {
            for (int m = 0; m < NPRIM; ++m) U.prim_new[m * n + c] = 0.0;
        } else {
            // [cell][16] accumulator: 13 sums; the first moments are kept as two half-range sums (slots 1..3: xi_d >= 0,
            // slots 13..15: xi_d < 0; the slice kernel leaves the latter 0), see sweep_tile.cu
            const double *r = U.raw + c * 16;
            const double rho = r[0];
            const double ir = 1.0 / rho;
            const double ux = (r[1] + r[13]) * ir, uy = (r[2] + r[14]) * ir, uz = (r[3] + r[15]) * ir;
            const double mxx = r[4], myy = r[5], mzz = r[6];
            const double mxy = r[7], mxz = r[8], myz = r[9];
            const double pxx = mxx - rho * ux * ux, pyy = myy - rho * uy * uy, pzz = mzz - rho * uz * uz;
            const double pxy = mxy - rho * ux * uy, pxz = mxz - rho * ux * uz, pyz = myz - rho * uy * uz;
            const double trP = pxx + pyy + pzz, trm = mxx + myy + mzz;
            const double u2 = ux * ux + uy * uy + uz * uz;
            const double T = (2.0 / 3.0) * trP * ir;
            const double qx = 0.5 * (r[10] - 2.0 * (ux * mxx + uy * mxy + uz * mxz) - ux * trm + 2.0 * rho * ux * u2);
            const double qy = 0.5 * (r[11] - 2.0 * (ux * mxy + uy * myy + uz * myz) - uy * trm + 2.0 * rho * uy * u2);
            const double qz = 0.5 * (r[12] - 2.0 * (ux * mxz + uy * myz + uz * mzz) - uz * trm + 2.0 * rho * uz * u2);
            double *o = U.prim_new;
            o[c] = rho; o[n + c] = ux; o[2 * n + c] = uy; o[3 * n + c] = uz; o[4 * n + c] = T;
            o[5 * n + c] = qx; o[6 * n + c] = qy; o[7 * n + c] = qz;
            const double p3 = trP * (1.0 / 3.0);
            o[8 * n + c] = pxx - p3; o[9 * n + c] = pyy - p3; o[10 * n + c] = pzz - p3;
            o[11 * n + c] = pxy; o[12 * n + c] = pxz; o[13 * n + c] = pyz;
            const int i = (int)(c % U.nx), j = (int)((c / U.nx) % U.ny), k = (int)(c / ((long long)U.nx * U.ny));
            mass = rho * (U.dx[i] * U.dy[j] * U.dz[k]);
        }
    }
    const double bs = block_sum(mass, sh);
    if (threadIdx.x == 0) U.part[blockIdx.x] = bs;
}

// single block: sum the mass partials in fixed order, publish the rescale factor
__global__ void __launch_bounds__(UB) mass_kernel(const UpdateParams U, int nparts)
{
    __shared__ double sh[UB / 32];
    double v = 0.0;
    for (int t = threadIdx.x; t < nparts; t += UB) v += U.part[t];
    const double tot = block_sum(v, sh);
    if (threadIdx.x == 0) {
        U.scal[0] = U.rescale ? U.mass0 / tot : 1.0;
        U.scal[1] = tot;
    }
}

__global__ void __launch_bounds__(UB) finish_kernel(const UpdateParams U)
{
    __shared__ double sh[UB / 32];
    const long long c = (long long)blockIdx.x * UB + threadIdx.x;
    const long long n = U.ncell;
    const double s = U.scal[0];
    double acc[6] = {0, 0, 0, 0, 0, 0};  // num_rho, den_rho, num_mom, den_mom, num_E, den_E
    if (c < n) {
        if (U.flags[c] & FLAG_SOLID) {
            for (int m = 0; m < NPRIM; ++m) U.prim[m * n + c] = 0.0;
            for (int m = 0; m < NCOEF; ++m) U.coef[m * n + c] = 0.0;
        } else {
            const double *pn = U.prim_new;
            double *po = U.prim;
            const double r1 = pn[c] * s, ux = pn[n + c], uy = pn[2 * n + c], uz = pn[3 * n + c], T1 = pn[4 * n + c];
            const double r0 = po[c], vx = po[n + c], vy = po[2 * n + c], vz = po[3 * n + c], T0 = po[4 * n + c];
            const double dmx = r1 * ux - r0 * vx, dmy = r1 * uy - r0 * vy, dmz = r1 * uz - r0 * vz;
            const double E1 = 0.75 * r1 * T1 + 0.5 * r1 * (ux * ux + uy * uy + uz * uz);
            const double E0 = 0.75 * r0 * T0 + 0.5 * r0 * (vx * vx + vy * vy + vz * vz);
            acc[0] = (r1 - r0) * (r1 - r0); acc[1] = r1 * r1;
            acc[2] = dmx * dmx + dmy * dmy + dmz * dmz;
            acc[3] = (r1 * ux) * (r1 * ux) + (r1 * uy) * (r1 * uy) + (r1 * uz) * (r1 * uz);
            acc[4] = (E1 - E0) * (E1 - E0); acc[5] = E1 * E1;
            const double qx = pn[5 * n + c] * s, qy = pn[6 * n + c] * s, qz = pn[7 * n + c] * s;
            po[c] = r1; po[n + c] = ux; po[2 * n + c] = uy; po[3 * n + c] = uz; po[4 * n + c] = T1;
            po[5 * n + c] = qx; po[6 * n + c] = qy; po[7 * n + c] = qz;
            for (int m = 8; m < NPRIM; ++m) po[m * n + c] = pn[m * n + c] * s;
            pack_cell(U, c, r1, ux, uy, uz, T1, qx, qy, qz);
        }
    }
    for (int m = 0; m < 6; ++m) {
        const double bs = block_sum(acc[m], sh);
        if (threadIdx.x == 0) U.part[(long long)(1 + m) * U.npart + blockIdx.x] = bs;
    }
}

// single block: residual of this iteration -> history[slot].  The slot is a device-side counter (scal[3], an exact small
// integer in a double) that the kernel advances itself, so that the launch parameters of an iteration do not change from
// one iteration to the next and the whole iteration can be replayed as a CUDA graph (dvm_api.cu).
__global__ void __launch_bounds__(UB) residual_kernel(const UpdateParams U, int nparts, int hist_cap)
{
    const int slot = (int)U.scal[3];
    __shared__ double sh[UB / 32];
    __shared__ double tot[6];
    for (int m = 0; m < 6; ++m) {
        double v = 0.0;
        for (int t = threadIdx.x; t < nparts; t += UB) v += U.part[(long long)(1 + m) * U.npart + t];
        const double bs = block_sum(v, sh);
        if (threadIdx.x == 0) tot[m] = bs;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int m = 0; m < 3; ++m) {
            const double num = tot[2 * m], den = tot[2 * m + 1];
            double r;
            if (den > 0.0) r = sqrt(num / den);
            else r = num > 0.0 ? __longlong_as_double(0x7ff0000000000000LL) : (num == 0.0 ? 0.0 : num);
            U.hist[3 * slot + m] = r;
        }
        U.hist_scale[slot] = U.scal[0];
        U.scal[3] = (double)((slot + 1) % hist_cap);
    }
}

__global__ void __launch_bounds__(UB) faces_kernel(const UpdateParams U)
{
    const int f = blockIdx.x * UB + threadIdx.x;
    if (f >= U.nface) return;
    const double pu = U.phi_unit[f];
    U.rho_w[f] = pu > 0.0 ? U.phi[f] / pu * U.scal[0] : 0.0;
}

// [cell][16] accumulator -> [13][ncell] (dvm_raw_moments)
__global__ void __launch_bounds__(UB) raw_export_kernel(const double *raw16, double *out13, long long n)
{
    const long long c = (long long)blockIdx.x * UB + threadIdx.x;
    if (c >= n) return;
    for (int m = 0; m < NRAW; ++m) out13[m * n + c] = raw16[c * 16 + m] + (m >= 1 && m <= 3 ? raw16[c * 16 + 12 + m] : 0.0);
}

// Wall-incident fluxes of Eq.(9) from the half-range first moments the tile sweep leaves in the accumulator
// rows: a face on side d of its cell is hit by the velocities moving towards d, Phi = sum w |xi_n| f over them.  With the
// second-order sweep (reading G21) the flux takes the value extrapolated to the face, f_c + psi (f_c - f_c1): the same
// combination of the half-range sums of the cell and of its upwind neighbour c1 (psi = 0 if c1 is not a fluid cell).
struct PhiGeom {
    int order, nx, ny, nz;
    const unsigned char *flags;
    const double *dx, *dy, *dz;
};
__global__ void __launch_bounds__(UB) phi_from_raw_kernel(const double *raw16, const int *face_cell, const int *face_dir, double *phi,
                                                          int nface, const PhiGeom G)
{
    const int f = blockIdx.x * UB + threadIdx.x;
    if (f >= nface) return;
    const int c = face_cell[f], d = face_dir[f];
    double v = 0.0;
    if (c >= 0) {
        const int slot = (d & 1) ? 1 + (d >> 1) : 13 + (d >> 1);
        const double sgn = (d & 1) ? 1.0 : -1.0;
        v = sgn * raw16[(long long)c * 16 + slot];
        if (G.order == 2 && !((G.flags[c] >> (d ^ 1)) & 1u)) {
            const int ax = d >> 1, s = (d & 1) ? 1 : -1;
            const int i = c % G.nx, j = (c / G.nx) % G.ny, k = c / (G.nx * G.ny);
            const int id = ax == 0 ? i : ax == 1 ? j : k;
            const double *w = ax == 0 ? G.dx : ax == 1 ? G.dy : G.dz;
            const long long stride = ax == 0 ? 1 : ax == 1 ? G.nx : (long long)G.nx * G.ny;
            const double psi = w[id] / (w[id] + w[id - s]);
            const double v1 = sgn * raw16[((long long)c - s * stride) * 16 + slot];
            v += psi * (v - v1);
        }
    }
    phi[f] = v;
}

static inline int nblk(long long n) { return (int)((n + UB - 1) / UB); }

cudaError_t launch_pack(const UpdateParams &U, cudaStream_t st)
{
    pack_kernel<<<nblk(U.ncell), UB, 0, st>>>(U);
    return cudaGetLastError();
}

cudaError_t launch_raw_export(const double *raw16, double *out13, long long n, cudaStream_t st)
{
    raw_export_kernel<<<nblk(n), UB, 0, st>>>(raw16, out13, n);
    return cudaGetLastError();
}

cudaError_t launch_phi_from_raw(const UpdateParams &U, const int *face_cell, const int *face_dir, double *phi, int order, cudaStream_t st)
{
    PhiGeom G{order, U.nx, U.ny, U.nz, U.flags, U.dx, U.dy, U.dz};
    phi_from_raw_kernel<<<nblk(U.nface), UB, 0, st>>>(U.raw, face_cell, face_dir, phi, U.nface, G);
    return cudaGetLastError();
}

cudaError_t launch_update(const UpdateParams &U, int hist_cap, cudaStream_t st, int *launches)
{
    const int nb = nblk(U.ncell);
    convert_kernel<<<nb, UB, 0, st>>>(U);
    mass_kernel<<<1, UB, 0, st>>>(U, nb);
    finish_kernel<<<nb, UB, 0, st>>>(U);
    residual_kernel<<<1, UB, 0, st>>>(U, nb, hist_cap);
    faces_kernel<<<nblk(U.nface), UB, 0, st>>>(U);
    *launches += 5;
    return cudaGetLastError();
}

}  // namespace dvm
