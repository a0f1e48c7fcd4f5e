// dvm_dev.cuh - device-side records shared by the kernels of the DVM iteration (arXiv 1810.00348).
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dvm {

constexpr int NCOEF = 9;   // per-cell pack: nu = 1/tau, A = rho/(pi T)^{3/2}, 1/T, ux, uy, uz, Qx, Qy, Qz
constexpr int NRAW = 13;   // raw velocity sums (Eq.(5), extended to the full second moment)
constexpr int NPRIM = 14;  // rho, u(3), T, q(3), sigma(6)

// cell flag bits
constexpr unsigned FLAG_SOLID = 1u << 6;  // bits 0..5: neighbour in direction d is not a fluid cell

struct BcParams {
    int type[7];
    double T[7], rho[7], u[7][3];
};

// one thread block of the sweep = a box of discrete velocities inside one octant (sign pattern)
struct BlockDesc {
    int ia0, na, ib0, nb, ic0, nc;  // box [ia0, ia0+na) x [ib0, ib0+nb) x [ic0, ic0+nc) of node indices
    int l0;                         // first flat local index (slice kernel)
    int sx, sy, sz;                 // sweep direction per axis: +1 ascending (xi >= 0), -1 descending
    int col0;                       // first column of this block in the f workspace (units of velocities)
    int pad;
};

struct SweepParams {
    int nx, ny, nz;
    long long ncell;
    const double *invdx, *invdy, *invdz;
    const double *dx, *dy, *dz;     // cell widths (second-order sweep)
    int order;                      // 1: first-order upwind Eq.(7); 2: second-order upwind (G21)
    long long fslice;               // order 2: offset (doubles) of the second stored slice in fbuf
    const unsigned char *flags;     // [ncell]
    const int *face_of;             // [6][ncell], face slot or -1
    const unsigned char *face_slot; // [nface] -> bc slot 0..6
    const double *coef;             // [NCOEF][ncell]
    const double *rho_w;            // [nface]
    double *phi;                    // [nface] wall-incident flux accumulators
    double *raw;                    // [ncell][16] accumulators (NRAW used)
    const double *xi_x, *xi_y, *xi_z, *w_x, *w_y, *w_z;
    const BlockDesc *blocks;
    double *fbuf;                   // distribution-function workspace (slices / tile faces)
    long long fstride;              // slice kernel: number of velocity columns (elements between cells)
    BcParams bc;
};

__device__ __forceinline__ double wall_maxwellian(const BcParams &bc, int b, double x, double y, double z)
{
    // Eq.(8), unit density, wall velocity in the exponent (G3)
    const double cx = x - bc.u[b][0], cy = y - bc.u[b][1], cz = z - bc.u[b][2];
    const double it = 1.0 / bc.T[b];
    const double pt = 3.14159265358979323846 * bc.T[b];
    return exp(-(cx * cx + cy * cy + cz * cz) * it) / (pt * sqrt(pt));
}

__device__ __forceinline__ double freestream_maxwellian(const BcParams &bc, int b, double x, double y, double z)
{
    return bc.rho[b] * wall_maxwellian(bc, b, x, y, z);
}

// value a ghost cell contributes per unit rho_w (wall) or in total (free stream); 0 for zero gradient
__device__ __forceinline__ double ghost_constant(const BcParams &bc, int b, double x, double y, double z)
{
    if (bc.type[b] == 0) return wall_maxwellian(bc, b, x, y, z);
    if (bc.type[b] == 1) return freestream_maxwellian(bc, b, x, y, z);
    return 0.0;
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

}  // namespace dvm
