// sweep_slice.cu - DVM_KERNEL_SLICE: the paper's thread mapping (Alg. 2),
// restated in fp64 for sm_100a with three changes: ONE in-place z-slice per velocity instead of two
// (cell (i,j) holds level k-1 until it is overwritten with level k), the equilibrium fused into the sweep
// from a 9-double per-cell pack staged row by row in shared memory, and the moment / wall-flux sums
// (Alg. 3) taken from registers right after each update, so the slice is never re-read.
// It is the baseline variant; the tile kernel (sweep_tile.cu) is the B200 design.
//
// order = 2 (DVM_OPT_ORDER; "extend the first order upwind scheme to second order by storing three
// consecutive slices"; reading G21 of DESIGN.md): the transport term of Eq.(7) along d becomes a_d (F(c) - F(c1)) with
// F = value at a cell's downwind face, extrapolated linearly from the two upwind centres (the cell value itself where the
// upwind neighbour is not a fluid cell).  A second in-place slice keeps level k-2 under level k-1, so with the slice being
// written this is the paper's three slices; the wall-incident flux of Eq.(9) takes the extrapolated face value.
#include "dvm_dev.cuh"

namespace dvm {

template <int NB>
__global__ void __launch_bounds__(NB) sweep_slice_kernel(const SweepParams P)
{
    extern __shared__ double sm[];
    double *s_coef = sm;                                        // [NCOEF][nx]
    unsigned char *s_flag = (unsigned char *)(sm + NCOEF * P.nx);  // [nx]

    const BlockDesc bd = P.blocks[blockIdx.x];
    const int nvel = bd.na * bd.nb * bd.nc;
    const int l = bd.l0 + (int)threadIdx.x;
    const bool active = l < nvel;
    const int ll = active ? l : 0;
    const int ia = bd.ia0 + ll % bd.na, ib = bd.ib0 + (ll / bd.na) % bd.nb, ic = bd.ic0 + ll / (bd.na * bd.nb);
    const double xx = P.xi_x[ia], xy = P.xi_y[ib], xz = P.xi_z[ic];
    const double w = active ? P.w_x[ia] * P.w_y[ib] * P.w_z[ic] : 0.0;
    const int sx = bd.sx, sy = bd.sy, sz = bd.sz;
    const int nx = P.nx, ny = P.ny, nz = P.nz;
    const long long nc = P.ncell;

    // upwind / downwind direction ids and flag bits
    const int upx = sx > 0 ? 0 : 1, upy = sy > 0 ? 2 : 3, upz = sz > 0 ? 4 : 5;
    const int dnx = upx ^ 1, dny = upy ^ 1, dnz = upz ^ 1;
    const double gx = ghost_constant(P.bc, upx, xx, xy, xz);
    const double gy = ghost_constant(P.bc, upy, xx, xy, xz);
    const double gz = ghost_constant(P.bc, upz, xx, xy, xz);
    const double gs = ghost_constant(P.bc, 6, xx, xy, xz);
    const int tx = P.bc.type[upx], ty = P.bc.type[upy], tz = P.bc.type[upz];
    const double axx = fabs(xx), axy = fabs(xy), axz = fabs(xz);
    const double xi2 = xx * xx + xy * xy + xz * xz;

    double *col = P.fbuf + (long long)bd.col0 + threadIdx.x;
    const long long S = P.fstride;
    const int lane = threadIdx.x & 31;

    for (int kk = 0; kk < nz; ++kk) {
        const int k = sz > 0 ? kk : nz - 1 - kk;
        const double az = axz * P.invdz[k];
        for (int jj = 0; jj < ny; ++jj) {
            const int j = sy > 0 ? jj : ny - 1 - jj;
            const double ay = axy * P.invdy[j];
            const long long row = ((long long)k * ny + j) * nx;
            __syncthreads();
            for (int t = threadIdx.x; t < NCOEF * nx; t += NB) {
                const int m = t / nx, i = t - m * nx;
                s_coef[t] = P.coef[m * nc + row + i];
            }
            for (int t = threadIdx.x; t < nx; t += NB) s_flag[t] = P.flags[row + t];
            __syncthreads();
            double fprev = 0.0, fprev2 = 0.0;
            unsigned flprev = 0xffu;   // flags of the cell fprev belongs to
            for (int ii = 0; ii < nx; ++ii) {
                const int i = sx > 0 ? ii : nx - 1 - ii;
                const unsigned fl = s_flag[i];
                if (fl & FLAG_SOLID) continue;
                const long long c = row + i;
                const double nu = s_coef[i], A = s_coef[nx + i], invT = s_coef[2 * nx + i];
                const double cx = xx - s_coef[3 * nx + i], cy = xy - s_coef[4 * nx + i], cz = xz - s_coef[5 * nx + i];
                const double c2 = cx * cx + cy * cy + cz * cz;
                const double Qc = s_coef[6 * nx + i] * cx + s_coef[7 * nx + i] * cy + s_coef[8 * nx + i] * cz;
                const double e = c2 * invT;
                const double fS = A * exp(-e) * (1.0 + Qc * (2.0 * e - 5.0));
                const double ax = axx * P.invdx[i];
                double num = nu * fS, den = nu;
                const bool o2 = P.order == 2;
                double px = 0.0, py = 0.0, pz = 0.0;     // psi of reading G21 per direction (0: first order there)
                double f1x = 0.0, f1y = 0.0, f1z = 0.0;  // value of the first upwind cell per direction
                // x upwind
                if (fl & (1u << upx)) {
                    const bool dom = (i == (sx > 0 ? 0 : nx - 1));
                    const int ty_ = dom ? tx : 0;
                    if (ty_ != 2) {
                        const int face = P.face_of[upx * nc + c];
                        const double g = dom ? (tx == 0 ? P.rho_w[face] * gx : gx) : P.rho_w[face] * gs;
                        num += ax * g; den += ax;
                    }
                } else if (!o2) { num += ax * fprev; den += ax; }
                else {
                    // G21: a_x [(1 + psi) f_c - psi f_c1 - F(c1)], F(c1) = f_c1 + psi_1 (f_c1 - f_c2) if c2 is a fluid cell
                    const double wc = P.dx[i], w1 = P.dx[i - sx];
                    px = wc / (wc + w1); f1x = fprev;
                    double Fup = fprev;
                    if (!(flprev & (1u << upx))) { const double w2 = P.dx[i - 2 * sx]; Fup = fprev + w1 / (w1 + w2) * (fprev - fprev2); }
                    num += ax * (px * fprev + Fup); den += ax * (1.0 + px);
                }
                // y upwind
                if (fl & (1u << upy)) {
                    const bool dom = (j == (sy > 0 ? 0 : ny - 1));
                    const int ty_ = dom ? ty : 0;
                    if (ty_ != 2) {
                        const int face = P.face_of[upy * nc + c];
                        const double g = dom ? (ty == 0 ? P.rho_w[face] * gy : gy) : P.rho_w[face] * gs;
                        num += ay * g; den += ay;
                    }
                } else if (!o2) { num += ay * col[((long long)(j - sy) * nx + i) * S]; den += ay; }
                else {
                    const double f1 = col[((long long)(j - sy) * nx + i) * S];
                    const double wc = P.dy[j], w1 = P.dy[j - sy];
                    py = wc / (wc + w1); f1y = f1;
                    double Fup = f1;
                    if (!(P.flags[c - (long long)sy * nx] & (1u << upy))) {
                        const double w2 = P.dy[j - 2 * sy];
                        Fup = f1 + w1 / (w1 + w2) * (f1 - col[((long long)(j - 2 * sy) * nx + i) * S]);
                    }
                    num += ay * (py * f1 + Fup); den += ay * (1.0 + py);
                }
                // z upwind: the in-place slice still holds level k -/+ 1 at (i, j)
                if (fl & (1u << upz)) {
                    const bool dom = (k == (sz > 0 ? 0 : nz - 1));
                    const int ty_ = dom ? tz : 0;
                    if (ty_ != 2) {
                        const int face = P.face_of[upz * nc + c];
                        const double g = dom ? (tz == 0 ? P.rho_w[face] * gz : gz) : P.rho_w[face] * gs;
                        num += az * g; den += az;
                    }
                } else if (!o2) { num += az * col[((long long)j * nx + i) * S]; den += az; }
                else {
                    const double f1 = col[((long long)j * nx + i) * S];
                    const double wc = P.dz[k], w1 = P.dz[k - sz];
                    pz = wc / (wc + w1); f1z = f1;
                    double Fup = f1;
                    if (!(P.flags[c - (long long)sz * nx * ny] & (1u << upz))) {
                        const double w2 = P.dz[k - 2 * sz];
                        Fup = f1 + w1 / (w1 + w2) * (f1 - col[P.fslice + ((long long)j * nx + i) * S]);
                    }
                    num += az * (pz * f1 + Fup); den += az * (1.0 + pz);
                }
                const double f = num / den;
                // second slice: level k-1 moves under the value being written (stale where k-1 is not fluid: never read)
                if (o2) col[P.fslice + ((long long)j * nx + i) * S] = col[((long long)j * nx + i) * S];
                col[((long long)j * nx + i) * S] = f;
                fprev2 = fprev; fprev = f; flprev = fl;

                // moments (Eq.(5)) reduced over the warp, one atomic per warp and moment
                const double wf = w * f;
                double m[NRAW];
                m[0] = wf; m[1] = wf * xx; m[2] = wf * xy; m[3] = wf * xz;
                m[4] = m[1] * xx; m[5] = m[2] * xy; m[6] = m[3] * xz;
                m[7] = m[1] * xy; m[8] = m[1] * xz; m[9] = m[2] * xz;
                m[10] = m[1] * xi2; m[11] = m[2] * xi2; m[12] = m[3] * xi2;
#pragma unroll
                for (int q = 0; q < NRAW; ++q) m[q] = warp_sum(m[q]);
                if (lane == 0) {
#pragma unroll
                    for (int q = 0; q < NRAW; ++q) atomicAdd(P.raw + c * 16 + q, m[q]);
                    // wall-incident flux (Eq.(9)): all velocities of the block share the sign of xi_d, so
                    // sum w |xi_d| f = s_d * (first-moment partial)
                    if (!o2) {
                        if (fl & (1u << dnx)) atomicAdd(P.phi + P.face_of[dnx * nc + c], sx * m[1]);
                        if (fl & (1u << dny)) atomicAdd(P.phi + P.face_of[dny * nc + c], sy * m[2]);
                        if (fl & (1u << dnz)) atomicAdd(P.phi + P.face_of[dnz * nc + c], sz * m[3]);
                    }
                }
                if (o2 && (fl & ((1u << dnx) | (1u << dny) | (1u << dnz)))) {
                    // order 2: the flux through a downwind boundary face takes the extrapolated face value (G21); the
                    // condition is the same for every thread (they all sit in the same cell)
                    const double hx = warp_sum(w * axx * (f + px * (f - f1x)));
                    const double hy = warp_sum(w * axy * (f + py * (f - f1y)));
                    const double hz = warp_sum(w * axz * (f + pz * (f - f1z)));
                    if (lane == 0) {
                        if (fl & (1u << dnx)) atomicAdd(P.phi + P.face_of[dnx * nc + c], hx);
                        if (fl & (1u << dny)) atomicAdd(P.phi + P.face_of[dny * nc + c], hy);
                        if (fl & (1u << dnz)) atomicAdd(P.phi + P.face_of[dnz * nc + c], hz);
                    }
                }
            }
        }
    }
}

cudaError_t launch_sweep_slice(const SweepParams &P, int nblocks, int nb, cudaStream_t st)
{
    const size_t smem = (size_t)NCOEF * P.nx * sizeof(double) + ((P.nx + 7) / 8) * 8;
    if (smem > 48 * 1024) {
        if (smem > 200 * 1024) return cudaErrorInvalidValue;   // one row of the per-cell pack must fit in shared memory
        cudaError_t e = nb == 128 ? cudaFuncSetAttribute(sweep_slice_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)
                      : nb == 64 ? cudaFuncSetAttribute(sweep_slice_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)
                                 : cudaFuncSetAttribute(sweep_slice_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    if (nb == 128) sweep_slice_kernel<128><<<nblocks, 128, smem, st>>>(P);
    else if (nb == 64) sweep_slice_kernel<64><<<nblocks, 64, smem, st>>>(P);
    else sweep_slice_kernel<32><<<nblocks, 32, smem, st>>>(P);
    return cudaGetLastError();
}

}  // namespace dvm
