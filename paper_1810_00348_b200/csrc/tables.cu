// tables.cu - the 1-D factor tables of the tile sweep kernel, rebuilt once per outer iteration from the per-cell pack
// of step n (a1/a2 of DESIGN.md): on the tensor velocity grid the source term of Eq.(7) factorises,
//   f^S / tau = [E_x E_y E_z] [1 + (Q_x + Q_y + Q_z)(e_x + e_y + e_z)]      (Eq.(2)),
// so one entry (E, Q, e, a) per (cell, 1-D node) is all the sweep needs: E = w exp(-(xi-u)^2/T) (the entries of table
// TX also carry rho (pi T)^{-3/2} / tau), Q = q'(xi-u), e = 2 (xi-u)^2/T (- 5 in TX), a = |xi| / cell width (Eq.(7),
// PAPER.md:77; 0 where the upwind face is a zero-gradient boundary, i.e. the term is dropped).  TX, TY, TZ hold the velocity
// axes T.ax[0..2]: TX the one that plays the wide role (A) in the sweep kernel, usually xi_x.
// order = 2 (DVM_OPT_ORDER, reading G21): the transport term of Eq.(7) along d is
// a_d (F(c) - F(c1)) with face values extrapolated from the two upwind centres, i.e. cd f_c - c1 f_c1 - c2 f_c2 with
//   c1 fluid: psi = w_c / (w_c + w_c1), psi1 = w_c1 / (w_c1 + w_c2) if c2 is fluid else 0,
//             cd = a (1 + psi), c1 = a (1 + psi + psi1), c2 = -a psi1;
//   c1 a wall / free-stream ghost: cd = c1 = a, c2 = 0;  zero gradient: all 0          (a = |xi| / w_c)
// and the entry is (E, Q, e, cd, c1, c2): all the boundary logic of the stencil is in these three numbers.
// The tables live on a grid padded by TILE_PAD dead cells (all-zero entries) so that every 4-cell row of a tile is one
// contiguous run the sweep kernel fetches with a single TMA bulk copy.  O(cells x (mx + my + mz)) work and bytes.
// Product code: shares nothing with oracle/.
#include "sweep_tile.cuh"

namespace dvm {

__global__ void __launch_bounds__(256) tables_kernel(const TableParams T)
{
    const int sx = T.nxb * T.na, sy = T.nyb * T.nbb, sz = T.nzb * T.ncb;
    const long long nslot = sx + sy + sz;
    const long long npc = (long long)T.nz * T.nyp * T.nxp;   // padded cells
    const long long n = T.ncell;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < n * nslot;
         idx += (long long)gridDim.x * blockDim.x) {
        const long long c = idx / nslot;
        const int sl = (int)(idx - c * nslot);
        const int i = (int)(c % T.nx), j = (int)((c / T.nx) % T.ny), k = (int)(c / ((long long)T.nx * T.ny));
        const long long pc = ((long long)k * T.nyp + (j + TILE_PAD)) * T.nxp + (i + TILE_PAD);
        int role, m, pos, width, blk;
        void *dst;
        if (sl < sx) { role = 0; width = T.na; blk = sl / width; pos = sl - blk * width; m = T.xnode[sl]; dst = T.TX; }
        else if (sl < sx + sy) { role = 1; width = T.nbb; const int t = sl - sx; blk = t / width; pos = t - blk * width; m = T.ynode[t]; dst = T.TY; }
        else { role = 2; width = T.ncb; const int t = sl - sx - sy; blk = t / width; pos = t - blk * width; m = T.znode[t]; dst = T.TZ; }
        const int d = T.ax[role];   // velocity axis (= direction of the transport term) this table belongs to
        const bool solid = T.flags[c] & FLAG_SOLID;
        const double nu = T.coef[c];
        double ent[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        if (!solid && m >= 0) {
            const double invT = T.coef[2 * n + c], u = T.coef[(3 + d) * n + c], q = T.coef[(6 + d) * n + c];
            const double xi = d == 0 ? T.xi_x[m] : d == 1 ? T.xi_y[m] : T.xi_z[m];
            double w = d == 0 ? T.w_x[m] : d == 1 ? T.w_y[m] : T.w_z[m];
            if (role == 0) w *= nu * T.coef[n + c];
            const int id = d == 0 ? i : d == 1 ? j : k, nd = d == 0 ? T.nx : d == 1 ? T.ny : T.nz;
            const double h = d == 0 ? T.invdx[i] : d == 1 ? T.invdy[j] : T.invdz[k];
            const bool pos_dir = xi >= 0.0;   // sweeps ascending: the upwind face is the low one
            const bool first = pos_dir ? id == 0 : id == nd - 1;
            const int up = 2 * d + (pos_dir ? 0 : 1);
            const bool drop = first && T.bc_type[up] == 2;
            const double c1 = xi - u, t = c1 * c1 * invT;
            ent[0] = w * exp(-t);
            ent[1] = q * c1;
            ent[2] = role == 0 ? 2.0 * t - 5.0 : 2.0 * t;
            const double a = drop ? 0.0 : fabs(xi) * h;
            ent[3] = a;
            if (T.order == 2) {
                ent[4] = a;
                if (!((T.flags[c] >> up) & 1u)) {
                    // the upwind neighbour c1 is a fluid cell: second order along d (reading G21)
                    const int s = pos_dir ? 1 : -1;
                    const long long stride = d == 0 ? 1 : d == 1 ? T.nx : (long long)T.nx * T.ny;
                    const double *wd = d == 0 ? T.dx : d == 1 ? T.dy : T.dz;
                    const double wc = wd[id], w1 = wd[id - s];
                    const double psi = wc / (wc + w1);
                    double psi1 = 0.0;
                    if (!((T.flags[c - s * stride] >> up) & 1u)) psi1 = w1 / (w1 + wd[id - 2 * s]);
                    ent[3] = a * (1.0 + psi);
                    ent[4] = a * (1.0 + psi + psi1);
                    ent[5] = -a * psi1;
                }
            }
        }
        const int es = T.order == 2 ? 6 : 4;
        const long long at = (((long long)blk * npc + pc) * width + pos) * es;
        if (T.f32) {
            // DVM_PREC_MIXED: the factors are evaluated in double and rounded once to single
            float *o = static_cast<float *>(dst) + at;
            for (int e = 0; e < es; ++e) o[e] = (float)ent[e];
        } else {
            double *o = static_cast<double *>(dst) + at;
            for (int e = 0; e < es; ++e) o[e] = ent[e];
        }
        if (sl == 0) { T.rec[pc].nu = solid ? 1.0 : nu; T.rec[pc].nu32 = solid ? 1.0f : (float)nu; }
    }
}

cudaError_t launch_tables(const TableParams &T, cudaStream_t st)
{
    const long long work = T.ncell * ((long long)T.nxb * T.na + (long long)T.nyb * T.nbb + (long long)T.nzb * T.ncb);
    const long long blocks = (work + 255) / 256;
    const int grid = (int)(blocks < 148LL * 32 ? blocks : 148LL * 32);
    tables_kernel<<<grid, 256, 0, st>>>(T);
    return cudaGetLastError();
}

}  // namespace dvm
