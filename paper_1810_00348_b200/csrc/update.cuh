// update.cuh - parameters of the moment-update / residual kernels (update.cu)
#pragma once
#include <cuda_runtime.h>

namespace dvm {

struct UpdateParams {
    int nx, ny, nz, nface;
    long long ncell;
    long long npart;            // stride of the partial-sum table (>= number of update blocks)
    const unsigned char *flags;
    const double *dx, *dy, *dz; // cell widths
    const double *raw;          // [ncell][16] velocity sums (13 used)
    double *prim;               // [14][ncell] state n -> n+1 (in place, in finish_kernel)
    double *prim_new;           // [14][ncell] unscaled conversion of this iteration
    double *coef;               // [9][ncell]
    double *part;               // [7][npart] block partials: mass, 6 residual sums
    double *scal;               // [0] rescale factor, [1] total mass before rescale
    double *hist;               // [cap][3] residual history ring
    double *hist_scale;         // [cap]
    const double *phi;          // [nface]
    const double *phi_unit;     // [nface] (0 where rho_w is not defined)
    double *rho_w;              // [nface]
    double omega, inv_cw_kn, shk, mass0;
    int rescale;
};

struct SweepParams;

cudaError_t launch_raw_export(const double *raw16, double *out13, long long n, cudaStream_t st);
cudaError_t launch_pack(const UpdateParams &U, cudaStream_t st);
cudaError_t launch_phi_from_raw(const UpdateParams &U, const int *face_cell, const int *face_dir, double *phi, int order, cudaStream_t st);
cudaError_t launch_update(const UpdateParams &U, int hist_cap, cudaStream_t st, int *launches);   // the history slot is a device-side counter
cudaError_t launch_sweep_slice(const SweepParams &P, int nblocks, int nb, cudaStream_t st);

}  // namespace dvm
