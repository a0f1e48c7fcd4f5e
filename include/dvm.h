/*
 * dvm.h - C ABI of the B200-native solver for ONE thing: the outer iteration of the memory-reduced
 * iterative discrete-velocity method (DVM) of arXiv 1810.00348 for the steady 3D3V Shakhov/BGK model
 * equation.  Citations are to /root/reference/PAPER.md (line, section, equation).
 *
 * One outer iteration (Alg. 1; Eq.(6)):
 *   every discrete velocity xi_alpha sweeps the physical grid along its characteristic direction with the
 *   first-order upwind formula Eq.(7), the Shakhov equilibrium f^S (Eq.(2))
 *   and the relaxation time tau = mu/p (Eq.(10)) being rebuilt on the fly from
 *   the macroscopic fields of step n; ghost values come from the Maxwell diffuse wall (Eq.(8)-(9),
 *   PAPER.md:211-219), the free stream or a zero-gradient outflow; the moments Eq.(5)
 *    and the wall-incident fluxes are reduced over velocity space as each value is produced
 *   (PAPER.md:81), so the 6-D distribution function is never stored; a moment-update step converts the
 *   sums to rho, u, T, q, sigma, rescales the mass of closed domains and evaluates the
 *   convergence residual.
 *
 * Units: speeds in v_m = sqrt(2 R T0), rho in rho0, T in T0, lengths in L, f in rho0/v_m^3, q in
 * rho0 v_m^3, sigma in rho0 v_m^2 (reading G2).
 *
 * Layout: cell index c = (k*ny + j)*nx + i (i fastest).  Fields are SoA: field m of cell c at [m*ncell + c].
 * Direction ids: 0 = x-, 1 = x+, 2 = y-, 3 = y+, 4 = z-, 5 = z+.
 * Boundary-face table (one slot per face whatever its type; see dvm_num_faces):
 *   the six domain faces first - x- [k*ny+j], x+ [k*ny+j], y- [k*nx+i], y+ [k*nx+i], z- [j*nx+i],
 *   z+ [j*nx+i] - then every face between a fluid cell and a solid (masked) cell inside the domain, ordered
 *   by (fluid cell index ascending, direction id ascending).
 *
 * Pointers: "host" = ordinary host memory, read during the call only (dvm_create copies what it needs);
 * "dev" = device memory on the solver's device, caller-owned, at least the stated size.
 * All device work is enqueued on the stream given at creation; only the calls marked (syncs) wait for it.
 * A solver lives on the CUDA device that is current when dvm_create is called; every later call switches to that
 * device for its duration and restores the caller's current device.
 * Every call returns 0 or a negative DVM_E* code; nothing throws or aborts across this boundary;
 * dvm_last_error() returns a thread-local message for the last failing call of this thread.
 * There is no CPU fallback: without a CUDA device dvm_create fails with DVM_ECUDA.
 */
#ifndef DVM_H
#define DVM_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DVM_OK          0
#define DVM_EINVAL     -1   /* NULL pointer, non-positive size, non-monotone faces or nodes, bad BC type */
#define DVM_ENOMEM     -2   /* the allocator returned NULL */
#define DVM_ECUDA      -3   /* a CUDA runtime call or kernel launch failed, or no device */
#define DVM_ENONFINITE -4   /* the residual reduction met NaN/Inf */

#define DVM_WALL_DIFFUSE  0 /* Eq.(8)-(9): ghost = rho_w g_w(xi), g_w Maxwellian at (T, u), rho_w lagged */
#define DVM_FREESTREAM    1 /* ghost = f^M(rho, u, T)(xi) */
#define DVM_ZERO_GRADIENT 2 /* ghost = the cell's own new value, i.e. the term drops out of Eq.(7) */

/* sweep-kernel variants (dvm_set_option DVM_OPT_KERNEL) */
#define DVM_KERNEL_AUTO   0
#define DVM_KERNEL_SLICE  1 /* the paper's mapping (thread = velocity, z-slice in HBM), fp64, in-place slice */
#define DVM_KERNEL_TILE   2 /* B200 design: z-column tiles with the plane in registers, faces via TMA */

#define DVM_OPT_KERNEL    1
#define DVM_OPT_MAX_F_MBYTES 2 /* tile kernel: cap (MiB) on the f workspace; velocity blocks then sweep in batches (0 = none) */
#define DVM_OPT_TILE_AXIS 6 /* tile kernel: velocity axis that plays the wide role (RV nodes per thread x 4 lane groups): 1 = xi_x,
                             2 = xi_y, 3 = xi_z; 0 = the library chooses the axis (and RV) that wastes the fewest lanes (default) */
#define DVM_OPT_ORDER     5 /* order of the upwind sweep: 1 = Eq.(7) (default); 2 = second-order upwind, the extension PAPER.md:393 names
                             ("second order by storing three consecutive slices"): Eq.(7) in flux-difference form with the value
                             at a cell's downwind face extrapolated linearly from the two upwind cell centres (the cell value
                             where the upwind neighbour is not a fluid cell; reading G21); the wall-incident flux of
                             Eq.(9) takes the extrapolated face value.  Tile kernel: two z-planes in registers and two-deep faces
                             (2 velocities per thread); slice kernel: two stored slices + the one being written */
#define DVM_OPT_MAX_CTAS  4 /* tile kernel: cap on the persistent grid (0 = every resident CTA); 1 runs the work items strictly in
                             hand-out order on one CTA - for tests of the dependency protocol, not for speed */
#define DVM_OPT_TILE_RV   3 /* tile kernel: velocities per thread, 4 (128-thread CTAs, velocity blocks of 16 x 8 x 4 nodes), 3 (128
                             threads, 12 x 8 x 4: fills sign halves of 12 k nodes) or 2 (256-thread CTAs, blocks of 8 x 8 x 8
                             nodes); 0 = the library chooses by lane use x measured speed of the variant (default) */

#define DVM_OPT_PRECISION 7 /* precision f is carried in by the sweep: DVM_PREC_F64 (default) or DVM_PREC_MIXED = the paper's timing
                             precision ("single precision computations"; reading G22): the factor tables, the
                             faces, the plane in registers and the arithmetic of Eq.(7) are IEEE single; the velocity sums of Eq.(5)
                             (tensor-core products, accumulator), the wall fluxes, the moment update and the residual stay double.
                             Tile kernel, order 1, 3 or 4 velocities per thread; every other combination: DVM_EINVAL at the first
                             dvm_iterate.  Fields then agree with the double result to 16 x 2^-24 x (nx + ny + nz) absolute
                             (units of DESIGN.md section 2), not to 1e-11 */
#define DVM_PREC_F64      0
#define DVM_PREC_MIXED    1
#define DVM_OPT_SHARD_COUNT 8 /* velocity-space sharding over several GPUs (the velocities are independent inside an
                             iteration; the paper's MPI program decomposes the velocity space): number of ranks n >= 1
                             (default 1).  With n > 1 this solver sweeps only the velocity blocks r, r + n, ... of the tile kernel
                             (r = DVM_OPT_SHARD_RANK), all macroscopic state is replicated, and an iteration is
                             dvm_sweep -> all-reduce (sum, fp64) of the buffer dvm_reduce_buffer names, over the ranks, by the caller
                             (NCCL) -> dvm_update; dvm_iterate / dvm_step_host then return DVM_EINVAL.  Tile kernel only */
#define DVM_OPT_SHARD_RANK  9 /* this solver's rank, 0 <= r < n; set DVM_OPT_SHARD_COUNT first */

typedef struct dvm_solver dvm_solver; /* opaque */

typedef struct {
    int nx, ny, nz;
    const double *xf, *yf, *zf;     /* host; face coordinates, nx+1 / ny+1 / nz+1 values, strictly increasing */
    const unsigned char *solid;     /* host; nz*ny*nx, 1 = solid cell; NULL = all fluid */
} dvm_grid;

typedef struct {
    int mx, my, mz;
    const double *xi_x, *xi_y, *xi_z; /* host; nodes per axis, strictly increasing (tensor grid) */
    const double *w_x, *w_y, *w_z;    /* host; 1-D quadrature weights >= 0; w_alpha = w_x w_y w_z (Eq.(5)) */
} dvm_vgrid;

typedef struct {
    double Kn, omega, Pr;           /* Pr = 1: BGK; 2/3: Shakhov */
    double rho0, u0[3], T0;         /* uniform initial state */
} dvm_gas;

typedef struct {
    int type;                       /* DVM_WALL_DIFFUSE | DVM_FREESTREAM | DVM_ZERO_GRADIENT */
    double T, rho, u[3];            /* wall: T, u ; free stream: rho, u, T ; zero gradient: unused */
} dvm_face_bc;

typedef struct {
    dvm_face_bc face[6];            /* x-, x+, y-, y+, z-, z+ */
    dvm_face_bc solid;              /* faces of masked cells (must be DVM_WALL_DIFFUSE) */
    int rescale_mass;               /* 1 = global density rescale of closed domains */
    int wall_norm;                  /* 0 = discrete half-flux normalisation (default), 1 = constant of Eq.(9) */
} dvm_bc;

typedef struct {
    void *stream;                               /* cudaStream_t (0 = default stream) */
    void *(*alloc)(size_t bytes, void *ctx);    /* device allocator, 256-byte aligned; NULL -> cudaMalloc */
    void (*free_)(void *ptr, void *ctx);        /* matching release; NULL -> cudaFree */
    void *ctx;
} dvm_device;

/* Build a solver: copies all host arrays, allocates its workspace through dev->alloc (no allocation scales
 * with ncell * nvel: the f workspace holds tile faces / one z-slice per in-flight velocity, the factor tables of the tile
 * kernel ncell * (mx + my + mz) entries), sets the uniform initial
 * state and rho_w^0 (DESIGN.md oracle step 1).  dev may be NULL (default stream, cudaMalloc). */
int dvm_create(const dvm_grid *grid, const dvm_vgrid *vgrid, const dvm_gas *gas, const dvm_bc *bc,
               const dvm_device *dev, dvm_solver **out);

/* n >= 0 outer iterations (Alg. 1 + moment update + residual), asynchronous on the stream.  Tile kernel: the first call captures
 * one iteration from the stream as a CUDA graph and every iteration is one graph launch from then on (DVM_GRAPH=0 in the
 * environment: plain kernel launches). */
int dvm_iterate(dvm_solver *s, int n);

/* The two halves of one outer iteration, for velocity-space sharding (DVM_OPT_SHARD_COUNT): dvm_sweep clears the velocity-sum
 * accumulator, rebuilds the factor tables and sweeps this rank's velocity blocks (rows a1-a5 of DESIGN.md); dvm_update converts
 * the sums to the state n+1, wall densities, mass rescale and residual (rows a5-a7) - every rank does it redundantly after the
 * all-reduce.  dvm_sweep; dvm_update with one rank is exactly dvm_iterate(1).  Asynchronous on the stream.  Tile kernel only
 * (DVM_EINVAL for the slice kernel, whose wall fluxes are separate atomics). */
int dvm_sweep(dvm_solver *s);
int dvm_update(dvm_solver *s);
/* The buffer the ranks must sum between dvm_sweep and dvm_update: *dev_ptr = the [ncell][16] fp64 accumulator (13 velocity
 * sums + the half-range first moments the wall fluxes are read from), *count = 16 * ncell doubles.  The pointer is the start
 * of an allocation made through dvm_device.alloc and stays valid for the life of the solver. */
int dvm_reduce_buffer(dvm_solver *s, double **dev_ptr, size_t *count);

/* Current macroscopic fields, dev_out[14][ncell]: rho, ux, uy, uz, T, qx, qy, qz, sxx, syy, szz, sxy, sxz, syz
 * (solid cells: zeros).  Asynchronous device-to-device copy on the stream. */
int dvm_moments(dvm_solver *s, double *dev_out);

/* (syncs) Residual of the last iteration, host_out3 = r_rho, r_mom, r_E (G9).
 * DVM_ENONFINITE if any of them is NaN/Inf; DVM_EINVAL before the first iteration. */
int dvm_residual(dvm_solver *s, double *host_out3);

/* ---- support calls ------------------------------------------------------------------------------ */
/* number of boundary-face slots (domain + solid), >= 0, or a negative error code */
int dvm_num_faces(const dvm_solver *s);
/* number of outer iterations done since creation */
int dvm_iterations_done(const dvm_solver *s);
/* State between iterations = checkpoint: dev_prim14 [14][ncell] (as dvm_moments), dev_rho_wall [nfaces].
 * Either pointer may be NULL to skip it.  Asynchronous. */
int dvm_get_state(dvm_solver *s, double *dev_prim14, double *dev_rho_wall);
/* Replace the state: dev_prim8 [8][ncell] = rho, u, T, q (sigma is output only); dev_rho_wall [nfaces] or NULL
 * (keep).  The reference mass of the rescale stays that of the initial state.  Asynchronous. */
int dvm_set_state(dvm_solver *s, const double *dev_prim8, const double *dev_rho_wall);
/* Raw velocity sums of the last iteration, dev_raw13 [13][ncell]:
 * sum_alpha w f {1, xi_x, xi_y, xi_z, xx, yy, zz, xy, xz, yz, xi_x|xi|^2, xi_y|xi|^2, xi_z|xi|^2}; before the
 * rescale.  Asynchronous. */
int dvm_raw_moments(dvm_solver *s, double *dev_raw13);
/* Wall-incident fluxes of the last iteration, dev_flux [nfaces] (before division by Phi_unit and rescale). */
int dvm_wall_flux(dvm_solver *s, double *dev_flux);
/* (syncs) Residual triples of the last min(max_n, iterations done, capacity) iterations, oldest first,
 * host_out[3*count]; returns count or a negative code. */
int dvm_residual_history(dvm_solver *s, double *host_out, int max_n);
/* (syncs) Mass-rescale factor of the last iteration (1 if rescale_mass = 0). */
int dvm_mass_scale(dvm_solver *s, double *host_out1);
/* (syncs) End-to-end step with HOST buffers: upload the state (host_prim8 [8][ncell], host_rho_wall [nfaces],
 * either may be NULL = keep), run n iterations, download prim14 [14][ncell] and rho_wall (either may be NULL). */
int dvm_step_host(dvm_solver *s, const double *host_prim8, const double *host_rho_wall, int n,
                  double *host_prim14_out, double *host_rho_wall_out);
/* Tuning / variant selection; must be called before the first dvm_iterate.  Unknown option: DVM_EINVAL. */
int dvm_set_option(dvm_solver *s, int option, int value);
/* Sweep-kernel variant in use: DVM_KERNEL_SLICE / DVM_KERNEL_TILE once the first dvm_iterate has planned the
 * workspace, the requested value (possibly DVM_KERNEL_AUTO) before. */
int dvm_kernel_used(const dvm_solver *s);
/* Velocities per thread of the tile kernel: 2, 3 or 4 once the first dvm_iterate has planned, the requested value before. */
int dvm_tile_rv(const dvm_solver *s);
/* 1 + velocity axis in the wide role of the tile kernel once planned (DVM_OPT_TILE_AXIS), the requested value before. */
int dvm_tile_axis(const dvm_solver *s);
/* DVM_PREC_F64 or DVM_PREC_MIXED (DVM_OPT_PRECISION). */
int dvm_precision(const dvm_solver *s);
/* Host-only (needs no device): the work decomposition the tile kernel would use for an nx x ny x nz grid and the
 * velocity nodes of v when target_ctas items should run concurrently, at most max_blocks velocity blocks are in
 * flight at once (0 = all; "smaller batches"), a thread carries rv velocities (2, 4, or 0 = the
 * library's choice for these nodes; 3 is a variant too), the sweep has the given order (1 or 2; order 2 needs rv = 2 or 0)
 * and wide_axis is as DVM_OPT_TILE_AXIS (0 = the library's choice).  counts5 = number of velocity blocks, tiles along x, tiles
 * along y, band height P, blocks per batch.  items9 (may be NULL) receives, for the first max_items work items in
 * hand-out order, {velocity block, tile x, tile y, predecessor in x, predecessor in y (for tile y = 0 of a later batch:
 * the last reader of the y-face slot), previous user of the x-face slot, x-face slot, octant bits, face-slot set};
 * predecessors are item indices or -1.  Returns the number of items. */
int dvm_plan_query(int nx, int ny, int nz, const dvm_vgrid *v, int target_ctas, int max_blocks, int rv, int order, int wide_axis,
                   int *counts5, int *items9, int max_items);
/* Host-only: the velocity blocks of the tile kernel for the nodes of v (rv, order as in dvm_plan_query), in block-id order (the
 * order of dvm_plan_query's items9[0]).  boxes8 (may be NULL) receives for the first max_blocks blocks {x0, nx, y0, ny, z0,
 * nz, NA + 65536 (1 + wide axis), 256 nbb + ncb}: the block holds the nodes [x0, x0+nx) x [y0, y0+ny) x [z0, z0+nz) of xi_x,
 * xi_y, xi_z, all of one sign octant, in a box of NA (along the wide axis) x nbb x ncb lanes.  Returns the number of blocks. */
int dvm_plan_vblocks(const dvm_vgrid *v, int rv, int order, int wide_axis, int *boxes8, int max_blocks);
/* The same for rank shard_rank of shard_count (DVM_OPT_SHARD_COUNT): only that rank's velocity blocks. */
int dvm_plan_shard_vblocks(const dvm_vgrid *v, int rv, int order, int wide_axis, int shard_rank, int shard_count, int *boxes8,
                           int max_blocks);
/* Bytes of device workspace held by the solver, and the part of it that holds distribution-function values. */
int dvm_workspace_bytes(const dvm_solver *s, size_t *total, size_t *f_bytes);
/* Number of kernel launches enqueued by this solver so far (bench.py's gpu_launches). */
long long dvm_launch_count(const dvm_solver *s);
/* How dvm_iterate issues an iteration: 1 = it replays the CUDA graph captured at the first dvm_iterate; 0 = plain kernel launches
 * because no graph is in use (before the first dvm_iterate, slice kernel, DVM_GRAPH=0, sharded solver); 2 = plain kernel launches
 * because the capture was tried and FAILED (e.g. the caller's stream was itself being captured) - results are the same, every
 * iteration costs twelve launches instead of one, and dvm_last_error() held the reason when the first dvm_iterate returned. */
int dvm_graph_active(const dvm_solver *s);
int dvm_destroy(dvm_solver *s);
const char *dvm_last_error(void);

/* ---- convergence residual without a solver and without any allocation ---------------------------------------------------
 * The residual of PAPER.md:269 (reading G9: r_rho = sqrt(sum (rho1 - rho0)^2 / sum rho1^2) over the cells, the same
 * for the momentum rho u and the energy rho E = 3/4 rho T + 1/2 rho |u|^2, unweighted sums) between two macroscopic states
 * the caller already holds, e.g. two outputs of dvm_moments.  It is the arithmetic and the two-level fixed-order reduction of
 * the solver's own residual kernels; what differs is where the per-block partial sums go.
 *
 * This call never enters the CUDA allocator (no cudaMalloc / cudaFree, no allocating library routine), so it is usable by
 * hosts that cannot allocate: a program that gave all device memory to its own pool at start-up (cudaMalloc would fail), a
 * latency-critical loop (cudaMalloc / cudaFree stall the whole device), or code called from a context where the allocator
 * may not be entered.  The partial sums live in a fixed 3 MiB array inside the library image; consequences:
 *   - every GPU onto which libdvm_b200.so is loaded holds those 3 MiB until the process exits;
 *   - ncell <= DVM_RESIDUAL_NOALLOC_MAX_CELLS (256^3); anything larger is refused with DVM_EINVAL and a message that names the
 *     limit - use a solver's dvm_residual there;
 *   - all calls share the array.  Calls are safe one after the other on one stream (no slot is read that the same call has not
 *     written first, so nothing needs clearing between calls); two calls that may run at the same time on one GPU (different
 *     streams, different host threads) race on it and return garbage - the caller serialises them;
 *   - the first call on each GPU also does the one-time set-up for that GPU (it asks the runtime for the array's device address,
 *     which makes the driver load the module).  Make that first call during start-up, before any stream capture begins.
 *
 * dev_prim_old, dev_prim_new: dev, SoA with field stride ncell, at least the first 5 fields of dvm_moments' layout (rho, ux, uy,
 * uz, T at [m*ncell + c]; a prim8 or prim14 buffer fits as it is); solid cells must hold zeros in both (dvm_moments writes
 * them so).  dev_out3: dev, 3 doubles = r_rho, r_mom, r_E; a zero denominator gives 0 (numerator 0) or +inf, a NaN in the
 * input propagates (no DVM_ENONFINITE here: nothing is read back).  stream: cudaStream_t (0 = default stream).  All three buffers
 * must belong to one GPU; the call runs there whatever device is current and restores the caller's device.  Asynchronous.
 * Errors: DVM_EINVAL (NULL, ncell <= 0 or beyond the limit, a buffer that is not device memory of that GPU), DVM_ECUDA. */
#define DVM_RESIDUAL_NOALLOC_MAX_CELLS 16777216LL
int dvm_residual_noalloc(const double *dev_prim_old, const double *dev_prim_new, long long ncell, double *dev_out3, void *stream);

/* ---- measurement aid (bench.py's roofline) ---------------------------------------------------------
 * (syncs) The fp64 rate this board sustains on a register-resident stream of fused multiply-adds: every SM full (2048 threads),
 * 8 independent chains per thread, `rounds` DFMAs per chain, no memory traffic, timed with CUDA events on the default stream of
 * the current device.  *host_lane_ops_per_s = executed fp64 thread-instructions per second (one DFMA = one lane-operation; the
 * nominal figure is 148 SM x 64 lanes x clock), *host_ms (may be NULL) = duration of the timed launch.  dev_sink: dev, >= 1 double,
 * never written in practice.  rounds = 2 000 000 runs for about 0.3 s on a B200. */
int dvm_fp64_peak_probe(double *dev_sink, long long rounds, double *host_lane_ops_per_s, double *host_ms);

#ifdef __cplusplus
}
#endif
#endif
