// sweep_tile.cuh - host interface and shared records of the tile sweep kernel (sweep_tile.cu, tile_plan.cu).
//
// DVM_KERNEL_TILE in one paragraph: the sweep of Eq.(7) is cut into
// work items (velocity block V, z-column tile (I', J')).  A velocity block is 512 discrete velocities of one
// sign octant (a box NA x nbb x ncb of node indices); a column tile is TX x TY = 4 x 4 cells wide and spans
// all nz levels.  One CTA owns an item: every thread carries RV velocities (consecutive xi_x nodes, same xi_y, xi_z)
// and keeps their 4 x 4 values of the current z-plane of the tile in REGISTERS, so the
// z-upwind and y-upwind operands never leave the register file; only the x- and y-faces of the column go to HBM
// (8 B per phase point instead of the 16 B of an in-place slice, 32 B in the paper's two-slice form,
// PAPER.md:104-106, 233-235).  Items are handed out by an atomic counter in an order that respects the upwind
// dependencies (x-face of (I'-1, J'), y-face of (I', J'-1)); done-flags in global memory gate the start of an item.
// The equilibrium enters through 1-D factor tables (tables.cu) staged by TMA with the faces; velocity blocks may
// sweep in batches that share face-slot sets when the f workspace is capped (DVM_OPT_MAX_F_MBYTES).
// Variants of the kernel (DVM_OPT_TILE_RV): RV = 4: CTAs of 128 threads, blocks of 16 x 32 nodes (nbb x ncb = 8 x 4
// or 4 x 8); RV = 3: 128 threads, blocks of 12 x 32 nodes; RV = 2: CTAs of 256 threads, blocks of 8 x 8 x 8 nodes, twice the
// warps per SM.
#pragma once
#include <cuda_runtime.h>
#include <vector>
#include "dvm_dev.cuh"

namespace dvm {

constexpr int TILE_TX = 4;                 // cells per tile along the sweep-relative x
#ifndef DVM_TILE_TY
#define DVM_TILE_TY 4
#endif
constexpr int TILE_TY = DVM_TILE_TY;        // cells per tile along the sweep-relative y
#ifndef DVM_TILE_F32_CTAS
#define DVM_TILE_F32_CTAS 3
#endif                                      // resident CTAs per SM the single-precision variants are compiled for
constexpr int TILE_NCELL = TILE_TX * TILE_TY;
constexpr int TILE_GA = 4;                 // xi_x groups per lane quad
constexpr int TILE_NVB = 512;              // velocities per block (incl. padding) = threads x RV, first-order kernels
constexpr int TILE_MAXBC = 16;             // nbb + ncb of a block
constexpr int TILE_PAD = 4;                // dead cells around the grid in the factor tables (tiles may overhang by 3)
// index ranges of the negative / non-negative nodes of one axis (nodes ascending): the two sweep directions
inline void split_axis(const std::vector<double> &xi, int lo[2], int cnt[2])
{
    int nneg = 0;
    while (nneg < (int)xi.size() && xi[nneg] < 0.0) ++nneg;
    lo[0] = 0; cnt[0] = nneg; lo[1] = nneg; cnt[1] = (int)xi.size() - nneg;
}
// Kernel variants: (rv, order) = (4, 1): 128 threads x 4 velocities; (3, 1): 128 x 3; (2, 1): 256 x 2; (2, 2): the second-order sweep
// (DVM_OPT_ORDER = 2) keeps two z-planes in registers: 128 threads x 2 velocities, 256 velocities per block.
inline int tile_threads(int rv, int order = 1) { return (order == 2 || rv >= 3) ? 128 : 256; }
inline int tile_nvb(int rv, int order = 1) { return tile_threads(rv, order) * rv; }   // velocities per block
inline int tile_na(int rv) { return TILE_GA * rv; }          // xi_x nodes per velocity block
inline int tile_npair(int rv, int order = 1) { return tile_threads(rv, order) / TILE_GA; }   // (xi_y, xi_z) pairs per block
inline int tile_entry_values(int order) { return order == 2 ? 6 : 4; }   // factor-table entry: (E, Q, e, a) or (E, Q, e, cd, c1, c2)
inline int tile_face_layers(int order) { return order == 2 ? 2 : 1; }     // upwind values per direction carried through a face

// per-cell record of the padded grid, fetched by TMA with the factor tables (48 bytes)
constexpr int REC_DEAD = 1 << 16;
struct CellRec {
    double nu;        // 1/tau of step n (written by the table kernel every iteration); 1 for dead cells
    int cidx;         // row of the [cell][16] accumulator the sums of this cell go to: the cell index; a dead cell (solid, or
                      // in the padding) produces exact zeros and names its own row / that of the nearest cell of the grid
    int flags;        // bits 0..5: neighbour in direction d is not fluid; bits 8..13: it is a solid cell; REC_DEAD
    int face[6];      // boundary-face slot in direction d or -1
    float nu32;       // nu rounded to single (DVM_PREC_MIXED)
    int pad;          // 48 bytes: every row of records starts on a 16-byte boundary (TMA)
};
static_assert(sizeof(CellRec) == 48, "CellRec rows must be 16-byte aligned");

// velocity block: node-index box [a0, a0+na) x [b0, b0+nb) x [c0, c0+nc) of the velocity axes in the roles A, B, C
// (TilePlan::ax; A = xi_x unless another axis fills the wide role better), na <= NA, nb <= nbb, nc <= ncb,
// nbb * ncb = pairs per block; lanes beyond the box carry weight 0
struct VBlock {
    int a0, na, b0, nb, c0, nc;
    int nbb, ncb;
    int sx, sy, sz;   // sweep direction per axis: +1 ascending (xi >= 0), -1 descending
    int xb, yb, zb;   // 1-D block ids: rows of the factor tables TX / TY / TZ this block reads
    int pad[2];
};

// work item; ti, tj are sweep-relative tile coordinates (0 = most upwind)
struct TileItem {
    int vb;
    int ti, tj;
    int pred_x;       // item index of (vb, ti-1, tj) or -1
    int pred_y;       // item index of (vb, ti, tj-1) or -1
    int pred_s;       // item index of the last reader of this item's x-face slot, (vb, ntx-1, tj-P), or -1
    int xslot;        // tj % P
    int fslot;        // face-slot set of the block: index within its batch
};

struct TilePlan {
    int ntx = 0, nty = 0, P = 1;
    int rv = 4, order = 1;             // kernel variant this plan is for: velocities per thread, order of the sweep
    int ax[3] = {0, 1, 2};             // velocity axis in the role A (the wide one: RV nodes per thread x 4 lane groups), B, C
    int batch = 0;                     // velocity blocks in flight at once (= face-slot sets)
    int nbb = 8, ncb = 4;              // one (xi_y, xi_z) block shape for the whole problem
    std::vector<int> xnode, ynode, znode;   // node index (of the axis in role A, B, C) per 1-D block slot (-1 = padding): [nxb][NA], [nyb][nbb], [nzb][ncb];
                                            // xnode is in table order: slot r*4 + ag holds node RV*ag + r of the block
    std::vector<VBlock> vblocks;
    std::vector<TileItem> items;
    size_t xface_values = 0, yface_values = 0;   // values of f the two face workspaces hold (8 or 4 bytes each)
};

struct TileParams {
    int nx, ny, nz, ntx, nty, P;
    int batch;                    // velocity blocks per batch: block vb uses face-slot set vb % batch
    long long ncell;
    const double *invdx, *invdy, *invdz;
    const unsigned char *flags;   // [ncell] bits 0..5: neighbour in direction d is not a fluid cell; bit 6: solid
    const unsigned char *sflags;  // [ncell] bits 0..5: neighbour in direction d is a solid cell; bit 6: solid
    const int *face_of;           // [6][ncell] boundary-face slot or -1
    const double *coef;           // [NCOEF][ncell]
    const double *rho_w;          // [nface]
    double *phi;                  // [nface]
    double *raw16;                // [ncell][16] velocity sums (13 used)
    const double *xi_x, *xi_y, *xi_z, *w_x, *w_y, *w_z;
    const double *gtab;           // [7][3][gstride] per BC slot and axis: weighted 1-D factors of the ghost Maxwellian
    int gstride;
    int bc_type[7];
    int foff[6];                  // first slot of each domain face in the boundary-face table
    const VBlock *vblocks;
    const TileItem *items;
    int nitems;
    int *done;                    // [nitems] epoch of completion
    int *counter;                 // next item
    int epoch;
    void *xface, *yface;          // double, or float when f is carried in single precision (DVM_PREC_MIXED)
    long long xslot_values, yslot_values;   // nz * layers * TILE_TY * NVB, nz * layers * TILE_TX * NVB
    // factor tables of step n (tables_kernel), padded grid nxp x nyp x nz, entries (E, Q, e, a) [order 2: (E, Q, e, cd, c1, c2)],
    // double or float like the faces:
    const void *TX, *TY, *TZ;     // [nxb][nz][nyp][nxp][NA][4 or 6], [nyb][nz][nyp][nxp][nbb][.], [nzb][nz][nyp][nxp][ncb][.]
    const CellRec *rec;           // [nz][nyp][nxp]
    int nxp, nyp, nbb, ncb;
};

struct TableParams {
    int nx, ny, nz, nxp, nyp, na, nbb, ncb, nxb, nyb, nzb, order;
    int f32;                      // 1: entries are written as float (DVM_PREC_MIXED)
    int ax[3];                    // velocity axis of the tables TX, TY, TZ (roles A, B, C)
    long long ncell;
    const double *coef;           // [NCOEF][ncell]
    const unsigned char *flags;   // bit 6: solid
    const double *invdx, *invdy, *invdz;
    const double *dx, *dy, *dz;   // cell widths (order 2)
    const double *xi_x, *xi_y, *xi_z, *w_x, *w_y, *w_z;
    const int *xnode, *ynode, *znode;
    int bc_type[6];
    void *TX, *TY, *TZ;
    CellRec *rec;
};

// Build velocity blocks, items and their order for a grid and a set of velocity nodes.  target_ctas = number of
// items that should be able to run concurrently (sets the band height P); max_blocks > 0 caps the velocity blocks in
// flight at once (batches).  Pure host code (tests call it through
// dvm_plan_query without a GPU).
// shard_rank / shard_count: the plan holds only the velocity blocks of that rank (velocity-space sharding; -1 if it has none).
int tile_plan(int nx, int ny, int nz, const std::vector<double> xi[3], int target_ctas, int max_blocks, int rv, int order,
              int wide_axis, TilePlan *plan, int shard_rank = 0, int shard_count = 1);

// f32: f carried in single precision (DVM_PREC_MIXED; order 1, rv 3 or 4)
bool tile_variant_exists(int rv, int order, bool f32);
size_t tile_smem_bytes(int rv, int order, bool f32);
cudaError_t tile_configure(int rv, int order, bool f32, int wide_axis, int *ctas_per_sm);
cudaError_t launch_sweep_tile(const TileParams &P, int rv, int order, bool f32, int wide_axis, int grid, cudaStream_t st);
cudaError_t launch_tables(const TableParams &T, cudaStream_t st);

}  // namespace dvm
