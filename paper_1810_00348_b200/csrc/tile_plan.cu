// tile_plan.cu - host planner of the tile sweep kernel: velocity blocks, work items, their hand-out order and
// the dependency edges (see sweep_tile.cuh).  Pure host code, no CUDA calls.
//
// Order.  Tile rows (sweep-relative tj) are grouped into bands of P rows.  Bands are processed one after the
// other; inside a band items are ordered by the diagonal d = ti + (tj mod P), then by row, then by velocity
// block.  Every predecessor of an item (the tile upwind in x, the tile upwind in y, and the last reader of the
// x-face slot the item is about to overwrite) is therefore earlier in the order, which - with items handed out
// by a monotone counter - rules out deadlock: an item only ever waits for items that are running or done.
#include "sweep_tile.cuh"

#include <algorithm>
#include <map>

namespace dvm {

namespace {

int ceil_div(int a, int b) { return (a + b - 1) / b; }

}  // namespace

int tile_plan(int nx, int ny, int nz, const std::vector<double> xi[3], int target_ctas, int max_blocks, int rv, int order,
              int wide_axis, TilePlan *plan, int shard_rank, int shard_count)
{
    if (nx <= 0 || ny <= 0 || nz <= 0 || !plan || (rv < 2 || rv > 4) || (order != 1 && order != 2) || (order == 2 && rv != 2) ||
        wide_axis < 0 || wide_axis > 2 || shard_count < 1 || shard_rank < 0 || shard_rank >= shard_count)
        return -1;
    const int NA = tile_na(rv), NVB = tile_nvb(rv, order), npair = tile_npair(rv, order), layers = tile_face_layers(order);
    plan->rv = rv; plan->order = order;
    // roles: A = the wide axis, B and C = the other two in ascending order
    const int ax[3] = {wide_axis, wide_axis == 0 ? 1 : 0, wide_axis == 2 ? 1 : 2};
    for (int r = 0; r < 3; ++r) plan->ax[r] = ax[r];
    plan->vblocks.clear();
    plan->items.clear();
    int lo[3][2], cnt[3][2];
    for (int d = 0; d < 3; ++d) split_axis(xi[d], lo[d], cnt[d]);

    // ---- (nbb, ncb) with nbb * ncb = pairs per block and nbb + ncb <= TILE_MAXBC: one shape for the whole problem (the
    //      factor tables are laid out by 1-D block), the one wasting the fewest lanes ----
    int best_bb = 8, best_cb = npair / 8;
    {
        long best = -1;
        const int shapes4[2][2] = {{8, 4}, {4, 8}}, shapes2[2][2] = {{8, 8}, {8, 8}};
        for (auto &s : (npair == 64 ? shapes2 : shapes4)) {
            long slots = 0;
            for (int oz = 0; oz < 2; ++oz) for (int oy = 0; oy < 2; ++oy)
                slots += (long)ceil_div(cnt[ax[1]][oy], s[0]) * ceil_div(cnt[ax[2]][oz], s[1]);
            if (best < 0 || slots < best) { best = slots; best_bb = s[0]; best_cb = s[1]; }
        }
    }
    plan->nbb = best_bb; plan->ncb = best_cb;
    // ---- 1-D blocks per axis and sign half; first block id of each half ----
    int first[3][2];
    const int width[3] = {NA, best_bb, best_cb};
    std::vector<int> *nodes[3] = {&plan->xnode, &plan->ynode, &plan->znode};
    for (int r = 0; r < 3; ++r) {
        const int d = ax[r];
        nodes[r]->clear();
        int nblk = 0;
        for (int h = 0; h < 2; ++h) {
            first[r][h] = nblk;
            for (int k0 = 0; k0 < cnt[d][h]; k0 += width[r], ++nblk)
                for (int sl = 0; sl < width[r]; ++sl) {
                    // A: table slot r*4 + ag holds node RV*ag + r of the block (conflict-free reads, sweep_tile.cu)
                    const int local = r == 0 ? rv * (sl & 3) + (sl >> 2) : sl;
                    nodes[r]->push_back(k0 + local < cnt[d][h] ? lo[d][h] + k0 + local : -1);
                }
        }
    }
    // ---- velocity blocks: per octant, chunks of NA x nbb x ncb node indices of the axes in the roles A, B, C ----
    for (int oc = 0; oc < 2; ++oc) for (int ob = 0; ob < 2; ++ob) for (int oa = 0; oa < 2; ++oa) {
        const int na = cnt[ax[0]][oa], nb = cnt[ax[1]][ob], nc = cnt[ax[2]][oc];
        if (na == 0 || nb == 0 || nc == 0) continue;
        int sgn[3];
        sgn[ax[0]] = oa ? 1 : -1; sgn[ax[1]] = ob ? 1 : -1; sgn[ax[2]] = oc ? 1 : -1;
        for (int c0 = 0; c0 < nc; c0 += best_cb) for (int b0 = 0; b0 < nb; b0 += best_bb)
            for (int a0 = 0; a0 < na; a0 += NA) {
                VBlock v{};
                v.a0 = lo[ax[0]][oa] + a0; v.na = std::min(NA, na - a0);
                v.b0 = lo[ax[1]][ob] + b0; v.nb = std::min(best_bb, nb - b0);
                v.c0 = lo[ax[2]][oc] + c0; v.nc = std::min(best_cb, nc - c0);
                v.nbb = best_bb; v.ncb = best_cb;
                v.sx = sgn[0]; v.sy = sgn[1]; v.sz = sgn[2];
                v.xb = first[0][oa] + a0 / NA; v.yb = first[1][ob] + b0 / best_bb; v.zb = first[2][oc] + c0 / best_cb;
                plan->vblocks.push_back(v);
            }
    }
    // velocity-space sharding (the paper's MPI program decomposes the velocity space): rank r
    // of n sweeps the velocity blocks r, r + n, r + 2n, ... of the list (every octant is spread over the ranks); the factor
    // tables stay complete
    if (shard_count > 1) {
        std::vector<VBlock> mine;
        for (size_t e = (size_t)shard_rank; e < plan->vblocks.size(); e += (size_t)shard_count) mine.push_back(plan->vblocks[e]);
        plan->vblocks.swap(mine);
    }
    const int nvb = (int)plan->vblocks.size();
    if (nvb == 0) return -1;
    const int ntx = ceil_div(nx, TILE_TX), nty = ceil_div(ny, TILE_TY);
    plan->ntx = ntx; plan->nty = nty;
    // velocity blocks in flight at once (smaller batches cap the memory of the stored f): the face
    // workspace holds one slot set per block of a batch; batches sweep the grid one after the other
    const int B = max_blocks > 0 ? std::min(max_blocks, nvb) : nvb;
    plan->batch = B;
    // band height: enough independent tiles per diagonal to keep target_ctas items in flight
    int P = ceil_div(std::max(target_ctas, 1) * 2, B);
    P = std::max(1, std::min(P, nty));
    plan->P = P;

    // ---- items in hand-out order: batch, band of P tile rows, diagonal, row, velocity block ----
    std::vector<int> index((size_t)nvb * ntx * nty, -1);
    auto at = [&](int vb, int ti, int tj) -> int & { return index[((size_t)vb * nty + tj) * ntx + ti]; };
    for (int v0 = 0; v0 < nvb; v0 += B)
        for (int band = 0; band * P < nty; ++band) {
            const int j0 = band * P, rows = std::min(P, nty - j0);
            for (int d = 0; d < ntx + rows - 1; ++d)
                for (int r = 0; r < rows; ++r) {
                    const int ti = d - r, tj = j0 + r;
                    if (ti < 0 || ti >= ntx) continue;
                    for (int vb = v0; vb < std::min(nvb, v0 + B); ++vb) {
                        TileItem it{};
                        it.vb = vb; it.ti = ti; it.tj = tj; it.xslot = tj % P; it.fslot = vb - v0;
                        it.pred_x = it.pred_y = it.pred_s = -1;
                        at(vb, ti, tj) = (int)plan->items.size();
                        plan->items.push_back(it);
                    }
                }
        }
    for (auto &it : plan->items) {
        if (it.ti > 0) it.pred_x = at(it.vb, it.ti - 1, it.tj);
        if (it.tj > 0) it.pred_y = at(it.vb, it.ti, it.tj - 1);
        if (it.ti == 0 && it.tj >= P) it.pred_s = at(it.vb, ntx - 1, it.tj - P);
        // face slots are shared with the block B places earlier (previous batch): wait for its last readers
        if (it.vb >= B) {
            if (it.tj == 0) it.pred_y = at(it.vb - B, it.ti, nty - 1);          // y-face slot (fslot, ti)
            if (it.ti == 0 && it.tj < P) {                                      // x-face slot (fslot, tj % P)
                const int last = it.tj + ((nty - 1 - it.tj) / P) * P;
                it.pred_s = at(it.vb - B, ntx - 1, last);
            }
        }
    }
    plan->xface_values = (size_t)B * P * nz * layers * TILE_TY * NVB;
    plan->yface_values = (size_t)B * ntx * nz * layers * TILE_TX * NVB;
    return 0;
}

}  // namespace dvm
