// dvm_api.cu - host side of the C ABI declared in include/dvm.h: validation, geometry / boundary-face tables,
// velocity-octant block tables, workspace management and the per-iteration launch sequence
// (Alg. 1: sweep all velocity groups, then update the moments).
// Product code: no CPU fallback and nothing shared with oracle/.
#include "../../include/dvm.h"
#include "dvm_dev.cuh"
#include "update.cuh"
#include "sweep_tile.cuh"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

using namespace dvm;

namespace {

thread_local std::string g_err;

int fail(int code, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
    return code;
}

#define CK(call)                                                                                     \
    do {                                                                                             \
        cudaError_t e_ = (call);                                                                     \
        if (e_ != cudaSuccess) return fail(DVM_ECUDA, "%s: %s (%s:%d)", #call, cudaGetErrorString(e_), \
                                           __FILE__, __LINE__);                                      \
    } while (0)

constexpr int HIST_CAP = 16384;

// Every entry point runs on the solver's device whatever device is current in the calling thread, and restores it.
struct DeviceGuard {
    int prev = -1, want;
    explicit DeviceGuard(int d) : want(d)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        if (prev != want) cudaSetDevice(want);
    }
    ~DeviceGuard()
    {
        if (prev >= 0 && prev != want) cudaSetDevice(prev);
    }
};
const double PI = 3.14159265358979323846;

}  // namespace

namespace dvm {
// for the other translation units of the library (residual_noalloc.cu): leave a message for dvm_last_error()
int report_error(int code, const char *msg)
{
    g_err = msg;
    return code;
}
}  // namespace dvm

struct dvm_solver {
    int nx = 0, ny = 0, nz = 0, mx = 0, my = 0, mz = 0, nface = 0;
    long long ncell = 0;
    std::vector<double> xf, yf, zf, xi[3], w[3];
    std::vector<unsigned char> solid;
    dvm_gas gas{};
    dvm_bc bc{};
    cudaStream_t stream = nullptr;
    int device = 0;               // CUDA device ordinal the solver lives on (current device at dvm_create)
    dvm_device dev{};
    std::vector<void *> allocs;
    size_t total_bytes = 0, f_bytes = 0;
    double mass0 = 0.0;
    int iters = 0;
    int kernel = DVM_KERNEL_AUTO;
    long long max_f_mbytes = 0;   // cap on the f workspace of the tile kernel (0 = none)
    int tile_rv = 0;              // velocities per thread of the tile kernel: 0 = choose, 2, 3, 4
    int tile_axis = 0;            // velocity axis in the wide role of the tile kernel: 0 = choose, 1 + axis
    int max_ctas = 0;             // cap on the persistent grid of the tile kernel (0 = all resident CTAs)
    int order = 1;                // 1: first-order upwind Eq.(7); 2: second-order upwind
    int precision = DVM_PREC_F64; // DVM_PREC_MIXED: f carried in single precision by the tile kernel
    int shard_rank = 0, shard_count = 1;   // velocity-space sharding (DVM_OPT_SHARD_COUNT / _RANK)
    bool swept = false;           // dvm_sweep done, dvm_update pending
    // one outer iteration of the tile kernel as a CUDA graph: captured at the first dvm_iterate, replayed afterwards (the
    // launch parameters of an iteration never change: constant flag epoch + flag reset, device-side history slot)
    cudaGraphExec_t graph_exec = nullptr;
    long long graph_launches = 0; // kernel launches inside the graph
    bool graph_off = false;       // DVM_GRAPH=0 in the environment, or the capture failed: plain launches
    bool graph_failed = false;    // the capture was tried and failed (dvm_graph_active reports it)
    size_t fvalue() const { return precision == DVM_PREC_MIXED ? sizeof(float) : sizeof(double); }
    bool planned = false;
    long long launches = 0;
    // device arrays
    double *d_invdx = nullptr, *d_invdy = nullptr, *d_invdz = nullptr, *d_dx = nullptr, *d_dy = nullptr, *d_dz = nullptr;
    unsigned char *d_flags = nullptr, *d_face_slot = nullptr;
    int *d_face_of = nullptr, *d_face_cell = nullptr, *d_face_dir = nullptr;
    double *d_xi[3] = {nullptr, nullptr, nullptr}, *d_w[3] = {nullptr, nullptr, nullptr};
    double *d_prim = nullptr, *d_prim_new = nullptr, *d_coef = nullptr, *d_raw = nullptr;
    double *d_rho_w = nullptr, *d_phi = nullptr, *d_phi_unit = nullptr;
    double *d_part = nullptr, *d_scal = nullptr, *d_hist = nullptr, *d_hist_scale = nullptr;
    long long npart = 0;
    // sweep plan
    std::vector<BlockDesc> blocks;
    BlockDesc *d_blocks = nullptr;
    double *d_fbuf = nullptr;
    long long fstride = 0, fslice = 0;
    int nb_threads = 128;
    TilePlan tile{};
    unsigned char *d_sflags = nullptr;
    double *d_gtab = nullptr;
    int gstride = 0;
    int foff[6] = {0, 0, 0, 0, 0, 0};
    VBlock *d_vblocks = nullptr;
    TileItem *d_items = nullptr;
    int *d_done = nullptr, *d_counter = nullptr;
    void *d_xface = nullptr, *d_yface = nullptr;
    int tile_grid = 0, epoch = 0;
    std::vector<double> h_rho_w0;
    // factor tables of the tile kernel (tables.cu)
    std::vector<CellRec> h_rec;
    CellRec *d_rec = nullptr;
    void *d_TX = nullptr, *d_TY = nullptr, *d_TZ = nullptr;
    int *d_xnode = nullptr, *d_ynode = nullptr, *d_znode = nullptr;
    int nxp = 0, nyp = 0, nxb = 0, nyb = 0, nzb = 0;
    size_t table_bytes = 0;

    void *dalloc(size_t bytes)
    {
        bytes = (bytes + 255) / 256 * 256;
        if (bytes == 0) bytes = 256;
        void *p = nullptr;
        if (dev.alloc) p = dev.alloc(bytes, dev.ctx);
        else if (cudaMalloc(&p, bytes) != cudaSuccess) p = nullptr;
        if (p) { allocs.push_back(p); total_bytes += bytes; }
        return p;
    }
    void dfree_all()
    {
        for (void *p : allocs) {
            if (dev.free_) dev.free_(p, dev.ctx);
            else if (!dev.alloc) cudaFree(p);
        }
        allocs.clear();
    }
};

namespace {

template <class T>
int upload(dvm_solver *s, T **dst, const T *src, size_t n)
{
    *dst = (T *)s->dalloc(n * sizeof(T));
    if (!*dst) return fail(DVM_ENOMEM, "device allocation of %zu bytes failed", n * sizeof(T));
    CK(cudaMemcpyAsync(*dst, src, n * sizeof(T), cudaMemcpyHostToDevice, s->stream));
    return 0;
}

template <class T>
int dzeros(dvm_solver *s, T **dst, size_t n)
{
    *dst = (T *)s->dalloc(n * sizeof(T));
    if (!*dst) return fail(DVM_ENOMEM, "device allocation of %zu bytes failed", n * sizeof(T));
    CK(cudaMemsetAsync(*dst, 0, n * sizeof(T), s->stream));
    return 0;
}

bool increasing(const double *a, int n)
{
    for (int i = 1; i < n; ++i)
        if (!(a[i] > a[i - 1])) return false;
    return true;
}

double host_wall_maxwellian(const dvm_face_bc &b, const double xi[3])
{
    const double cx = xi[0] - b.u[0], cy = xi[1] - b.u[1], cz = xi[2] - b.u[2];
    return std::exp(-(cx * cx + cy * cy + cz * cz) / b.T) / std::pow(PI * b.T, 1.5);
}

const dvm_face_bc &slot_bc(const dvm_bc &bc, int b) { return b < 6 ? bc.face[b] : bc.solid; }

UpdateParams update_params(dvm_solver *s)
{
    UpdateParams U{};
    U.nx = s->nx; U.ny = s->ny; U.nz = s->nz; U.nface = s->nface; U.ncell = s->ncell; U.npart = s->npart;
    U.flags = s->d_flags; U.dx = s->d_dx; U.dy = s->d_dy; U.dz = s->d_dz;
    U.raw = s->d_raw; U.prim = s->d_prim; U.prim_new = s->d_prim_new; U.coef = s->d_coef;
    U.part = s->d_part; U.scal = s->d_scal; U.hist = s->d_hist; U.hist_scale = s->d_hist_scale;
    U.phi = s->d_phi; U.phi_unit = s->d_phi_unit; U.rho_w = s->d_rho_w;
    U.omega = s->gas.omega;
    const double cw = 15.0 * std::sqrt(PI) / ((5.0 - 2.0 * s->gas.omega) * (7.0 - 2.0 * s->gas.omega));
    U.inv_cw_kn = 1.0 / (cw * s->gas.Kn);
    U.shk = (1.0 - s->gas.Pr) * 0.8;
    U.mass0 = s->mass0;
    U.rescale = s->bc.rescale_mass;
    return U;
}

SweepParams sweep_params(dvm_solver *s)
{
    SweepParams P{};
    P.nx = s->nx; P.ny = s->ny; P.nz = s->nz; P.ncell = s->ncell;
    P.invdx = s->d_invdx; P.invdy = s->d_invdy; P.invdz = s->d_invdz;
    P.dx = s->d_dx; P.dy = s->d_dy; P.dz = s->d_dz; P.order = s->order; P.fslice = s->fslice;
    P.flags = s->d_flags; P.face_of = s->d_face_of; P.face_slot = s->d_face_slot;
    P.coef = s->d_coef; P.rho_w = s->d_rho_w; P.phi = s->d_phi; P.raw = s->d_raw;
    P.xi_x = s->d_xi[0]; P.xi_y = s->d_xi[1]; P.xi_z = s->d_xi[2];
    P.w_x = s->d_w[0]; P.w_y = s->d_w[1]; P.w_z = s->d_w[2];
    P.blocks = s->d_blocks; P.fbuf = s->d_fbuf; P.fstride = s->fstride;
    for (int b = 0; b < 7; ++b) {
        const dvm_face_bc &f = slot_bc(s->bc, b);
        P.bc.type[b] = f.type; P.bc.T[b] = f.T; P.bc.rho[b] = f.rho;
        for (int d = 0; d < 3; ++d) P.bc.u[b][d] = f.u[d];
    }
    return P;
}

TileParams tile_params(dvm_solver *s)
{
    TileParams P{};
    P.nx = s->nx; P.ny = s->ny; P.nz = s->nz; P.ntx = s->tile.ntx; P.nty = s->tile.nty; P.P = s->tile.P;
    P.batch = s->tile.batch;
    P.ncell = s->ncell;
    P.invdx = s->d_invdx; P.invdy = s->d_invdy; P.invdz = s->d_invdz;
    P.flags = s->d_flags; P.sflags = s->d_sflags; P.face_of = s->d_face_of;
    P.coef = s->d_coef; P.rho_w = s->d_rho_w; P.phi = s->d_phi; P.raw16 = s->d_raw;
    P.xi_x = s->d_xi[0]; P.xi_y = s->d_xi[1]; P.xi_z = s->d_xi[2];
    P.w_x = s->d_w[0]; P.w_y = s->d_w[1]; P.w_z = s->d_w[2];
    P.gtab = s->d_gtab; P.gstride = s->gstride;
    for (int b = 0; b < 7; ++b) P.bc_type[b] = slot_bc(s->bc, b).type;
    for (int d = 0; d < 6; ++d) P.foff[d] = s->foff[d];
    P.vblocks = s->d_vblocks; P.items = s->d_items; P.nitems = (int)s->tile.items.size();
    P.done = s->d_done; P.counter = s->d_counter; P.epoch = s->epoch;
    P.xface = s->d_xface; P.yface = s->d_yface;
    const int nvb = tile_nvb(s->tile.rv, s->tile.order), layers = tile_face_layers(s->tile.order);
    P.xslot_values = (long long)s->nz * layers * TILE_TY * nvb;
    P.yslot_values = (long long)s->nz * layers * TILE_TX * nvb;
    P.TX = s->d_TX; P.TY = s->d_TY; P.TZ = s->d_TZ; P.rec = s->d_rec;
    P.nxp = s->nxp; P.nyp = s->nyp; P.nbb = s->tile.nbb; P.ncb = s->tile.ncb;
    return P;
}

TableParams table_params(dvm_solver *s)
{
    TableParams T{};
    T.nx = s->nx; T.ny = s->ny; T.nz = s->nz; T.nxp = s->nxp; T.nyp = s->nyp;
    for (int r = 0; r < 3; ++r) T.ax[r] = s->tile.ax[r];
    T.order = s->tile.order; T.f32 = s->precision == DVM_PREC_MIXED; T.dx = s->d_dx; T.dy = s->d_dy; T.dz = s->d_dz;
    T.na = tile_na(s->tile.rv); T.nbb = s->tile.nbb; T.ncb = s->tile.ncb; T.nxb = s->nxb; T.nyb = s->nyb; T.nzb = s->nzb;
    T.ncell = s->ncell; T.coef = s->d_coef; T.flags = s->d_flags;
    T.invdx = s->d_invdx; T.invdy = s->d_invdy; T.invdz = s->d_invdz;
    T.xi_x = s->d_xi[0]; T.xi_y = s->d_xi[1]; T.xi_z = s->d_xi[2];
    T.w_x = s->d_w[0]; T.w_y = s->d_w[1]; T.w_z = s->d_w[2];
    T.xnode = s->d_xnode; T.ynode = s->d_ynode; T.znode = s->d_znode;
    for (int d = 0; d < 6; ++d) T.bc_type[d] = s->bc.face[d].type;
    T.TX = s->d_TX; T.TY = s->d_TY; T.TZ = s->d_TZ; T.rec = s->d_rec;
    return T;
}

// Variant of the tile kernel for a velocity grid when the caller leaves the choice open: the (velocities per thread, wide
// axis) pair with the highest expected throughput = (share of its lanes that carry a velocity: blocks of 16 x 32, 12 x 32
// or 8 x 64 nodes per sign octant, the wide side along the chosen velocity axis) x (measured throughput of the variant
// relative to RV = 4 when all fill their blocks).  rv / axis > 0 (resp. >= 0) fix that part.
constexpr double RV_SPEED[5] = {0.0, 0.0, 0.80, 0.90, 1.0};
void choose_variant(const std::vector<double> xi[3], int order, int rv_fixed, int axis_fixed, int *rv_out, int *axis_out, bool f32 = false)
{
    if (order == 2) rv_fixed = 2;
    const long long nvel = (long long)xi[0].size() * xi[1].size() * xi[2].size();
    int best_rv = rv_fixed ? rv_fixed : 4, best_ax = axis_fixed >= 0 ? axis_fixed : 0;
    double best_score = -1.0;
    for (int rv = 4; rv >= 2; --rv) {
        if (rv_fixed && rv != rv_fixed) continue;
        if (!rv_fixed && !tile_variant_exists(rv, order, f32)) continue;
        for (int ax = 0; ax < 3; ++ax) {
            if (axis_fixed >= 0 && ax != axis_fixed) continue;
            TilePlan tp;
            if (tile_plan(4, 4, 1, xi, 1, 0, rv, order, ax, &tp)) continue;
            const double fill = (double)nvel / ((double)tp.vblocks.size() * tile_nvb(rv, order));
            if (fill * RV_SPEED[rv] > best_score * 1.0000001) { best_score = fill * RV_SPEED[rv]; best_rv = rv; best_ax = ax; }
        }
    }
    *rv_out = best_rv; *axis_out = best_ax;
}

int plan_once(dvm_solver *s);

// Decide the kernel variant and build the block table + f workspace (once, before the first iteration).  A failed attempt
// gives back what it allocated and puts back what the caller had requested (kernel, velocities per thread, wide axis: plan_once
// replaces "the library chooses" by its choice), so that the call can be repeated, e.g. with another workspace cap or
// precision, and is planned afresh.
int plan(dvm_solver *s)
{
    if (s->planned) return 0;
    const size_t nalloc = s->allocs.size(), bytes = s->total_bytes;
    const int req_kernel = s->kernel, req_rv = s->tile_rv, req_axis = s->tile_axis;
    const int rc = plan_once(s);
    if (rc != 0) {
        cudaStreamSynchronize(s->stream);
        for (size_t e = nalloc; e < s->allocs.size(); ++e) {
            if (s->dev.free_) s->dev.free_(s->allocs[e], s->dev.ctx);
            else if (!s->dev.alloc) cudaFree(s->allocs[e]);
        }
        s->allocs.resize(nalloc);
        s->total_bytes = bytes;
        s->f_bytes = 0;
        s->table_bytes = 0;
        s->kernel = req_kernel; s->tile_rv = req_rv; s->tile_axis = req_axis;
        // everything plan_once may have pointed at the memory just released
        s->d_fbuf = nullptr; s->d_blocks = nullptr; s->d_xface = nullptr; s->d_yface = nullptr;
        s->d_TX = nullptr; s->d_TY = nullptr; s->d_TZ = nullptr; s->d_rec = nullptr;
        s->d_xnode = nullptr; s->d_ynode = nullptr; s->d_znode = nullptr;
        s->d_vblocks = nullptr; s->d_items = nullptr; s->d_done = nullptr; s->d_counter = nullptr;
    }
    return rc;
}

int plan_once(dvm_solver *s)
{
    const long long nvel = (long long)s->mx * s->my * s->mz;
    int kernel = s->kernel;
    if (kernel == DVM_KERNEL_AUTO) kernel = DVM_KERNEL_TILE;
    if (kernel == DVM_KERNEL_TILE && s->order == 2 && s->tile_rv > 2)
        return fail(DVM_EINVAL, "the second-order tile kernel carries 2 velocities per thread (DVM_OPT_TILE_RV = 2 or 0)");
    const bool f32 = s->precision == DVM_PREC_MIXED;
    if (f32 && (kernel != DVM_KERNEL_TILE || s->order != 1 || s->tile_rv == 2))
        return fail(DVM_EINVAL, "DVM_PREC_MIXED is a mode of the first-order tile kernel with 3 or 4 velocities per thread");
    if (s->shard_count > 1 && kernel != DVM_KERNEL_TILE)
        return fail(DVM_EINVAL, "velocity-space sharding (DVM_OPT_SHARD_COUNT) is a mode of the tile kernel");
    s->kernel = kernel;
    int lo[3][2], cnt[3][2];
    for (int d = 0; d < 3; ++d) split_axis(s->xi[d], lo[d], cnt[d]);
    s->blocks.clear();
    if (kernel == DVM_KERNEL_SLICE) {
        int nb = 128;
        if (nvel / 128 < 296) nb = 64;
        if (nvel / 64 < 296) nb = 32;
        s->nb_threads = nb;
        int col = 0;
        for (int oz = 0; oz < 2; ++oz) for (int oy = 0; oy < 2; ++oy) for (int ox = 0; ox < 2; ++ox) {
            const int n = cnt[0][ox] * cnt[1][oy] * cnt[2][oz];
            for (int l0 = 0; l0 < n; l0 += nb) {
                BlockDesc b{};
                b.ia0 = lo[0][ox]; b.na = cnt[0][ox]; b.ib0 = lo[1][oy]; b.nb = cnt[1][oy];
                b.ic0 = lo[2][oz]; b.nc = cnt[2][oz]; b.l0 = l0;
                b.sx = ox ? 1 : -1; b.sy = oy ? 1 : -1; b.sz = oz ? 1 : -1;
                b.col0 = col; col += nb;
                s->blocks.push_back(b);
            }
        }
        s->fstride = col;
        s->fslice = s->order == 2 ? (long long)col * s->nx * s->ny : 0;
        const size_t fbytes = (size_t)col * s->nx * s->ny * sizeof(double) * (s->order == 2 ? 2 : 1);
        s->d_fbuf = (double *)s->dalloc(fbytes);
        if (!s->d_fbuf) return fail(DVM_ENOMEM, "slice workspace of %zu bytes failed", fbytes);
        s->f_bytes = fbytes;
    } else {
        int per_sm = 0, dev = 0, nsm = 0;
        const int order = s->order;
        int rv = 0, wide = 0;
        choose_variant(s->xi, order, s->tile_rv, s->tile_axis - 1, &rv, &wide, f32);
        s->tile_rv = rv; s->tile_axis = wide + 1;
        CK(tile_configure(rv, order, f32, wide, &per_sm));
        CK(cudaGetDevice(&dev));
        CK(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
        if (per_sm < 1) return fail(DVM_ECUDA, "tile kernel does not fit on an SM");
        const int resident = per_sm * nsm;
        if (tile_plan(s->nx, s->ny, s->nz, s->xi, resident, 0, rv, order, wide, &s->tile, s->shard_rank, s->shard_count))
            return fail(DVM_EINVAL, s->shard_count > 1 ? "tile plan failed (more shards than velocity blocks?)" : "tile plan failed");
        if (s->max_f_mbytes > 0) {
            // cap on the f workspace: fewer velocity blocks in flight (batches); the band height P
            // grows as the batch shrinks, so iterate to a fixed point; one block is the floor
            const double vbytes = (double)s->fvalue();
            const double cap = (double)s->max_f_mbytes * 1048576.0, lvl = (double)s->nz * tile_nvb(rv, order) * tile_face_layers(order) * vbytes;
            int B = (int)s->tile.vblocks.size();
            for (int pass = 0; pass < 8; ++pass) {
                const double need = (double)(s->tile.xface_values + s->tile.yface_values) * vbytes;
                if (need <= cap || B == 1) break;
                B = std::max(1, std::min(B - 1, (int)(cap / ((s->tile.P * TILE_TY + s->tile.ntx * TILE_TX) * lvl))));
                if (tile_plan(s->nx, s->ny, s->nz, s->xi, resident, B, rv, order, wide, &s->tile, s->shard_rank, s->shard_count))
                    return fail(DVM_EINVAL, "tile plan failed");
            }
            const double need = (double)(s->tile.xface_values + s->tile.yface_values) * vbytes;
            if (need > cap)
                return fail(DVM_EINVAL, "the f workspace needs %.1f MiB even with one velocity block in flight: the cap of %lld MiB "
                            "(DVM_OPT_MAX_F_MBYTES) cannot be met", need / 1048576.0, s->max_f_mbytes);
        }
        const size_t nitems = s->tile.items.size();
        s->tile_grid = (int)std::min<size_t>((size_t)resident, nitems);
        if (s->max_ctas > 0) s->tile_grid = std::min(s->tile_grid, s->max_ctas);
        const size_t fbytes = (s->tile.xface_values + s->tile.yface_values) * s->fvalue();
        s->d_xface = s->dalloc(s->tile.xface_values * s->fvalue());
        s->d_yface = s->dalloc(s->tile.yface_values * s->fvalue());
        if (!s->d_xface || !s->d_yface) return fail(DVM_ENOMEM, "tile face workspace of %zu bytes failed", fbytes);
        s->f_bytes = fbytes;
        // factor tables on the padded grid: [1-D block][nz][nyp][nxp][width] entries of 32 bytes, zero in the padding
        {
            s->nxb = (int)s->tile.xnode.size() / tile_na(rv);
            s->nyb = (int)s->tile.ynode.size() / s->tile.nbb;
            s->nzb = (int)s->tile.znode.size() / s->tile.ncb;
            const size_t npc = (size_t)s->nz * s->nyp * s->nxp;
            const size_t eb = (size_t)tile_entry_values(order) * s->fvalue();   // bytes per entry
            const size_t ex = npc * s->tile.xnode.size() * eb, ey = npc * s->tile.ynode.size() * eb, ez = npc * s->tile.znode.size() * eb;
            unsigned char *tx = nullptr, *ty = nullptr, *tz = nullptr;
            if (dzeros(s, &tx, ex) || dzeros(s, &ty, ey) || dzeros(s, &tz, ez)) return DVM_ENOMEM;
            s->d_TX = tx; s->d_TY = ty; s->d_TZ = tz;
            s->table_bytes = ex + ey + ez;
            if (upload(s, &s->d_rec, s->h_rec.data(), s->h_rec.size())) return DVM_ENOMEM;
            if (upload(s, &s->d_xnode, s->tile.xnode.data(), s->tile.xnode.size())) return DVM_ENOMEM;
            if (upload(s, &s->d_ynode, s->tile.ynode.data(), s->tile.ynode.size())) return DVM_ENOMEM;
            if (upload(s, &s->d_znode, s->tile.znode.data(), s->tile.znode.size())) return DVM_ENOMEM;
        }
        if (upload(s, &s->d_vblocks, s->tile.vblocks.data(), s->tile.vblocks.size())) return DVM_ENOMEM;
        if (upload(s, &s->d_items, s->tile.items.data(), nitems)) return DVM_ENOMEM;
        if (dzeros(s, &s->d_done, nitems)) return DVM_ENOMEM;
        if (dzeros(s, &s->d_counter, 64)) return DVM_ENOMEM;
        CK(cudaStreamSynchronize(s->stream));  // the host vectors above are read asynchronously
        s->h_rec.clear(); s->h_rec.shrink_to_fit();
        s->planned = true;
        return 0;
    }
    if (upload(s, &s->d_blocks, s->blocks.data(), s->blocks.size())) return DVM_ENOMEM;
    s->planned = true;
    return 0;
}

}  // namespace

extern "C" {

const char *dvm_last_error(void) { return g_err.c_str(); }

int dvm_create(const dvm_grid *g, const dvm_vgrid *v, const dvm_gas *gas, const dvm_bc *bc, const dvm_device *dev,
               dvm_solver **out)
{
    if (!g || !v || !gas || !bc || !out) return fail(DVM_EINVAL, "NULL argument");
    *out = nullptr;
    if (g->nx <= 0 || g->ny <= 0 || g->nz <= 0 || v->mx <= 0 || v->my <= 0 || v->mz <= 0)
        return fail(DVM_EINVAL, "non-positive grid size");
    if (!g->xf || !g->yf || !g->zf || !v->xi_x || !v->xi_y || !v->xi_z || !v->w_x || !v->w_y || !v->w_z)
        return fail(DVM_EINVAL, "NULL array");
    if ((long long)g->nx * g->ny * g->nz > 2000000000LL) return fail(DVM_EINVAL, "too many cells");
    if (!increasing(g->xf, g->nx + 1) || !increasing(g->yf, g->ny + 1) || !increasing(g->zf, g->nz + 1))
        return fail(DVM_EINVAL, "face coordinates must be strictly increasing");
    if (!increasing(v->xi_x, v->mx) || !increasing(v->xi_y, v->my) || !increasing(v->xi_z, v->mz))
        return fail(DVM_EINVAL, "velocity nodes must be strictly increasing");
    for (int d = 0; d < 3; ++d) {
        const double *w = d == 0 ? v->w_x : d == 1 ? v->w_y : v->w_z;
        const int m = d == 0 ? v->mx : d == 1 ? v->my : v->mz;
        for (int i = 0; i < m; ++i)
            if (!(w[i] >= 0.0)) return fail(DVM_EINVAL, "quadrature weights must be >= 0");
    }
    if (!(gas->Kn > 0) || !(gas->rho0 > 0) || !(gas->T0 > 0) || !(gas->Pr > 0))
        return fail(DVM_EINVAL, "Kn, Pr, rho0, T0 must be positive");
    for (int b = 0; b < 7; ++b) {
        const dvm_face_bc &f = slot_bc(*bc, b);
        if (f.type < 0 || f.type > 2) return fail(DVM_EINVAL, "bad boundary type %d in slot %d", f.type, b);
        if (f.type != DVM_ZERO_GRADIENT && !(f.T > 0)) return fail(DVM_EINVAL, "boundary temperature must be > 0");
    }
    if (g->solid && bc->solid.type != DVM_WALL_DIFFUSE) return fail(DVM_EINVAL, "solid faces must be diffuse walls");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(DVM_ECUDA, "no CUDA device: this library has no CPU fallback");
    }

    dvm_solver *s = new (std::nothrow) dvm_solver;
    if (!s) return fail(DVM_ENOMEM, "host allocation failed");
    s->nx = g->nx; s->ny = g->ny; s->nz = g->nz; s->mx = v->mx; s->my = v->my; s->mz = v->mz;
    s->ncell = (long long)g->nx * g->ny * g->nz;
    s->xf.assign(g->xf, g->xf + g->nx + 1); s->yf.assign(g->yf, g->yf + g->ny + 1); s->zf.assign(g->zf, g->zf + g->nz + 1);
    s->xi[0].assign(v->xi_x, v->xi_x + v->mx); s->xi[1].assign(v->xi_y, v->xi_y + v->my); s->xi[2].assign(v->xi_z, v->xi_z + v->mz);
    s->w[0].assign(v->w_x, v->w_x + v->mx); s->w[1].assign(v->w_y, v->w_y + v->my); s->w[2].assign(v->w_z, v->w_z + v->mz);
    s->solid.assign((size_t)s->ncell, 0);
    if (g->solid) for (long long c = 0; c < s->ncell; ++c) s->solid[c] = g->solid[c] ? 1 : 0;
    s->gas = *gas; s->bc = *bc;
    if (dev) { s->dev = *dev; s->stream = (cudaStream_t)dev->stream; }
    if (cudaGetDevice(&s->device) != cudaSuccess) { delete s; return fail(DVM_ECUDA, "cudaGetDevice failed"); }

    auto bail = [&](int rc) { cudaStreamSynchronize(s->stream); s->dfree_all(); delete s; return rc; };

    const int nx = s->nx, ny = s->ny, nz = s->nz;
    const long long n = s->ncell;
    // ---- geometry ----
    std::vector<double> dx(nx), dy(ny), dz(nz), idx(nx), idy(ny), idz(nz);
    for (int i = 0; i < nx; ++i) { dx[i] = s->xf[i + 1] - s->xf[i]; idx[i] = 1.0 / dx[i]; }
    for (int j = 0; j < ny; ++j) { dy[j] = s->yf[j + 1] - s->yf[j]; idy[j] = 1.0 / dy[j]; }
    for (int k = 0; k < nz; ++k) { dz[k] = s->zf[k + 1] - s->zf[k]; idz[k] = 1.0 / dz[k]; }
    // ---- cell flags, boundary-face table (order stated in dvm.h) ----
    std::vector<unsigned char> flags((size_t)n, 0), sflags((size_t)n, 0);
    std::vector<int> face_of((size_t)6 * n, -1);
    const int off[6] = {0, ny * nz, 2 * ny * nz, 2 * ny * nz + nx * nz, 2 * ny * nz + 2 * nx * nz,
                        2 * ny * nz + 2 * nx * nz + nx * ny};
    const int ndom = off[5] + nx * ny;
    std::vector<unsigned char> face_slot((size_t)ndom, 6);
    std::vector<int> face_cell((size_t)ndom, -1), face_dir((size_t)ndom, 0);
    static const int di[6] = {-1, 1, 0, 0, 0, 0}, dj[6] = {0, 0, -1, 1, 0, 0}, dk[6] = {0, 0, 0, 0, -1, 1};
    auto sol = [&](int i, int j, int k) { return s->solid[((size_t)k * ny + j) * nx + i] != 0; };
    double mass0 = 0.0;
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
        const long long c = ((long long)k * ny + j) * nx + i;
        const bool cs = sol(i, j, k);
        if (cs) { flags[c] |= FLAG_SOLID; sflags[c] |= FLAG_SOLID; }
        else mass0 += gas->rho0 * (dx[i] * dy[j] * dz[k]);
        for (int d = 0; d < 6; ++d) {
            const int ii = i + di[d], jj = j + dj[d], kk = k + dk[d];
            const bool outside = ii < 0 || ii >= nx || jj < 0 || jj >= ny || kk < 0 || kk >= nz;
            if (outside) {
                int f;
                switch (d) {
                    case 0: case 1: f = off[d] + k * ny + j; break;
                    case 2: case 3: f = off[d] + k * nx + i; break;
                    default: f = off[d] + j * nx + i; break;
                }
                face_slot[f] = (unsigned char)d; face_dir[f] = d;
                flags[c] |= (unsigned char)(1u << d);
                if (!cs) { face_cell[f] = (int)c; face_of[(size_t)d * n + c] = f; }
            } else if (sol(ii, jj, kk)) {
                flags[c] |= (unsigned char)(1u << d);
                sflags[c] |= (unsigned char)(1u << d);
                if (!cs) {
                    const int f = (int)face_slot.size();
                    face_slot.push_back(6); face_cell.push_back((int)c); face_dir.push_back(d);
                    face_of[(size_t)d * n + c] = f;
                }
            }
        }
    }
    s->nface = (int)face_slot.size();
    s->mass0 = mass0;
    // per-cell records of the padded grid for the tile kernel (static part; nu is written every iteration)
    s->nxp = nx + 2 * TILE_PAD; s->nyp = ny + 2 * TILE_PAD;
    {
        s->h_rec.resize((size_t)nz * s->nyp * s->nxp);
        for (int k = 0; k < nz; ++k) for (int jp = 0; jp < s->nyp; ++jp) for (int ip = 0; ip < s->nxp; ++ip) {
            const int i = ip - TILE_PAD, j = jp - TILE_PAD;
            const bool inside = i >= 0 && i < nx && j >= 0 && j < ny;
            const int ic = std::min(std::max(i, 0), nx - 1), jc = std::min(std::max(j, 0), ny - 1);
            const long long c = ((long long)k * ny + jc) * nx + ic;
            CellRec &r = s->h_rec[((size_t)k * s->nyp + jp) * s->nxp + ip];
            r.nu = 1.0; r.nu32 = 1.0f; r.cidx = (int)c; r.flags = REC_DEAD; r.pad = 0;
            for (int d = 0; d < 6; ++d) r.face[d] = -1;
            if (!inside || s->solid[c]) continue;
            r.flags = (int)(flags[c] & 63) | ((int)(sflags[c] & 63) << 8);
            for (int d = 0; d < 6; ++d) r.face[d] = face_of[(size_t)d * n + c];
        }
    }
    for (int d = 0; d < 6; ++d) s->foff[d] = off[d];
    // ---- 1-D factors of the ghost distributions (tile kernel): per BC slot and axis, w(xi) exp(-(xi-u)^2/T), with
    //      (pi T)^{-3/2} (and rho of a free stream) folded into the x factor; zero for zero-gradient slots ----
    s->gstride = std::max(s->mx, std::max(s->my, s->mz));
    std::vector<double> gtab((size_t)7 * 3 * s->gstride, 0.0);
    for (int b = 0; b < 7; ++b) {
        const dvm_face_bc &f = slot_bc(*bc, b);
        if (f.type == DVM_ZERO_GRADIENT) continue;
        for (int d = 0; d < 3; ++d) {
            const double pref = d == 0 ? (f.type == DVM_FREESTREAM ? f.rho : 1.0) / std::pow(PI * f.T, 1.5) : 1.0;
            for (size_t m = 0; m < s->xi[d].size(); ++m) {
                const double c1 = s->xi[d][m] - f.u[d];
                gtab[((size_t)b * 3 + d) * s->gstride + m] = pref * s->w[d][m] * std::exp(-c1 * c1 / f.T);
            }
        }
    }
    // ---- Phi_unit per (bc slot, direction) and Phi^0 per direction (oracle step 1; Eq.(9) with weights) ----
    double tab[7][6] = {}, phi0[6] = {};
    {
        long double t[7][6] = {}, p0[6] = {};
        dvm_face_bc init{};
        init.T = gas->T0; init.u[0] = gas->u0[0]; init.u[1] = gas->u0[1]; init.u[2] = gas->u0[2];
        for (int ic = 0; ic < s->mz; ++ic) for (int ib = 0; ib < s->my; ++ib) for (int ia = 0; ia < s->mx; ++ia) {
            const double xi[3] = {s->xi[0][ia], s->xi[1][ib], s->xi[2][ic]};
            const double w = s->w[0][ia] * s->w[1][ib] * s->w[2][ic];
            const double f0 = gas->rho0 * host_wall_maxwellian(init, xi);
            for (int d = 0; d < 6; ++d) {
                const double toward = xi[d / 2] * ((d & 1) ? 1.0 : -1.0);  // > 0: moving towards side d
                if (toward > 0) p0[d] += (long double)(w * toward * f0);
            }
            for (int b = 0; b < 7; ++b) {
                const dvm_face_bc &f = slot_bc(*bc, b);
                if (f.type != DVM_WALL_DIFFUSE) continue;
                const double gw = host_wall_maxwellian(f, xi);
                for (int d = 0; d < 6; ++d) {
                    const double away = xi[d / 2] * ((d & 1) ? -1.0 : 1.0);  // > 0: leaving a wall on side d
                    if (away > 0) t[b][d] += (long double)(w * away * gw);
                }
            }
        }
        for (int b = 0; b < 7; ++b) for (int d = 0; d < 6; ++d) tab[b][d] = (double)t[b][d];
        for (int d = 0; d < 6; ++d) phi0[d] = (double)p0[d];
    }
    std::vector<double> phi_unit((size_t)s->nface, 0.0), rho_w0((size_t)s->nface, 0.0);
    for (int f = 0; f < s->nface; ++f) {
        const int b = face_slot[f];
        const dvm_face_bc &fb = slot_bc(*bc, b);
        if (fb.type != DVM_WALL_DIFFUSE || face_cell[f] < 0) continue;
        phi_unit[f] = bc->wall_norm == 1 ? std::sqrt(fb.T / (4.0 * PI)) : tab[b][face_dir[f]];
        if (!(phi_unit[f] > 0.0)) { return bail(fail(DVM_EINVAL, "no velocity node leaves wall face %d", f)); }
        rho_w0[f] = phi0[face_dir[f]] / phi_unit[f];
    }
    s->h_rho_w0 = rho_w0;

    // ---- device state ----
    int rc = 0;
    rc |= upload(s, &s->d_invdx, idx.data(), nx); rc |= upload(s, &s->d_invdy, idy.data(), ny);
    rc |= upload(s, &s->d_invdz, idz.data(), nz);
    rc |= upload(s, &s->d_dx, dx.data(), nx); rc |= upload(s, &s->d_dy, dy.data(), ny); rc |= upload(s, &s->d_dz, dz.data(), nz);
    rc |= upload(s, &s->d_flags, flags.data(), (size_t)n);
    rc |= upload(s, &s->d_sflags, sflags.data(), (size_t)n);
    rc |= upload(s, &s->d_gtab, gtab.data(), gtab.size());
    rc |= upload(s, &s->d_face_of, face_of.data(), (size_t)6 * n);
    rc |= upload(s, &s->d_face_slot, face_slot.data(), (size_t)s->nface);
    rc |= upload(s, &s->d_face_cell, face_cell.data(), (size_t)s->nface);
    rc |= upload(s, &s->d_face_dir, face_dir.data(), (size_t)s->nface);
    for (int d = 0; d < 3; ++d) {
        rc |= upload(s, &s->d_xi[d], s->xi[d].data(), s->xi[d].size());
        rc |= upload(s, &s->d_w[d], s->w[d].data(), s->w[d].size());
    }
    rc |= upload(s, &s->d_phi_unit, phi_unit.data(), (size_t)s->nface);
    rc |= upload(s, &s->d_rho_w, rho_w0.data(), (size_t)s->nface);
    rc |= dzeros(s, &s->d_phi, (size_t)s->nface);
    rc |= dzeros(s, &s->d_prim_new, (size_t)NPRIM * n);
    rc |= dzeros(s, &s->d_coef, (size_t)NCOEF * n);
    rc |= dzeros(s, &s->d_raw, (size_t)16 * n);
    s->npart = (n + 255) / 256;
    rc |= dzeros(s, &s->d_part, (size_t)7 * s->npart);
    rc |= dzeros(s, &s->d_scal, 8);
    rc |= dzeros(s, &s->d_hist, (size_t)3 * HIST_CAP);
    rc |= dzeros(s, &s->d_hist_scale, (size_t)HIST_CAP);
    if (rc) return bail(rc == DVM_ENOMEM ? DVM_ENOMEM : DVM_ECUDA);
    {
        std::vector<double> prim((size_t)NPRIM * n, 0.0);
        for (long long c = 0; c < n; ++c) {
            if (s->solid[c]) continue;
            prim[c] = gas->rho0; prim[n + c] = gas->u0[0]; prim[2 * n + c] = gas->u0[1]; prim[3 * n + c] = gas->u0[2];
            prim[4 * n + c] = gas->T0;
        }
        if (upload(s, &s->d_prim, prim.data(), prim.size())) return bail(DVM_ENOMEM);
        if (cudaStreamSynchronize(s->stream) != cudaSuccess) return bail(fail(DVM_ECUDA, "upload failed"));
    }
    {
        UpdateParams U = update_params(s);
        if (launch_pack(U, s->stream) != cudaSuccess) return bail(fail(DVM_ECUDA, "pack kernel launch failed"));
        s->launches += 1;
    }
    if (cudaStreamSynchronize(s->stream) != cudaSuccess) return bail(fail(DVM_ECUDA, "initialisation failed: %s", cudaGetErrorString(cudaGetLastError())));
    *out = s;
    return DVM_OK;
}

int dvm_set_option(dvm_solver *s, int option, int value)
{
    if (!s) return fail(DVM_EINVAL, "NULL solver");
    if (option == DVM_OPT_KERNEL) {
        if (s->planned) return fail(DVM_EINVAL, "kernel variant must be chosen before the first iteration");
        if (value < DVM_KERNEL_AUTO || value > DVM_KERNEL_TILE) return fail(DVM_EINVAL, "unknown kernel variant %d", value);
        s->kernel = value;
        return DVM_OK;
    }
    if (option == DVM_OPT_TILE_RV) {
        if (s->planned) return fail(DVM_EINVAL, "the tile-kernel variant must be chosen before the first iteration");
        if (value != 0 && (value < 2 || value > 4)) return fail(DVM_EINVAL, "velocities per thread must be 0 (choose), 2, 3 or 4");
        s->tile_rv = value;
        return DVM_OK;
    }
    if (option == DVM_OPT_TILE_AXIS) {
        if (s->planned) return fail(DVM_EINVAL, "the wide axis of the tile kernel must be chosen before the first iteration");
        if (value < 0 || value > 3) return fail(DVM_EINVAL, "wide axis: 0 (choose), 1 = xi_x, 2 = xi_y, 3 = xi_z");
        s->tile_axis = value;
        return DVM_OK;
    }
    if (option == DVM_OPT_ORDER) {
        if (s->planned) return fail(DVM_EINVAL, "the order of the sweep must be chosen before the first iteration");
        if (value != 1 && value != 2) return fail(DVM_EINVAL, "the order of the upwind sweep is 1 or 2");
        s->order = value;
        return DVM_OK;
    }
    if (option == DVM_OPT_PRECISION) {
        if (s->planned) return fail(DVM_EINVAL, "the precision of the sweep must be chosen before the first iteration");
        if (value != DVM_PREC_F64 && value != DVM_PREC_MIXED) return fail(DVM_EINVAL, "precision: DVM_PREC_F64 or DVM_PREC_MIXED");
        s->precision = value;
        return DVM_OK;
    }
    if (option == DVM_OPT_SHARD_COUNT || option == DVM_OPT_SHARD_RANK) {
        if (s->planned) return fail(DVM_EINVAL, "sharding must be set before the first iteration");
        if (option == DVM_OPT_SHARD_COUNT) {
            if (value < 1) return fail(DVM_EINVAL, "shard count must be >= 1");
            s->shard_count = value;
            if (s->shard_rank >= value) s->shard_rank = 0;
        } else {
            if (value < 0 || value >= s->shard_count) return fail(DVM_EINVAL, "shard rank must be in [0, shard count)");
            s->shard_rank = value;
        }
        return DVM_OK;
    }
    if (option == DVM_OPT_MAX_CTAS) {
        if (s->planned) return fail(DVM_EINVAL, "the grid cap must be set before the first iteration");
        if (value < 0) return fail(DVM_EINVAL, "negative grid cap");
        s->max_ctas = value;
        return DVM_OK;
    }
    if (option == DVM_OPT_MAX_F_MBYTES) {
        if (s->planned) return fail(DVM_EINVAL, "the workspace cap must be set before the first iteration");
        if (value < 0) return fail(DVM_EINVAL, "negative workspace cap");
        s->max_f_mbytes = value;
        return DVM_OK;
    }
    return fail(DVM_EINVAL, "unknown option %d", option);
}

namespace {

// first half of an outer iteration: clear the accumulators, (tile kernel) rebuild the factor tables, sweep
int sweep_phase(dvm_solver *s)
{
    CK(cudaMemsetAsync(s->d_raw, 0, (size_t)16 * s->ncell * sizeof(double), s->stream));
    CK(cudaMemsetAsync(s->d_phi, 0, (size_t)s->nface * sizeof(double), s->stream));
    if (s->kernel == DVM_KERNEL_SLICE) {
        const SweepParams P = sweep_params(s);
        CK(launch_sweep_slice(P, (int)s->blocks.size(), s->nb_threads, s->stream));
    } else {
        CK(launch_tables(table_params(s), s->stream));
        s->launches += 1;
        CK(cudaMemsetAsync(s->d_counter, 0, sizeof(int), s->stream));
        // completion flags back to 0; the epoch they are compared with stays 1 (constant launch parameters: CUDA graph)
        CK(cudaMemsetAsync(s->d_done, 0, s->tile.items.size() * sizeof(int), s->stream));
        s->epoch = 1;
        const TileParams TP = tile_params(s);
        CK(launch_sweep_tile(TP, s->tile_rv, s->order, s->precision == DVM_PREC_MIXED, s->tile.ax[0], s->tile_grid, s->stream));
    }
    s->launches += 1;
    return 0;
}

// (syncs) The history slot the NEXT residual_kernel will write, read from the counter that kernel advances itself (scal[3]):
// the host's iteration count is not used to address the ring, so the two cannot drift apart.
int history_next_slot(dvm_solver *s, int *next)
{
    double v = 0.0;
    CK(cudaMemcpyAsync(&v, s->d_scal + 3, sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    if (!(v >= 0.0 && v < (double)HIST_CAP)) return fail(DVM_ECUDA, "history counter on the device is corrupt (%g)", v);
    *next = (int)v;
    return 0;
}

// second half: wall fluxes from the half-range sums (tile kernel), conversion, wall densities, rescale, residual
int update_phase(dvm_solver *s)
{
    const UpdateParams U = update_params(s);
    if (s->kernel != DVM_KERNEL_SLICE) {
        CK(launch_phi_from_raw(U, s->d_face_cell, s->d_face_dir, s->d_phi, s->order, s->stream));
        s->launches += 1;
    }
    int l = 0;
    CK(launch_update(U, HIST_CAP, s->stream, &l));
    s->launches += l;
    s->iters += 1;
    return 0;
}

}  // namespace

int dvm_iterate(dvm_solver *s, int niter)
{
    if (!s || niter < 0) return fail(DVM_EINVAL, "bad argument");
    if (niter == 0) return DVM_OK;
    if (s->shard_count > 1)
        return fail(DVM_EINVAL, "this solver holds 1 of %d velocity shards: iterate with dvm_sweep / all-reduce / dvm_update", s->shard_count);
    if (s->swept) return fail(DVM_EINVAL, "dvm_sweep without dvm_update");
    DeviceGuard guard(s->device);
    if (int rc = plan(s)) return rc;
    if (s->kernel == DVM_KERNEL_TILE && !s->graph_off && !s->graph_exec) {
        // capture one iteration (3 + 1 memsets, factor tables, sweep, wall fluxes, 5 update kernels) and replay it from now
        // on: one launch per iteration instead of twelve (configs 0 and 1 are launch-bound: 0.14 ms per iteration)
        if (const char *e = std::getenv("DVM_GRAPH")) s->graph_off = std::atoi(e) == 0;
        if (!s->graph_off) {
            const long long l0 = s->launches;
            const int it0 = s->iters;
            cudaGraph_t g = nullptr;
            // The capture runs on a stream of its own, not on the solver's: the solver's stream is very often the legacy
            // default stream (torch's current stream, dvm_device.stream = 0), which cannot be captured at all.  Nothing
            // executes during a capture, so the stream it is recorded on does not matter; the graph is launched on the
            // solver's stream.
            cudaStream_t user = s->stream, cap = nullptr;
            bool ok = cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking) == cudaSuccess;
            if (ok) {
                s->stream = cap;
                ok = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
                if (ok) {
                    const int rc1 = sweep_phase(s), rc2 = rc1 ? rc1 : update_phase(s);
                    ok = cudaStreamEndCapture(cap, &g) == cudaSuccess && rc2 == 0 && g != nullptr;
                }
                s->stream = user;
            }
            if (ok) ok = cudaGraphInstantiate(&s->graph_exec, g, 0) == cudaSuccess;
            if (g) cudaGraphDestroy(g);
            if (cap) cudaStreamDestroy(cap);
            s->graph_launches = s->launches - l0;
            s->launches = l0; s->iters = it0;           // nothing ran yet
            if (!ok) {
                // not an error of the iteration (plain launches follow), but it must not go unnoticed: dvm_graph_active() = 0
                // and the reason stays readable through dvm_last_error() until the next failing call of this thread
                const cudaError_t ce = cudaGetLastError();
                s->graph_exec = nullptr; s->graph_off = true; s->graph_failed = true;
                fail(DVM_OK, "CUDA-graph capture of the iteration failed (%s): iterating with plain kernel launches",
                     ce == cudaSuccess ? "a launch inside the capture was refused" : cudaGetErrorString(ce));
            }
        }
    }
    for (int it = 0; it < niter; ++it) {
        if (s->graph_exec) {
            CK(cudaGraphLaunch(s->graph_exec, s->stream));
            s->launches += s->graph_launches;
            s->iters += 1;
            continue;
        }
        if (int rc = sweep_phase(s)) return rc;
        if (int rc = update_phase(s)) return rc;
    }
    return DVM_OK;
}

int dvm_sweep(dvm_solver *s)
{
    if (!s) return fail(DVM_EINVAL, "NULL solver");
    if (s->swept) return fail(DVM_EINVAL, "dvm_sweep twice without dvm_update");
    DeviceGuard guard(s->device);
    if (int rc = plan(s)) return rc;
    if (s->kernel == DVM_KERNEL_SLICE) return fail(DVM_EINVAL, "dvm_sweep / dvm_update are calls of the tile kernel");
    if (int rc = sweep_phase(s)) return rc;
    s->swept = true;
    return DVM_OK;
}

int dvm_update(dvm_solver *s)
{
    if (!s) return fail(DVM_EINVAL, "NULL solver");
    if (!s->swept) return fail(DVM_EINVAL, "dvm_update without dvm_sweep");
    DeviceGuard guard(s->device);
    if (int rc = update_phase(s)) return rc;
    s->swept = false;
    return DVM_OK;
}

int dvm_reduce_buffer(dvm_solver *s, double **dev_ptr, size_t *count)
{
    if (!s || !dev_ptr || !count) return fail(DVM_EINVAL, "NULL argument");
    *dev_ptr = s->d_raw;
    *count = (size_t)16 * (size_t)s->ncell;
    return DVM_OK;
}

int dvm_moments(dvm_solver *s, double *dev_out)
{
    if (!s || !dev_out) return fail(DVM_EINVAL, "NULL argument");
    DeviceGuard guard(s->device);
    CK(cudaMemcpyAsync(dev_out, s->d_prim, (size_t)NPRIM * s->ncell * sizeof(double), cudaMemcpyDeviceToDevice, s->stream));
    return DVM_OK;
}

int dvm_residual(dvm_solver *s, double *host_out3)
{
    if (!s || !host_out3) return fail(DVM_EINVAL, "NULL argument");
    DeviceGuard guard(s->device);
    if (s->iters == 0) return fail(DVM_EINVAL, "no iteration done yet");
    int next = 0;
    if (int rc = history_next_slot(s, &next)) return rc;
    const int slot = (next + HIST_CAP - 1) % HIST_CAP;
    CK(cudaMemcpyAsync(host_out3, s->d_hist + 3 * slot, 3 * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    for (int m = 0; m < 3; ++m)
        if (!std::isfinite(host_out3[m])) return fail(DVM_ENONFINITE, "residual %d is not finite", m);
    return DVM_OK;   // (an earlier iteration's NaN stays visible in dvm_residual_history)
}

int dvm_num_faces(const dvm_solver *s) { return s ? s->nface : fail(DVM_EINVAL, "NULL solver"); }
int dvm_iterations_done(const dvm_solver *s) { return s ? s->iters : fail(DVM_EINVAL, "NULL solver"); }
int dvm_kernel_used(const dvm_solver *s) { return s ? s->kernel : fail(DVM_EINVAL, "NULL solver"); }
int dvm_tile_rv(const dvm_solver *s) { return s ? s->tile_rv : fail(DVM_EINVAL, "NULL solver"); }
int dvm_tile_axis(const dvm_solver *s) { return s ? s->tile_axis : fail(DVM_EINVAL, "NULL solver"); }
int dvm_precision(const dvm_solver *s) { return s ? s->precision : fail(DVM_EINVAL, "NULL solver"); }
long long dvm_launch_count(const dvm_solver *s) { return s ? s->launches : -1; }
int dvm_graph_active(const dvm_solver *s)
{
    if (!s) return fail(DVM_EINVAL, "NULL solver");
    return s->graph_exec ? 1 : (s->graph_failed ? 2 : 0);
}

int dvm_get_state(dvm_solver *s, double *dev_prim14, double *dev_rho_wall)
{
    if (!s) return fail(DVM_EINVAL, "NULL solver");
    DeviceGuard guard(s->device);
    if (dev_prim14) CK(cudaMemcpyAsync(dev_prim14, s->d_prim, (size_t)NPRIM * s->ncell * sizeof(double), cudaMemcpyDeviceToDevice, s->stream));
    if (dev_rho_wall) CK(cudaMemcpyAsync(dev_rho_wall, s->d_rho_w, (size_t)s->nface * sizeof(double), cudaMemcpyDeviceToDevice, s->stream));
    return DVM_OK;
}

int dvm_set_state(dvm_solver *s, const double *dev_prim8, const double *dev_rho_wall)
{
    if (!s || !dev_prim8) return fail(DVM_EINVAL, "NULL argument");
    if (s->swept) return fail(DVM_EINVAL, "dvm_sweep without dvm_update: the state cannot be replaced between the two");
    DeviceGuard guard(s->device);
    CK(cudaMemcpyAsync(s->d_prim, dev_prim8, (size_t)8 * s->ncell * sizeof(double), cudaMemcpyDeviceToDevice, s->stream));
    CK(cudaMemsetAsync(s->d_prim + 8 * s->ncell, 0, (size_t)6 * s->ncell * sizeof(double), s->stream));
    if (dev_rho_wall) CK(cudaMemcpyAsync(s->d_rho_w, dev_rho_wall, (size_t)s->nface * sizeof(double), cudaMemcpyDeviceToDevice, s->stream));
    const UpdateParams U = update_params(s);
    CK(launch_pack(U, s->stream));
    s->launches += 1;
    return DVM_OK;
}

int dvm_raw_moments(dvm_solver *s, double *dev_raw13)
{
    if (!s || !dev_raw13) return fail(DVM_EINVAL, "NULL argument");
    DeviceGuard guard(s->device);
    CK(launch_raw_export(s->d_raw, dev_raw13, s->ncell, s->stream));
    s->launches += 1;
    return DVM_OK;
}

int dvm_wall_flux(dvm_solver *s, double *dev_flux)
{
    if (!s || !dev_flux) return fail(DVM_EINVAL, "NULL argument");
    DeviceGuard guard(s->device);
    CK(cudaMemcpyAsync(dev_flux, s->d_phi, (size_t)s->nface * sizeof(double), cudaMemcpyDeviceToDevice, s->stream));
    return DVM_OK;
}

int dvm_residual_history(dvm_solver *s, double *host_out, int max_n)
{
    if (!s || !host_out || max_n < 0) return fail(DVM_EINVAL, "bad argument");
    DeviceGuard guard(s->device);
    const int count = std::min(std::min(max_n, s->iters), HIST_CAP);
    if (count > 0) {
        int next = 0;
        if (int rc = history_next_slot(s, &next)) return rc;
        const int slot = ((next - count) % HIST_CAP + HIST_CAP) % HIST_CAP;
        const int run1 = std::min(count, HIST_CAP - slot);
        CK(cudaMemcpyAsync(host_out, s->d_hist + 3 * slot, (size_t)3 * run1 * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
        if (count > run1)
            CK(cudaMemcpyAsync(host_out + 3 * run1, s->d_hist, (size_t)3 * (count - run1) * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    }
    CK(cudaStreamSynchronize(s->stream));
    return count;
}

int dvm_mass_scale(dvm_solver *s, double *host_out1)
{
    if (!s || !host_out1) return fail(DVM_EINVAL, "NULL argument");
    DeviceGuard guard(s->device);
    if (s->iters == 0) { *host_out1 = 1.0; return DVM_OK; }
    CK(cudaMemcpyAsync(host_out1, s->d_scal, sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    return DVM_OK;
}

int dvm_step_host(dvm_solver *s, const double *host_prim8, const double *host_rho_wall, int n,
                  double *host_prim14_out, double *host_rho_wall_out)
{
    if (!s || n < 0) return fail(DVM_EINVAL, "bad argument");
    // refuse before the state is touched: a sharded solver's replicated state must not change on one rank only
    if (s->shard_count > 1 && n > 0)
        return fail(DVM_EINVAL, "this solver holds 1 of %d velocity shards: iterate with dvm_sweep / all-reduce / dvm_update", s->shard_count);
    if (s->swept) return fail(DVM_EINVAL, "dvm_sweep without dvm_update: the state cannot be replaced between the two");
    DeviceGuard guard(s->device);
    if (host_prim8) {
        CK(cudaMemcpyAsync(s->d_prim, host_prim8, (size_t)8 * s->ncell * sizeof(double), cudaMemcpyHostToDevice, s->stream));
        CK(cudaMemsetAsync(s->d_prim + 8 * s->ncell, 0, (size_t)6 * s->ncell * sizeof(double), s->stream));
        const UpdateParams U = update_params(s);
        CK(launch_pack(U, s->stream));
        s->launches += 1;
    }
    if (host_rho_wall) CK(cudaMemcpyAsync(s->d_rho_w, host_rho_wall, (size_t)s->nface * sizeof(double), cudaMemcpyHostToDevice, s->stream));
    if (int rc = dvm_iterate(s, n)) return rc;
    if (host_prim14_out) CK(cudaMemcpyAsync(host_prim14_out, s->d_prim, (size_t)NPRIM * s->ncell * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    if (host_rho_wall_out) CK(cudaMemcpyAsync(host_rho_wall_out, s->d_rho_w, (size_t)s->nface * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    return DVM_OK;
}

int dvm_plan_query(int nx, int ny, int nz, const dvm_vgrid *v, int target_ctas, int max_blocks, int rv, int order, int wide_axis,
                   int *counts5, int *items9, int max_items)
{
    if (wide_axis < 0 || wide_axis > 3) return fail(DVM_EINVAL, "bad argument");
    if (!v || !counts5 || max_blocks < 0 || (rv != 0 && (rv < 2 || rv > 4)) || (order != 1 && order != 2) || (order == 2 && rv > 2) || nx <= 0 || ny <= 0 || nz <= 0 || v->mx <= 0 || v->my <= 0 || v->mz <= 0 || !v->xi_x || !v->xi_y || !v->xi_z)
        return fail(DVM_EINVAL, "bad argument");
    std::vector<double> xi[3];
    xi[0].assign(v->xi_x, v->xi_x + v->mx); xi[1].assign(v->xi_y, v->xi_y + v->my); xi[2].assign(v->xi_z, v->xi_z + v->mz);
    TilePlan tp;
    int wide = 0;
    choose_variant(xi, order, rv, wide_axis - 1, &rv, &wide);
    if (tile_plan(nx, ny, nz, xi, target_ctas, max_blocks, rv, order, wide, &tp)) return fail(DVM_EINVAL, "tile plan failed");
    counts5[0] = (int)tp.vblocks.size(); counts5[1] = tp.ntx; counts5[2] = tp.nty; counts5[3] = tp.P; counts5[4] = tp.batch;
    const int n = (int)tp.items.size();
    if (items9) {
        for (int e = 0; e < n && e < max_items; ++e) {
            const TileItem &it = tp.items[e];
            const VBlock &vb = tp.vblocks[it.vb];
            int *o = items9 + 9 * e;
            o[0] = it.vb; o[1] = it.ti; o[2] = it.tj; o[3] = it.pred_x; o[4] = it.pred_y; o[5] = it.pred_s; o[6] = it.xslot;
            o[7] = (vb.sx > 0) | ((vb.sy > 0) << 1) | ((vb.sz > 0) << 2);
            o[8] = it.fslot;
        }
    }
    return n;
}

int dvm_plan_vblocks(const dvm_vgrid *v, int rv, int order, int wide_axis, int *boxes8, int max_blocks)
{
    if (wide_axis < 0 || wide_axis > 3) return fail(DVM_EINVAL, "bad argument");
    if (!v || max_blocks < 0 || (rv != 0 && (rv < 2 || rv > 4)) || (order != 1 && order != 2) || (order == 2 && rv > 2) || v->mx <= 0 || v->my <= 0 || v->mz <= 0 || !v->xi_x || !v->xi_y || !v->xi_z)
        return fail(DVM_EINVAL, "bad argument");
    std::vector<double> xi[3];
    xi[0].assign(v->xi_x, v->xi_x + v->mx); xi[1].assign(v->xi_y, v->xi_y + v->my); xi[2].assign(v->xi_z, v->xi_z + v->mz);
    int wide = 0;
    choose_variant(xi, order, rv, wide_axis - 1, &rv, &wide);
    TilePlan tp;
    if (tile_plan(4, 4, 1, xi, 1, 0, rv, order, wide, &tp)) return fail(DVM_EINVAL, "tile plan failed");
    const int n = (int)tp.vblocks.size();
    if (boxes8)
        for (int e = 0; e < n && e < max_blocks; ++e) {
            const VBlock &b = tp.vblocks[e];
            int *o = boxes8 + 8 * e;
            // node ranges in the order xi_x, xi_y, xi_z whatever the roles are
            const int lo[3] = {b.a0, b.b0, b.c0}, cn[3] = {b.na, b.nb, b.nc};
            for (int r = 0; r < 3; ++r) { o[2 * tp.ax[r]] = lo[r]; o[2 * tp.ax[r] + 1] = cn[r]; }
            o[6] = tile_na(rv) + 65536 * (tp.ax[0] + 1); o[7] = b.nbb * 256 + b.ncb;
        }
    return n;
}

int dvm_plan_shard_vblocks(const dvm_vgrid *v, int rv, int order, int wide_axis, int shard_rank, int shard_count, int *boxes8,
                           int max_blocks)
{
    if (wide_axis < 0 || wide_axis > 3 || shard_count < 1 || shard_rank < 0 || shard_rank >= shard_count) return fail(DVM_EINVAL, "bad argument");
    if (!v || max_blocks < 0 || (rv != 0 && (rv < 2 || rv > 4)) || (order != 1 && order != 2) || (order == 2 && rv > 2) || v->mx <= 0 || v->my <= 0 || v->mz <= 0 || !v->xi_x || !v->xi_y || !v->xi_z)
        return fail(DVM_EINVAL, "bad argument");
    std::vector<double> xi[3];
    xi[0].assign(v->xi_x, v->xi_x + v->mx); xi[1].assign(v->xi_y, v->xi_y + v->my); xi[2].assign(v->xi_z, v->xi_z + v->mz);
    int wide = 0;
    choose_variant(xi, order, rv, wide_axis - 1, &rv, &wide);
    TilePlan tp;
    if (tile_plan(4, 4, 1, xi, 1, 0, rv, order, wide, &tp, shard_rank, shard_count)) return fail(DVM_EINVAL, "tile plan failed (more shards than velocity blocks?)");
    const int n = (int)tp.vblocks.size();
    if (boxes8)
        for (int e = 0; e < n && e < max_blocks; ++e) {
            const VBlock &b = tp.vblocks[e];
            int *o = boxes8 + 8 * e;
            const int lo[3] = {b.a0, b.b0, b.c0}, cn[3] = {b.na, b.nb, b.nc};
            for (int r = 0; r < 3; ++r) { o[2 * tp.ax[r]] = lo[r]; o[2 * tp.ax[r] + 1] = cn[r]; }
            o[6] = tile_na(rv) + 65536 * (tp.ax[0] + 1); o[7] = b.nbb * 256 + b.ncb;
        }
    return n;
}

int dvm_workspace_bytes(const dvm_solver *s, size_t *total, size_t *f_bytes)
{
    if (!s) return fail(DVM_EINVAL, "NULL solver");
    if (total) *total = s->total_bytes;
    if (f_bytes) *f_bytes = s->f_bytes;
    return DVM_OK;
}

int dvm_destroy(dvm_solver *s)
{
    if (!s) return DVM_OK;
    DeviceGuard guard(s->device);
    cudaStreamSynchronize(s->stream);
    if (s->graph_exec) cudaGraphExecDestroy(s->graph_exec);
    s->dfree_all();
    delete s;
    return DVM_OK;
}

}  // extern "C"
