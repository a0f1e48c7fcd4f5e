// sweep_tile.cu - DVM_KERNEL_TILE: the B200 sweep kernel of the DVM iteration (arXiv 1810.00348).
//
// What it computes is exactly Alg. 1-3 of the paper: for every discrete velocity the
// first-order upwind recurrence Eq.(7) over the whole physical grid with the Shakhov
// equilibrium Eq.(2) rebuilt on the fly, diffuse-wall / free-stream / zero-gradient ghosts
// (Eq.(8)-(9)), and the velocity sums Eq.(5) plus the wall-incident fluxes
// taken as each value is produced, so that f is never stored.  How it computes it is new:
//
//  * work item = (velocity block of 512 velocities of one sign octant) x (4 x 4 z-column of cells); a CTA of 128
//    threads owns an item, a thread owns 4 velocities (consecutive xi_x nodes) and keeps the 4 x 4 x 4 values of
//    the current z-plane in registers: x-, y- and z-upwind operands of interior cells are register operands;
//  * what is carried is g = w_alpha f_alpha (the recurrence is linear in f), so quadrature weights cost nothing;
//  * exp(-|xi-U|^2/T) and the Shakhov polynomial factorise per axis on the tensor velocity grid: tables.cu tabulates
//    one entry (E, Q, e, a) per (cell, 1-D node) once per iteration; per level the CTA receives the 16 + nbb + ncb
//    entries of its 16 cells as TMA row copies, together with the cell records (1/tau, cell index, faces);
//  * the division of Eq.(7) is MUFU.RCP64H + one cubic Newton step (3 DFMA, < 1 ulp);
//  * the 13 velocity sums use the tensor structure: 4 power sums over the thread's xi_x nodes (4 DFMA / point),
//    a lane-quad exchange over the 16 xi_x nodes of the block, then each lane expands its share of the 16
//    (power of xi_x) x (monomial of xi_y, xi_z) products and a transposing butterfly over the 8 lane groups leaves
//    one partial per lane, which goes to the [cell][16] accumulator in L2/HBM as one coalesced fp64 RED per
//    (2 cells, warp);
//  * the 4 rows of a level are a loop with rotating register slots: the level loop must fit the 32 KB instruction
//    cache (profiles/r01_ifetch_microbench.txt), the fully unrolled level did not;
//  * the x- and y-faces of the column are the only f-traffic: written with coalesced 32-byte stores per thread,
//    read back by the downwind item with TMA bulk copies (cp.async.bulk + mbarrier) two levels ahead;
//  * items are handed out by an atomic counter in dependency order (tile_plan.cu); done-flags gate their start.
//
// Product code: shares nothing with oracle/.
#include "sweep_tile.cuh"

#include <cstdint>
#include <cstdio>

namespace dvm {

namespace {

constexpr int NVB = TILE_NVB;
constexpr int NCELL = TILE_NCELL;
constexpr int RB = 4;                                  // cells of a row whose moment reductions are interleaved
constexpr int XLEVEL_DOUBLES = TILE_TY * NVB;          // one level of an x-face slot
constexpr int YLEVEL_DOUBLES = TILE_TX * NVB;          // one level of a y-face slot
constexpr unsigned XLEVEL_BYTES = XLEVEL_DOUBLES * 8u, YLEVEL_BYTES = YLEVEL_DOUBLES * 8u;

constexpr unsigned XROW_BYTES = 4 * TILE_NA * 32u;      // one 4-cell row of x entries
constexpr unsigned REC_ROW_BYTES = 4 * (unsigned)sizeof(CellRec);

struct __align__(128) TileSmem {
    // ---- staged by TMA two levels ahead (index = level parity) ----
    double xface[2][TILE_TY][NVB];                 // x-face input of the level
    double yface[2][TILE_TX][NVB];                 // y-face input
    double4 xtab[2][NCELL][TILE_NA];               // per (cell', xi_x node): E, Q, e, a   (slot r*4 + ag); cell' = row * 4 +
    double4 ytab[2][NCELL * 8];                    // position of the cell in ascending absolute x;  [cell'][nbb]
    double4 ztab[2][NCELL * 8];                    // [cell'][ncb]
    CellRec rec[2][NCELL];                         // per cell': 1/tau, cell index, neighbour flags, boundary faces
    // ---- decoded per level by 16 threads (sweep-relative cell = jj * 4 + ii) ----
    double nu[2][NCELL];                           // 1/tau (1 for dead cells)
    double4 spec[2][NCELL];                        // rho_w of a solid ghost in x, y, z (slow-path levels)
    int code[2][NCELL];                            // 1: x-up solid ghost, 2: y-up, 4: z-up, 8: dead cell
    int cidx[2][NCELL];                            // global cell index or -1 (dead)
    int dnface[2][NCELL][4];                       // wall face downwind in x, y, z (or -1); [3] = -1
    double rwb[2][8];                              // ghost densities of the domain faces: 4 x-face rows, 4 y-face columns
    // ---- per item ----
    double xi_a[TILE_NA];                          // nodes of the block (0 beyond the box)
    double xi_bc[TILE_MAXBC];
    double g[4][3][16];                            // ghost Maxwellian 1-D factors: upwind x, y, z face and solid
    unsigned long long mbar[2];
    int item;
};

// ---- PTX helpers -----------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long *b, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *b, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *b, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(b)), "r"(parity) : "memory");
}
// TMA 1-D bulk copy global -> shared, completion counted on an mbarrier
__device__ __forceinline__ void tma_load(void *dst, const void *src, unsigned bytes, unsigned long long *b)
{
#ifdef DVM_DEBUG_TMA
    if ((smem_u32(dst) & 15u) || ((unsigned long long)src & 15ull) || (bytes & 15u) || bytes == 0)
        printf("tma misaligned: dst %u src %p bytes %u (thread %d)\n", smem_u32(dst), src, bytes, (int)threadIdx.x);
#endif
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(b))
                 : "memory");
}
__device__ __forceinline__ void fence_proxy_async()
{
    asm volatile("fence.proxy.async;" ::: "memory");
}
// generic-proxy accesses to global / shared memory ordered before later async-proxy (TMA) accesses to the same space
__device__ __forceinline__ void fence_proxy_async_global()
{
    asm volatile("fence.proxy.async.global;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ int ld_acquire(const int *p)
{
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(int *p, int v)
{
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// 1/d: MUFU.RCP64H seed (about 20 bits) + one cubic Newton step: e = 1 - d y, y (1 + e + e^2); error ~ e^3
__device__ __forceinline__ double fast_rcp(double d)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(d));
    const double e = fma(-d, y, 1.0);
    const double t = fma(e, e, e);
    return fma(y, t, y);
}
__device__ __forceinline__ double shx(double v, int m) { return __shfl_xor_sync(0xffffffffu, v, m); }

// moment index (order of dvm_raw_moments) of output j of lane type q = lane & 3
//   q = 0: S0 {1, xi_y, xi_z, xi_y^2}        q = 1: S1 {1, xi_y, xi_z, xi_y^2 + xi_z^2}
//   q = 2: S0 {xi_z^2, xi_y xi_z, xi_y r2, xi_z r2}   q = 3: S2 {1, xi_y, xi_z}, S3 {1}
__constant__ int c_mom[4][4] = {{0, 2, 3, 5}, {1, 7, 8, 10}, {6, 9, 11, 12}, {4, 11, 12, 10}};

// per-item constants, uniform over the CTA
struct ItemCtx {
    int sx, sy, sz;
    int i0, j0;          // sweep-relative origin of the tile
    int upx, upy, upz;   // direction ids of the upwind sides
    int tpx, tpy, tpz;   // BC types of the upwind domain faces
    int first_x, first_y;
    int nbb, ncb;
};

__device__ __forceinline__ bool cell_of(const TileParams &P, const ItemCtx &I, int ii, int jj, int kp, int &i, int &j,
                                        int &k)
{
    const int ip = I.i0 + ii, jp = I.j0 + jj;
    i = I.sx > 0 ? ip : P.nx - 1 - ip;
    j = I.sy > 0 ? jp : P.ny - 1 - jp;
    k = I.sz > 0 ? kp : P.nz - 1 - kp;
    return ip < P.nx && jp < P.ny;
}

// ghost density of a domain face cell: rho_w of a wall, 1 for a free stream (rho_inf is folded into the factors),
// 0 for a dropped (zero-gradient) term
__device__ __forceinline__ double face_density(const TileParams &P, int type, int slot)
{
    if (type == 0) return P.rho_w[slot];
    return type == 1 ? 1.0 : 0.0;
}

// Ghost densities of the domain faces of level kp for a tile at the upwind x / y edge of the domain (one value per
// thread 32..39), loaded two levels ahead into a register and written to shared memory by rwb_store.
__device__ __forceinline__ double rwb_load(const TileParams &P, const ItemCtx &I, int kp, int tid)
{
    double v = 0.0;
    if (kp >= P.nz) return v;
    int i, j, k;
    if (tid >= 32 && tid < 32 + TILE_TY) {
        if (I.first_x && cell_of(P, I, 0, tid - 32, kp, i, j, k)) v = face_density(P, I.tpx, P.foff[I.upx] + k * P.ny + j);
    } else if (tid >= 36 && tid < 40) {
        if (I.first_y && cell_of(P, I, tid - 36, 0, kp, i, j, k)) v = face_density(P, I.tpy, P.foff[I.upy] + k * P.nx + i);
    }
    return v;
}

__device__ __forceinline__ void rwb_store(TileSmem &s, int b, int tid, double v)
{
    if (tid >= 32 && tid < 40) s.rwb[b][tid - 32] = v;
}

// TMA copies of level kp into buffer b = kp & 1: the x- / y-face input and, per 4-cell row, the x, y, z factor-table
// rows and the cell records (tables.cu; every row is one contiguous run of the padded grid).  Executed by threads
// 64..79 (one row copy each); thread 64 also posts the byte count and fetches the faces.
__device__ __forceinline__ void issue_level(const TileParams &P, const ItemCtx &I, TileSmem &s, const VBlock &vb, int kp,
                                            int tid, const double *xsrc, const double *ysrc)
{
    const int b = kp & 1, q = tid - 64;
    if (q < 0 || q >= 4 * TILE_TY) return;
    const unsigned ybytes = 4u * vb.nbb * 32u, zbytes = 4u * vb.ncb * 32u;
    if (q == 0) {
        const unsigned faces = (I.first_x ? 0u : XLEVEL_BYTES) + (I.first_y ? 0u : YLEVEL_BYTES);
        mbar_expect_tx(&s.mbar[b], faces + (unsigned)TILE_TY * (XROW_BYTES + ybytes + zbytes + REC_ROW_BYTES));
        if (!I.first_x) tma_load(&s.xface[b][0][0], xsrc + (long long)kp * XLEVEL_DOUBLES, XLEVEL_BYTES, &s.mbar[b]);
        if (!I.first_y) tma_load(&s.yface[b][0][0], ysrc + (long long)kp * YLEVEL_DOUBLES, YLEVEL_BYTES, &s.mbar[b]);
    }
    const int jj = q % TILE_TY, kind = q / TILE_TY;
    // first cell (lowest absolute x) of row jj on the padded grid; rows may lie in the dead padding
    const int jp = I.j0 + jj, ip0 = I.i0;
    const int j = I.sy > 0 ? jp : P.ny - 1 - jp;
    const int i = I.sx > 0 ? ip0 : P.nx - 4 - ip0;
    const int k = I.sz > 0 ? kp : P.nz - 1 - kp;
    const long long npc = (long long)P.nz * P.nyp * P.nxp;
    const long long pc = ((long long)k * P.nyp + (j + TILE_PAD)) * P.nxp + (i + TILE_PAD);
    if (kind == 0) tma_load(&s.xtab[b][jj * 4][0], P.TX + ((long long)vb.xb * npc + pc) * TILE_NA, XROW_BYTES, &s.mbar[b]);
    else if (kind == 1) tma_load(&s.ytab[b][jj * 4 * vb.nbb], P.TY + ((long long)vb.yb * npc + pc) * vb.nbb, ybytes, &s.mbar[b]);
    else if (kind == 2) tma_load(&s.ztab[b][jj * 4 * vb.ncb], P.TZ + ((long long)vb.zb * npc + pc) * vb.ncb, zbytes, &s.mbar[b]);
    else tma_load(&s.rec[b][jj * 4], P.rec + pc, REC_ROW_BYTES, &s.mbar[b]);
}

// Per-cell records of level kp (buffer b = kp & 1) decoded from the staged CellRec rows by threads 96..111; the caller
// has waited for the level's TMA copies.  Returns 1 if this thread saw a fluid cell with a solid upwind ghost.
__device__ __forceinline__ int decode_records(const TileParams &P, const ItemCtx &I, TileSmem &s, int kp, int tid)
{
    const int b = kp & 1;
    int special = 0;
    if (tid >= 96 && tid < 96 + NCELL) {
        const int cell = tid - 96, ii = cell & 3, jj = cell >> 2;
        const CellRec &r = s.rec[b][jj * 4 + (I.sx > 0 ? ii : 3 - ii)];
        const bool dead = r.cidx < 0;
        const int flags = r.flags & 0xff, sfl = (r.flags >> 8) & 0xff;
        int code = 8;
        double4 sp = make_double4(0.0, 0.0, 0.0, 0.0);
        int dn[3] = {-1, -1, -1};
        if (!dead) {
            code = ((sfl >> I.upx) & 1) | (((sfl >> I.upy) & 1) << 1) | (((sfl >> I.upz) & 1) << 2);
            if (code & 1) sp.x = P.rho_w[r.face[I.upx]];
            if (code & 2) sp.y = P.rho_w[r.face[I.upy]];
            if (code & 4) sp.z = P.rho_w[r.face[I.upz]];
            if ((flags >> (I.upx ^ 1)) & 1) dn[0] = r.face[I.upx ^ 1];
            if ((flags >> (I.upy ^ 1)) & 1) dn[1] = r.face[I.upy ^ 1];
            if ((flags >> (I.upz ^ 1)) & 1) dn[2] = r.face[I.upz ^ 1];
        }
        s.code[b][cell] = code;
        s.spec[b][cell] = sp;
        s.cidx[b][cell] = r.cidx;
        s.nu[b][cell] = dead ? 1.0 : r.nu;
        s.dnface[b][cell][0] = dn[0]; s.dnface[b][cell][1] = dn[1]; s.dnface[b][cell][2] = dn[2];
        s.dnface[b][cell][3] = -1;
        special = (code & 7) != 0;
    }
    return special;
}

// Ghost values of the domain faces of level kp (buffer b) for a tile at the upwind x / y edge of the domain
__device__ __forceinline__ void fill_faces(const ItemCtx &I, TileSmem &s, int b, int tid, int ag, int yidx, int zidx)
{
    if (I.first_x) {
        const double gyz = s.g[0][1][yidx] * s.g[0][2][zidx];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const double G = s.g[0][0][4 * ag + r] * gyz;
#pragma unroll
            for (int jj = 0; jj < TILE_TY; ++jj) s.xface[b][jj][tid * 4 + r] = s.rwb[b][jj] * G;
        }
    }
    if (I.first_y) {
        const double gyz = s.g[1][1][yidx] * s.g[1][2][zidx];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const double G = s.g[1][0][4 * ag + r] * gyz;
#pragma unroll
            for (int ii = 0; ii < 4; ++ii) s.yface[b][ii][tid * 4 + r] = s.rwb[b][4 + ii] * G;
        }
    }
}

// Reduction of the four power sums S_p = sum_r xi_x^p g_r of a lane over the 4 x-groups of a lane quad and the
// (xi_y, xi_z) pairs with lane bits 2 and 3 (see the header comment), for N cells at once, stage by stage, so that
// the shuffle latency of one cell is covered by the other cells' instructions.  Leaves, in every lane, the partial
// sum over its half-warp of one of the 16 products of the cell; lane & 15 names it (c_mom).  S[c][p] = power sum p of cell c; k[c] = result of cell c.
template <int N>
__device__ __forceinline__ void reduce_halfN(const double (&S)[N][4], const double (&cf)[4], const int vsel, int lane,
                                             double (&k)[N])
{
    const bool b0 = lane & 1, b1 = lane & 2;
    double a0[N], u[N], v[N];
#pragma unroll
    for (int c = 0; c < N; ++c) a0[c] = S[c][0] + shx(S[c][0], 1);
#pragma unroll
    for (int c = 0; c < N; ++c) u[c] = (b1 ? S[c][2] : S[c][1]) + shx(b1 ? S[c][1] : S[c][2], 2);
#pragma unroll
    for (int c = 0; c < N; ++c) v[c] = S[c][3] + shx(b1 ? 0.0 : S[c][3], 2);
#pragma unroll
    for (int c = 0; c < N; ++c) a0[c] += shx(a0[c], 2);
#pragma unroll
    for (int c = 0; c < N; ++c) u[c] += shx(u[c], 1);
#pragma unroll
    for (int c = 0; c < N; ++c) v[c] += shx(v[c], 1);
    // Pair stage without selects between the shuffles: the lane with pair bits m = 2 b2 + b3 keeps its four products in
    // the order r_k = o_(k xor m) (cf is stored permuted), so that both exchange steps send fixed registers; only the
    // operand of the S3 product (lane role 3, product 3, register 3 xor m: bit k of vsel) is chosen per register.
    const bool s0 = vsel & 1, s1 = vsel & 2, s2 = vsel & 4, s3 = vsel & 8;
    double r0[N], r1[N];
#pragma unroll
    for (int c = 0; c < N; ++c) {
        const double U = b0 ? u[c] : a0[c];
        const double p0 = cf[0] * (s0 ? v[c] : U), p1 = cf[1] * (s1 ? v[c] : U);
        const double p2 = cf[2] * (s2 ? v[c] : U), p3 = cf[3] * (s3 ? v[c] : U);
        r0[c] = p0 + shx(p2, 4);
        r1[c] = p1 + shx(p3, 4);
    }
#pragma unroll
    for (int c = 0; c < N; ++c) k[c] = r0[c] + shx(r1[c], 8);
}

// per-thread constants of an item
struct ThreadCtx {
    double X1[4], X2[4], X3[4];  // xi_x, xi_x^2, xi_x^3 of the thread's nodes
    double cf[4];                // expansion coefficients of this lane, in the order cf[k] = c[k xor m] (reduce_halfN)
    int vsel;                    // bit k: product k of this lane takes the S3 sum
    double dsgn;                 // sign of the wall-flux contribution of this lane
    double *rawm;                // raw16 + moment slot of this lane
    int ag, yi, zi;              // xi_x group, rows of the thread's xi_y and xi_z nodes in xi_bc / g
    int yl, zl, nbb, ncb;        // local xi_y / xi_z index in the block, block shape
    int xrev;                    // 3 if the sweep runs against x (table rows are in ascending absolute x), else 0
    int dsel;                    // wall-flux direction (3 = none) of this lane
};

// velocity sums of two cells (A: lower half-warp keeps it, B: upper half-warp) -> accumulators, one RED per lane
__device__ __forceinline__ void emit_pair(const TileParams &P, TileSmem &s, const int b, const int cellA, double kA, double kB,
                                          const ThreadCtx &T, const int lane)
{
    const bool hi = lane & 16;
    const double keep = hi ? kB : kA, send = hi ? kA : kB;
    const double tot = keep + shx(send, 16);
    const int cell = cellA + (hi ? 1 : 0);
    const int c = s.cidx[b][cell];
    if (c >= 0) {
        atomicAdd(T.rawm + (long long)c * 16, tot);
        const int f = s.dnface[b][cell][T.dsel];
        if (f >= 0) atomicAdd(P.phi + f, T.dsgn * tot);
    }
}

// One level of the column, fast path (no solid ghost in the level): 4 rows x 4 cells x 4 velocities per thread,
// fully unrolled so that the plane lives in registers.  Dead cells (outside the domain / solid) have all-zero table
// entries and nu = 1, so they produce g = 0 by the same arithmetic.
__device__ __forceinline__ void compute_level(const TileParams &P, TileSmem &s, const int b, double (&pl)[TILE_TY][4][4],
                                              const ThreadCtx &T, const int tid, const int lane, double *xout,
                                              double *yout)
{
    // The 4 rows of the tile are a real loop: the B200 instruction cache holds 32 KB, and a level loop larger than
    // that is fetch-bound at 1/3 instruction per clock and scheduler (profiles/r01_ifetch_microbench.txt); the
    // fully unrolled level was 48 KB.  The plane stays in registers with static indices: every iteration works on
    // row slot 0 (old values of row jj -> new values) with the new row jj - 1 in slot 3, then the slots rotate.
    // y-upwind operands of the row: the staged y-face for the first row, then the row just computed
    double yu[4][4];
#pragma unroll
    for (int ii = 0; ii < 4; ++ii) {
        const double2 *p = reinterpret_cast<const double2 *>(&s.yface[b][ii][tid * 4]);
        const double2 v0 = p[0], v1 = p[1];
        yu[ii][0] = v0.x; yu[ii][1] = v0.y; yu[ii][2] = v1.x; yu[ii][3] = v1.y;
    }
#pragma unroll 1
    for (int jj = 0; jj < TILE_TY; ++jj) {
        double fx[4];
        {
            const double2 *p = reinterpret_cast<const double2 *>(&s.xface[b][jj][tid * 4]);
            const double2 v0 = p[0], v1 = p[1];
            fx[0] = v0.x; fx[1] = v0.y; fx[2] = v1.x; fx[3] = v1.y;
        }
        double SR[RB][4];
#pragma unroll
        for (int ii = 0; ii < 4; ++ii) {
            const int cell = jj * 4 + ii;
            const int cp = jj * 4 + (ii ^ T.xrev);   // position of the cell in the staged table rows
            const double4 yt = s.ytab[b][cp * T.nbb + T.yl];
            const double4 zt = s.ztab[b][cp * T.ncb + T.zl];
            const double Eyz = yt.x * zt.x, Qyz = yt.y + zt.y, eyz = yt.z + zt.z;
            const double ay = yt.w, az = zt.w;
            const double dyz = (ay + az) + s.nu[b][cell];
            double S0 = 0.0, S1 = 0.0, S2 = 0.0, S3 = 0.0;
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const double4 xt = s.xtab[b][cp][r * 4 + T.ag];
                const double src = (xt.x * Eyz) * fma(xt.y + Qyz, xt.z + eyz, 1.0);
                const double inv = fast_rcp(xt.w + dyz);
                double num = fma(ay, yu[ii][r], src);
                num = fma(az, pl[0][ii][r], num);
                num = fma(xt.w, fx[r], num);
                const double gg = num * inv;
                fx[r] = gg;
                pl[0][ii][r] = gg;
                yu[ii][r] = gg;
                S0 += gg;
                S1 = fma(T.X1[r], gg, S1);
                S2 = fma(T.X2[r], gg, S2);
                S3 = fma(T.X3[r], gg, S3);
            }
            SR[ii % RB][0] = S0; SR[ii % RB][1] = S1; SR[ii % RB][2] = S2; SR[ii % RB][3] = S3;
            if (ii % RB == RB - 1) {
                double k[RB];
                reduce_halfN<RB>(SR, T.cf, T.vsel, lane, k);
#pragma unroll
                for (int c = 0; c < RB; c += 2) emit_pair(P, s, b, cell - (RB - 1) + c, k[c], k[c + 1], T, lane);
            }
        }
        if (xout) {
            double2 *p = reinterpret_cast<double2 *>(xout + jj * NVB + tid * 4);
            p[0] = make_double2(fx[0], fx[1]);
            p[1] = make_double2(fx[2], fx[3]);
        }
        // rotate the row slots: (0, 1, 2, 3) <- (1, 2, 3, 0); after the 4th iteration the rows are back in place
#pragma unroll
        for (int ii = 0; ii < 4; ++ii)
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const double t = pl[0][ii][r];
#pragma unroll
                for (int q = 0; q + 1 < TILE_TY; ++q) pl[q][ii][r] = pl[q + 1][ii][r];
                pl[TILE_TY - 1][ii][r] = t;
            }
    }
    if (yout) {
#pragma unroll
        for (int ii = 0; ii < 4; ++ii) {
            double2 *p = reinterpret_cast<double2 *>(yout + ii * NVB + tid * 4);
            p[0] = make_double2(pl[TILE_TY - 1][ii][0], pl[TILE_TY - 1][ii][1]);
            p[1] = make_double2(pl[TILE_TY - 1][ii][2], pl[TILE_TY - 1][ii][3]);
        }
    }
}

// One level that holds a solid ghost (a fluid cell whose upwind neighbour is a masked cell): the same arithmetic
// written as compact loops over a copy of the plane in local memory.  Rare (the surface of a masked body), so its
// speed does not matter; keeping it out of the unrolled path halves the code the instruction cache has to hold.
__device__ __forceinline__ void compute_level_slow(const TileParams &P, TileSmem &s, const int b, double *pl,
                                                   const ThreadCtx &T, const int tid, const int lane, double *xout,
                                                   double *yout)
{
    const double gyz = s.g[3][1][T.yi] * s.g[3][2][T.zi];
#pragma unroll 1
    for (int jj = 0; jj < TILE_TY; ++jj) {
        double fx[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) fx[r] = s.xface[b][jj][tid * 4 + r];
        double kprev = 0.0;
#pragma unroll 1
        for (int ii = 0; ii < 4; ++ii) {
            const int cell = jj * 4 + ii;
            const int cp = jj * 4 + (ii ^ T.xrev);   // position of the cell in the staged table rows
            const double4 yt = s.ytab[b][cp * T.nbb + T.yl];
            const double4 zt = s.ztab[b][cp * T.ncb + T.zl];
            const double Eyz = yt.x * zt.x, Qyz = yt.y + zt.y, eyz = yt.z + zt.z;
            const double ay = yt.w, az = zt.w;
            const double dyz = (ay + az) + s.nu[b][cell];
            const int code = s.code[b][cell];
            const double4 sp = s.spec[b][cell];
            double S0 = 0.0, S1 = 0.0, S2 = 0.0, S3 = 0.0;
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const double Pg = s.g[3][0][4 * T.ag + r] * gyz;
                const double4 xt = s.xtab[b][cp][r * 4 + T.ag];
                double xu = fx[r], zu = pl[cell * 4 + r];
                double yu = jj == 0 ? s.yface[b][ii][tid * 4 + r] : pl[(cell - 4) * 4 + r];
                if (code & 1) xu = sp.x * Pg;
                if (code & 2) yu = sp.y * Pg;
                if (code & 4) zu = sp.z * Pg;
                const double src = (xt.x * Eyz) * fma(xt.y + Qyz, xt.z + eyz, 1.0);
                const double inv = fast_rcp(xt.w + dyz);
                double num = fma(ay, yu, src);
                num = fma(az, zu, num);
                num = fma(xt.w, xu, num);
                double gg = num * inv;
                if (code & 8) gg = 0.0;
                fx[r] = gg;
                pl[cell * 4 + r] = gg;
                S0 += gg;
                S1 = fma(T.X1[r], gg, S1);
                S2 = fma(T.X2[r], gg, S2);
                S3 = fma(T.X3[r], gg, S3);
            }
            const double S1c[1][4] = {{S0, S1, S2, S3}};
            double k1[1];
            reduce_halfN<1>(S1c, T.cf, T.vsel, lane, k1);
            const double kk = k1[0];
            if (ii & 1) emit_pair(P, s, b, cell - 1, kprev, kk, T, lane);
            else kprev = kk;
        }
        if (xout) {
#pragma unroll
            for (int r = 0; r < 4; ++r) xout[jj * NVB + tid * 4 + r] = fx[r];
        }
    }
    if (yout) {
#pragma unroll 1
        for (int ii = 0; ii < 4; ++ii)
#pragma unroll
            for (int r = 0; r < 4; ++r) yout[ii * NVB + tid * 4 + r] = pl[((TILE_TY - 1) * 4 + ii) * 4 + r];
    }
}

__global__ void __launch_bounds__(TILE_THREADS, TILE_MIN_CTAS) sweep_tile_kernel(const TileParams P)
{
    // dynamic shared memory starts at offset 0 of the CTA's window (no static __shared__ in this kernel), so the
    // 128-byte alignment holds; casting without pointer arithmetic keeps the address space visible (LDS / STS)
    extern __shared__ __align__(128) unsigned char smem_raw[];
    TileSmem &s = *reinterpret_cast<TileSmem *>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) {
        mbar_init(&s.mbar[0], 1);
        mbar_init(&s.mbar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_proxy_async();
    }
    __syncthreads();
    unsigned par[2] = {0u, 0u};

    for (;;) {
        // ---- next item (dependency order), wait for its upwind items ----
        if (tid == 0) {
            const int n = atomicAdd(P.counter, 1);
            s.item = n;
            if (n < P.nitems) {
                const TileItem it = P.items[n];
                const int pred[3] = {it.pred_x, it.pred_y, it.pred_s};
#pragma unroll
                for (int q = 0; q < 3; ++q)
                    if (pred[q] >= 0)
                        while (ld_acquire(P.done + pred[q]) != P.epoch) __nanosleep(64);
            }
        }
        __syncthreads();
        // every thread reads the same value; the lane-0 broadcast tells the compiler it is warp-uniform
        const int n = __shfl_sync(0xffffffffu, s.item, 0);
        if (n >= P.nitems) break;
        const TileItem it = P.items[n];
        const VBlock vb = P.vblocks[it.vb];
        ItemCtx I;
        I.sx = vb.sx; I.sy = vb.sy; I.sz = vb.sz;
        I.i0 = it.ti * TILE_TX; I.j0 = it.tj * TILE_TY;
        I.upx = vb.sx > 0 ? 0 : 1; I.upy = vb.sy > 0 ? 2 : 3; I.upz = vb.sz > 0 ? 4 : 5;
        I.tpx = P.bc_type[I.upx]; I.tpy = P.bc_type[I.upy]; I.tpz = P.bc_type[I.upz];
        I.first_x = it.ti == 0; I.first_y = it.tj == 0;
        I.nbb = vb.nbb; I.ncb = vb.ncb;
        double *xdst = P.xface + ((long long)(it.vb % P.batch) * P.P + it.xslot) * P.xslot_doubles;
        double *ydst = P.yface + ((long long)(it.vb % P.batch) * P.ntx + it.ti) * P.yslot_doubles;

        // ---- TMA copies of levels 0 and 1 (the staging buffers are free: every thread passed the end-of-item
        //      barrier; the upwind items' face stores were made with the generic proxy) ----
        if (tid >= 64 && tid < 64 + 4 * TILE_TY) {
            fence_proxy_async_global();
            issue_level(P, I, s, vb, 0, tid, xdst, ydst);
            if (P.nz > 1) issue_level(P, I, s, vb, 1, tid, xdst, ydst);
        }
        // ---- per-item tables: nodes, ghost factors; ghost densities of the domain faces of levels 0 and 1 ----
        {
            const int slotid[4] = {I.upx, I.upy, I.upz, 6};
            if (tid < 16) {
                const bool ok = tid < vb.na;
                const int idx = vb.a0 + tid;
                s.xi_a[tid] = ok ? P.xi_x[idx] : 0.0;
#pragma unroll
                for (int f = 0; f < 4; ++f) s.g[f][0][tid] = ok ? P.gtab[(long long)(slotid[f] * 3 + 0) * P.gstride + idx] : 0.0;
            } else if (tid < 16 + vb.nbb) {
                const int bl = tid - 16;
                const bool ok = bl < vb.nb;
                const int idx = vb.b0 + bl;
                s.xi_bc[bl] = ok ? P.xi_y[idx] : 0.0;
#pragma unroll
                for (int f = 0; f < 4; ++f) s.g[f][1][bl] = ok ? P.gtab[(long long)(slotid[f] * 3 + 1) * P.gstride + idx] : 0.0;
            } else if (tid >= 32 && tid < 32 + vb.ncb) {
                const int cl = tid - 32;
                const bool ok = cl < vb.nc;
                const int idx = vb.c0 + cl;
                s.xi_bc[vb.nbb + cl] = ok ? P.xi_z[idx] : 0.0;
#pragma unroll
                for (int f = 0; f < 4; ++f)
                    s.g[f][2][vb.nbb + cl] = ok ? P.gtab[(long long)(slotid[f] * 3 + 2) * P.gstride + idx] : 0.0;
            }
            rwb_store(s, 0, tid, rwb_load(P, I, 0, tid));
            rwb_store(s, 1, tid, rwb_load(P, I, 1, tid));
        }
        __syncthreads();

        ThreadCtx T;
        T.ag = lane & 3;
        T.nbb = vb.nbb; T.ncb = vb.ncb;
        T.xrev = vb.sx > 0 ? 0 : 3;
        {
            const int pair = warp * 8 + (lane >> 2);
            T.yl = pair % vb.nbb; T.zl = pair / vb.nbb;
            T.yi = T.yl;
            T.zi = vb.nbb + T.zl;
            const double xb = s.xi_bc[T.yi], xc = s.xi_bc[T.zi], r2 = xb * xb + xc * xc;
            const int q = lane & 3, j = ((lane >> 2) & 1) * 2 + ((lane >> 3) & 1);
            double cq[4];
            if (q == 0) { cq[0] = 1.0; cq[1] = xb; cq[2] = xc; cq[3] = xb * xb; }
            else if (q == 1) { cq[0] = 1.0; cq[1] = xb; cq[2] = xc; cq[3] = r2; }
            else if (q == 2) { cq[0] = xc * xc; cq[1] = xb * xc; cq[2] = xb * r2; cq[3] = xc * r2; }
            else { cq[0] = 1.0; cq[1] = xb; cq[2] = xc; cq[3] = 1.0; }
#pragma unroll
            for (int k = 0; k < 4; ++k) {   // static indices only: cf[k] = cq[k ^ j]
                T.cf[k] = j == 0 ? cq[k] : j == 1 ? cq[k ^ 1] : j == 2 ? cq[k ^ 2] : cq[k ^ 3];
            }
            T.vsel = q == 3 ? 1 << (3 ^ j) : 0;
            T.rawm = P.raw16 + c_mom[q][j];
            T.dsel = 3; T.dsgn = 0.0;
            if (q == 1 && j == 0) { T.dsel = 0; T.dsgn = (double)vb.sx; }
            if (q == 0 && j == 1) { T.dsel = 1; T.dsgn = (double)vb.sy; }
            if (q == 0 && j == 2) { T.dsel = 2; T.dsgn = (double)vb.sz; }
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const double x = s.xi_a[4 * T.ag + r];
                T.X1[r] = x; T.X2[r] = x * x; T.X3[r] = x * x * x;
            }
        }

        // records and boundary faces of level 0 (its copies were issued above; the wait does not consume the phase)
        int special = 0;
        if (tid >= 96 && tid < 96 + NCELL) {
            mbar_wait(&s.mbar[0], par[0]);
            special = decode_records(P, I, s, 0, tid);
        }
        fill_faces(I, s, 0, tid, T.ag, T.yi, T.zi);
        // plane = ghost of the upwind z face of the domain
        double pl[TILE_TY][4][4];
        {
            const double gyz = s.g[2][1][T.yi] * s.g[2][2][T.zi];
            double G[4];
#pragma unroll
            for (int r = 0; r < 4; ++r) G[r] = s.g[2][0][4 * T.ag + r] * gyz;
#pragma unroll
            for (int jj = 0; jj < TILE_TY; ++jj)
#pragma unroll
                for (int ii = 0; ii < 4; ++ii) {
                    int i, j, k;
                    double rw = 0.0;
                    if (cell_of(P, I, ii, jj, 0, i, j, k)) rw = face_density(P, I.tpz, P.foff[I.upz] + j * P.nx + i);
#pragma unroll
                    for (int r = 0; r < 4; ++r) pl[jj][ii][r] = rw * G[r];
                }
        }
        special = __shfl_sync(0xffffffffu, __syncthreads_or(special), 0);

        const bool write_x = it.ti < P.ntx - 1, write_y = it.tj < P.nty - 1;

        for (int kp = 0; kp < P.nz; ++kp) {
            const int b = kp & 1;
            const double vrw = rwb_load(P, I, kp + 2, tid);
            mbar_wait(&s.mbar[b], par[b]);
            par[b] ^= 1u;
            double *xout = write_x ? xdst + (long long)kp * XLEVEL_DOUBLES : nullptr;
            double *yout = write_y ? ydst + (long long)kp * YLEVEL_DOUBLES : nullptr;
            if (special) {
                double tmp[NCELL * 4];
#pragma unroll
                for (int c = 0; c < NCELL; ++c)
#pragma unroll
                    for (int r = 0; r < 4; ++r) tmp[c * 4 + r] = pl[c >> 2][c & 3][r];
                compute_level_slow(P, s, b, tmp, T, tid, lane, xout, yout);
#pragma unroll
                for (int c = 0; c < NCELL; ++c)
#pragma unroll
                    for (int r = 0; r < 4; ++r) pl[c >> 2][c & 3][r] = tmp[c * 4 + r];
            } else {
                compute_level(P, s, b, pl, T, tid, lane, xout, yout);
            }
            rwb_store(s, b, tid, vrw);
            int sp = 0;
            if (kp + 1 < P.nz) {
                if (tid >= 96 && tid < 96 + NCELL) {
                    mbar_wait(&s.mbar[b ^ 1], par[b ^ 1]);   // level kp + 1 has landed (issued a level ago)
                    sp = decode_records(P, I, s, kp + 1, tid);
                }
                fill_faces(I, s, b ^ 1, tid, T.ag, T.yi, T.zi);
            }
            special = __shfl_sync(0xffffffffu, __syncthreads_or(sp), 0);
            if (tid >= 64 && tid < 64 + 4 * TILE_TY && kp + 2 < P.nz) {
                fence_proxy_async_smem();  // this level's reads of the staging buffers before the TMA overwrites them
                issue_level(P, I, s, vb, kp + 2, tid, xdst, ydst);
            }
        }
        // ---- publish: faces of this item are complete ----
        __threadfence();
        __syncthreads();
        if (tid == 0) st_release(P.done + n, P.epoch);
    }
}

}  // namespace

size_t tile_smem_bytes() { return sizeof(TileSmem); }

cudaError_t tile_configure(int *ctas_per_sm)
{
    cudaError_t e = cudaFuncSetAttribute(sweep_tile_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tile_smem_bytes());
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, sweep_tile_kernel, TILE_THREADS, tile_smem_bytes());
}

cudaError_t launch_sweep_tile(const TileParams &P, int grid, cudaStream_t st)
{
    sweep_tile_kernel<<<grid, TILE_THREADS, tile_smem_bytes(), st>>>(P);
    return cudaGetLastError();
}

}  // namespace dvm
