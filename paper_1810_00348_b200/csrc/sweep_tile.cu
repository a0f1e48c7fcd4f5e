// sweep_tile.cu - DVM_KERNEL_TILE: the B200 sweep kernel of the DVM iteration (arXiv 1810.00348).
//
// What it computes is exactly Alg. 1-3 of the paper: for every discrete velocity the
// first-order upwind recurrence Eq.(7) over the whole physical grid with the Shakhov
// equilibrium Eq.(2) rebuilt on the fly, diffuse-wall / free-stream / zero-gradient ghosts
// (Eq.(8)-(9)), and the velocity sums Eq.(5) plus the wall-incident fluxes
// taken as each value is produced, so that f is never stored.  How it computes it is new:
//
//  * work item = (velocity block of 512 velocities of one sign octant) x (4 x 4 z-column of cells); a CTA owns an
//    item, a thread owns RV velocities (consecutive xi_x nodes) and keeps their 4 x 4 values of the current z-plane
//    in registers: x-, y- and z-upwind operands of interior cells are register operands.  Variants: RV = 4 (128
//    threads, blocks of 16 x 32 nodes, 8 warps per SM), RV = 3 (128 threads, blocks of 12 x 32 nodes: fills 24-node sign
//    halves), RV = 2 (256 threads, blocks of 8 x 64 nodes, 16 warps per SM), and RV = 2 at order 2 (128 threads);
//  * what is carried is g = w_alpha f_alpha (the recurrence is linear in f), so quadrature weights cost nothing;
//  * exp(-|xi-U|^2/T) and the Shakhov polynomial factorise per axis on the tensor velocity grid: tables.cu tabulates
//    one entry (E, Q, e, a) per (cell, 1-D node) once per iteration; per level the CTA receives the entries of its
//    16 cells as TMA row copies, together with the cell records (1/tau, cell index, faces);
//  * the cell value is written as g = (a_x g_xup + N) / den, so that the recurrence along x is one fp64 FMA and one
//    multiplication per value and everything else (N: source term + y- and z-upwind terms; 1 / den by MUFU.RCP64H + one
//    cubic Newton step) is independent work, done for the RV nodes of a thread in lock step;
//  * the 13 velocity sums are two small matrix products on the fp64 tensor cores (mma.sync m8n8k4 = SASS DMMA, a
//    pipe of its own beside the fp64 FMA pipe): powers of xi_x times the values over the lane quad, then monomials
//    of (xi_y, xi_z) over the 8 pairs of a warp; results go to the [cell][16] accumulator in L2 / HBM as fp64 REDs;
//  * the x- and y-faces of the column are the only f-traffic: written with ordered 16-byte stores,
//    read back by the downwind item with TMA bulk copies (cp.async.bulk + mbarrier) two levels ahead;
//  * items are handed out by an atomic counter in dependency order (tile_plan.cu); done-flags gate their start.
//
//  * R = the type f is carried in: double, or float for DVM_OPT_PRECISION = DVM_PREC_MIXED (the paper's timing precision,
//    PAPER.md:313; reading G22): factor tables, faces, the plane in registers and the arithmetic of Eq.(7) are then
//    IEEE single, the velocity sums (DMMA operands, accumulator, REDs) stay double.
//
// Product code: shares nothing with oracle/.
#include "sweep_tile.cuh"

#include <cstddef>
#include <cstdint>
#include <cstdio>

namespace dvm {

namespace {

constexpr int NCELL = TILE_NCELL;
constexpr int GA = TILE_GA;
constexpr unsigned REC_ROW_BYTES = 4 * (unsigned)sizeof(CellRec);

// vector types of the carried type
template <typename R> struct Vec;
template <> struct Vec<double> { using v2 = double2; using v4 = double4; };
template <> struct Vec<float> { using v2 = float2; using v4 = float4; };

// Kernel variant: RV velocities per thread, ORD = order of the upwind sweep, R = type f is carried in (sweep_tile.cuh)
template <int RV, int ORD, typename R>
struct KC {
    static constexpr int THREADS = (ORD == 2 || RV >= 3) ? 128 : 256;
    static constexpr int WARPS = THREADS / 32;
    static constexpr int NVB = THREADS * RV;                 // velocities per block
    static constexpr int ES = (ORD == 2 ? 6 : 4) * (int)sizeof(R);   // bytes of a factor-table entry
    static constexpr int LAYERS = ORD;                       // upwind values per direction carried through a face
    static constexpr int XLEVEL_VALUES = LAYERS * TILE_TY * NVB;   // one level of an x-face slot
    static constexpr int YLEVEL_VALUES = LAYERS * TILE_TX * NVB;   // one level of a y-face slot
    static constexpr unsigned XLEVEL_BYTES = XLEVEL_VALUES * (unsigned)sizeof(R), YLEVEL_BYTES = YLEVEL_VALUES * (unsigned)sizeof(R);
    // resident CTAs per SM the kernel is compiled for: the double plane takes 128 registers of a thread (2 CTAs of 128
    // threads x 255 registers), the single plane half of that
    static constexpr int MIN_CTAS = sizeof(R) == 4 ? DVM_TILE_F32_CTAS : 2;
};

// One TMA bulk copy per level: source of level 0, byte step per level, destination in a LevelBuf; bytes = 0: skipped.
struct CopyDesc {
    const unsigned char *src;
    long long step;
    unsigned dst, bytes;
    unsigned pad[2];
};
constexpr int NCOPY = 4 * TILE_TY + 2;              // per row: x, y, z factor rows and cell records; x-face and y-face input

// One tile row (4 cells along x) of one level: everything the row's arithmetic reads sits at a static offset from the
// row's base address, whatever the row index and the level parity are.
template <int RV, int ORD, typename R>
struct __align__(128) RowBuf {
    // ---- staged by TMA two levels ahead ----
    alignas(16) unsigned char xtab[4 * GA * RV * KC<RV, ORD, R>::ES];   // per (cell', xi_x node): E, Q, e, a [order 2: E, Q, e, cd, c1,
    alignas(16) unsigned char ytab[4 * 8 * KC<RV, ORD, R>::ES];         // c2] (slot r*4 + ag); cell' = position of the cell in ascending
    alignas(16) unsigned char ztab[4 * 8 * KC<RV, ORD, R>::ES];         // absolute x;  y: [cell'][nbb], z: [cell'][ncb]
    CellRec rec[4];                                // per cell': 1/tau, accumulator row, neighbour flags, boundary faces
    // ---- decoded by 16 threads on levels that hold a solid ghost (slow path; sweep-relative cell ii) ----
    double4 spec[4];                               // rho_w of a solid ghost in x, y, z
    int code[4];                                   // 1: x-up solid ghost, 2: y-up, 4: z-up, 8: dead cell
};

template <int RV, int ORD, typename R>
struct __align__(128) LevelBuf {
    RowBuf<RV, ORD, R> row[TILE_TY];
    alignas(16) R xface[KC<RV, ORD, R>::LAYERS][TILE_TY][KC<RV, ORD, R>::NVB];   // x-face input of the level (layer 0: nearest upwind cell)
    alignas(16) R yface[KC<RV, ORD, R>::LAYERS][TILE_TX][KC<RV, ORD, R>::NVB];   // y-face input of the level
    double rwb[8];                                 // ghost densities of the domain faces: 4 x-face rows, 4 y-face columns
};

template <int RV, int ORD, typename R>
struct __align__(128) TileSmem {
    LevelBuf<RV, ORD, R> lv[2];                            // index = level parity
    // ---- per item ----
    double xi_a[16];                               // nodes of the block (0 beyond the box)
    double xi_bc[TILE_MAXBC];
    double g[4][3][16];                            // ghost Maxwellian 1-D factors: upwind x, y, z face and solid
    CopyDesc desc[NCOPY];                          // the TMA copies of one level of this item (issue_level)
    unsigned long long mbar[2];
    unsigned txbytes;                              // bytes the copies of one level deliver
    int item;
    int special[2];                                // the level in buffer b holds a fluid cell with a solid upwind ghost
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
__device__ __forceinline__ float fast_rcp(float d)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(d));   // MUFU.RCP: 1 ulp
    return y;
}
// MUFU seed of 1 / d in the carried type
__device__ __forceinline__ double rcp_seed(double d)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(d));
    return y;
}
__device__ __forceinline__ float rcp_seed(float d) { return fast_rcp(d); }
// Global REDs and face stores are volatile asm statements: they keep their program order, so ptxas cannot sink the
// stores of a whole level to its end, where the burst would stall the warp on the load/store unit.
__device__ __forceinline__ void red_f64(double *addr, double v)
{
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(addr), "d"(v));
}
__device__ __forceinline__ void st_f64x2(double *addr, double a, double b)
{
    asm volatile("st.global.v2.f64 [%0], {%1, %2};" ::"l"(addr), "d"(a), "d"(b));
}
__device__ __forceinline__ void st_f64(double *addr, double a)
{
    asm volatile("st.global.f64 [%0], %1;" ::"l"(addr), "d"(a));
}
__device__ __forceinline__ void st_f32x4(float *addr, float a, float b, float c, float d)
{
    asm volatile("st.global.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(d));
}
__device__ __forceinline__ void st_f32x2(float *addr, float a, float b)
{
    asm volatile("st.global.v2.f32 [%0], {%1, %2};" ::"l"(addr), "f"(a), "f"(b));
}
__device__ __forceinline__ void st_f32(float *addr, float a)
{
    asm volatile("st.global.f32 [%0], %1;" ::"l"(addr), "f"(a));
}

// Lane <-> velocity mapping.  The fp64 MMA contracts over lane & 3, and stage 1 of the velocity sums contracts over the
// xi_x groups, so the MMA wants the value of (xi_x group ag, pair n) in lane 4 n + ag, and by default the thread in that lane
// owns that velocity.  A 128-bit shared-memory load whose address is shared by NON-adjacent lanes costs 4 wavefronts whatever
// the number of distinct addresses (1 - 2 when ADJACENT lanes share it; micro-benchmark in profiles/r02_sweep_tile.md), and the
// entries of the xi_x table - 3/4 of the shared-memory wavefronts - are shared by the lanes of one xi_x group.
// -DDVM_TILE_XPOSE=1 gives the thread in lane l the velocity (ag = l >> 3, pair = l & 7) instead - the 8 lanes of a group are
// adjacent - and hands every new value to the lane the MMA wants it in with one shuffle: 38 % fewer shared-memory wavefronts,
// parity-green, and 7 % SLOWER on every config (cfg4 3.79e11 against 4.08e11): the shared-memory pipe is the most used unit
// but not what limits the kernel.  Kept as a compile-time switch for the record; off.
#ifndef DVM_TILE_XPOSE
#define DVM_TILE_XPOSE 0
#endif
__device__ __forceinline__ int lane_ag(int lane) { return DVM_TILE_XPOSE ? lane >> 3 : lane & 3; }
__device__ __forceinline__ int lane_pair(int lane) { return DVM_TILE_XPOSE ? lane & 7 : lane >> 2; }
// the value the MMA wants from this lane (B fragment: k = lane & 3 = xi_x group, n = lane >> 2 = pair), widened to double
__device__ __forceinline__ double mma_operand(double g, int lane)
{
    return DVM_TILE_XPOSE ? __shfl_sync(0xffffffffu, g, (lane & 3) * 8 + (lane >> 2)) : g;
}
__device__ __forceinline__ double mma_operand(float g, int lane)
{
    return (double)(DVM_TILE_XPOSE ? __shfl_sync(0xffffffffu, g, (lane & 3) * 8 + (lane >> 2)) : g);
}

// D (8 x 8) += A (8 x 4, row-major) * B (4 x 8, column-major) in fp64 on the tensor cores (DMMA).  Fragments of lane l:
// A[l >> 2][l & 3], B[l & 3][l >> 2], C/D[l >> 2][2 (l & 3) + {0, 1}].
__device__ __forceinline__ void dmma(double &c0, double &c1, const double a, const double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// the first product of a chain: D = A * B (the zero accumulator is the zero register, not two moves)
__device__ __forceinline__ void dmma0(double &c0, double &c1, const double a, const double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%4, %4};" : "=d"(c0), "=d"(c1) : "d"(a), "d"(b), "d"(0.0));
}

// Velocity sums of Eq.(5) as two small matrix products per pair of cells (A, B) and warp.
//   stage 1, once per computed value g (RV per cell and thread): C[p][pair] += X[p][ag] * g[ag][pair], the lane supplying
//     its own g as the B fragment (k = its xi_x group ag = lane & 3, n = its (xi_y, xi_z) pair lane >> 2) and xi_x^p of
//     its own node as the A fragment (p = (lane >> 2) & 3: rows 4..7 repeat rows 0..3).  After the RV products
//     C[p][pair] = sum over the xi_x nodes of the block of xi_x^p g, for the warp's 8 pairs.  Cell A and cell B have
//     an accumulator each; lanes 0..15 (rows 0..3) then keep A's, lanes 16..31 (rows 4..7) B's.
//   stage 2, once per cell pair: D[row][j] = sum_pair C[row][pair] * M_j(pair), M = {1, y^2, y, z^2, z, yz, y r2, z r2},
//     r2 = y^2 + z^2.  The C fragment of stage 1 (columns 2q, 2q + 1) is the A fragment of the two k-steps (pairs 0, 2, 4, 6
//     and 1, 3, 5, 7) as it stands; every lane supplies M_(lane >> 2) of pairs 2q and 2q + 1 as B fragments.
// 17 of the 32 values D[p][j] of a cell are products the 13 sums need; each lane adds its two results (j = 2q and
// 2q + 1, p = (lane >> 2) & 3, q = lane & 3) to the [cell][16] accumulator row in L2 / HBM with a fp64 RED; sums made of
// several products (xi_x |xi|^2 ...) simply receive several REDs.  Slots of the row: 0..12 = the 13 sums in the order of
// dvm_raw_moments, except that slots 1, 2, 3 hold the first moments of the velocities with xi_d >= 0 only and slots 13,
// 14, 15 those of xi_d < 0: every velocity block lies in one sign octant, so this costs nothing, and the half-range
// sums are the wall-incident fluxes of Eq.(9): update.cu reads them from here, the sweep needs no flux
// atomics.  c_slot0 / c_slot1: slot of the first / second result; c_use: 1 if the sums need it (a result they do not
// need is added as 0 to a slot no other lane of the same instruction targets).
__constant__ signed char c_slot0[4][4] = {{0, 2, 3, 11}, {1, 7, 8, 5}, {4, 11, 12, 6}, {10, 9, 2, 3}};
__constant__ signed char c_use0[4][4] = {{1, 1, 1, 1}, {1, 1, 1, 0}, {1, 1, 1, 0}, {1, 0, 0, 0}};
__constant__ signed char c_slot1[4][4] = {{5, 6, 9, 12}, {10, 10, 0, 1}, {2, 3, 4, 7}, {8, 11, 13, 14}};
__constant__ signed char c_use1[4][4] = {{1, 1, 1, 1}, {1, 1, 0, 0}, {0, 0, 0, 0}, {0, 0, 0, 0}};

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

template <int RV, int ORD, typename R>
__device__ __forceinline__ void rwb_store(TileSmem<RV, ORD, R> &s, int b, int tid, double v)
{
    if (tid >= 32 && tid < 40) s.lv[b].rwb[tid - 32] = v;
}

// The TMA copies of a level are described once per item (setup_copies: per 4-cell row the x, y, z factor-table rows and
// the cell records - tables.cu; every row is one contiguous run of the padded grid - plus the x- and y-face input) and
// issued per level by lane q / WARPS of warp q % WARPS for copy q (issue_level), so the copies are spread over the warps.
template <int RV, int ORD, typename R>
__device__ __forceinline__ int copy_of_thread(int tid) { return (tid & 31) * KC<RV, ORD, R>::WARPS + (tid >> 5); }

template <int RV, int ORD, typename R>
__device__ __forceinline__ void setup_copies(const TileParams &P, const ItemCtx &I, TileSmem<RV, ORD, R> &s, const VBlock &vb, int tid,
                                             const R *xsrc, const R *ysrc)
{
    using RB = RowBuf<RV, ORD, R>;
    using LB = LevelBuf<RV, ORD, R>;
    constexpr int NA = GA * RV, ES = KC<RV, ORD, R>::ES;
    constexpr unsigned XLEVEL_BYTES = KC<RV, ORD, R>::XLEVEL_BYTES, YLEVEL_BYTES = KC<RV, ORD, R>::YLEVEL_BYTES;
    const int q = copy_of_thread<RV, ORD, R>(tid);
    if (q >= NCOPY) return;
    const unsigned xbytes = 4u * NA * ES, ybytes = 4u * vb.nbb * ES, zbytes = 4u * vb.ncb * ES;
    CopyDesc d;
    d.pad[0] = d.pad[1] = 0;
    if (q == 4 * TILE_TY) {
        d.src = reinterpret_cast<const unsigned char *>(xsrc); d.step = XLEVEL_BYTES;
        d.dst = (unsigned)offsetof(LB, xface); d.bytes = I.first_x ? 0u : XLEVEL_BYTES;
    } else if (q == 4 * TILE_TY + 1) {
        d.src = reinterpret_cast<const unsigned char *>(ysrc); d.step = YLEVEL_BYTES;
        d.dst = (unsigned)offsetof(LB, yface); d.bytes = I.first_y ? 0u : YLEVEL_BYTES;
    } else {
        const int jj = q % TILE_TY, kind = q / TILE_TY;
        // first cell (lowest absolute x) of row jj on the padded grid at level 0; rows may lie in the dead padding
        const int jp = I.j0 + jj, ip0 = I.i0;
        const int j = I.sy > 0 ? jp : P.ny - 1 - jp;
        const int i = I.sx > 0 ? ip0 : P.nx - 4 - ip0;
        const int k = I.sz > 0 ? 0 : P.nz - 1;
        const long long npc = (long long)P.nz * P.nyp * P.nxp, lvl = (long long)P.nyp * P.nxp * I.sz;
        const long long pc = ((long long)k * P.nyp + (j + TILE_PAD)) * P.nxp + (i + TILE_PAD);
        const unsigned rowoff = (unsigned)(offsetof(LB, row) + jj * sizeof(RowBuf<RV, ORD, R>));
        if (kind == 0) {
            d.src = reinterpret_cast<const unsigned char *>(P.TX) + ((long long)vb.xb * npc + pc) * NA * ES;
            d.step = lvl * NA * ES; d.dst = rowoff + (unsigned)offsetof(RB, xtab); d.bytes = xbytes;
        } else if (kind == 1) {
            d.src = reinterpret_cast<const unsigned char *>(P.TY) + ((long long)vb.yb * npc + pc) * vb.nbb * ES;
            d.step = lvl * vb.nbb * ES; d.dst = rowoff + (unsigned)offsetof(RB, ytab); d.bytes = ybytes;
        } else if (kind == 2) {
            d.src = reinterpret_cast<const unsigned char *>(P.TZ) + ((long long)vb.zb * npc + pc) * vb.ncb * ES;
            d.step = lvl * vb.ncb * ES; d.dst = rowoff + (unsigned)offsetof(RB, ztab); d.bytes = zbytes;
        } else {
            d.src = reinterpret_cast<const unsigned char *>(P.rec + pc);
            d.step = lvl * (long long)sizeof(CellRec); d.dst = rowoff + (unsigned)offsetof(RB, rec); d.bytes = REC_ROW_BYTES;
        }
    }
    s.desc[q] = d;
    if (q == 0)
        s.txbytes = (I.first_x ? 0u : XLEVEL_BYTES) + (I.first_y ? 0u : YLEVEL_BYTES) +
                    (unsigned)TILE_TY * (xbytes + ybytes + zbytes + REC_ROW_BYTES);
}

// issue the copies of level kp into buffer kp & 1 (the descriptors were written by the same threads)
template <int RV, int ORD, typename R>
__device__ __forceinline__ void issue_level(TileSmem<RV, ORD, R> &s, int kp, int tid)
{
    const int q = copy_of_thread<RV, ORD, R>(tid);
    if (q >= NCOPY) return;
    const int b = kp & 1;
    if (q == 0) mbar_expect_tx(&s.mbar[b], s.txbytes);
    const CopyDesc d = s.desc[q];
    if (d.bytes) tma_load(reinterpret_cast<unsigned char *>(&s.lv[b]) + d.dst, d.src + (long long)kp * d.step, d.bytes, &s.mbar[b]);
}

// Does the level staged in buffer b hold a fluid cell whose upwind neighbour is a masked cell?  Asked by lanes 0..15 of
// warp 0 (one record each) right after they have waited for the level's copies; the answer reaches the other threads
// through the CTA barrier that ends the level before.
template <int RV, int ORD, typename R>
__device__ __forceinline__ void detect_special(const ItemCtx &I, TileSmem<RV, ORD, R> &s, int b, int lane)
{
    const CellRec &r = s.lv[b].row[lane >> 2].rec[lane & 3];
    const int upmask = (1 << I.upx) | (1 << I.upy) | (1 << I.upz);
    const bool hit = (((r.flags >> 8) & 0x3f) & upmask) != 0;
    const unsigned any = __ballot_sync(0x0000ffffu, hit);
    if (lane == 0) s.special[b] = any != 0u;
}

// Slow path only: per-cell ghost codes of the level in buffer b, decoded from the staged records by the first 16 threads
// of the last warp.
template <int RV, int ORD, typename R>
__device__ __forceinline__ void decode_records(const TileParams &P, const ItemCtx &I, TileSmem<RV, ORD, R> &s, int b, int tid)
{
    constexpr int T0 = KC<RV, ORD, R>::THREADS - 32;
    if (tid >= T0 && tid < T0 + NCELL) {
        const int cell = tid - T0, ii = cell & 3, jj = cell >> 2;
        RowBuf<RV, ORD, R> &Rw = s.lv[b].row[jj];
        const CellRec &r = Rw.rec[I.sx > 0 ? ii : 3 - ii];
        const bool dead = (r.flags & REC_DEAD) != 0;
        const int sfl = (r.flags >> 8) & 0xff;
        int code = 8;
        double4 sp = make_double4(0.0, 0.0, 0.0, 0.0);
        if (!dead) {
            code = ((sfl >> I.upx) & 1) | (((sfl >> I.upy) & 1) << 1) | (((sfl >> I.upz) & 1) << 2);
            if (code & 1) sp.x = P.rho_w[r.face[I.upx]];
            if (code & 2) sp.y = P.rho_w[r.face[I.upy]];
            if (code & 4) sp.z = P.rho_w[r.face[I.upz]];
        }
        Rw.code[ii] = code;
        Rw.spec[ii] = sp;
    }
}

// The RV values of a thread in a face row of NVB doubles are stored as RV / 2 pairs, pair h of thread t at double
// (h * threads + t) * 2 (odd RV: the last value of thread t follows the pairs, at pairs + t): every 16-byte access of a
// warp then covers 512 contiguous bytes (full sectors in L2 / HBM, no bank conflict in shared memory).  row = start of the
// face row.
// Single values with RV = 4: the four values of a thread are one 16-byte quad at tid * 4.
__device__ __forceinline__ void st_pair(double *a, double x, double y) { st_f64x2(a, x, y); }
__device__ __forceinline__ void st_pair(float *a, float x, float y) { st_f32x2(a, x, y); }
__device__ __forceinline__ void st_one(double *a, double x) { st_f64(a, x); }
__device__ __forceinline__ void st_one(float *a, float x) { st_f32(a, x); }
template <int RV, int ORD, typename R>
__device__ __forceinline__ int face_index(int tid, int r)
{
    constexpr int TH = KC<RV, ORD, R>::THREADS;
    if (sizeof(R) == 4 && RV == 4) return tid * 4 + r;
    return r < 2 * (RV / 2) ? ((r >> 1) * TH + tid) * 2 + (r & 1) : (RV / 2) * TH * 2 + tid;
}
template <int RV, int ORD, typename R>
__device__ __forceinline__ void load_face(const R *row, int tid, R (&v)[RV])
{
    constexpr int TH = KC<RV, ORD, R>::THREADS;
    using V2 = typename Vec<R>::v2;
    if (sizeof(R) == 4 && RV == 4) {
        const float4 t = reinterpret_cast<const float4 *>(row)[tid];
        v[0] = t.x; v[1] = t.y; v[2 % RV] = t.z; v[3 % RV] = t.w;
    } else {
#pragma unroll
        for (int h = 0; h < RV / 2; ++h) {
            const V2 t = reinterpret_cast<const V2 *>(row)[h * TH + tid];
            v[2 * h] = t.x; v[2 * h + 1] = t.y;
        }
        if (RV & 1) v[RV - 1] = row[(RV / 2) * TH * 2 + tid];
    }
}
template <int RV, int ORD, typename R>
__device__ __forceinline__ void store_face(R *row, int tid, const R (&v)[RV])
{
    constexpr int TH = KC<RV, ORD, R>::THREADS;
    if (sizeof(R) == 4 && RV == 4) {
        st_f32x4(reinterpret_cast<float *>(row) + tid * 4, (float)v[0], (float)v[1], (float)v[2 % RV], (float)v[3 % RV]);
    } else {
#pragma unroll
        for (int h = 0; h < RV / 2; ++h) st_pair(row + (h * TH + tid) * 2, v[2 * h], v[2 * h + 1]);
        if (RV & 1) st_one(row + (RV / 2) * TH * 2 + tid, v[RV - 1]);
    }
}

// Ghost values of the domain faces of level kp (buffer b) for a tile at the upwind x / y edge of the domain
template <int RV, int ORD, typename R>
__device__ __forceinline__ void fill_faces(const ItemCtx &I, TileSmem<RV, ORD, R> &s, int b, int tid, int ag, int yidx, int zidx)
{
    LevelBuf<RV, ORD, R> &L = s.lv[b];
    if (I.first_x) {
        const double gyz = s.g[0][1][yidx] * s.g[0][2][zidx];
#pragma unroll
        for (int r = 0; r < RV; ++r) {
            const double G = s.g[0][0][RV * ag + r] * gyz;
#pragma unroll
            for (int jj = 0; jj < TILE_TY; ++jj) {
                L.xface[0][jj][face_index<RV, ORD, R>(tid, r)] = (R)(L.rwb[jj] * G);
                if (ORD == 2) L.xface[ORD - 1][jj][face_index<RV, ORD, R>(tid, r)] = (R)0;   // second upwind value: its coefficient is 0
            }
        }
    }
    if (I.first_y) {
        const double gyz = s.g[1][1][yidx] * s.g[1][2][zidx];
#pragma unroll
        for (int r = 0; r < RV; ++r) {
            const double G = s.g[1][0][RV * ag + r] * gyz;
#pragma unroll
            for (int ii = 0; ii < 4; ++ii) {
                L.yface[0][ii][face_index<RV, ORD, R>(tid, r)] = (R)(L.rwb[4 + ii] * G);
                if (ORD == 2) L.yface[ORD - 1][ii][face_index<RV, ORD, R>(tid, r)] = (R)0;
            }
        }
    }
}

// per-thread constants of an item
template <int RV, int ORD, typename R>
struct ThreadCtx {
    double aX[RV];               // stage-1 A fragments per node r: xi_x^p, p = (lane >> 2) & 3
    double yz0, yz1;             // stage-2 B fragments: monomial lane >> 2 of the warp's pairs 2 (lane & 3), 2 (lane & 3) + 1
    double *raw0, *raw1;         // raw16 + accumulator slot of the lane's two results
    double use0, use1;           // 1 if the result is one of the products the sums need, else 0 (the RED then adds 0)
    int xo[4], yo[4], zo[4];     // byte offsets in a RowBuf of the thread's table entries of cell ii (r = 0 for x)
    int ro[4];                   // byte offset in a RowBuf of the record of cell ii
    int ag, yi, zi;              // xi_x group, rows of the thread's xi_y and xi_z nodes in xi_bc / g
    int xrev;                    // 3 if the sweep runs against x (table rows are in ascending absolute x), else 0
};

template <int RV, int ORD, typename R>
__device__ __forceinline__ const typename Vec<R>::v4 &entry(const RowBuf<RV, ORD, R> &B, int byte_off)
{
    return *reinterpret_cast<const typename Vec<R>::v4 *>(reinterpret_cast<const unsigned char *>(&B) + byte_off);
}
// order 2: the two stencil coefficients c1, c2 that follow (E, Q, e, cd) in an entry
template <int RV, int ORD, typename R>
__device__ __forceinline__ const typename Vec<R>::v2 &entry_c(const RowBuf<RV, ORD, R> &B, int byte_off)
{
    return *reinterpret_cast<const typename Vec<R>::v2 *>(reinterpret_cast<const unsigned char *>(&B) + byte_off + 4 * sizeof(R));
}
template <int RV, int ORD, typename R>
__device__ __forceinline__ const CellRec &record(const RowBuf<RV, ORD, R> &B, int byte_off)
{
    return *reinterpret_cast<const CellRec *>(reinterpret_cast<const unsigned char *>(&B) + byte_off);
}
// 1/tau of a cell in the carried type (the record holds it in both)
__device__ __forceinline__ void rec_nu(const CellRec &r, double &nu) { nu = r.nu; }
__device__ __forceinline__ void rec_nu(const CellRec &r, float &nu) { nu = r.nu32; }

// stage 2 for a pair of cells (A, B; roA, roB: their records) of a row and the REDs of its results (lanes 0..15: cell A,
// 16..31: cell B).
// No predicates and no branches (the row stays one basic block): a result the sums do not need is multiplied by 0 and
// added to a slot no other lane of the instruction targets; dead cells have g = 0 and name a row of their own or, in
// the padding, of the nearest cell of the grid.
template <int RV, int ORD, typename R>
__device__ __forceinline__ void emit_pair(const RowBuf<RV, ORD, R> &Rw, const int roA, const int roB, const double a0, const double a1,
                                          const double b0, const double b1, const ThreadCtx<RV, ORD, R> &T, const int lane)
{
    const bool hi = lane & 16;
    double d0, d1;
    dmma0(d0, d1, hi ? b0 : a0, T.yz0);
    dmma(d0, d1, hi ? b1 : a1, T.yz1);
    const long long c = record<RV, ORD, R>(Rw, hi ? roB : roA).cidx;
    red_f64(T.raw0 + c * 16, d0 * T.use0);
    red_f64(T.raw1 + c * 16, d1 * T.use1);
}

// One row (4 cells along the sweep-relative x) of a level, fast path: zrow holds the values of the row in the previous
// z-plane (the z-upwind operands) and receives the new ones, yup holds the y-upwind operands (the staged y-face for the
// first row of the tile, else the row just computed).  Dead cells (outside the domain / solid) have all-zero table
// entries and nu = 1, so they produce g = 0 by the same arithmetic.  The last row of the tile (LAST) also writes the
// y-face output, cell by cell, so that the stores are spread over the row.
// ORD = 2 (second-order upwind, G21): z2row / yup2 / the second x-face layer hold the second upwind values; the
// table entries carry the stencil coefficients (cd, c1, c2) per direction, so the cell value is
// g = [src + sum_d (c1_d g_1d + c2_d g_2d)] / (nu + sum_d cd_d); the recurrence along x is still one DFMA per value
// (the c2 term uses the value two cells back, known a cell earlier).  YL: y-face layer this row's values go to (-1: none).
template <int RV, int ORD, int AX, int YL, typename R>
__device__ __forceinline__ void compute_row(const RowBuf<RV, ORD, R> &Rw, const R *xin, const R *xin2, R (&zrow)[4][RV],
                                            R (&z2row)[4][RV], const R (&yup)[4][RV], const R (&yup2)[4][RV],
                                            const ThreadCtx<RV, ORD, R> &T, const int tid, const int lane, R *xout, const bool wx,
                                            R *yout, const bool wy)
{
    using V4 = typename Vec<R>::v4;
    using V2 = typename Vec<R>::v2;
    constexpr int NVB = KC<RV, ORD, R>::NVB, ES = KC<RV, ORD, R>::ES;
    constexpr R ONE = (R)1, ZERO = (R)0;
    R fx[RV], fx2[RV];
    load_face<RV, ORD, R>(xin, tid, fx);
    if (ORD == 2) load_face<RV, ORD, R>(xin2, tid, fx2);
    double acc[2][2];
#pragma unroll
    for (int ii = 0; ii < 4; ++ii) {
        const V4 yt = entry<RV, ORD, R>(Rw, T.yo[ii]);
        const V4 zt = entry<RV, ORD, R>(Rw, T.zo[ii]);
        R nu;
        rec_nu(record<RV, ORD, R>(Rw, T.ro[ii]), nu);
        const R Eyz = yt.x * zt.x, Qyz = yt.y + zt.y, eyz = yt.z + zt.z;
        const R dyz = (yt.w + zt.w) + nu;
        // stencil coefficients of the entries of the roles B and C (one per cell) - and, below, A (one per node)
        R c1B = yt.w, c1C = zt.w, c2B = ZERO, c2C = ZERO;
        if (ORD == 2) {
            const V2 yc = entry_c<RV, ORD, R>(Rw, T.yo[ii]), zc = entry_c<RV, ORD, R>(Rw, T.zo[ii]);
            c1B = yc.x; c2B = yc.y; c1C = zc.x; c2C = zc.y;
        }
        // Everything that does not depend on the x-upwind value, for the RV nodes of the thread in lock step (the fp64
        // pipe has a latency of ~10 clocks): the cell value is g = (W g_xup + V) / den with W = a_x and
        // V = a_y g_yup + a_z g_zup + src, Eq.(7) PAPER.md:75-79.
        V4 xt[RV];
        V2 xc[RV];
        R t1[RV], t2[RV], d[RV], y0[RV], sE[RV], e[RV], W[RV], V[RV];
#pragma unroll
        for (int r = 0; r < RV; ++r) xt[r] = entry<RV, ORD, R>(Rw, T.xo[ii] + r * GA * ES);
        if (ORD == 2) {
#pragma unroll
            for (int r = 0; r < RV; ++r) xc[r] = entry_c<RV, ORD, R>(Rw, T.xo[ii] + r * GA * ES);
        }
#pragma unroll
        for (int r = 0; r < RV; ++r) d[r] = xt[r].w + dyz;
#pragma unroll
        for (int r = 0; r < RV; ++r) t1[r] = xt[r].y + Qyz;
#pragma unroll
        for (int r = 0; r < RV; ++r) y0[r] = rcp_seed(d[r]);
#pragma unroll
        for (int r = 0; r < RV; ++r) t2[r] = xt[r].z + eyz;
#pragma unroll
        for (int r = 0; r < RV; ++r) sE[r] = xt[r].x * Eyz;
        if (sizeof(R) == 8) {
#pragma unroll
            for (int r = 0; r < RV; ++r) e[r] = fma(-d[r], y0[r], ONE);
        }
#pragma unroll
        for (int r = 0; r < RV; ++r) t1[r] = fma(t1[r], t2[r], ONE);
        if (sizeof(R) == 8) {
#pragma unroll
            for (int r = 0; r < RV; ++r) e[r] = fma(e[r], e[r], e[r]);
        }
#pragma unroll
        for (int r = 0; r < RV; ++r) V[r] = sE[r] * t1[r];
        if (sizeof(R) == 8) {
#pragma unroll
            for (int r = 0; r < RV; ++r) y0[r] = fma(y0[r], e[r], y0[r]);   // 1 / den (MUFU seed + cubic Newton step; single: the seed is exact to 1 ulp)
        }
        // The entry of role A belongs to velocity axis AX, B and C to the other two in ascending order; the coefficient of the
        // x- / y- / z-upwind value is the one of the entry that holds xi_x / xi_y / xi_z (compile-time selection).
        R c1A[RV], c2A[RV];
#pragma unroll
        for (int r = 0; r < RV; ++r) { c1A[r] = ORD == 2 ? xc[r].x : xt[r].w; c2A[r] = ORD == 2 ? xc[r].y : ZERO; }
#pragma unroll
        for (int r = 0; r < RV; ++r) V[r] = fma(AX == 0 ? c1B : AX == 1 ? c1A[r] : c1C, yup[ii][r], V[r]);
        if (ORD == 2) {
#pragma unroll
            for (int r = 0; r < RV; ++r) V[r] = fma(AX == 0 ? c2B : AX == 1 ? c2A[r] : c2C, yup2[ii][r], V[r]);
        }
#pragma unroll
        for (int r = 0; r < RV; ++r) W[r] = AX == 0 ? c1A[r] : c1B;
#pragma unroll
        for (int r = 0; r < RV; ++r) V[r] = fma(AX == 2 ? c1A[r] : c1C, zrow[ii][r], V[r]);
        if (ORD == 2) {
#pragma unroll
            for (int r = 0; r < RV; ++r) V[r] = fma(AX == 2 ? c2A[r] : c2C, z2row[ii][r], V[r]);
#pragma unroll
            for (int r = 0; r < RV; ++r) V[r] = fma(AX == 0 ? c2A[r] : c2B, fx2[r], V[r]);
        }
        // the recurrence along x: one FMA and the multiplication by 1 / den per value (scaling W and V by 1 / den beforehand
        // would take the multiplication off the recurrence at the price of one more per value: measured 3 % slower - the
        // chain of a row is short against the work of a level)
#pragma unroll
        for (int r = 0; r < RV; ++r) {
            const R gg = fma(W[r], fx[r], V[r]) * y0[r];
            if (ORD == 2) { fx2[r] = fx[r]; z2row[ii][r] = zrow[ii][r]; }
            fx[r] = gg;
            zrow[ii][r] = gg;
        }
        // velocity sums: always in double (a single value is widened exactly)
        dmma0(acc[ii & 1][0], acc[ii & 1][1], T.aX[0], mma_operand(zrow[ii][0], lane));
#pragma unroll
        for (int r = 1; r < RV; ++r) dmma(acc[ii & 1][0], acc[ii & 1][1], T.aX[r], mma_operand(zrow[ii][r], lane));
        if (ii & 1) emit_pair<RV, ORD, R>(Rw, T.ro[ii - 1], T.ro[ii], acc[0][0], acc[0][1], acc[1][0], acc[1][1], T, lane);
        if (YL >= 0 && wy) store_face<RV, ORD, R>(yout + (YL * TILE_TX + ii) * NVB, tid, zrow[ii]);
    }
    if (wx) {
        store_face<RV, ORD, R>(xout, tid, fx);
        if (ORD == 2) store_face<RV, ORD, R>(xout + TILE_TY * NVB, tid, fx2);
    }
}

// One level of the column, fast path (no solid ghost in the level): 4 rows x 4 cells x RV velocities per thread with the
// plane in registers (static indices only); the rows are unrolled, the y-upwind operands of a row are the registers of
// the row before.  The B200 instruction cache holds 32 KB, and a level loop larger than that is fetch-bound at 1/3
// instruction per clock and scheduler (profiles/r01_ifetch_microbench.txt): the instructions a level executes on
// this path (about 1900 for RV = 4) stay below that; rolled variants with rotating row slots were slower (profiles/).
template <int RV, int ORD, int AX, typename R>
__device__ __forceinline__ void compute_level(const LevelBuf<RV, ORD, R> &L, R (&pl)[TILE_TY][4][RV], R (&pl2)[ORD == 2 ? TILE_TY : 1][4][RV],
                                              const ThreadCtx<RV, ORD, R> &T, const int tid, const int lane, R *xout, const bool wx,
                                              R *yout, const bool wy)
{
    constexpr int NVB = KC<RV, ORD, R>::NVB, L2 = ORD - 1;
    static_assert(TILE_TY >= 2 || ORD == 1, "the second-order tile kernel needs at least two rows per tile");
    R yu[4][RV], yu2[4][RV];
#pragma unroll
    for (int ii = 0; ii < 4; ++ii) load_face<RV, ORD, R>(&L.yface[0][ii][0], tid, yu[ii]);
    if (ORD == 2) {
#pragma unroll
        for (int ii = 0; ii < 4; ++ii) load_face<RV, ORD, R>(&L.yface[L2][ii][0], tid, yu2[ii]);
    }
    // y-face layer a row's values go to: the last row -> layer 0, the one before (order 2) -> layer 1
    if (TILE_TY == 1) {
        compute_row<RV, ORD, AX, 0, R>(L.row[0], L.xface[0][0], L.xface[L2][0], pl[0], pl2[0], yu, yu2, T, tid, lane, xout, wx, yout, wy);
    } else {
        compute_row<RV, ORD, AX, (ORD == 2 && TILE_TY == 2) ? 1 : -1, R>(L.row[0], L.xface[0][0], L.xface[L2][0], pl[0], pl2[0], yu, yu2, T, tid, lane,
                                                                xout, wx, yout, wy);
#pragma unroll
        for (int jj = 1; jj < TILE_TY - 1; ++jj) {
            if (ORD == 2 && jj == TILE_TY - 2)
                compute_row<RV, ORD, AX, 1, R>(L.row[jj], L.xface[0][jj], L.xface[L2][jj], pl[jj], pl2[ORD == 2 ? jj : 0], pl[jj - 1], jj >= 2 ? pl[jj >= 2 ? jj - 2 : 0] : yu,
                                        T, tid, lane, xout + jj * NVB, wx, yout, wy);
            else
                compute_row<RV, ORD, AX, -1, R>(L.row[jj], L.xface[0][jj], L.xface[L2][jj], pl[jj], pl2[ORD == 2 ? jj : 0], pl[jj - 1], jj >= 2 ? pl[jj >= 2 ? jj - 2 : 0] : yu,
                                         T, tid, lane, xout + jj * NVB, wx, yout, wy);
        }
        constexpr int J = TILE_TY - 1;
        compute_row<RV, ORD, AX, 0, R>(L.row[J], L.xface[0][J], L.xface[L2][J], pl[J], pl2[ORD == 2 ? J : 0], pl[J - 1], J >= 2 ? pl[J >= 2 ? J - 2 : 0] : yu, T, tid, lane,
                                xout + J * NVB, wx, yout, wy);
    }
}

// One level that holds a solid ghost (a fluid cell whose upwind neighbour is a masked cell): the same arithmetic
// written as compact loops over a copy of the plane(s) in local memory.  Rare (the surface of a masked body), so its
// speed does not matter; keeping it out of the unrolled path halves the code the instruction cache has to hold.
// A solid ghost replaces the first upwind value; the coefficient of the second one is 0 there (tables.cu).
template <int RV, int ORD, int AX, typename R>
__device__ __forceinline__ void compute_level_slow(TileSmem<RV, ORD, R> &s, const LevelBuf<RV, ORD, R> &L, R *pl, R *pl2,
                                                   const ThreadCtx<RV, ORD, R> &T, const int tid, const int lane, R *xout, R *yout)
{
    using V4 = typename Vec<R>::v4;
    using V2 = typename Vec<R>::v2;
    constexpr int NVB = KC<RV, ORD, R>::NVB, ES = KC<RV, ORD, R>::ES, L2 = ORD - 1;
    constexpr R ONE = (R)1, ZERO = (R)0;
    const double gyz = s.g[3][1][T.yi] * s.g[3][2][T.zi];
#pragma unroll 1
    for (int jj = 0; jj < TILE_TY; ++jj) {
        const RowBuf<RV, ORD, R> &Rw = L.row[jj];
        R fx[RV], fx2[RV];
#pragma unroll
        for (int r = 0; r < RV; ++r) {
            fx[r] = L.xface[0][jj][face_index<RV, ORD, R>(tid, r)];
            fx2[r] = ORD == 2 ? L.xface[L2][jj][face_index<RV, ORD, R>(tid, r)] : ZERO;
        }
        double accA0 = 0.0, accA1 = 0.0;
        int roPrev = 0;
#pragma unroll 1
        for (int ii = 0; ii < 4; ++ii) {
            const int cell = jj * 4 + ii;
            const int xo = ii == 0 ? T.xo[0] : ii == 1 ? T.xo[1] : ii == 2 ? T.xo[2] : T.xo[3];
            const int yo = ii == 0 ? T.yo[0] : ii == 1 ? T.yo[1] : ii == 2 ? T.yo[2] : T.yo[3];
            const int zo = ii == 0 ? T.zo[0] : ii == 1 ? T.zo[1] : ii == 2 ? T.zo[2] : T.zo[3];
            const V4 yt = entry<RV, ORD, R>(Rw, yo);
            const V4 zt = entry<RV, ORD, R>(Rw, zo);
            const R Eyz = yt.x * zt.x, Qyz = yt.y + zt.y, eyz = yt.z + zt.z;
            R c1B = yt.w, c1C = zt.w, c2B = ZERO, c2C = ZERO;
            if (ORD == 2) {
                const V2 yc = entry_c<RV, ORD, R>(Rw, yo), zc = entry_c<RV, ORD, R>(Rw, zo);
                c1B = yc.x; c2B = yc.y; c1C = zc.x; c2C = zc.y;
            }
            const int ro = ii == 0 ? T.ro[0] : ii == 1 ? T.ro[1] : ii == 2 ? T.ro[2] : T.ro[3];
            R nu;
            rec_nu(record<RV, ORD, R>(Rw, ro), nu);
            const R dyz = (yt.w + zt.w) + nu;
            const int code = Rw.code[ii];
            const double4 sp = Rw.spec[ii];
            double c0 = 0.0, c1 = 0.0;
#pragma unroll
            for (int r = 0; r < RV; ++r) {
                const double Pg = s.g[3][0][RV * T.ag + r] * gyz;
                const V4 xt = entry<RV, ORD, R>(Rw, xo + r * GA * ES);
                R c1A = xt.w, c2A = ZERO;
                if (ORD == 2) { const V2 xc = entry_c<RV, ORD, R>(Rw, xo + r * GA * ES); c1A = xc.x; c2A = xc.y; }
                const R c1x = AX == 0 ? c1A : c1B, c1y = AX == 0 ? c1B : AX == 1 ? c1A : c1C, c1z = AX == 2 ? c1A : c1C;
                const R c2x = AX == 0 ? c2A : c2B, c2y = AX == 0 ? c2B : AX == 1 ? c2A : c2C, c2z = AX == 2 ? c2A : c2C;
                R xu = fx[r], zu = pl[cell * RV + r];
                R yu = jj == 0 ? L.yface[0][ii][face_index<RV, ORD, R>(tid, r)] : pl[(cell - 4) * RV + r];
                R xu2 = fx2[r], zu2 = ZERO, yu2 = ZERO;
                if (ORD == 2) {
                    zu2 = pl2[cell * RV + r];
                    yu2 = jj == 0 ? L.yface[L2][ii][face_index<RV, ORD, R>(tid, r)]
                        : jj == 1 ? L.yface[0][ii][face_index<RV, ORD, R>(tid, r)] : pl[(cell - 8) * RV + r];
                }
                if (code & 1) xu = (R)(sp.x * Pg);
                if (code & 2) yu = (R)(sp.y * Pg);
                if (code & 4) zu = (R)(sp.z * Pg);
                const R src = (xt.x * Eyz) * fma(xt.y + Qyz, xt.z + eyz, ONE);
                const R inv = fast_rcp(xt.w + dyz);
                R num = fma(c1y, yu, src);
                num = fma(c1z, zu, num);
                num = fma(c1x, xu, num);
                if (ORD == 2) {
                    num = fma(c2y, yu2, num);
                    num = fma(c2z, zu2, num);
                    num = fma(c2x, xu2, num);
                }
                R gg = num * inv;
                if (code & 8) gg = ZERO;
                fx2[r] = fx[r];
                fx[r] = gg;
                if (ORD == 2) pl2[cell * RV + r] = pl[cell * RV + r];
                pl[cell * RV + r] = gg;
                dmma(c0, c1, T.aX[r], mma_operand(gg, lane));
            }
            if (ii & 1) {
                emit_pair<RV, ORD, R>(Rw, roPrev, ro, accA0, accA1, c0, c1, T, lane);
            } else {
                accA0 = c0; accA1 = c1;
            }
            roPrev = ro;
        }
        if (xout) {
#pragma unroll
            for (int r = 0; r < RV; ++r) {
                xout[jj * NVB + face_index<RV, ORD, R>(tid, r)] = fx[r];
                if (ORD == 2) xout[(TILE_TY + jj) * NVB + face_index<RV, ORD, R>(tid, r)] = fx2[r];
            }
        }
    }
    if (yout) {
#pragma unroll 1
        for (int ii = 0; ii < 4; ++ii)
#pragma unroll
            for (int r = 0; r < RV; ++r) {
                yout[ii * NVB + face_index<RV, ORD, R>(tid, r)] = pl[((TILE_TY - 1) * 4 + ii) * RV + r];
                if (ORD == 2) yout[(TILE_TX + ii) * NVB + face_index<RV, ORD, R>(tid, r)] = pl[((TILE_TY >= 2 ? TILE_TY - 2 : 0) * 4 + ii) * RV + r];
            }
    }
}

template <int RV, int ORD, int AX, typename R>
__global__ void __launch_bounds__(KC<RV, ORD, R>::THREADS, KC<RV, ORD, R>::MIN_CTAS) sweep_tile_kernel(const TileParams P)
{
    constexpr int NA = GA * RV, THREADS = KC<RV, ORD, R>::THREADS, XLEVEL_VALUES = KC<RV, ORD, R>::XLEVEL_VALUES, YLEVEL_VALUES = KC<RV, ORD, R>::YLEVEL_VALUES;
    (void)THREADS;
    using RB = RowBuf<RV, ORD, R>;
    // velocity axis in the role A (AX), B, C and their node arrays
    constexpr int AXB = AX == 0 ? 1 : 0, AXC = AX == 2 ? 1 : 2;
    const double *xiA = AX == 0 ? P.xi_x : AX == 1 ? P.xi_y : P.xi_z;
    const double *xiB = AXB == 0 ? P.xi_x : P.xi_y, *xiC = AXC == 1 ? P.xi_y : P.xi_z;
    // dynamic shared memory starts at offset 0 of the CTA's window (no static __shared__ in this kernel), so the
    // 128-byte alignment holds; casting without pointer arithmetic keeps the address space visible (LDS / STS)
    extern __shared__ __align__(128) unsigned char smem_raw[];
    TileSmem<RV, ORD, R> &s = *reinterpret_cast<TileSmem<RV, ORD, R> *>(smem_raw);
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
        R *xdst = static_cast<R *>(P.xface) + ((long long)(it.vb % P.batch) * P.P + it.xslot) * P.xslot_values;
        R *ydst = static_cast<R *>(P.yface) + ((long long)(it.vb % P.batch) * P.ntx + it.ti) * P.yslot_values;

        // ---- TMA copies of levels 0 and 1 (the staging buffers are free: every thread passed the end-of-item
        //      barrier; the upwind items' face stores were made with the generic proxy) ----
        setup_copies<RV, ORD, R>(P, I, s, vb, tid, xdst, ydst);
        if (copy_of_thread<RV, ORD, R>(tid) < NCOPY) {
            fence_proxy_async_global();
            issue_level<RV, ORD, R>(s, 0, tid);
            if (P.nz > 1) issue_level<RV, ORD, R>(s, 1, tid);
        }
        // ---- per-item tables: nodes, ghost factors; ghost densities of the domain faces of levels 0 and 1 ----
        {
            const int slotid[4] = {I.upx, I.upy, I.upz, 6};
            if (tid < 16) {
                const bool ok = tid < vb.na;
                const int idx = vb.a0 + tid;
                s.xi_a[tid] = ok ? xiA[idx] : 0.0;
#pragma unroll
                for (int f = 0; f < 4; ++f) s.g[f][0][tid] = ok ? P.gtab[(long long)(slotid[f] * 3 + AX) * P.gstride + idx] : 0.0;
            } else if (tid < 16 + vb.nbb) {
                const int bl = tid - 16;
                const bool ok = bl < vb.nb;
                const int idx = vb.b0 + bl;
                s.xi_bc[bl] = ok ? xiB[idx] : 0.0;
#pragma unroll
                for (int f = 0; f < 4; ++f) s.g[f][1][bl] = ok ? P.gtab[(long long)(slotid[f] * 3 + AXB) * P.gstride + idx] : 0.0;
            } else if (tid >= 32 && tid < 32 + vb.ncb) {
                const int cl = tid - 32;
                const bool ok = cl < vb.nc;
                const int idx = vb.c0 + cl;
                s.xi_bc[vb.nbb + cl] = ok ? xiC[idx] : 0.0;
#pragma unroll
                for (int f = 0; f < 4; ++f)
                    s.g[f][2][vb.nbb + cl] = ok ? P.gtab[(long long)(slotid[f] * 3 + AXC) * P.gstride + idx] : 0.0;
            }
            rwb_store<RV, ORD, R>(s, 0, tid, rwb_load(P, I, 0, tid));
            rwb_store<RV, ORD, R>(s, 1, tid, rwb_load(P, I, 1, tid));
        }
        __syncthreads();

        ThreadCtx<RV, ORD, R> T;
        T.ag = lane_ag(lane);
        T.xrev = vb.sx > 0 ? 0 : 3;
        {
            const int pair = warp * 8 + lane_pair(lane);
            const int yl = pair % vb.nbb, zl = pair / vb.nbb;
            T.yi = yl;
            T.zi = vb.nbb + zl;
            // table entries of the thread in a row buffer: cell ii sits at position ii ^ xrev of the staged rows
#pragma unroll
            for (int ii = 0; ii < 4; ++ii) {
                const int cp = ii ^ T.xrev;
                T.xo[ii] = (int)offsetof(RB, xtab) + (cp * NA + T.ag) * KC<RV, ORD, R>::ES;
                T.yo[ii] = (int)offsetof(RB, ytab) + (cp * vb.nbb + yl) * KC<RV, ORD, R>::ES;
                T.zo[ii] = (int)offsetof(RB, ztab) + (cp * vb.ncb + zl) * KC<RV, ORD, R>::ES;
                T.ro[ii] = (int)offsetof(RB, rec) + cp * (int)sizeof(CellRec);
            }
            // stage-1 A fragments: xi_x^p of the thread's own nodes, p = (lane >> 2) & 3
            const int row = lane >> 2, pw = row & 3;
#pragma unroll
            for (int r = 0; r < RV; ++r) {
                const double x = s.xi_a[RV * (lane & 3) + r];      // the MMA's view: k = lane & 3
                T.aX[r] = pw == 0 ? 1.0 : pw == 1 ? x : pw == 2 ? x * x : x * x * x;
            }
            // stage-2 B fragments: monomial j = lane >> 2 of the (xi_y, xi_z) nodes of pairs 2q and 2q + 1 of this warp
            const int j = lane >> 2, q = lane & 3;
            double mono[2];
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int pr = warp * 8 + 2 * q + e;
                const double y = s.xi_bc[pr % vb.nbb], z = s.xi_bc[vb.nbb + pr / vb.nbb], r2 = y * y + z * z;
                mono[e] = j == 0 ? 1.0 : j == 1 ? y * y : j == 2 ? y : j == 3 ? z * z : j == 4 ? z : j == 5 ? y * z
                        : j == 6 ? y * r2 : z * r2;
            }
            T.yz0 = mono[0]; T.yz1 = mono[1];
            // results of this lane: D[p][2q], D[p][2q + 1] and their accumulator slots.  c_slot names the sums in terms of the
            // roles (A, B, C) = (xi_AX, xi_AXB, xi_AXC); the accumulator row is in terms of (xi_x, xi_y, xi_z)
            int s0 = c_slot0[pw][q], s1 = c_slot1[pw][q];
            const bool u0 = c_use0[pw][q], u1 = c_use1[pw][q];
            const int axr[3] = {AX, AXB, AXC}, sgn[3] = {vb.sx, vb.sy, vb.sz};
            auto physical = [&](int sl) {
                if (sl >= 1 && sl <= 3) return 1 + axr[sl - 1];
                if (sl >= 4 && sl <= 6) return 4 + axr[sl - 4];
                if (sl == 7) return 6 + AX + AXB;      // {0,1} -> 7, {0,2} -> 8, {1,2} -> 9
                if (sl == 8) return 6 + AX + AXC;
                if (sl == 9) return 6 + AXB + AXC;
                if (sl >= 10 && sl <= 12) return 10 + axr[sl - 10];
                if (sl >= 13) return 13 + axr[sl - 13];
                return sl;
            };
            if (s0 >= 1 && s0 <= 3) {
                // first moments: half-range slot by the sign of the block; an unneeded result goes to the other one
                if ((sgn[axr[s0 - 1]] < 0) == u0) s0 += 12;
            }
            s0 = physical(s0); s1 = physical(s1);
            T.raw0 = P.raw16 + s0; T.raw1 = P.raw16 + s1;
            T.use0 = u0 ? 1.0 : 0.0; T.use1 = u1 ? 1.0 : 0.0;
        }

        // Level 0 has landed?  Only lanes 0..15 of warp 0 ever wait on the mbarrier of a level's copies (a try_wait round
        // trip costs several hundred clocks); they do so one level ahead, look for solid ghosts in the staged records, and
        // the CTA barrier that follows hands their observation of the completed copies on to every other thread.
        if (tid < NCELL) {
            mbar_wait(&s.mbar[0], par[0]);
            par[0] ^= 1u;
            detect_special<RV, ORD, R>(I, s, 0, lane);
        }
        fill_faces<RV, ORD, R>(I, s, 0, tid, T.ag, T.yi, T.zi);
        // plane = ghost of the upwind z face of the domain (order 2: the plane before it is never used, its coefficient
        // is 0 in the first level; it must only be finite)
        R pl[TILE_TY][4][RV], pl2[ORD == 2 ? TILE_TY : 1][4][RV];
#pragma unroll
        for (int jj = 0; jj < (ORD == 2 ? TILE_TY : 1); ++jj)
#pragma unroll
            for (int ii = 0; ii < 4; ++ii)
#pragma unroll
                for (int r = 0; r < RV; ++r) pl2[jj][ii][r] = (R)0;
        {
            const double gyz = s.g[2][1][T.yi] * s.g[2][2][T.zi];
            double G[RV];
#pragma unroll
            for (int r = 0; r < RV; ++r) G[r] = s.g[2][0][RV * T.ag + r] * gyz;
#pragma unroll
            for (int jj = 0; jj < TILE_TY; ++jj)
#pragma unroll
                for (int ii = 0; ii < 4; ++ii) {
                    int i, j, k;
                    double rw = 0.0;
                    if (cell_of(P, I, ii, jj, 0, i, j, k)) rw = face_density(P, I.tpz, P.foff[I.upz] + j * P.nx + i);
#pragma unroll
                    for (int r = 0; r < RV; ++r) pl[jj][ii][r] = (R)(rw * G[r]);
                }
        }
        __syncthreads();

        const bool write_x = it.ti < P.ntx - 1, write_y = it.tj < P.nty - 1;
        const bool edge = I.first_x | I.first_y;

        for (int kp = 0; kp < P.nz; ++kp) {
            const int b = kp & 1;
            // level kp + 1 (issued a level ago): wait for it and look for solid ghosts, for the barrier at the end
            if (tid < NCELL && kp + 1 < P.nz) {
                mbar_wait(&s.mbar[b ^ 1], par[b ^ 1]);
                par[b ^ 1] ^= 1u;
                detect_special<RV, ORD, R>(I, s, b ^ 1, lane);
            }
            double vrw = 0.0;
            if (edge) vrw = rwb_load(P, I, kp + 2, tid);
            const int special = __shfl_sync(0xffffffffu, s.special[b], 0);
            R *xout = xdst + (long long)kp * XLEVEL_VALUES, *yout = ydst + (long long)kp * YLEVEL_VALUES;
            if (special) {
                // every thread of the CTA takes this branch together
                decode_records<RV, ORD, R>(P, I, s, b, tid);
                __syncthreads();
                R tmp[NCELL * RV], tmp2[ORD == 2 ? NCELL * RV : 1];
#pragma unroll
                for (int c = 0; c < NCELL; ++c)
#pragma unroll
                    for (int r = 0; r < RV; ++r) {
                        tmp[c * RV + r] = pl[c >> 2][c & 3][r];
                        if (ORD == 2) tmp2[c * RV + r] = pl2[ORD == 2 ? c >> 2 : 0][c & 3][r];
                    }
                compute_level_slow<RV, ORD, AX, R>(s, s.lv[b], tmp, tmp2, T, tid, lane, write_x ? xout : nullptr, write_y ? yout : nullptr);
#pragma unroll
                for (int c = 0; c < NCELL; ++c)
#pragma unroll
                    for (int r = 0; r < RV; ++r) {
                        pl[c >> 2][c & 3][r] = tmp[c * RV + r];
                        if (ORD == 2) pl2[ORD == 2 ? c >> 2 : 0][c & 3][r] = tmp2[c * RV + r];
                    }
            } else {
                compute_level<RV, ORD, AX, R>(s.lv[b], pl, pl2, T, tid, lane, xout, write_x, yout, write_y);
            }
            if (edge) {
                rwb_store<RV, ORD, R>(s, b, tid, vrw);
                if (kp + 1 < P.nz) fill_faces<RV, ORD, R>(I, s, b ^ 1, tid, T.ag, T.yi, T.zi);
            }
            __syncthreads();
            if (copy_of_thread<RV, ORD, R>(tid) < NCOPY && kp + 2 < P.nz) {
                fence_proxy_async_smem();  // this level's reads of the staging buffers before the TMA overwrites them
                issue_level<RV, ORD, R>(s, kp + 2, tid);
            }
        }
        // ---- publish: faces of this item are complete ----
        asm volatile("" ::: "memory");
        __threadfence();
        __syncthreads();
        if (tid == 0) st_release(P.done + n, P.epoch);
    }
}

template <int RV, int ORD, int AX, typename R>
cudaError_t configure1(int *ctas_per_sm)
{
    cudaError_t e = cudaFuncSetAttribute(sweep_tile_kernel<RV, ORD, AX, R>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(TileSmem<RV, ORD, R>));
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, sweep_tile_kernel<RV, ORD, AX, R>, KC<RV, ORD, R>::THREADS, sizeof(TileSmem<RV, ORD, R>));
}
template <int RV, int ORD, typename R>
cudaError_t configure(int ax, int *ctas_per_sm)
{
    return ax == 1 ? configure1<RV, ORD, 1, R>(ctas_per_sm) : ax == 2 ? configure1<RV, ORD, 2, R>(ctas_per_sm) : configure1<RV, ORD, 0, R>(ctas_per_sm);
}
template <int RV, int ORD, typename R>
void launch(const TileParams &P, int ax, int grid, cudaStream_t st)
{
    if (ax == 1) sweep_tile_kernel<RV, ORD, 1, R><<<grid, KC<RV, ORD, R>::THREADS, sizeof(TileSmem<RV, ORD, R>), st>>>(P);
    else if (ax == 2) sweep_tile_kernel<RV, ORD, 2, R><<<grid, KC<RV, ORD, R>::THREADS, sizeof(TileSmem<RV, ORD, R>), st>>>(P);
    else sweep_tile_kernel<RV, ORD, 0, R><<<grid, KC<RV, ORD, R>::THREADS, sizeof(TileSmem<RV, ORD, R>), st>>>(P);
}

}  // namespace

// (rv, order, f32): the variants that exist: double (4 | 3 | 2, 1), (2, 2); single (4 | 3, 1)
bool tile_variant_exists(int rv, int order, bool f32)
{
    if (f32) return order == 1 && (rv == 3 || rv == 4);
    return order == 2 ? rv == 2 : (rv >= 2 && rv <= 4);
}

size_t tile_smem_bytes(int rv, int order, bool f32)
{
    if (f32) return rv == 3 ? sizeof(TileSmem<3, 1, float>) : sizeof(TileSmem<4, 1, float>);
    return order == 2 ? sizeof(TileSmem<2, 2, double>) : rv == 2 ? sizeof(TileSmem<2, 1, double>) : rv == 3 ? sizeof(TileSmem<3, 1, double>) : sizeof(TileSmem<4, 1, double>);
}

cudaError_t tile_configure(int rv, int order, bool f32, int wide_axis, int *ctas_per_sm)
{
    if (!tile_variant_exists(rv, order, f32)) return cudaErrorInvalidValue;
    if (f32) return rv == 3 ? configure<3, 1, float>(wide_axis, ctas_per_sm) : configure<4, 1, float>(wide_axis, ctas_per_sm);
    return order == 2 ? configure<2, 2, double>(wide_axis, ctas_per_sm) : rv == 2 ? configure<2, 1, double>(wide_axis, ctas_per_sm)
         : rv == 3 ? configure<3, 1, double>(wide_axis, ctas_per_sm) : configure<4, 1, double>(wide_axis, ctas_per_sm);
}

cudaError_t launch_sweep_tile(const TileParams &P, int rv, int order, bool f32, int wide_axis, int grid, cudaStream_t st)
{
    if (!tile_variant_exists(rv, order, f32)) return cudaErrorInvalidValue;
    if (f32) {
        if (rv == 3) launch<3, 1, float>(P, wide_axis, grid, st);
        else launch<4, 1, float>(P, wide_axis, grid, st);
    } else if (order == 2) launch<2, 2, double>(P, wide_axis, grid, st);
    else if (rv == 2) launch<2, 1, double>(P, wide_axis, grid, st);
    else if (rv == 3) launch<3, 1, double>(P, wide_axis, grid, st);
    else launch<4, 1, double>(P, wide_axis, grid, st);
    return cudaGetLastError();
}

}  // namespace dvm
