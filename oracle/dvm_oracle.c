/*
 * dvm_oracle.c - CPU ORACLE (test infrastructure, see dvm_oracle.h) for one outer iteration of the
 * iterative discrete-velocity method of arXiv 1810.00348.
 *
 * Written step by step in the order of DESIGN.md "Oracle steps 0-7", each citing the passage of
 * /root/reference/PAPER.md it restates.  Deliberately plain: one full 3-D array f per velocity (the
 * form of ref. [60]), direct exp() / pow() / division per phase point, long-double
 * accumulation of the velocity sums in a fixed alpha order per thread.  OpenMP over velocities only
 * (velocities are independent inside an iteration).
 *
 * order = 2 ("extend the first order upwind scheme to second order by
 * storing three consecutive slices"): the paper gives no formula; reading G21 of DESIGN.md is the finite-volume
 * second-order upwind scheme, i.e. Eq.(7) with the cell values at the two faces of a cell replaced by values
 * extrapolated linearly from the two upwind cell centres, first order where the second upwind cell is missing.
 */
#include "dvm_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define PI 3.14159265358979323846264338327950288

typedef struct {
    int nface;
    int *face_of[6]; /* face_of[dir][cell] = face index if the neighbour in direction dir is not fluid, else -1 */
    int *bc_slot;    /* per face: 0..5 domain face, 6 solid */
    int *cell;       /* per face: adjacent fluid cell or -1 */
    int *dir;        /* per face: direction id seen from the cell */
    double *area;
} face_tab;

static int is_solid(const odvm_problem *p, int i, int j, int k)
{
    return p->solid && p->solid[((size_t)k * p->ny + j) * p->nx + i] != 0;
}

static void free_faces(face_tab *t)
{
    for (int d = 0; d < 6; ++d) free(t->face_of[d]);
    free(t->bc_slot); free(t->cell); free(t->dir); free(t->area);
}

/* Face table in the order stated in dvm_oracle.h */
static int build_faces(const odvm_problem *p, face_tab *t)
{
    const int nx = p->nx, ny = p->ny, nz = p->nz;
    const size_t n = (size_t)nx * ny * nz;
    memset(t, 0, sizeof *t);
    for (int d = 0; d < 6; ++d) {
        t->face_of[d] = (int *)malloc(n * sizeof(int));
        if (!t->face_of[d]) return -1;
        for (size_t c = 0; c < n; ++c) t->face_of[d][c] = -1;
    }
    const int off0 = 0, off1 = ny * nz, off2 = 2 * ny * nz, off3 = off2 + nx * nz, off4 = off3 + nx * nz,
              off5 = off4 + nx * ny, ndom = off5 + nx * ny;
    /* count solid-adjacent faces */
    int nsol = 0;
    static const int di[6] = {-1, 1, 0, 0, 0, 0}, dj[6] = {0, 0, -1, 1, 0, 0}, dk[6] = {0, 0, 0, 0, -1, 1};
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
        if (is_solid(p, i, j, k)) continue;
        for (int d = 0; d < 6; ++d) {
            int ii = i + di[d], jj = j + dj[d], kk = k + dk[d];
            if (ii < 0 || ii >= nx || jj < 0 || jj >= ny || kk < 0 || kk >= nz) continue;
            if (is_solid(p, ii, jj, kk)) ++nsol;
        }
    }
    t->nface = ndom + nsol;
    t->bc_slot = (int *)malloc(t->nface * sizeof(int));
    t->cell = (int *)malloc(t->nface * sizeof(int));
    t->dir = (int *)malloc(t->nface * sizeof(int));
    t->area = (double *)malloc(t->nface * sizeof(double));
    if (!t->bc_slot || !t->cell || !t->dir || !t->area) return -1;
    for (int f = 0; f < t->nface; ++f) { t->cell[f] = -1; t->dir[f] = 0; t->bc_slot[f] = 6; t->area[f] = 0; }
    int next = ndom;
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
        const int c = (k * ny + j) * nx + i;
        const double dx = p->xf[i + 1] - p->xf[i], dy = p->yf[j + 1] - p->yf[j], dz = p->zf[k + 1] - p->zf[k];
        const double ar[6] = {dy * dz, dy * dz, dx * dz, dx * dz, dx * dy, dx * dy};
        /* domain faces get their slot whether or not the cell is fluid */
        int dom[6] = {-1, -1, -1, -1, -1, -1};
        if (i == 0) dom[0] = off0 + k * ny + j;
        if (i == nx - 1) dom[1] = off1 + k * ny + j;
        if (j == 0) dom[2] = off2 + k * nx + i;
        if (j == ny - 1) dom[3] = off3 + k * nx + i;
        if (k == 0) dom[4] = off4 + j * nx + i;
        if (k == nz - 1) dom[5] = off5 + j * nx + i;
        const int sol = is_solid(p, i, j, k);
        for (int d = 0; d < 6; ++d) {
            if (dom[d] >= 0) {
                const int f = dom[d];
                t->bc_slot[f] = d; t->dir[f] = d; t->area[f] = ar[d];
                if (!sol) { t->cell[f] = c; t->face_of[d][c] = f; }
            } else if (!sol) {
                int ii = i + di[d], jj = j + dj[d], kk = k + dk[d];
                if (is_solid(p, ii, jj, kk)) {
                    const int f = next++;
                    t->bc_slot[f] = 6; t->dir[f] = d; t->area[f] = ar[d]; t->cell[f] = c;
                    t->face_of[d][c] = f;
                }
            }
        }
    }
    return 0;
}

int odvm_num_faces(const odvm_problem *p)
{
    face_tab t;
    if (build_faces(p, &t)) { free_faces(&t); return -1; }
    int n = t.nface;
    free_faces(&t);
    return n;
}

int odvm_face_table(const odvm_problem *p, int *cell, int *dir, double *area)
{
    face_tab t;
    if (build_faces(p, &t)) { free_faces(&t); return -1; }
    for (int f = 0; f < t.nface; ++f) { cell[f] = t.cell[f]; dir[f] = t.dir[f]; area[f] = t.area[f]; }
    int n = t.nface;
    free_faces(&t);
    return n;
}

/* ---- Step 0: constants (Eq.(2), 261-263 Eq.(10)) ------------------------------------ */
double odvm_c_omega(double omega)
{
    return 15.0 * sqrt(PI) / ((5.0 - 2.0 * omega) * (7.0 - 2.0 * omega));
}

double odvm_tau(const odvm_problem *p, double rho, double T)
{
    /* tau = mu/p with mu = mu_ref (T/T_ref)^omega, mu_ref from Eq.(10), lambda_ref = Kn L */
    return odvm_c_omega(p->omega) * p->Kn * pow(T, p->omega - 1.0) / rho;
}

double odvm_feq(const odvm_problem *p, const double *W, const double *xi)
{
    const double rho = W[0], T = W[4];
    const double cx = xi[0] - W[1], cy = xi[1] - W[2], cz = xi[2] - W[3];
    const double c2 = cx * cx + cy * cy + cz * cz;
    const double cq = cx * W[5] + cy * W[6] + cz * W[7];
    /* f^M = rho/(2 pi R T)^{3/2} exp(-c^2/(2RT)), with RT -> T/2 in v_m units */
    const double fM = rho / pow(PI * T, 1.5) * exp(-c2 / T);
    /* (1-Pr) c.q/(5 p R T) (c^2/(RT) - 5), p = rho T/2, RT = T/2 */
    return fM * (1.0 + (1.0 - p->Pr) * (4.0 / 5.0) * cq / (rho * T * T) * (2.0 * c2 / T - 5.0));
}

double odvm_gwall(const odvm_problem *p, int b, const double *xi)
{
    /* Eq.(8) with unit density and the wall velocity in the exponent (reading G3) */
    const double Tw = p->bc_T[b];
    const double cx = xi[0] - p->bc_u[b][0], cy = xi[1] - p->bc_u[b][1], cz = xi[2] - p->bc_u[b][2];
    return exp(-(cx * cx + cy * cy + cz * cz) / Tw) / pow(PI * Tw, 1.5);
}

static double ghost_freestream(const odvm_problem *p, int b, const double *xi)
{
    double W[8] = {p->bc_rho[b], p->bc_u[b][0], p->bc_u[b][1], p->bc_u[b][2], p->bc_T[b], 0, 0, 0};
    return odvm_feq(p, W, xi);
}

static void velocity(const odvm_problem *p, int ia, int ib, int ic, double *xi, double *w)
{
    xi[0] = p->xi_x[ia]; xi[1] = p->xi_y[ib]; xi[2] = p->xi_z[ic];
    *w = p->w_x[ia] * p->w_y[ib] * p->w_z[ic];
}

/* Phi_unit(face) = sum over velocities leaving the wall of w |xi_n| g_w  (Eq.(9) with weights, G4) */
static void phi_unit_faces(const odvm_problem *p, const face_tab *t, double *phi)
{
    /* one value per (bc slot, direction) pair is enough; compute the 7 x 6 table then scatter */
    long double tab[7][6];
    for (int b = 0; b < 7; ++b) for (int d = 0; d < 6; ++d) tab[b][d] = 0;
    for (int ic = 0; ic < p->mz; ++ic) for (int ib = 0; ib < p->my; ++ib) for (int ia = 0; ia < p->mx; ++ia) {
        double xi[3], w;
        velocity(p, ia, ib, ic, xi, &w);
        for (int b = 0; b < 7; ++b) {
            if (p->bc_type[b] != ODVM_WALL_DIFFUSE) continue;
            const double g = odvm_gwall(p, b, xi);
            for (int d = 0; d < 6; ++d) {
                /* wall lies on side d of the cell: its normal into the gas is -e_d; leaving the wall
                 * means xi.(-e_d) > 0 */
                const double xin = xi[d / 2] * ((d & 1) ? -1.0 : 1.0);
                if (xin > 0) tab[b][d] += (long double)(w * xin * g);
            }
        }
    }
    for (int f = 0; f < t->nface; ++f) {
        const int b = t->bc_slot[f];
        if (p->bc_type[b] != ODVM_WALL_DIFFUSE) { phi[f] = 0.0; continue; }
        phi[f] = p->wall_norm == 1 ? sqrt(p->bc_T[b] / (4.0 * PI)) : (double)tab[b][t->dir[f]];
    }
}

int odvm_phi_unit(const odvm_problem *p, double *phi_unit)
{
    face_tab t;
    if (build_faces(p, &t)) { free_faces(&t); return -1; }
    phi_unit_faces(p, &t, phi_unit);
    free_faces(&t);
    return 0;
}

int odvm_rho_equilibrium(const odvm_problem *p, const double *prim8, double *rhoS)
{
    const size_t n = (size_t)p->nx * p->ny * p->nz;
    for (size_t c = 0; c < n; ++c) {
        if (p->solid && p->solid[c]) { rhoS[c] = 0; continue; }
        double W[8];
        for (int m = 0; m < 8; ++m) W[m] = prim8[m * n + c];
        long double s = 0;
        for (int ic = 0; ic < p->mz; ++ic) for (int ib = 0; ib < p->my; ++ib) for (int ia = 0; ia < p->mx; ++ia) {
            double xi[3], w;
            velocity(p, ia, ib, ic, xi, &w);
            s += (long double)(w * odvm_feq(p, W, xi));
        }
        rhoS[c] = (double)s;
    }
    return 0;
}

double odvm_total_mass(const odvm_problem *p, const double *rho)
{
    long double m = 0;
    for (int k = 0; k < p->nz; ++k) for (int j = 0; j < p->ny; ++j) for (int i = 0; i < p->nx; ++i) {
        if (is_solid(p, i, j, k)) continue;
        const double V = (p->xf[i + 1] - p->xf[i]) * (p->yf[j + 1] - p->yf[j]) * (p->zf[k + 1] - p->zf[k]);
        m += (long double)(rho[((size_t)k * p->ny + j) * p->nx + i] * V);
    }
    return (double)m;
}

/* ---- Step 1: initial state ---------------------------------------------------------- */
int odvm_init_state(const odvm_problem *p, double rho0, const double *u0, double T0,
                    double *prim8, double *rho_w, double *mass0)
{
    const size_t n = (size_t)p->nx * p->ny * p->nz;
    face_tab t;
    if (build_faces(p, &t)) { free_faces(&t); return -1; }
    const double W0[8] = {rho0, u0[0], u0[1], u0[2], T0, 0, 0, 0};
    for (size_t c = 0; c < n; ++c) {
        const int sol = p->solid && p->solid[c];
        for (int m = 0; m < 8; ++m) prim8[m * n + c] = sol ? 0.0 : W0[m];
    }
    /* rho_w^0 = Phi^0 / Phi_unit, Phi^0 = flux of f^M(W^0) of the adjacent cell onto the wall */
    double *phi_u = (double *)malloc(t.nface * sizeof(double));
    if (!phi_u) { free_faces(&t); return -1; }
    phi_unit_faces(p, &t, phi_u);
    long double phi0[6] = {0, 0, 0, 0, 0, 0};
    for (int ic = 0; ic < p->mz; ++ic) for (int ib = 0; ib < p->my; ++ib) for (int ia = 0; ia < p->mx; ++ia) {
        double xi[3], w;
        velocity(p, ia, ib, ic, xi, &w);
        const double f0 = odvm_feq(p, W0, xi);
        for (int d = 0; d < 6; ++d) {
            const double xin = xi[d / 2] * ((d & 1) ? 1.0 : -1.0); /* towards side d */
            if (xin > 0) phi0[d] += (long double)(w * xin * f0);
        }
    }
    for (int f = 0; f < t.nface; ++f) {
        const int b = t.bc_slot[f];
        rho_w[f] = (p->bc_type[b] == ODVM_WALL_DIFFUSE && t.cell[f] >= 0) ? (double)phi0[t.dir[f]] / phi_u[f] : 0.0;
    }
    *mass0 = odvm_total_mass(p, prim8);
    free(phi_u);
    free_faces(&t);
    return 0;
}

/* ---- Step 2: sweep of one velocity (Eq.(7); Alg.2) --------------- */
typedef struct {
    long double *raw;      /* [13][ncell] or NULL */
    long double *flux_out; /* [nface] or NULL */
    long double *flux_in;  /* [nface] or NULL */
} accum;

static void sweep_one(const odvm_problem *p, const face_tab *t, const double *prim8, const double *rho_w,
                      const double *xi, double w, double *f, accum *acc)
{
    const int nx = p->nx, ny = p->ny, nz = p->nz;
    const size_t n = (size_t)nx * ny * nz;
    const int sx = xi[0] >= 0 ? 1 : -1, sy = xi[1] >= 0 ? 1 : -1, sz = xi[2] >= 0 ? 1 : -1;
    const int s[3] = {sx, sy, sz};
    const size_t stride[3] = {1, (size_t)nx, (size_t)nx * ny};
    /* ghost values that do not depend on the cell */
    double gw[7], gfs[7];
    for (int b = 0; b < 7; ++b) {
        gw[b] = p->bc_type[b] == ODVM_WALL_DIFFUSE ? odvm_gwall(p, b, xi) : 0.0;
        gfs[b] = p->bc_type[b] == ODVM_FREESTREAM ? ghost_freestream(p, b, xi) : 0.0;
    }
    const double xi2 = xi[0] * xi[0] + xi[1] * xi[1] + xi[2] * xi[2];
    /* f32 = 1 (reading G22 of DESIGN.md; "single precision computations"): the sweep runs in IEEE single.
     * Every number the update of Eq.(7) takes in or produces - tau, f^S, the coefficients a_d, the ghost values, the
     * running numerator and denominator, the quotient f_c - is rounded to single after the operation that makes it
     * (a double operation on singles followed by this rounding IS the single operation for + - * /).  The velocity
     * sums below stay in extended precision: only f is single. */
    const int f32 = p->f32 != 0;
#define SGL(x) (f32 ? (double)(float)(x) : (x))
    for (int b = 0; b < 7; ++b) { gw[b] = SGL(gw[b]); gfs[b] = SGL(gfs[b]); }
    for (int kk = 0; kk < nz; ++kk) {
        const int k = sz > 0 ? kk : nz - 1 - kk;
        for (int jj = 0; jj < ny; ++jj) {
            const int j = sy > 0 ? jj : ny - 1 - jj;
            for (int ii = 0; ii < nx; ++ii) {
                const int i = sx > 0 ? ii : nx - 1 - ii;
                const size_t c = ((size_t)k * ny + j) * nx + i;
                if (p->solid && p->solid[c]) { f[c] = 0.0; continue; }
                double W[8];
                for (int m = 0; m < 8; ++m) W[m] = prim8[m * n + c];
                const double tau = SGL(odvm_tau(p, W[0], W[4]));
                const double a[3] = {SGL(fabs(xi[0]) / (p->xf[i + 1] - p->xf[i])),
                                     SGL(fabs(xi[1]) / (p->yf[j + 1] - p->yf[j])),
                                     SGL(fabs(xi[2]) / (p->zf[k + 1] - p->zf[k]))};
                double num = SGL(SGL(odvm_feq(p, W, xi)) / tau);
                double den = SGL(1.0 / tau);
                int zg_face[3] = {-1, -1, -1};
                double psi[3] = {0.0, 0.0, 0.0}, f1v[3] = {0.0, 0.0, 0.0};
                for (int d = 0; d < 3; ++d) {
                    const int up = 2 * d + (s[d] > 0 ? 0 : 1); /* side of the cell the flow comes from */
                    const int face = t->face_of[up][c];
                    double fu;
                    if (face < 0) {
                        const size_t c1 = c - (size_t)((long)s[d] * (long)stride[d]);
                        fu = f[c1];
                        if (p->order == 2) {
                            /* Reading G21.  Value at the downwind face of a cell = its value extrapolated linearly
                             * from the two upwind centres: F(c) = f_c + psi_c (f_c - f_c1), psi_c = w_c / (w_c + w_c1)
                             * (w = cell widths along d); F(c) = f_c if c1 is not a fluid cell.  The transport term of
                             * Eq.(7) along d becomes a_d (F(c) - F(c1)); F(c1) likewise needs c2. */
                            const int idx[3] = {i, j, k};
                            const double *xfd = d == 0 ? p->xf : d == 1 ? p->yf : p->zf;
                            const int q = idx[d], q1 = q - s[d];
                            const double wc = xfd[q + 1] - xfd[q], w1 = xfd[q1 + 1] - xfd[q1];
                            psi[d] = wc / (wc + w1);
                            f1v[d] = fu;
                            double Fup = fu;
                            if (t->face_of[up][c1] < 0) {
                                const size_t c2 = c1 - (size_t)((long)s[d] * (long)stride[d]);
                                const int q2 = q1 - s[d];
                                const double w2 = xfd[q2 + 1] - xfd[q2];
                                Fup = fu + w1 / (w1 + w2) * (fu - f[c2]);
                            }
                            /* a_d [(1 + psi) f_c - psi f_c1 - Fup] : the f_c part goes to the denominator */
                            num += a[d] * (psi[d] * fu + Fup);
                            den += a[d] * (1.0 + psi[d]);
                            continue;
                        }
                    } else {
                        const int b = t->bc_slot[face];
                        if (p->bc_type[b] == ODVM_WALL_DIFFUSE) fu = SGL(rho_w[face] * gw[b]);
                        else if (p->bc_type[b] == ODVM_FREESTREAM) fu = gfs[b];
                        else { zg_face[d] = face; continue; } /* zero gradient: drop the term */
                        if (acc && acc->flux_in) acc->flux_in[face] += (long double)(w * fabs(xi[d]) * fu);
                    }
                    num = SGL(num + SGL(a[d] * fu));
                    den = SGL(den + a[d]);
                }
                const double fc = SGL(num / den);
                f[c] = fc;
                if (!acc) continue;
                /* value at the downwind faces of the cell: f_c (order 1), extrapolated (order 2, G21) */
                double Fdn[3];
                for (int d = 0; d < 3; ++d) Fdn[d] = fc + psi[d] * (fc - f1v[d]);
                for (int d = 0; d < 3; ++d)
                    if (zg_face[d] >= 0 && acc->flux_in) acc->flux_in[zg_face[d]] += (long double)(w * fabs(xi[d]) * Fdn[d]);
                /* ---- Step 3: raw moments (Eq.(5)) ---- */
                if (acc->raw) {
                    const long double wf = (long double)w * (long double)fc;
                    long double *r = acc->raw;
                    r[0 * n + c] += wf;
                    r[1 * n + c] += wf * xi[0];
                    r[2 * n + c] += wf * xi[1];
                    r[3 * n + c] += wf * xi[2];
                    r[4 * n + c] += wf * (xi[0] * xi[0]);
                    r[5 * n + c] += wf * (xi[1] * xi[1]);
                    r[6 * n + c] += wf * (xi[2] * xi[2]);
                    r[7 * n + c] += wf * (xi[0] * xi[1]);
                    r[8 * n + c] += wf * (xi[0] * xi[2]);
                    r[9 * n + c] += wf * (xi[1] * xi[2]);
                    r[10 * n + c] += wf * (xi[0] * xi2);
                    r[11 * n + c] += wf * (xi[1] * xi2);
                    r[12 * n + c] += wf * (xi[2] * xi2);
                }
                /* ---- Step 4: flux onto the downwind boundary faces (Eq.(9)) ---- */
                if (acc->flux_out) {
                    for (int d = 0; d < 3; ++d) {
                        const int dn = 2 * d + (s[d] > 0 ? 1 : 0);
                        const int face = t->face_of[dn][c];
                        if (face >= 0) acc->flux_out[face] += (long double)(w * fabs(xi[d]) * Fdn[d]);
                    }
                }
            }
        }
    }
#undef SGL
}

int odvm_sweep_velocity(const odvm_problem *p, const double *prim8_in, const double *rho_w_in,
                        int ia, int ib, int ic, double *f_out)
{
    face_tab t;
    if (build_faces(p, &t)) { free_faces(&t); return -1; }
    double xi[3], w;
    velocity(p, ia, ib, ic, xi, &w);
    sweep_one(p, &t, prim8_in, rho_w_in, xi, w, f_out, NULL);
    free_faces(&t);
    return 0;
}

/* ---- Steps 2-7 ------------------------------------------------------------------------------------ */
int odvm_step(const odvm_problem *p, const double *prim8_in, const double *rho_w_in, double mass0,
              double *raw13_out, double *prim14_out, double *rho_w_out,
              double *flux_out, double *flux_in, double *resid3, double *scale, int nthreads)
{
    const int nx = p->nx, ny = p->ny, nz = p->nz;
    const size_t n = (size_t)nx * ny * nz;
    const long nvel = (long)p->mx * p->my * p->mz;
    face_tab t;
    if (p->f32 && p->order == 2) return -2; /* the single-precision sweep is stated for Eq.(7) only (G22) */
    if (build_faces(p, &t)) { free_faces(&t); return -1; }
    const int nface = t.nface;
    int nt = 1;
#ifdef _OPENMP
    nt = nthreads > 0 ? nthreads : omp_get_max_threads();
#endif
    if (nt > nvel) nt = (int)nvel;
    long double **raw_t = (long double **)calloc(nt, sizeof *raw_t);
    long double **fo_t = (long double **)calloc(nt, sizeof *fo_t);
    long double **fi_t = (long double **)calloc(nt, sizeof *fi_t);
    int fail = 0;
#pragma omp parallel num_threads(nt)
    {
#ifdef _OPENMP
        const int tid = omp_get_thread_num();
#else
        const int tid = 0;
#endif
        double *f = (double *)malloc(n * sizeof(double));
        raw_t[tid] = (long double *)calloc(13 * n, sizeof(long double));
        fo_t[tid] = (long double *)calloc(nface, sizeof(long double));
        fi_t[tid] = (long double *)calloc(nface, sizeof(long double));
        if (!f || !raw_t[tid] || !fo_t[tid] || !fi_t[tid]) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp barrier
        if (!fail) {
            accum acc = {raw_t[tid], fo_t[tid], fi_t[tid]};
            /* contiguous alpha blocks per thread, alpha = (ic*my + ib)*mx + ia, ascending */
            const long lo = nvel * tid / nt, hi = nvel * (tid + 1) / nt;
            for (long al = lo; al < hi; ++al) {
                const int ia = (int)(al % p->mx), ib = (int)((al / p->mx) % p->my), ic = (int)(al / ((long)p->mx * p->my));
                double xi[3], w;
                velocity(p, ia, ib, ic, xi, &w);
                if (w == 0.0) continue;
                sweep_one(p, &t, prim8_in, rho_w_in, xi, w, f, &acc);
            }
        }
        free(f);
    }
    if (fail) {
        for (int q = 0; q < nt; ++q) { free(raw_t[q]); free(fo_t[q]); free(fi_t[q]); }
        free(raw_t); free(fo_t); free(fi_t); free_faces(&t);
        return -2;
    }
    /* combine the per-thread partial sums in thread order */
    for (size_t e = 0; e < 13 * n; ++e) {
        long double sum = 0;
        for (int q = 0; q < nt; ++q) sum += raw_t[q][e];
        raw13_out[e] = (double)sum;
    }
    double *phi_u = (double *)malloc(nface * sizeof(double));
    phi_unit_faces(p, &t, phi_u);
    for (int f = 0; f < nface; ++f) {
        long double so = 0, si = 0;
        for (int q = 0; q < nt; ++q) { so += fo_t[q][f]; si += fi_t[q][f]; }
        if (flux_out) flux_out[f] = (double)so;
        if (flux_in) flux_in[f] = (double)si;
        const int b = t.bc_slot[f];
        rho_w_out[f] = (p->bc_type[b] == ODVM_WALL_DIFFUSE && t.cell[f] >= 0) ? (double)so / phi_u[f] : 0.0;
    }
    for (int q = 0; q < nt; ++q) { free(raw_t[q]); free(fo_t[q]); free(fi_t[q]); }
    free(raw_t); free(fo_t); free(fi_t); free(phi_u);

    /* ---- Step 5: raw -> primitive (Eq.(3)) ---- */
    for (size_t c = 0; c < n; ++c) {
        if (p->solid && p->solid[c]) { for (int m = 0; m < 14; ++m) prim14_out[m * n + c] = 0.0; continue; }
        const double *r = raw13_out;
        const double rho = r[c];
        const double U[3] = {r[1 * n + c] / rho, r[2 * n + c] / rho, r[3 * n + c] / rho};
        const double m2[3][3] = {{r[4 * n + c], r[7 * n + c], r[8 * n + c]},
                                 {r[7 * n + c], r[5 * n + c], r[9 * n + c]},
                                 {r[8 * n + c], r[9 * n + c], r[6 * n + c]}};
        const double m3[3] = {r[10 * n + c], r[11 * n + c], r[12 * n + c]};
        double P[3][3];
        for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) P[a][b] = m2[a][b] - rho * U[a] * U[b];
        const double trP = P[0][0] + P[1][1] + P[2][2];
        const double trm2 = m2[0][0] + m2[1][1] + m2[2][2];
        const double U2 = U[0] * U[0] + U[1] * U[1] + U[2] * U[2];
        const double T = (2.0 / 3.0) * trP / rho; /* p = rho T/2 = trP/3 */
        double q[3];
        for (int a = 0; a < 3; ++a) {
            const double Um2 = U[0] * m2[a][0] + U[1] * m2[a][1] + U[2] * m2[a][2];
            q[a] = 0.5 * (m3[a] - 2.0 * Um2 - U[a] * trm2 + 2.0 * rho * U[a] * U2);
        }
        double *o = prim14_out;
        o[0 * n + c] = rho; o[1 * n + c] = U[0]; o[2 * n + c] = U[1]; o[3 * n + c] = U[2]; o[4 * n + c] = T;
        o[5 * n + c] = q[0]; o[6 * n + c] = q[1]; o[7 * n + c] = q[2];
        o[8 * n + c] = P[0][0] - trP / 3.0; o[9 * n + c] = P[1][1] - trP / 3.0; o[10 * n + c] = P[2][2] - trP / 3.0;
        o[11 * n + c] = P[0][1]; o[12 * n + c] = P[0][2]; o[13 * n + c] = P[1][2];
    }

    /* ---- Step 6: global mass rescale for closed domains (reading G8) ---- */
    double sfac = 1.0;
    if (p->rescale_mass) {
        sfac = mass0 / odvm_total_mass(p, prim14_out);
        static const int lin[10] = {0, 5, 6, 7, 8, 9, 10, 11, 12, 13}; /* rho, q, sigma: linear in f */
        for (int m = 0; m < 10; ++m) for (size_t c = 0; c < n; ++c) prim14_out[lin[m] * n + c] *= sfac;
        for (int f = 0; f < nface; ++f) rho_w_out[f] *= sfac;
    }
    if (scale) *scale = sfac;

    /* ---- Step 7: residual (reading G9) ---- */
    if (resid3) {
        long double num[3] = {0, 0, 0}, den[3] = {0, 0, 0};
        for (size_t c = 0; c < n; ++c) {
            if (p->solid && p->solid[c]) continue;
            const double r1 = prim14_out[c], r0 = prim8_in[c];
            const double T1 = prim14_out[4 * n + c], T0 = prim8_in[4 * n + c];
            double u1s = 0, u0s = 0;
            for (int a = 0; a < 3; ++a) {
                const double u1 = prim14_out[(1 + a) * n + c], u0 = prim8_in[(1 + a) * n + c];
                const double dm = r1 * u1 - r0 * u0;
                num[1] += (long double)(dm * dm);
                den[1] += (long double)((r1 * u1) * (r1 * u1));
                u1s += u1 * u1; u0s += u0 * u0;
            }
            const double E1 = 0.75 * r1 * T1 + 0.5 * r1 * u1s, E0 = 0.75 * r0 * T0 + 0.5 * r0 * u0s;
            num[0] += (long double)((r1 - r0) * (r1 - r0)); den[0] += (long double)(r1 * r1);
            num[2] += (long double)((E1 - E0) * (E1 - E0)); den[2] += (long double)(E1 * E1);
        }
        for (int m = 0; m < 3; ++m) {
            if (den[m] > 0) resid3[m] = (double)sqrtl(num[m] / den[m]);
            else resid3[m] = num[m] > 0 ? INFINITY : 0.0;
        }
    }
    free_faces(&t);
    return nt;
}
