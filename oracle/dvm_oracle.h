/*
 * dvm_oracle.h - CPU ORACLE for one outer iteration of the iterative discrete-velocity method of
 * arXiv 1810.00348 (steady 3D3V Shakhov/BGK model equation, first-order upwind sweep; second-order upwind as the
 * paper's stated extension).
 *
 * THIS IS TEST INFRASTRUCTURE.  It is a plain, slow, obviously-correct restatement of the paper's
 * scheme (one full 3-D array f[k][j][i] per discrete velocity, direct exp/pow, division, no slices, no
 * batching, no tiling).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / reference
 * legs may call it.  It shares no code with the CUDA path under paper_1810_00348_b200/csrc and neither
 * side includes or imports the other.
 *
 * Units (reading G2): speeds in v_m = sqrt(2 R T0), density in rho0, temperature in T0,
 * lengths in L, f in rho0 / v_m^3, heat flux in rho0 v_m^3, stress in rho0 v_m^2.
 *
 * Cell index c = (k*ny + j)*nx + i.  Direction ids: 0 = x-, 1 = x+, 2 = y-, 3 = y+, 4 = z-, 5 = z+.
 * Boundary-face table (one rho_w / flux slot per face, whatever its BC type):
 *   domain faces first: x- [k*ny+j], x+ [k*ny+j], y- [k*nx+i], y+ [k*nx+i], z- [j*nx+i], z+ [j*nx+i],
 *   then the faces between a fluid cell and a solid cell inside the domain, ordered by
 *   (fluid cell index ascending, direction id ascending).
 *
 * Pins (run with -m "not gpu"): tests/test_oracle_pins.py (P1-P16 of DESIGN.md), tests/test_oracle_order2.py (order = 2),
 * tests/test_oracle_f32.py (f32 = 1).  Every function here is pinned.  The converged solution is pinned against its closed form in
 * the free-molecular limit (P17, P18); for the cavity / cube fields at finite Kn the paper prints no value to pin against
 * (PAPER.md:271, 295).
 */
#ifndef DVM_ORACLE_H
#define DVM_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

enum { ODVM_WALL_DIFFUSE = 0, ODVM_FREESTREAM = 1, ODVM_ZERO_GRADIENT = 2 };

typedef struct {
    int nx, ny, nz;
    const double *xf, *yf, *zf;     /* face coordinates, n+1 each */
    const unsigned char *solid;     /* nz*ny*nx, 1 = solid, or NULL */
    int mx, my, mz;
    const double *xi_x, *xi_y, *xi_z; /* velocity nodes per axis */
    const double *w_x, *w_y, *w_z;    /* 1-D weights; w_alpha = product */
    double Kn, omega, Pr;
    int    bc_type[7];              /* 0..5 domain faces, 6 = faces of solid cells */
    double bc_T[7], bc_rho[7], bc_u[7][3];
    int rescale_mass;               /* 1 = apply the global mass rescale */
    int wall_norm;                  /* 0 = discrete Phi_unit (G4), 1 = analytic constant of Eq.(9) */
    int order;                      /* 1 = first-order upwind, Eq.(7); 2 = second-order upwind (reading G21) */
    int f32;                        /* 0 = everything in double; 1 = the sweep of Eq.(7) in IEEE single, velocity sums in extended
                                     * precision (the paper's timing precision; reading G22); order 1 only */
} odvm_problem;

/* number of boundary faces (domain + solid); fills nothing */
int odvm_num_faces(const odvm_problem *p);
/* for every face: adjacent fluid cell (or -1 if that domain-face cell is solid), direction id seen from
 * that cell, face area */
int odvm_face_table(const odvm_problem *p, int *cell, int *dir, double *area);

/* C_omega = 15 sqrt(pi) / ((5-2w)(7-2w))  - Eq.(10) */
double odvm_c_omega(double omega);
/* relaxation time tau = C_omega Kn T^(omega-1) / rho  - PAPER.md:43, 261-263 */
double odvm_tau(const odvm_problem *p, double rho, double T);
/* Shakhov equilibrium f^S (Eq.(2)) at velocity xi[3] for W = rho,ux,uy,uz,T,qx,qy,qz */
double odvm_feq(const odvm_problem *p, const double *W8, const double *xi3);
/* wall Maxwellian of unit density g_w (Eq.(8), reading G3) for BC slot b (0..6) */
double odvm_gwall(const odvm_problem *p, int b, const double *xi3);
/* Phi_unit per face (0 for non-wall faces) - Eq.(9) with weights, reading G4 */
int odvm_phi_unit(const odvm_problem *p, double *phi_unit);
/* discrete density of the equilibrium: rhoS[c] = sum_alpha w_alpha f^S_alpha(W_c) (used by pin P4) */
int odvm_rho_equilibrium(const odvm_problem *p, const double *prim8, double *rhoS);

/* Step 1: uniform state -> prim8 [8][ncell], rho_w [nface], *mass0 = sum rho V */
int odvm_init_state(const odvm_problem *p, double rho0, const double *u0, double T0,
                    double *prim8, double *rho_w, double *mass0);

/* total mass sum_c rho_c V_c over fluid cells */
double odvm_total_mass(const odvm_problem *p, const double *rho);

/* Steps 2-7: one outer iteration  (W^n, rho_w^n) -> (raw13, prim14^{n+1}, rho_w^{n+1}, residual).
 *   prim8_in  [8][ncell]  rho,ux,uy,uz,T,qx,qy,qz           rho_w_in [nface]
 *   raw13_out [13][ncell] sum w f {1, xi_x,xi_y,xi_z, xx,yy,zz,xy,xz,yz, x|xi|^2,y|xi|^2,z|xi|^2}
 *   prim14_out[14][ncell] rho,ux,uy,uz,T,qx,qy,qz,sxx,syy,szz,sxy,sxz,syz (after the rescale)
 *   rho_w_out [nface], flux_out [nface] = sum_{leaving the domain} w |xi_n| f_face (f_face = f_cell for order 1),
 *   flux_in [nface] = sum_{entering} w |xi_n| f_ghost (diagnostic for pin P4),
 *   resid[3] = r_rho, r_mom, r_E;  *scale = mass-rescale factor s (1 if off).
 * Velocities whose weight is exactly 0 are skipped.  nthreads <= 0 -> all OpenMP threads.
 * Returns the number of threads used, or < 0 on error. */
int odvm_step(const odvm_problem *p, const double *prim8_in, const double *rho_w_in, double mass0,
              double *raw13_out, double *prim14_out, double *rho_w_out,
              double *flux_out, double *flux_in, double *resid3, double *scale, int nthreads);

/* the field f[k][j][i] of ONE velocity (ia, ib, ic) for the given state (pins P5, P6, P9) */
int odvm_sweep_velocity(const odvm_problem *p, const double *prim8_in, const double *rho_w_in,
                        int ia, int ib, int ic, double *f_out);

#ifdef __cplusplus
}
#endif
#endif
