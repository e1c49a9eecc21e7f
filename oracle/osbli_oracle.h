/* osbli_oracle.h -- CPU ORACLE for the OpenSBLI residual + RK3 hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares
 * no code, header, table or helper with the CUDA path (include/osbli.h,
 * paper_2007_14933_b200/csrc); its parameter struct below is deliberately its own.
 *
 * Source of truth: /root/reference/PAPER.md (Lusher, Jammy & Sandham, arXiv 2007.14933),
 * cited as PAPER.md:<line>.  Where the paper is silent or garbled the reading taken is the
 * one listed in DESIGN.md ("Readings", Q1..Q31).
 *
 * Arithmetic: IEEE binary64, built with -O2 -ffp-contract=off (no FMA contraction, no
 * fast-math).  The only parallelism is an OpenMP "parallel for" over independent grid lines
 * (every output point is written by exactly one iteration, no reductions), so results are
 * bit-identical for any thread count.
 *
 * Array layout ("oracle layout", dense, not the GPU's padded layout): a scalar field is a
 * C-ordered array [NZ][NY][NX] with N_d = n_d + 2 h_d, h_d = 3 if n_d > 1 else 0 (halo
 * depth, "ghost (halo) points required by the shock-capturing schemes");
 * node (i,j,k) lives at ((k+h_z) NY + (j+h_y)) NX + (i+h_x).  A state is 5 such fields
 * back to back: rho, rho*u, rho*v, rho*w, rho*E (eq. 1-3).
 *
 * Pins (tests/test_oracle_*.py, all "-m 'not gpu'"): every function here is pinned, nothing
 * is "parity unpinned" -- see DESIGN.md "Pins".
 */
#ifndef OSBLI_ORACLE_H
#define OSBLI_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { ORACLE_WENOZ5 = 0, ORACLE_TENO5 = 1, ORACLE_TENO6 = 2, ORACLE_WENOJS5 = 3, ORACLE_CENTRAL4 = 4,
       ORACLE_WENOZ3 = 5, ORACLE_WENOZ7 = 6 /* 7th-order WENO-Z, four ghost points */ };
enum { ORACLE_VISC_NONE = 0, ORACLE_VISC_CONST = 1, ORACLE_VISC_SUTHERLAND = 2 };
enum { ORACLE_BC_PERIODIC = 0, ORACLE_BC_EXTRAP0 = 1, ORACLE_BC_DIRICHLET = 2, ORACLE_BC_WALL_ISOTHERMAL = 3,
       ORACLE_BC_WALL_ADIABATIC = 4 };
enum { ORACLE_PART_INVISCID = 1, ORACLE_PART_VISCOUS = 2 };
enum { ORACLE_AVG_ROE = 0, ORACLE_AVG_SIMPLE = 1 };            /* PAPER.md:104 step 2(a)                    */
enum { ORACLE_RK3_WILLIAMSON = 0, ORACLE_RK3_SSP = 1 };        /* PAPER.md:232, 242 (refs [23], [44])       */

typedef struct {
  int32_t n[3];           /* interior points nx, ny, nz; n_d == 1 => direction inactive             */
  double  delta[3];       /* grid spacing per direction (uniform mode)                              */
  int32_t curvilinear;    /* 0: uniform Cartesian; 1: metric arrays below are used                  */
  const double *D[3][3];  /* D[k][j] = d xi_k / d x_j, unit computational spacing    */
  const double *detJ;     /* det(d x / d xi)                                                        */
  const double *E[3][6];  /* E[l][ij] = d2 xi_l / dx_i dx_j, ij in {xx,xy,xz,yy,yz,zz}              */
  double  gamma, Re, Pr, Minf;
  int32_t scheme;         /* ORACLE_WENOZ5 | ORACLE_TENO5 | ORACLE_TENO6 | ORACLE_WENOJS5           */
  double  teno_ct;        /* C_T                                                      */
  double  eps;            /* epsilon of eq. (22), (25)                           */
  int32_t visc;           /* ORACLE_VISC_*                                                          */
  double  suth_ratio;     /* SuthT/RefT of the listing at                          */
  int32_t bc[3][2];       /* [direction][side]                                    */
  double  wall_T[3][2];   /* T_w of eq. (41)                                                        */
  const double *dirichlet;/* full state (oracle layout) holding frozen boundary values, or NULL     */
  int32_t nthreads;       /* OpenMP threads for the outer line loops (>= 1)                         */
  double  force[3];       /* constant body force per unit volume (channel case):  */
                          /* R_{rho u_i} += f_i, R_{rho E} += u_i f_i (Q34)               */
  int32_t averaging;      /* ORACLE_AVG_*: interface state of step 2(a) (Q11, Q38)        */
  int32_t rk3_form;       /* ORACLE_RK3_*: coefficients used by oracle_rk3_step (Q15, Q39) */
} oracle_params;

/* ---- building blocks, exposed so that the pins can reach them one by one ---------------- */

/* W(a,b,c,d,e): WENO-Z5 / TENO5 reconstruction at the interface between c and d, upwind side
 * a,b,c.  PAPER.md:117-128 (eq. 14-15), 138-143 (eq. 17-19), 165-167 (eq. 22), 173-190
 * (eq. 23-26).  *margin (may be NULL) receives min_r |chi_r/C_T - 1| for TENO (Q14),
 * +inf for WENO-Z. */
double oracle_reconstruct(int32_t scheme, double a, double b, double c, double d, double e,
                          double eps, double teno_ct, double *margin);

/* W6(a,b,c,d,e,f): TENO6 reconstruction at the interface between c and d, upwind side a,b,c
 * (eq. 23-25 and 27; candidates, ideal weights and beta_3: DESIGN.md Q32). */
double oracle_reconstruct6(double a, double b, double c, double d, double e, double f,
                           double eps, double teno_ct, double *margin);

/* beta_0 (R), beta_1 (C), beta_2 (L), beta_3 (4-point) and tau_6 of W6, for the pins. */
/* WENO-7Z value at i+1/2 from v7 = nodes i-3..i+3; out5 (may be NULL) = beta_0..beta_3, tau_7 */
double oracle_reconstruct7(const double *v7, double eps, double *out5);
void oracle_teno6_indicators(double a, double b, double c, double d, double e, double f, double *out5);

/* Roe-averaged eigensystem at an interface (step 2a-2b).  QL, QR: the two
 * 5-component conservative states; nhat: unit normal.  Outputs row-major 5x5 L (rows = left
 * eigenvectors), R (columns = right eigenvectors), and the Roe state (u,v,w,H,a). */
void oracle_eigensystem(double gamma, const double *QL, const double *QR, const double *nhat,
                        double *L, double *R, double *roe);

/* Same with the averaging of step 2(a) selectable (ORACLE_AVG_*; Q38). */
void oracle_eigensystem_avg(double gamma, int32_t averaging, const double *QL, const double *QR,
                            const double *nhat, double *L, double *R, double *roe);

/* 4th-order central first / second difference of a 1-D array f[0..n-1] at node i
 * (eq. 28 (sign corrected), 29, 30-35).  periodic != 0: f must carry 2
 * valid points either side of [0,n) (pass a pointer into a padded array). */
double oracle_d1(const double *f, int32_t n, int32_t i, int32_t periodic, double delta);
double oracle_d2(const double *f, int32_t n, int32_t i, int32_t periodic, double delta);

/* Reconstructed interface flux f^_{i+1/2} along direction dir at node (i,j,k), i.e. between
 * node (i,j,k) and its +1 neighbour along dir (steps 1-2).  Halos of Q must
 * be filled.  margin may be NULL. */
void oracle_interface_flux(const oracle_params *p, const double *Q, int32_t dir,
                           int32_t i, int32_t j, int32_t k, double *fhat, double *margin);

/* ---- the path --------------------------------------------------------------------------- */

int32_t oracle_halo(const oracle_params *p, int32_t *h);          /* h[3]                    */
int64_t oracle_field_size(const oracle_params *p);                /* NX*NY*NZ                */

/* Fill halos and boundary planes of Q in place.  Order: x, then
 * y over the x-extended range, then z over the x,y-extended range. */
int32_t oracle_bc(const oracle_params *p, double *Q);

/* R = dQ/dt on interior nodes (halo entries of R are left untouched).  parts: bit mask of
 * ORACLE_PART_*.  margin: NULL or one field (oracle layout) receiving, per node, the minimum
 * TENO margin over every reconstruction feeding that node. */
int32_t oracle_rhs(const oracle_params *p, const double *Q, double *R, int32_t parts, double *margin);

/* Same residual at npts listed nodes only (ijk = npts x 3 int32); out = npts x 5. */
int32_t oracle_rhs_points(const oracle_params *p, const double *Q, int32_t parts,
                          int64_t npts, const int32_t *ijk, double *out);

/* Metric terms from node coordinates ("evaluated by the same central interior
 * and boundary schemes ... computed once at the start").  coords: 3 fields x,y,z in oracle
 * layout whose halos hold the periodic continuation in periodic directions.  Outputs: D[9]
 * (D[k*3+j] = d xi_k/d x_j), detJ, E[18] (E[l*6+ij]) fields in oracle layout, halos filled.
 * Uses only p->n, p->bc (periodicity), p->delta (inactive directions) and p->nthreads. */
int32_t oracle_metrics(const oracle_params *p, const double *coords,
                       double *const *D, double *detJ, double *const *E);

/* One RK3 stage update on `count` contiguous values: dU = A_s dU + dt R; U += B_s dU
 * (eq. 36-37; s = 0,1,2).  oracle_rk3_step applies exactly this per x-line. */
void oracle_rk3_update(int32_t s, double dt, int64_t count, double *U, double *dU, const double *R);

/* The SSP member of the 3rd-order family (coefficients: DESIGN.md Q39). */
void oracle_rk3ssp_update(int32_t s, double dt, int64_t count, double *U, double *dU, const double *R);

/* One low-storage RK3 step (eq. 36-38): for s in 0..2 { bc(Q); R = rhs(Q);
 * dU = A_s dU + dt R; Q += B_s dU }; bc(Q).  dU and R are caller-provided scratch states.
 * p->rk3_form selects the coefficient set (Williamson [23] or SSP [44]). */
int32_t oracle_rk3_step(const oracle_params *p, double *Q, double *dU, double *R, double dt);

/* Five-stage 4th-order member of the same family (Q35). */
void oracle_rk4_update(int32_t s, double dt, int64_t count, double *U, double *dU, const double *R);
int32_t oracle_rk4_step(const oracle_params *p, double *Q, double *dU, double *R, double dt);

#ifdef __cplusplus
}
#endif
#endif
