/* osbli.h -- C ABI of libosbli: the per-RK-stage residual + low-storage RK3 hot path of
 * OpenSBLI's method (Lusher, Jammy & Sandham, arXiv 2007.14933; cited as PAPER.md:<line>)
 * for one NVIDIA B200 (sm_100a), fp64.
 *
 * What the library computes (every step runs in hand-written CUDA kernels; there is no CPU
 * fallback and no other back-end):
 *   - osbli_bc        halo / boundary-plane fill                 PAPER.md:363-385 (eq. 40-46), 503, 586
 *   - osbli_rhs       R = -sum_d delta_d f^_d + viscous terms     PAPER.md:100-111 (steps 1-4),
 *                     characteristic WENO-Z5 / TENO5 + LLF         117-194 (eq. 14-26), 85-98 (eq. 11-13),
 *                     + 4th-order central viscous / heat flux      45-57 (eq. 1-5), 198-228 (eq. 28-35)
 *   - osbli_rk3_step  3-stage low-storage Runge-Kutta step         PAPER.md:232-242 (eq. 36-38)
 *   - osbli_rk4_step  5-stage 4th-order member of the same family
 *   - osbli_rk3_step_static  osbli_rk3_step without a handle or a caller workspace (static scratch, <= 64 MiB)
 *   - osbli_advance_host  same, from/to HOST memory (copies inside)
 *
 * Conventions
 *   - All functions return an int status (OSBLI_OK = 0).  No exceptions, no global state.
 *   - "device pointer" = address valid on the current CUDA device; "host pointer" = ordinary
 *     (preferably pinned) host memory.  Each argument below says which.
 *   - cuda_stream is a cudaStream_t passed as void* (NULL = legacy default stream).
 *   - osbli_bc / osbli_rhs / osbli_rk3_step only ENQUEUE work on the stream and return; they
 *     never synchronise.  osbli_advance_host synchronises the stream before returning.
 *   - Ownership: the caller owns every buffer (state arrays, workspace, metric fields, the
 *     Dirichlet state).  The library borrows the pointers given to osbli_init for the life of
 *     the handle and never allocates or frees device memory.
 *
 * State layout ("padded SoA", described by osbli_layout): a state is 5 scalar fields back to
 * back -- rho, rho*u, rho*v, rho*w, rho*E -- each a 3-D array, x fastest.
 * Node (i,j,k) of variable c, with i in [-halo[0], nx+halo[0]) etc., lives at
 *     c*stride_var + (k+halo[2])*stride_z + (j+halo[1])*stride_y + x_offset + i        (doubles)
 * halo[d] = 3 for an active direction (n_d > 1; "ghost points required by the
 * shock-capturing schemes"; 4 with OSBLI_SCHEME_WENOZ7, stencil i-3..i+4), 0 for an inactive one (n_d == 1: no halo, no sweep).  x_offset and
 * stride_y are multiples of 16 doubles so that interior node i = 0 of every row is 128-byte
 * aligned when the base pointer is.  Metric fields and the Dirichlet state use the same layout
 * (one field / five fields).  Entries that are neither interior nor halo are never read.
 */
#ifndef OSBLI_H
#define OSBLI_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct osbli_ctx *osbli_handle;

enum { OSBLI_OK = 0, OSBLI_EINVAL = 1, OSBLI_EUNSUPPORTED = 2, OSBLI_ECUDA = 3, OSBLI_EWORKSPACE = 4,
       OSBLI_ESTATIC = 5 /* osbli_rk3_step_static only: the problem exceeds OSBLI_STATIC_SCRATCH_BYTES */ };
enum { OSBLI_SCHEME_WENOZ5 = 0, OSBLI_SCHEME_TENO5 = 1, OSBLI_SCHEME_TENO6 = 2,
       OSBLI_SCHEME_WENOJS5 = 3 /* eq. (20)-(21); set eps = 1e-6 */,
       OSBLI_SCHEME_CENTRAL4 = 4 /* eq. (28) on the flux vectors, no shock capturing; uniform grids */,
       OSBLI_SCHEME_WENOZ3 = 5 /* third-order WENO-Z */,
       OSBLI_SCHEME_WENOZ7 = 6 /* seventh-order WENO-Z: halo 4, untuned sweeps,
                                  separate stage update */ };
enum { OSBLI_VISC_NONE = 0 /* Euler */, OSBLI_VISC_CONST = 1 /* mu = 1 */,
       OSBLI_VISC_SUTHERLAND = 2 /* PAPER.md:59-63, 317-318 */ };
enum { OSBLI_BC_PERIODIC = 0, OSBLI_BC_EXTRAP0 = 1, OSBLI_BC_DIRICHLET = 2,
       OSBLI_BC_WALL_ISOTHERMAL = 3, OSBLI_BC_WALL_ADIABATIC = 4 };
enum { OSBLI_AVG_ROE = 0 /* sqrt(rho)-weighted u_j, H */,
       OSBLI_AVG_SIMPLE = 1 /* U_{i+1/2} = (U_i + U_{i+1})/2 */ };               /* PAPER.md:104 step 2(a) */
enum { OSBLI_RK3_WILLIAMSON = 0 /* coefficients of ref. [23] */,
       OSBLI_RK3_SSP = 1 /* strong-stability-preserving set of ref. [44] */ };

/* Curvilinear metric fields, DEVICE pointers, each one scalar field in the
 * padded layout with halos filled.  Unit computational spacing in every direction. */
typedef struct {
  const double *D[3][3];   /* D[k][j] = d xi_k / d x_j                                          */
  const double *detJ;      /* det(d x / d xi)                                                    */
  const double *E[3][6];   /* E[l][ij] = d2 xi_l / dx_i dx_j, ij in {xx,xy,xz,yy,yz,zz};
                              read only when visc != OSBLI_VISC_NONE                             */
} osbli_metrics;

typedef struct {
  int32_t nx, ny, nz;      /* interior points per direction; n_d == 1 => direction inactive;
                              an active direction needs n_d >= 5                                 */
  double  dx, dy, dz;      /* uniform spacings, used when metrics == NULL                        */
  const osbli_metrics *metrics;  /* HOST pointer to a struct of DEVICE pointers, or NULL for a
                              uniform Cartesian grid.  The struct is copied by osbli_init.       */
  double  gamma, Re, Pr, Minf;
  int32_t scheme;          /* OSBLI_SCHEME_*                                                     */
  double  teno_ct;         /* TENO cut-off C_T, eq. (23)-(24), PAPER.md:177, 194 (e.g. 1e-6)     */
  double  eps;             /* epsilon of eq. (22), (25), PAPER.md:167, 188 (e.g. 1e-16); must be
                              >= 1e-18: the division-free weight forms raise (beta+eps) to the
                              18th power, which must stay inside the binary64 range; for the
                              same reason characteristic-variable jumps must stay below ~1e7
                              (non-dimensional variables, as everywhere in the paper)            */
  int32_t visc;            /* OSBLI_VISC_*                                                       */
  double  suth_ratio;      /* SuthT/RefT of PAPER.md:317-318                                     */
  int32_t bc[3][2];        /* [direction][side]; PERIODIC must be set on both sides or neither   */
  double  wall_T[3][2];    /* T_w of eq. (41) where bc == OSBLI_BC_WALL_ISOTHERMAL               */
  const double *dirichlet; /* DEVICE pointer to a full state (padded layout) holding the frozen
                              boundary values, required iff some bc == OSBLI_BC_DIRICHLET        */
  double  force[3];        /* constant body force per unit volume (laminar channel):
                              dQ/dt gains f_i in the momentum and u_i f_i in the energy equation  */
  int32_t averaging;       /* OSBLI_AVG_*: interface state whose eigenvectors diagonalise the fluxes,
                              PAPER.md:104 "either simple or Roe averaging"                        */
  int32_t rk3_form;        /* OSBLI_RK3_*: coefficient set A_i, B_i used by osbli_rk3_step          */
} osbli_params;

typedef struct {
  int32_t halo[3];
  int64_t x_offset, stride_y, stride_z, stride_var, total_doubles;  /* total = 5 * stride_var   */
} osbli_layout;

/* Layout of a state for these grid dimensions.  Host only, pure (reads nx, ny, nz).
 * OSBLI_EINVAL if a dimension is < 1 or an active one is < 5. */
int osbli_get_layout(const osbli_params *p, osbli_layout *out);

/* Bytes of device workspace osbli_init needs: three states (the residual R and the two
 * intermediate states Q2, Q3 of osbli_rk3_step, see there) and, when visc != NONE, the staged
 * primitive fields u, v, w, T (and mu for Sutherland) with their first differences along x, y, z
 * (16 or 20 scalar fields; "store some"). */
int osbli_workspace_bytes(const osbli_params *p, size_t *out);

/* Validates *p, records it and the workspace (DEVICE pointer, 256-byte aligned, >= the size
 * above, else OSBLI_EWORKSPACE).  Errors: OSBLI_EINVAL (sizes, enum values, periodic flags not
 * paired, gamma <= 1, eps < 1e-18, missing dirichlet / metrics pointers), OSBLI_EUNSUPPORTED
 * (nx == 1: x is the contiguous direction and must be active; boundary types of an inactive
 * direction are ignored), OSBLI_ECUDA (no sm_100 device / runtime failure). */
/* A handle whose configuration takes the general viscous path (non-periodic, curvilinear or Sutherland) also owns one
 * CUDA stream and two events: osbli_rhs / osbli_rk3_step form the staged primitive fields and their first differences
 * on it, next to the first sweeps, forked from and joined back into the caller's stream by events (nothing is
 * synchronised on the host; to the caller the work stays ordered on the stream it passed). */
int osbli_init(const osbli_params *p, void *d_workspace, size_t workspace_bytes, osbli_handle *out);

/* Fill the halos (depth layout.halo) (and, for DIRICHLET / WALL, the boundary plane) of device state Q in
 * place: x, then y over the x-extended range, then z over the x,y-extended range, so edges and
 * corners are defined.  PERIODIC: wrap.  EXTRAP0: zero-order extrapolation of the boundary
 * node.  DIRICHLET: boundary plane + halos copied from params.dirichlet
 * (PAPER.md:493, 586).  WALL_ISOTHERMAL: eq. (40)-(46).  WALL_ADIABATIC: the same
 * with T_w = (48 T_1 - 36 T_2 + 16 T_3 - 3 T_4)/25 from the interior nodes of the wall-normal line
 * (one-sided 4th-order dT/dn = 0). */
int osbli_bc(osbli_handle h, double *d_Q, void *cuda_stream);

/* d_R <- dQ/dt on interior nodes (halo / pad entries of R untouched):
 * R = -sum over active directions of (f^_{i+1/2} - f^_{i-1/2})/Delta (or /detJ)
 * eq. (10), with f^ from the characteristic reconstruction of PAPER.md:100-111, plus the
 * viscous and heat-flux terms of eq. (2)-(5) when visc != NONE.  Halos of d_Q must be filled
 * (osbli_bc).  d_R must not alias d_Q.  Uses the primitive-field part of the workspace. */
int osbli_rhs(osbli_handle h, const double *d_Q, double *d_R, void *cuda_stream);

/* One low-storage RK3 step, eq. (36)-(38): for s in 0..2 { bc(Q); R = rhs(Q);
 * Qtmp = A_s Qtmp + dt R; Q += B_s Qtmp } then bc(Q).  d_Qtmp is the dU accumulator of eq. (36);
 * it is overwritten (A_0 = 0) and need not be initialised.  R lives in the workspace.
 * A_i, B_i: params.rk3_form (Williamson's 2N-storage scheme, or the SSP set whose A_3 is 0 as well).
 * With two or more active directions the update is done by the last sweep kernel of each stage
 * (no separate pass over R), which cannot update in place: the state moves d_Q -> Q2 -> Q3 ->
 * d_Q through two workspace states; the result is in d_Q with its halos filled.  The viscous
 * terms are added in front of the last sweep.  1-D problems update d_Q in place. */
int osbli_rk3_step(osbli_handle h, double *d_Q, double *d_Qtmp, double dt, void *cuda_stream);

/* The same with the five-stage 4th-order member of the family eq. (36)-(38) ("The 3rd and
 * 4th order schemes have three and five sub-stages per iteration"): Q -> Q2 -> Q3 -> Q2 -> Q3 -> Q. */
int osbli_rk4_step(osbli_handle h, double *d_Q, double *d_Qtmp, double dt, void *cuda_stream);

/* osbli_rk3_step for callers that cannot allocate device memory or keep a handle (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc): the same RK3 step (eq. (36)-(38), same kernels, same
 * order, same result as osbli_init + osbli_rk3_step), with the workspace (R, Q2, Q3, staged primitives) in a
 * file-scope static device array of OSBLI_STATIC_SCRATCH_BYTES inside the library instead of a caller-provided one.
 * The call allocates nothing on the host or the device (no cudaMalloc / cudaFree, no handle); every device that
 * loads the library holds the array until the process exits.
 *   p        host pointer; read during the call only.  p->dirichlet / p->metrics: device pointers as for osbli_init.
 *   d_Q      device pointer, state in the padded layout of osbli_get_layout(p): advanced in place, halos filled.
 *   d_Qtmp   device pointer, dU accumulator (overwritten, need not be initialised); both stay owned by the caller.
 * Limit: osbli_workspace_bytes(p) <= OSBLI_STATIC_SCRATCH_BYTES (64 MiB: e.g. the 1-D cases, 64^3 with the fast
 * viscous path, 48^3 with the general one); beyond it the call returns OSBLI_ESTATIC and launches nothing.  Other
 * errors as osbli_init.  All calls on a device share the one array, which keeps the last call's contents (the part
 * a call uses is cleared on the stream first): calls that may overlap on the GPU (different streams, or threads)
 * race and must be serialised by the caller.  The per-device set-up (array address, shared-memory attributes)
 * happens on the first call on each device, with that device current. */
#define OSBLI_STATIC_SCRATCH_BYTES ((size_t)64 << 20)
size_t osbli_static_scratch_bytes(void);
int osbli_rk3_step_static(const osbli_params *p, double *d_Q, double *d_Qtmp, double dt, void *cuda_stream);

/* End-to-end convenience with HOST buffers: copies the interior nodes of h_Q (host, padded layout,
 * total_doubles doubles) to d_Q, runs nsteps RK3 steps of size dt (halos are rebuilt on the device),
 * copies the interior nodes of the result back into h_Q and synchronises the stream.  Halo and padding
 * entries of h_Q are neither read nor written (5 * nx * ny * nz doubles cross the bus each way).
 * d_Q, d_Qtmp: device scratch states owned by the caller. */
int osbli_advance_host(osbli_handle h, double *h_Q, double *d_Q, double *d_Qtmp, double dt,
                       int32_t nsteps, void *cuda_stream);

/* The same for a batch of independent states, pipelined: h_Q[b] (b = 0..nbatch-1, HOST pointers, padded layout,
 * pinned memory for the copies to be asynchronous) are each advanced by nsteps RK3 steps in place.  Three device
 * states d_Q[0..2] (DEVICE pointers owned by the caller) rotate through host->device copy, compute and
 * device->host copy on three streams (the caller's stream computes; two internal non-blocking streams copy), so
 * that in steady state the cost per state is max(copy in, compute, copy out) instead of their sum.  Host
 * buffers may repeat with period 3 (h_Q[b] == h_Q[b+3]): the copy-in of b+3 is ordered after the copy-out of b.
 * Returns after everything has completed (the stream is synchronised).  Results are bit-identical to
 * osbli_advance_host on each state. */
int osbli_advance_host_batch(osbli_handle h, double *const *h_Q, int32_t nbatch, double *const *d_Q,
                             double *d_Qtmp, double dt, int32_t nsteps, void *cuda_stream);

/* Number of kernel launches the handle has enqueued so far (host counter; for bench.py). */
int osbli_launch_count(osbli_handle h, int64_t *out);

/* Kernel classes of the path: a0 halo fill, a1 staged primitives (viscous path),
 * a2+a3 characteristic sweep per direction, a4 viscous terms, a5 RK3 stage update. */
enum { OSBLI_K_BC = 0, OSBLI_K_PRIM = 1, OSBLI_K_SWEEP_X = 2, OSBLI_K_SWEEP_Y = 3, OSBLI_K_SWEEP_Z = 4,
       OSBLI_K_VISCOUS = 5, OSBLI_K_RK = 6, OSBLI_K_COUNT = 7 };

/* Per-kernel device timing without a profiler: between osbli_profile_begin and osbli_profile_end
 * every launch of the handle is bracketed by two CUDA events on its stream.  osbli_profile_end
 * synchronises the stream and writes, per kernel class, the summed elapsed milliseconds and the
 * launch count into two HOST arrays of OSBLI_K_COUNT entries. */
int osbli_profile_begin(osbli_handle h);
int osbli_profile_end(osbli_handle h, void *cuda_stream, double *ms_per_class, int64_t *launches_per_class);

/* Measured fp64 peak of the current device: a register-only DFMA kernel (8 independent chains per
 * thread, 2 x 1024 threads per SM) timed with CUDA events on the stream; *tflops (HOST) receives
 * the best of 5 runs, counting 2 flop per DFMA.  d_scratch: DEVICE pointer to >= 8 bytes.
 * Synchronises.  This is the denominator of bench.py's "alu" roofline. */
int osbli_measure_fp64_peak(void *d_scratch, void *cuda_stream, double *tflops);

int osbli_destroy(osbli_handle h);
const char *osbli_strerror(int status);

#ifdef __cplusplus
}
#endif
#endif
