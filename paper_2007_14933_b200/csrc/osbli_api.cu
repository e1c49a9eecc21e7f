// osbli_api.cu -- host side of the C ABI declared in include/osbli.h: layout, parameter
// validation, launch sequencing on the caller's stream.  No device allocation, no synchronisation
// (except osbli_advance_host), no CPU fallback.
#include <mutex>
#include "../../include/osbli.h"
#include "osbli_kernels.h"

#include <cmath>
#include <cstring>
#include <new>
#include <vector>

using namespace osbli;

struct ProfiledLaunch { int cls; cudaEvent_t t0, t1; };

struct osbli_ctx {
  DevParams P;
  double *R;          // residual state in the workspace (used by osbli_rk3_step)
  double *Q2, *Q3;    // two more states in the workspace: targets of the fused sweep + stage update
  double *prim;       // staged u, v, w, T (, mu) fields in the workspace
  int64_t launches;
  bool profiling;
  std::vector<ProfiledLaunch> *prof;   // events around every launch while profiling
  TmapCache tmaps;                     // tensor maps of the states seen by the fast viscous kernel
  cudaStream_t s_in, s_out;            // copy streams of osbli_advance_host_batch (created on first use)
  cudaEvent_t ev_h2d[3], ev_cmp[3], ev_d2h[3];
  bool pipe_ready;
  // general viscous path: the staged primitives and their first differences depend on Q only and are formed on a side
  // stream next to the first sweeps (created by osbli_init; absent in osbli_rk3_step_static, which creates nothing)
  cudaStream_t s_side;
  cudaEvent_t ev_fork, ev_join;
  bool side_ready;
};

#ifndef OSBLI_SIDE_STREAM
#define OSBLI_SIDE_STREAM 1    // general viscous path: primitives + first differences on a side stream next to the first sweeps
#endif
#ifndef OSBLI_CURV_TILED_X
#define OSBLI_CURV_TILED_X 1   // curvilinear grids: the x sweep runs on the tiled kernel of osbli_weno7.cu (config 4: 0.180 -> 0.149 ms;
#endif                        // the y and z sweeps lose there: 0.134 -> 0.178, 0.139 -> 0.301 with 8 nodes along z)

namespace {

int make_layout(const osbli_params *p, Layout *L) {
  const int n[3] = {p->nx, p->ny, p->nz};
  for (int d = 0; d < 3; ++d) {
    if (n[d] < 1) return OSBLI_EINVAL;
    if (n[d] > 1 && n[d] < 5) return OSBLI_EINVAL;
    L->n[d] = n[d];
    L->h[d] = n[d] > 1 ? (p->scheme == OSBLI_SCHEME_WENOZ7 ? kHalo7 : kHalo) : 0;
  }
  L->xoff = kXOffset;
  const long long rowlen = kXOffset + (long long)n[0] + kXTail;
  L->sy = (rowlen + 15) / 16 * 16;
  L->sz = L->sy * (n[1] + 2 * L->h[1]);
  L->sv = L->sz * (n[2] + 2 * L->h[2]);
  return OSBLI_OK;
}

// workspace fields of the general viscous path: staged u, v, w, T (, mu) and their first differences along x, y, z
// (none on the fast path -- uniform grid, mu = 1, three active periodic directions -- whose kernels read Q directly)
int nprim(const osbli_params *p) {
  if (p->visc == OSBLI_VISC_NONE) return 0;
  bool fast = !p->metrics && p->visc == OSBLI_VISC_CONST;
  const int n[3] = {p->nx, p->ny, p->nz};
  for (int d = 0; d < 3; ++d)
    if (n[d] <= 1 || p->bc[d][0] != OSBLI_BC_PERIODIC || p->bc[d][1] != OSBLI_BC_PERIODIC) fast = false;
  return fast ? 0 : 4 * (p->visc == OSBLI_VISC_SUTHERLAND ? 5 : 4);
}

int validate(const osbli_params *p) {
  if (!p) return OSBLI_EINVAL;
  Layout L;
  if (int rc = make_layout(p, &L)) return rc;
  if (p->nx == 1) return OSBLI_EUNSUPPORTED;                       // x is the contiguous direction; it must be active
  if (p->scheme < OSBLI_SCHEME_WENOZ5 || p->scheme > OSBLI_SCHEME_WENOZ7) return OSBLI_EINVAL;
  if (p->scheme == OSBLI_SCHEME_CENTRAL4 && p->metrics) return OSBLI_EUNSUPPORTED;   // central convective terms: uniform grids
  if (p->visc < OSBLI_VISC_NONE || p->visc > OSBLI_VISC_SUTHERLAND) return OSBLI_EINVAL;
  if (p->averaging != OSBLI_AVG_ROE && p->averaging != OSBLI_AVG_SIMPLE) return OSBLI_EINVAL;
  if (p->rk3_form != OSBLI_RK3_WILLIAMSON && p->rk3_form != OSBLI_RK3_SSP) return OSBLI_EINVAL;
  if (!(p->gamma > 1.0)) return OSBLI_EINVAL;
  if (!(p->eps >= 1e-18) || !(p->teno_ct > 0.0)) return OSBLI_EINVAL;
  if (p->visc != OSBLI_VISC_NONE && (!(p->Re > 0.0) || !(p->Pr > 0.0) || !(p->Minf > 0.0))) return OSBLI_EINVAL;
  bool need_dirichlet = false;
  for (int d = 0; d < 3; ++d) {
    const int n = d == 0 ? p->nx : (d == 1 ? p->ny : p->nz);
    for (int s = 0; s < 2; ++s) {
      const int b = p->bc[d][s];
      if (b < OSBLI_BC_PERIODIC || b > OSBLI_BC_WALL_ADIABATIC) return OSBLI_EINVAL;
      if (n > 1 && b == OSBLI_BC_WALL_ADIABATIC && !(p->Minf > 0.0)) return OSBLI_EINVAL;
      if (n > 1 && b == OSBLI_BC_DIRICHLET) need_dirichlet = true;
      if (n > 1 && b == OSBLI_BC_WALL_ISOTHERMAL && !(p->wall_T[d][s] > 0.0)) return OSBLI_EINVAL;
      if (n > 1 && b == OSBLI_BC_WALL_ISOTHERMAL && !(p->Minf > 0.0)) return OSBLI_EINVAL;
    }
    if ((p->bc[d][0] == OSBLI_BC_PERIODIC) != (p->bc[d][1] == OSBLI_BC_PERIODIC)) return OSBLI_EINVAL;
  }
  if (need_dirichlet && !p->dirichlet) return OSBLI_EINVAL;
  if (!p->metrics) {
    const double dl[3] = {p->dx, p->dy, p->dz};
    for (int d = 0; d < 3; ++d)
      if (L.n[d] > 1 && !(dl[d] > 0.0)) return OSBLI_EINVAL;
  } else {
    const osbli_metrics *m = p->metrics;
    if (!m->detJ) return OSBLI_EINVAL;
    for (int k = 0; k < 3; ++k) {
      for (int j = 0; j < 3; ++j)
        if (!m->D[k][j]) return OSBLI_EINVAL;
      if (p->visc != OSBLI_VISC_NONE)
        for (int e = 0; e < 6; ++e)
          if (!m->E[k][e]) return OSBLI_EINVAL;
    }
  }
  return OSBLI_OK;
}

inline cudaStream_t as_stream(void *s) { return reinterpret_cast<cudaStream_t>(s); }

// Every kernel launch goes through here: counted, and (only while osbli_profile_begin is in
// effect) bracketed by two events on the same stream so that bench.py can attribute device time
// to kernel classes without a profiler attached.
#define OSBLI_LAUNCH(h, cls, st, call)                                   \
  do {                                                                   \
    ProfiledLaunch pl_ = {cls, nullptr, nullptr};                        \
    if ((h)->profiling) {                                                \
      if (cudaEventCreate(&pl_.t0) != cudaSuccess) return OSBLI_ECUDA;   \
      if (cudaEventCreate(&pl_.t1) != cudaSuccess) { cudaEventDestroy(pl_.t0); return OSBLI_ECUDA; } \
      cudaEventRecord(pl_.t0, st);                                       \
    }                                                                    \
    if ((call) != cudaSuccess) return OSBLI_ECUDA;                       \
    if ((h)->profiling) { cudaEventRecord(pl_.t1, st); (h)->prof->push_back(pl_); } \
    ++(h)->launches;                                                     \
  } while (0)

int do_bc(osbli_ctx *h, double *Q, cudaStream_t st) {
  for (int d = 0; d < 3; ++d)
    if (h->P.L.n[d] > 1) OSBLI_LAUNCH(h, OSBLI_K_BC, st, launch_bc(h->P, d, Q, st));
  return OSBLI_OK;
}

// Residual of one stage.  Order: every sweep but the last, the viscous terms, the last sweep.
// With rk != nullptr the last sweep (y or z) also does the stage update (RkArgs) and R is left
// without the last direction's flux difference.
int do_rhs(osbli_ctx *h, const double *Q, double *R, const RkArgs *rk, cudaStream_t st) {
  const DevParams &P = h->P;
  const bool fast_visc = viscous_fast_path(P);
  const bool general_visc = P.visc != OSBLI_VISC_NONE && !fast_visc;
  int last = 0;
  for (int d = 0; d < 3; ++d)
    if (P.L.n[d] > 1) last = d;
  // fork: primitives and first differences on the side stream while the first sweeps run (2-D / 3-D sweeps path only)
  const bool fork = OSBLI_SIDE_STREAM && general_visc && h->side_ready && last > 0 && P.scheme != OSBLI_SCHEME_CENTRAL4;
  if (fork) {
    if (cudaEventRecord(h->ev_fork, st) != cudaSuccess || cudaStreamWaitEvent(h->s_side, h->ev_fork, 0) != cudaSuccess) return OSBLI_ECUDA;
    OSBLI_LAUNCH(h, OSBLI_K_PRIM, h->s_side, launch_primitives(P, Q, h->prim, h->s_side));
    OSBLI_LAUNCH(h, OSBLI_K_VISCOUS, h->s_side, launch_gradients(P, h->prim, h->s_side));
    if (cudaEventRecord(h->ev_join, h->s_side) != cudaSuccess) return OSBLI_ECUDA;
  } else if (general_visc) {
    OSBLI_LAUNCH(h, OSBLI_K_PRIM, st, launch_primitives(P, Q, h->prim, st));
  }
  if (P.scheme == OSBLI_SCHEME_CENTRAL4) {                            // no sweeps: central convective terms, then the rest
    if (rk) return OSBLI_EINVAL;
    OSBLI_LAUNCH(h, OSBLI_K_SWEEP_X, st, launch_central(P, Q, R, st));
    if (fast_visc) OSBLI_LAUNCH(h, OSBLI_K_VISCOUS, st, launch_viscous_fast(P, Q, R, &h->tmaps, st));
    else if (P.visc != OSBLI_VISC_NONE) {
      OSBLI_LAUNCH(h, OSBLI_K_VISCOUS, st, launch_viscous(P, Q, h->prim, R, 1, st));
      ++h->launches;                                                // launch_viscous = gradients_kernel + viscous_kernel
    }
    if (P.has_force) OSBLI_LAUNCH(h, OSBLI_K_VISCOUS, st, launch_force(P, Q, R, st));
    return OSBLI_OK;
  }
  int accumulate = 0;
  for (int d = 0; d < 3; ++d) {
    if (P.L.n[d] <= 1) continue;
    if (d == last && last > 0) {                                    // viscous terms go in front of the last sweep
      if (fast_visc) OSBLI_LAUNCH(h, OSBLI_K_VISCOUS, st, launch_viscous_fast(P, Q, R, &h->tmaps, st));
      else if (fork) {                                              // join: the first differences are there
        if (cudaStreamWaitEvent(st, h->ev_join, 0) != cudaSuccess) return OSBLI_ECUDA;
        OSBLI_LAUNCH(h, OSBLI_K_VISCOUS, st, launch_viscous_assemble(P, h->prim, R, accumulate, st));
      } else if (P.visc != OSBLI_VISC_NONE) {
        OSBLI_LAUNCH(h, OSBLI_K_VISCOUS, st, launch_viscous(P, Q, h->prim, R, accumulate, st));
        ++h->launches;                                              // launch_viscous = gradients_kernel + viscous_kernel
      }
      if (P.has_force) OSBLI_LAUNCH(h, OSBLI_K_VISCOUS, st, launch_force(P, Q, R, st));
    }
    if (P.scheme == OSBLI_SCHEME_WENOZ7) {                          // side scheme: its own untuned sweeps, no fused update
      if (rk) return OSBLI_EINVAL;
      OSBLI_LAUNCH(h, OSBLI_K_SWEEP_X + d, st, launch_sweep7(P, d, Q, R, accumulate, st));
    } else if (OSBLI_CURV_TILED_X && P.curvilinear && d == 0 && !(d == last && rk) &&
               (long long)((P.L.n[1] * P.L.n[2] + 31) / 32) * ((P.L.n[0] + 63) / 64) < 148LL * 8) {
      // curvilinear x sweep on grids whose 64-node line segments do not fill the chip's warp slots (config 4): the tiled
      // kernel, one thread per interface, instead of the march with 16-node segments
      OSBLI_LAUNCH(h, OSBLI_K_SWEEP_X + d, st, launch_sweep_tiled(P, d, Q, R, accumulate, st));
    } else
      OSBLI_LAUNCH(h, OSBLI_K_SWEEP_X + d, st, launch_sweep(P, d, Q, R, accumulate, d == last ? rk : nullptr, st));
    accumulate = 1;
  }
  if (last == 0 && P.visc != OSBLI_VISC_NONE)                       // 1-D: the x sweep, then the viscous terms
  {
    OSBLI_LAUNCH(h, OSBLI_K_VISCOUS, st, launch_viscous(P, Q, h->prim, R, accumulate, st));
    ++h->launches;                                                  // launch_viscous = gradients_kernel + viscous_kernel
  }
  if (last == 0 && P.has_force) OSBLI_LAUNCH(h, OSBLI_K_VISCOUS, st, launch_force(P, Q, R, st));
  return OSBLI_OK;
}

// One low-storage Runge-Kutta step, eq. (36)-(38), nstages = 3 (RK3) or 5 (4th order).  With two or more
// active directions the update is fused into the last sweep of every stage, which cannot update in place,
// so the state moves Q -> Q2 -> Q3 (-> Q2 -> Q3) -> Q through two workspace states; 1-D problems use the
// separate in-place update kernel.  The result is in Q either way.
int do_step(osbli_ctx *h, int nstages, double *Q, double *Qtmp, double dt, cudaStream_t st) {
  if (central_fused_path(h->P)) {
    // central scheme on a uniform triply periodic grid: one kernel per stage (convective + viscous terms, stage
    // update, periodic images of the new state), Q -> Q2 -> Q3 (-> Q2 -> Q3) -> Q; one halo fill per step
    for (int s = 0; s < nstages; ++s) {
      double *src = s == 0 ? Q : ((s & 1) ? h->Q2 : h->Q3);
      double *dst = s == nstages - 1 ? Q : ((s & 1) ? h->Q3 : h->Q2);
      if (s == 0)
        if (int rc = do_bc(h, src, st)) return rc;
      RkArgs rk;
      rk_coefficients(nstages, h->P.rk3_form, s, &rk.A, &rk.B);
      rk.dt = dt; rk.Qtmp = Qtmp; rk.Qout = dst; rk.first = (rk.A == 0.0); rk.wrap = 1;
      OSBLI_LAUNCH(h, OSBLI_K_SWEEP_Z, st, launch_central_fused(h->P, src, rk, &h->tmaps, st));
    }
    return OSBLI_OK;
  }
  const bool fuse = (h->P.L.n[1] > 1 || h->P.L.n[2] > 1) && h->P.scheme != OSBLI_SCHEME_CENTRAL4 &&
                    h->P.scheme != OSBLI_SCHEME_WENOZ7;
  bool wrap = fuse;                  // every active direction periodic: the fused update fills the halos itself
  for (int d = 0; d < 3; ++d)
    if (h->P.L.n[d] > 1 && !h->P.periodic[d]) wrap = false;
  for (int s = 0; s < nstages; ++s) {
    if (fuse) {
      double *src = s == 0 ? Q : ((s & 1) ? h->Q2 : h->Q3);
      double *dst = s == nstages - 1 ? Q : ((s & 1) ? h->Q3 : h->Q2);
      if (s == 0 || !wrap)
        if (int rc = do_bc(h, src, st)) return rc;
      RkArgs rk;
      rk_coefficients(nstages, h->P.rk3_form, s, &rk.A, &rk.B);
      rk.dt = dt; rk.Qtmp = Qtmp; rk.Qout = dst; rk.first = (rk.A == 0.0); rk.wrap = wrap ? 1 : 0;   // A_s = 0: dU is not read
      if (int rc = do_rhs(h, src, h->R, &rk, st)) return rc;
    } else {
      if (int rc = do_bc(h, Q, st)) return rc;
      if (int rc = do_rhs(h, Q, h->R, nullptr, st)) return rc;
      OSBLI_LAUNCH(h, OSBLI_K_RK, st, launch_rk_update(h->P, nstages, s, dt, Q, Qtmp, h->R, st));
    }
  }
  return wrap ? OSBLI_OK : do_bc(h, Q, st);
}

// A context from validated parameters and a workspace of osbli_workspace_bytes(p) bytes (no allocation; the
// profiling list is the caller's business).
void fill_ctx(const osbli_params *p, void *d_workspace, osbli_ctx *h) {
  std::memset(h, 0, sizeof(*h));
  DevParams &P = h->P;
  make_layout(p, &P.L);
  P.curvilinear = p->metrics ? 1 : 0;
  const double dl[3] = {p->dx, p->dy, p->dz};
  for (int d = 0; d < 3; ++d) {
    const double delta = (P.L.n[d] > 1 && !P.curvilinear) ? dl[d] : 1.0;
    P.inv_delta[d] = 1.0 / delta;
    P.inv12d[d] = 1.0 / (12.0 * delta);
    P.inv12d2[d] = 1.0 / (12.0 * delta * delta);
    P.periodic[d] = p->bc[d][0] == OSBLI_BC_PERIODIC;
    for (int s = 0; s < 2; ++s) { P.bc[d][s] = p->bc[d][s]; P.wall_T[d][s] = p->wall_T[d][s]; }
  }
  P.gamma = p->gamma; P.gm1 = p->gamma - 1.0;
  P.Re = p->Re; P.inv_Re = p->visc != OSBLI_VISC_NONE ? 1.0 / p->Re : 0.0;
  P.Pr = p->Pr; P.Minf = p->Minf; P.gM2 = p->gamma * p->Minf * p->Minf;
  P.cq = p->visc != OSBLI_VISC_NONE ? 1.0 / ((p->gamma - 1.0) * p->Minf * p->Minf * p->Pr * p->Re) : 0.0;
  P.scheme = p->scheme; P.visc = p->visc;
  P.ct = p->teno_ct; P.eps = p->eps; P.suth = p->suth_ratio;
  const double nstencils = p->scheme == OSBLI_SCHEME_TENO6 ? 4.0 : 3.0;
  P.teno_kfast = (std::pow(nstencils * p->teno_ct, -1.0 / 6.0) - 1.0) * (1.0 - 1e-6);
  P.dirichlet = p->dirichlet;
  for (int a = 0; a < 3; ++a) P.force[a] = p->force[a];
  P.has_force = (p->force[0] != 0.0 || p->force[1] != 0.0 || p->force[2] != 0.0) ? 1 : 0;
  P.averaging = p->averaging;
  P.rk3_form = p->rk3_form;
  if (p->metrics) {
    for (int k = 0; k < 3; ++k) {
      for (int j = 0; j < 3; ++j) P.D[k][j] = p->metrics->D[k][j];
      for (int e = 0; e < 6; ++e) P.E[k][e] = p->metrics->E[k][e];
    }
    P.detJ = p->metrics->detJ;
  }
  h->R = static_cast<double *>(d_workspace);
  h->Q2 = h->R + 5 * P.L.sv;
  h->Q3 = h->Q2 + 5 * P.L.sv;
  h->prim = h->Q3 + 5 * P.L.sv;
}

}  // namespace

extern "C" {

int osbli_get_layout(const osbli_params *p, osbli_layout *out) {
  if (!p || !out) return OSBLI_EINVAL;
  Layout L;
  if (int rc = make_layout(p, &L)) return rc;
  for (int d = 0; d < 3; ++d) out->halo[d] = L.h[d];
  out->x_offset = L.xoff;
  out->stride_y = L.sy;
  out->stride_z = L.sz;
  out->stride_var = L.sv;
  out->total_doubles = 5 * L.sv;
  return OSBLI_OK;
}

int osbli_workspace_bytes(const osbli_params *p, size_t *out) {
  if (!p || !out) return OSBLI_EINVAL;
  Layout L;
  if (int rc = make_layout(p, &L)) return rc;
  if (p->visc < OSBLI_VISC_NONE || p->visc > OSBLI_VISC_SUTHERLAND) return OSBLI_EINVAL;
  *out = (size_t)(15 + nprim(p)) * (size_t)L.sv * sizeof(double);   // R, Q2, Q3, staged primitives
  return OSBLI_OK;
}

int osbli_init(const osbli_params *p, void *d_workspace, size_t workspace_bytes, osbli_handle *out) {
  if (!out) return OSBLI_EINVAL;
  *out = nullptr;
  if (int rc = validate(p)) return rc;
  size_t need = 0;
  osbli_workspace_bytes(p, &need);
  if (!d_workspace || workspace_bytes < need || (reinterpret_cast<uintptr_t>(d_workspace) & 255u)) return OSBLI_EWORKSPACE;

  int dev = 0;
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return OSBLI_ECUDA;
  if (prop.major != 10) return OSBLI_ECUDA;                      // sm_100a code only; no other path exists
  // opt-in shared-memory sizes are per device: set them for the device this handle lives on
  if (sweep_set_attributes() != cudaSuccess || viscous_set_attributes() != cudaSuccess || central_set_attributes() != cudaSuccess) return OSBLI_ECUDA;

  osbli_ctx *h = new (std::nothrow) osbli_ctx;
  if (!h) return OSBLI_EINVAL;
  fill_ctx(p, d_workspace, h);
  h->prof = new (std::nothrow) std::vector<ProfiledLaunch>();
  if (!h->prof) { delete h; return OSBLI_EINVAL; }
  if (nprim(p) > 0) {                                              // side stream of the general viscous path
    if (cudaStreamCreateWithFlags(&h->s_side, cudaStreamNonBlocking) == cudaSuccess &&
        cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming) == cudaSuccess &&
        cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming) == cudaSuccess)
      h->side_ready = true;
    else { delete h->prof; delete h; return OSBLI_ECUDA; }
  }
  *out = h;
  return OSBLI_OK;
}

int osbli_bc(osbli_handle h, double *d_Q, void *cuda_stream) {
  if (!h || !d_Q) return OSBLI_EINVAL;
  return do_bc(h, d_Q, as_stream(cuda_stream));
}

int osbli_rhs(osbli_handle h, const double *d_Q, double *d_R, void *cuda_stream) {
  if (!h || !d_Q || !d_R || d_Q == d_R) return OSBLI_EINVAL;
  return do_rhs(h, d_Q, d_R, nullptr, as_stream(cuda_stream));
}

int osbli_rk3_step(osbli_handle h, double *d_Q, double *d_Qtmp, double dt, void *cuda_stream) {
  if (!h || !d_Q || !d_Qtmp || d_Q == d_Qtmp) return OSBLI_EINVAL;
  return do_step(h, 3, d_Q, d_Qtmp, dt, as_stream(cuda_stream));
}

int osbli_rk4_step(osbli_handle h, double *d_Q, double *d_Qtmp, double dt, void *cuda_stream) {
  if (!h || !d_Q || !d_Qtmp || d_Q == d_Qtmp) return OSBLI_EINVAL;
  return do_step(h, 5, d_Q, d_Qtmp, dt, as_stream(cuda_stream));
}

// interior nodes of the five variables between a host and a device state of the same padded layout
static cudaError_t copy_interior(const Layout &L, double *dst, const double *src, cudaMemcpyKind kind, cudaStream_t st) {
  const size_t pitch = (size_t)L.sy * sizeof(double);
  const size_t rows = (size_t)(L.n[1] + 2 * L.h[1]);
  for (int c = 0; c < 5; ++c) {
    cudaMemcpy3DParms p = {};
    p.srcPtr = make_cudaPitchedPtr(const_cast<double *>(src) + (size_t)c * L.sv, pitch, pitch, rows);
    p.dstPtr = make_cudaPitchedPtr(dst + (size_t)c * L.sv, pitch, pitch, rows);
    p.srcPos = make_cudaPos((size_t)L.xoff * sizeof(double), (size_t)L.h[1], (size_t)L.h[2]);
    p.dstPos = p.srcPos;
    p.extent = make_cudaExtent((size_t)L.n[0] * sizeof(double), (size_t)L.n[1], (size_t)L.n[2]);
    p.kind = kind;
    if (cudaError_t e = cudaMemcpy3DAsync(&p, st)) return e;
  }
  return cudaSuccess;
}

int osbli_advance_host(osbli_handle h, double *h_Q, double *d_Q, double *d_Qtmp, double dt, int32_t nsteps,
                       void *cuda_stream) {
  if (!h || !h_Q || !d_Q || !d_Qtmp || d_Q == d_Qtmp || nsteps < 0) return OSBLI_EINVAL;
  cudaStream_t st = as_stream(cuda_stream);
  // only interior nodes cross the bus (halos are rebuilt on the device by the first halo fill): 15 % fewer bytes at 256^3
  if (copy_interior(h->P.L, d_Q, h_Q, cudaMemcpyHostToDevice, st) != cudaSuccess) return OSBLI_ECUDA;
  if (nsteps == 0)
    if (int rc = do_bc(h, d_Q, st)) return rc;
  for (int s = 0; s < nsteps; ++s)
    if (int rc = do_step(h, 3, d_Q, d_Qtmp, dt, st)) return rc;
  if (copy_interior(h->P.L, h_Q, d_Q, cudaMemcpyDeviceToHost, st) != cudaSuccess) return OSBLI_ECUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return OSBLI_ECUDA;
  return OSBLI_OK;
}

static int pipe_setup(osbli_ctx *h) {
  if (h->pipe_ready) return OSBLI_OK;
  if (cudaStreamCreateWithFlags(&h->s_in, cudaStreamNonBlocking) != cudaSuccess) return OSBLI_ECUDA;
  if (cudaStreamCreateWithFlags(&h->s_out, cudaStreamNonBlocking) != cudaSuccess) return OSBLI_ECUDA;
  for (int s = 0; s < 3; ++s)
    if (cudaEventCreateWithFlags(&h->ev_h2d[s], cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_cmp[s], cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_d2h[s], cudaEventDisableTiming) != cudaSuccess)
      return OSBLI_ECUDA;
  h->pipe_ready = true;
  return OSBLI_OK;
}

int osbli_advance_host_batch(osbli_handle h, double *const *h_Q, int32_t nbatch, double *const *d_Q,
                             double *d_Qtmp, double dt, int32_t nsteps, void *cuda_stream) {
  if (!h || !h_Q || !d_Q || !d_Qtmp || nbatch < 0 || nsteps < 0) return OSBLI_EINVAL;
  for (int s = 0; s < 3; ++s) {
    if (!d_Q[s] || d_Q[s] == d_Qtmp) return OSBLI_EINVAL;
    for (int t = 0; t < s; ++t)
      if (d_Q[s] == d_Q[t]) return OSBLI_EINVAL;
  }
  for (int b = 0; b < nbatch; ++b)
    if (!h_Q[b]) return OSBLI_EINVAL;
  if (int rc = pipe_setup(h)) return rc;
  cudaStream_t st = as_stream(cuda_stream);
  const Layout &L = h->P.L;
  // work already queued on the caller's stream (it may still use d_Q / d_Qtmp) comes first
  if (cudaEventRecord(h->ev_cmp[0], st) != cudaSuccess) return OSBLI_ECUDA;
  if (cudaStreamWaitEvent(h->s_in, h->ev_cmp[0], 0) != cudaSuccess) return OSBLI_ECUDA;
  for (int b = 0; b < nbatch; ++b) {
    const int s = b % 3;
    if (b >= 3 && cudaStreamWaitEvent(h->s_in, h->ev_d2h[s], 0) != cudaSuccess) return OSBLI_ECUDA;   // slot s (and h_Q[b-3]) are free
    if (copy_interior(L, d_Q[s], h_Q[b], cudaMemcpyHostToDevice, h->s_in) != cudaSuccess) return OSBLI_ECUDA;
    if (cudaEventRecord(h->ev_h2d[s], h->s_in) != cudaSuccess) return OSBLI_ECUDA;
    if (cudaStreamWaitEvent(st, h->ev_h2d[s], 0) != cudaSuccess) return OSBLI_ECUDA;
    if (nsteps == 0)
      if (int rc = do_bc(h, d_Q[s], st)) return rc;
    for (int k = 0; k < nsteps; ++k)
      if (int rc = do_step(h, 3, d_Q[s], d_Qtmp, dt, st)) return rc;
    if (cudaEventRecord(h->ev_cmp[s], st) != cudaSuccess) return OSBLI_ECUDA;
    if (cudaStreamWaitEvent(h->s_out, h->ev_cmp[s], 0) != cudaSuccess) return OSBLI_ECUDA;
    if (copy_interior(L, h_Q[b], d_Q[s], cudaMemcpyDeviceToHost, h->s_out) != cudaSuccess) return OSBLI_ECUDA;
    if (cudaEventRecord(h->ev_d2h[s], h->s_out) != cudaSuccess) return OSBLI_ECUDA;
  }
  for (int s = 0; s < 3 && s < nbatch; ++s)
    if (cudaStreamWaitEvent(st, h->ev_d2h[s], 0) != cudaSuccess) return OSBLI_ECUDA;   // the caller's stream ends after the last copy-out
  if (cudaStreamSynchronize(st) != cudaSuccess) return OSBLI_ECUDA;
  return OSBLI_OK;
}

int osbli_launch_count(osbli_handle h, int64_t *out) {
  if (!h || !out) return OSBLI_EINVAL;
  *out = h->launches;
  return OSBLI_OK;
}

int osbli_profile_begin(osbli_handle h) {
  if (!h || h->profiling) return OSBLI_EINVAL;
  h->profiling = true;
  return OSBLI_OK;
}

int osbli_profile_end(osbli_handle h, void *cuda_stream, double *ms_per_class, int64_t *launches_per_class) {
  if (!h || !h->profiling || !ms_per_class || !launches_per_class) return OSBLI_EINVAL;
  h->profiling = false;
  int rc = OSBLI_OK;
  if (cudaStreamSynchronize(as_stream(cuda_stream)) != cudaSuccess) rc = OSBLI_ECUDA;
  for (int c = 0; c < OSBLI_K_COUNT; ++c) { ms_per_class[c] = 0.0; launches_per_class[c] = 0; }
  for (ProfiledLaunch &pl : *h->prof) {
    float ms = 0.f;
    if (rc == OSBLI_OK && cudaEventElapsedTime(&ms, pl.t0, pl.t1) != cudaSuccess) rc = OSBLI_ECUDA;
    ms_per_class[pl.cls] += ms;
    ++launches_per_class[pl.cls];
    cudaEventDestroy(pl.t0);
    cudaEventDestroy(pl.t1);
  }
  h->prof->clear();
  return rc;
}

int osbli_measure_fp64_peak(void *d_scratch, void *cuda_stream, double *tflops) {
  if (!d_scratch || !tflops) return OSBLI_EINVAL;
  return measure_fp64_peak(static_cast<double *>(d_scratch), as_stream(cuda_stream), tflops) == cudaSuccess
             ? OSBLI_OK : OSBLI_ECUDA;
}

int osbli_destroy(osbli_handle h) {
  if (!h) return OSBLI_EINVAL;
  if (h->prof) {
    for (ProfiledLaunch &pl : *h->prof) { cudaEventDestroy(pl.t0); cudaEventDestroy(pl.t1); }
    delete h->prof;
  }
  if (h->side_ready) {
    cudaStreamDestroy(h->s_side);
    cudaEventDestroy(h->ev_fork);
    cudaEventDestroy(h->ev_join);
  }
  if (h->pipe_ready) {
    cudaStreamDestroy(h->s_in);
    cudaStreamDestroy(h->s_out);
    for (int s = 0; s < 3; ++s) { cudaEventDestroy(h->ev_h2d[s]); cudaEventDestroy(h->ev_cmp[s]); cudaEventDestroy(h->ev_d2h[s]); }
  }
  delete h;
  return OSBLI_OK;
}

// ---- osbli_rk3_step_static: one RK3 step with the workspace in a static device array (include/osbli.h) ----------
// Every device that loads the library holds these OSBLI_STATIC_SCRATCH_BYTES until the process exits.  In host code
// the name g_static_scratch is a host-side stand-in, not a device address: the address a kernel can use comes from
// cudaGetSymbolAddress, once per device, with that device current (static_scratch_setup).
}  // extern "C"

static __device__ __align__(256) double g_static_scratch[OSBLI_STATIC_SCRATCH_BYTES / sizeof(double)];

namespace {
constexpr int kMaxDevices = 64;
std::mutex g_static_mu;
double *g_static_ptr[kMaxDevices];     // device address of g_static_scratch on each device ordinal (nullptr: not set up)

// Once per device, with that device current: opt-in shared-memory sizes of the kernels and the array's device address.
int static_scratch_setup(int dev, double **out) {
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_ptr[dev]) {
    int major = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess || major != 10) return OSBLI_ECUDA;
    if (sweep_set_attributes() != cudaSuccess || viscous_set_attributes() != cudaSuccess || central_set_attributes() != cudaSuccess) return OSBLI_ECUDA;
    double *ptr = nullptr;
    if (cudaGetSymbolAddress(reinterpret_cast<void **>(&ptr), g_static_scratch) != cudaSuccess || !ptr) return OSBLI_ECUDA;
    if (reinterpret_cast<uintptr_t>(ptr) & 255u) return OSBLI_ECUDA;
    g_static_ptr[dev] = ptr;
  }
  *out = g_static_ptr[dev];
  return OSBLI_OK;
}
}  // namespace

extern "C" {

size_t osbli_static_scratch_bytes(void) { return OSBLI_STATIC_SCRATCH_BYTES; }

int osbli_rk3_step_static(const osbli_params *p, double *d_Q, double *d_Qtmp, double dt, void *cuda_stream) {
  if (!d_Q || !d_Qtmp || d_Q == d_Qtmp) return OSBLI_EINVAL;
  if (int rc = validate(p)) return rc;
  size_t need = 0;
  if (int rc = osbli_workspace_bytes(p, &need)) return rc;
  if (need > OSBLI_STATIC_SCRATCH_BYTES) return OSBLI_ESTATIC;     // the problem does not fit the static array
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return OSBLI_ECUDA;
  double *ws = nullptr;
  if (int rc = static_scratch_setup(dev, &ws)) return rc;
  cudaStream_t st = as_stream(cuda_stream);
  // the array keeps the last call's contents (possibly of another problem shape): start from zeros
  if (cudaMemsetAsync(ws, 0, need, st) != cudaSuccess) return OSBLI_ECUDA;
  osbli_ctx ctx;                                                    // on the stack: no handle, nothing to free
  fill_ctx(p, ws, &ctx);
  return do_step(&ctx, 3, d_Q, d_Qtmp, dt, st);
}

const char *osbli_strerror(int status) {
  switch (status) {
    case OSBLI_OK: return "ok";
    case OSBLI_EINVAL: return "invalid argument";
    case OSBLI_EUNSUPPORTED: return "unsupported configuration";
    case OSBLI_ECUDA: return "CUDA error (no sm_100 device, or a launch / copy failed)";
    case OSBLI_EWORKSPACE: return "workspace missing, too small or not 256-byte aligned";
    case OSBLI_ESTATIC: return "problem too large for osbli_rk3_step_static: its workspace exceeds OSBLI_STATIC_SCRATCH_BYTES (64 MiB)";
    default: return "unknown status";
  }
}

}  // extern "C"
