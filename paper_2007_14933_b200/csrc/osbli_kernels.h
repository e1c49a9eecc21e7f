// osbli_kernels.h -- host-side launchers of the CUDA kernels (internal to libosbli).
#pragma once
#include "osbli_common.cuh"

namespace osbli {

// Runge-Kutta stage update fused into the last sweep of a stage (eq. (36)-(37)):
// dU = A dU + dt R, Qout = Q + B dU; `first` = stage 1 (A = 0, dU not read).  Qout != Q.
// wrap != 0 (all active directions periodic): the periodic images of the boundary-near nodes are
// written into the halos of Qout as well, which replaces the halo fill of the next stage.
struct RkArgs { double A, B, dt; double *Qtmp, *Qout; int first, wrap; };
void rk_coefficients(int nstages, int form, int stage, double *A, double *B);   // nstages = 3 (RK3; form = OSBLI_RK3_*) or 5 (RK4)

// R (-)= flux difference of the characteristic reconstruction along `dir` (osbli_sweep.cu).
// rk != nullptr (dir 1 or 2, accumulate = 1 only): R is read but not written, the stage update is done instead.
cudaError_t launch_sweep(const DevParams &P, int dir, const double *Q, double *R, int accumulate, const RkArgs *rk,
                         cudaStream_t st);

// 7th-order WENO-Z sweeps (scheme 6, osbli_weno7.cu): R (-)= flux difference along `dir`; no fused update
cudaError_t launch_sweep7(const DevParams &P, int dir, const double *Q, double *R, int accumulate, cudaStream_t st);
// the same tiled kernel for the 5th/6th-order schemes on curvilinear grids (no fused update)
cudaError_t launch_sweep_tiled(const DevParams &P, int dir, const double *Q, double *R, int accumulate, cudaStream_t st);

// staged primitive fields u, v, w, T (, mu) on the halo-extended grid, then R += viscous terms (osbli_visc.cu)
cudaError_t launch_primitives(const DevParams &P, const double *Q, double *prim, cudaStream_t st);
cudaError_t launch_viscous(const DevParams &P, const double *Q, const double *prim, double *R, int accumulate, cudaStream_t st);
// its two kernels on their own: the first differences of the staged fields (depend on Q only), then the assembly (R +=)
cudaError_t launch_gradients(const DevParams &P, const double *prim, cudaStream_t st);
cudaError_t launch_viscous_assemble(const DevParams &P, const double *prim, double *R, int accumulate, cudaStream_t st);

// fused fast path (uniform grid, mu = 1, three periodic directions): reads Q directly, R += viscous terms
bool viscous_fast_path(const DevParams &P);
struct TmapCache {                    // tensor maps of the states the fast viscous kernel has been launched on (host side)
  static constexpr int kSlots = 6;
  struct alignas(64) Map { unsigned long long opaque[16]; } map[kSlots];   // CUtensorMap (128 bytes, 64-byte aligned)
  const double *ptr[kSlots];
  int rows[kSlots];                   // box height the map was encoded for
  int count, next;
};
cudaError_t launch_viscous_fast(const DevParams &P, const double *Q, double *R, TmapCache *cache, cudaStream_t st);

// Per-device one-time set-up (opt-in dynamic shared-memory sizes): called by osbli_init for the current device.
cudaError_t sweep_set_attributes();
cudaError_t viscous_set_attributes();

// scheme 4 on uniform triply periodic grids with mu = 1 (osbli_central.cu): convective + viscous terms + stage update
// + periodic write-through in one kernel per stage; Q -> rk.Qout, dU = rk.Qtmp in place
bool central_fused_path(const DevParams &P);
cudaError_t central_set_attributes();
cudaError_t launch_central_fused(const DevParams &P, const double *Q, const RkArgs &rk, TmapCache *cache, cudaStream_t st);

// central convective terms, scheme 4 (osbli_visc.cu): R = - sum_d delta_d F_d on interior nodes (writes R)
cudaError_t launch_central(const DevParams &P, const double *Q, double *R, cudaStream_t st);

// constant body force (osbli_bc_rk.cu): R_{rho u_i} += f_i, R_{rho E} += u_i f_i on interior nodes
cudaError_t launch_force(const DevParams &P, const double *Q, double *R, cudaStream_t st);

// halo fill along one direction (osbli_bc_rk.cu); returns the number of launches through *nl
cudaError_t launch_bc(const DevParams &P, int dir, double *Q, cudaStream_t st);

// RK3 stage update, eq. (36)-(37): Qtmp = A Qtmp + dt R; Q += B Qtmp on interior nodes
cudaError_t launch_rk_update(const DevParams &P, int nstages, int stage, double dt, double *Q, double *Qtmp, const double *R, cudaStream_t st);

// DFMA micro-benchmark (osbli_peak.cu): measured fp64 TFLOP/s of this device; d_scratch >= 8 bytes
cudaError_t measure_fp64_peak(double *d_scratch, cudaStream_t st, double *tflops);

}  // namespace osbli
