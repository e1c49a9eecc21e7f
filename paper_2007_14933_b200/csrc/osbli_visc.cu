// osbli_visc.cu -- viscous and heat-flux terms of eq. (2)-(5), discretised with the
// 4th-order central differences of eq. (28)-(29) (eq. (28) with its sign corrected, Q1)
// and the one-sided closures of eq. (30)-(35), next to non-periodic boundaries;
// metric chain rule on curvilinear grids.
//
// General path, three kernels (the paper's "store some" idea: "the derivatives of the velocity
// components ... are stored ... to be reused in the mixed derivatives", everything else is recomputed):
// (1) point-wise u, v, w, T (, mu) staged once per stage on the halo-extended grid; (2) their first
// differences delta_l f along every active direction (closures included), stored where a mixed difference
// will read them; (3) one thread per node: second differences from the staged fields, mixed differences
// delta_k(delta_l f) as ONE five-point stencil over the stored first differences (4-5 loads instead of the
// 16-25 of a nested evaluation: the curvilinear chain rule needs all 12 of them), assembly of
// d_j tau_ij,  d_j(u_i tau_ij) - d_j q_j  and R +=.
#include "osbli_kernels.h"

#include "osbli_tma.cuh"
#include <type_traits>

namespace osbli {

// eq. (7): p = (gamma-1)(rhoE - rho u.u/2), T = gamma M^2 p / rho;
// mu = T^1.5 (1+S)/(T+S), S = SuthT/RefT.
template <bool SUTH>
__global__ void __launch_bounds__(256)
primitives_kernel(const __grid_constant__ DevParams P, const double *__restrict__ Q, double *__restrict__ prim) {
  const Layout &L = P.L;
  const int i = blockIdx.x * blockDim.x + threadIdx.x - L.h[0];
  const int j = (int)blockIdx.y - L.h[1];
  const int k = (int)blockIdx.z - L.h[2];
  if (i >= L.n[0] + L.h[0]) return;
  const long long at = L.at(i, j, k);
  const double r = __ldg(Q + at), mx = __ldg(Q + L.sv + at), my = __ldg(Q + 2 * L.sv + at);
  const double mz = __ldg(Q + 3 * L.sv + at), E = __ldg(Q + 4 * L.sv + at);
  const double ir = 1.0 / r;
  const double u = mx * ir, v = my * ir, w = mz * ir;
  const double p = P.gm1 * (E - 0.5 * (mx * u + my * v + mz * w));
  const double T = P.gM2 * p * ir;
  prim[at] = u;
  prim[L.sv + at] = v;
  prim[2 * L.sv + at] = w;
  prim[3 * L.sv + at] = T;
  if constexpr (SUTH) prim[4 * L.sv + at] = T * sqrt(T) * (1.0 + P.suth) / (T + P.suth);
}

// Coefficients (times 12 Delta) of the first difference at node i of a line of n nodes and the
// offset of the first stencil node.  Interior eq. (28); ends eq. (30)-(33).
__device__ __forceinline__ int d1_stencil(int n, int i, int per, double (&c)[5]) {
  if (!per) {
    if (i == 0)     { c[0] = -25.0; c[1] = 48.0;  c[2] = -36.0; c[3] = 16.0;  c[4] = -3.0; return 0; }
    if (i == 1)     { c[0] = -3.0;  c[1] = -10.0; c[2] = 18.0;  c[3] = -6.0;  c[4] = 1.0;  return -1; }
    if (i == n - 2) { c[0] = -1.0;  c[1] = 6.0;   c[2] = -18.0; c[3] = 10.0;  c[4] = 3.0;  return -3; }
    if (i == n - 1) { c[0] = 3.0;   c[1] = -16.0; c[2] = 36.0;  c[3] = -48.0; c[4] = 25.0; return -4; }
  }
  c[0] = 1.0; c[1] = -8.0; c[2] = 0.0; c[3] = 8.0; c[4] = -1.0;
  return -2;
}
// Second difference: interior eq. (29); ends eq. (34)-(35) and their mirror images.
__device__ __forceinline__ int d2_stencil(int n, int i, int per, double (&c)[5]) {
  if (!per) {
    if (i == 0)     { c[0] = 35.0; c[1] = -104.0; c[2] = 114.0; c[3] = -56.0;  c[4] = 11.0; return 0; }
    if (i == 1)     { c[0] = 11.0; c[1] = -20.0;  c[2] = 6.0;   c[3] = 4.0;    c[4] = -1.0; return -1; }
    if (i == n - 2) { c[0] = -1.0; c[1] = 4.0;    c[2] = 6.0;   c[3] = -20.0;  c[4] = 11.0; return -3; }
    if (i == n - 1) { c[0] = 11.0; c[1] = -56.0;  c[2] = 114.0; c[3] = -104.0; c[4] = 35.0; return -4; }
  }
  c[0] = -1.0; c[1] = 16.0; c[2] = -30.0; c[3] = 16.0; c[4] = -1.0;
  return -2;
}

// grad[(f * 3 + l) * sv + at] = delta_l f (computational difference incl. the 1/(12 Delta) factor) at every node whose
// l-index is interior and whose other indices lie in the interior extended by 2 along periodic directions
// (where the mixed differences of interior nodes reach).
template <int NF>
__global__ void __launch_bounds__(128)
gradients_kernel(const __grid_constant__ DevParams P, const double *__restrict__ prim, double *__restrict__ grad, int curv) {
  const Layout &L = P.L;
  int ext[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) ext[d] = (L.n[d] > 1 && P.periodic[d]) ? 2 : 0;
  const int nd[3] = {(int)(blockIdx.x * blockDim.x + threadIdx.x) - ext[0], (int)blockIdx.y - ext[1], (int)blockIdx.z - ext[2]};
  if (nd[0] >= L.n[0] + ext[0]) return;
  const long long at = L.at(nd[0], nd[1], nd[2]);
  const long long sv = L.sv;
  const long long st[3] = {1, L.sy, L.sz};
#pragma unroll
  for (int l = 0; l < 3; ++l) {
    if (L.n[l] <= 1 || nd[l] < 0 || nd[l] >= L.n[l]) continue;
    double a[5];
    const int o = d1_stencil(L.n[l], nd[l], P.periodic[l], a);
    const double sc = curv ? (1.0 / 12.0) : P.inv12d[l];
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      double acc = 0.0;
#pragma unroll
      for (int m = 0; m < 5; ++m) acc = fma(a[m] * sc, __ldg(prim + f * sv + at + (long long)(o + m) * st[l]), acc);
      grad[(f * 3 + l) * sv + at] = acc;
    }
  }
}

// Stencil tables (times 12 Delta resp. 12 Delta^2) by node class: 0 interior eq. (28)/(29), 1..4 the one-sided
// closures eq. (30)-(35) at nodes 0, 1, n-2, n-1; c_off = offset of the first stencil node.  Kept in constant memory
// and indexed by the class of the node so that no coefficient array waits in registers.
static __constant__ double c_d1[5][5] = {{1.0, -8.0, 0.0, 8.0, -1.0}, {-25.0, 48.0, -36.0, 16.0, -3.0}, {-3.0, -10.0, 18.0, -6.0, 1.0},
                                         {-1.0, 6.0, -18.0, 10.0, 3.0}, {3.0, -16.0, 36.0, -48.0, 25.0}};
static __constant__ double c_d2[5][5] = {{-1.0, 16.0, -30.0, 16.0, -1.0}, {35.0, -104.0, 114.0, -56.0, 11.0}, {11.0, -20.0, 6.0, 4.0, -1.0},
                                         {-1.0, 4.0, 6.0, -20.0, 11.0}, {11.0, -56.0, 114.0, -104.0, 35.0}};
static __constant__ int c_off[5] = {-2, 0, -1, -3, -4};
__device__ __forceinline__ int node_class(int n, int i, int per) {
  if (per) return 0;
  return i == 0 ? 1 : (i == 1 ? 2 : (i == n - 2 ? 3 : (i == n - 1 ? 4 : 0)));
}

// One thread per node.  Written so that little waits in registers (the first version held the coefficient
// arrays, all first and all second differences of all fields at once: 206 registers, 8 warps per SM, every load a
// full-latency stall): the physical first derivatives of u, v, w, T (, mu) are formed from the stored first
// differences; then ONE field at a time its second / mixed differences are formed and folded straight into the
// Laplacians and into d_i(div u).
// INTERIOR: the node uses the interior stencils eq. (28)-(29) in every direction (all but the two nodes next to each
// non-periodic boundary): coefficients and offsets are compile-time constants, nothing is fetched from the tables.
template <bool CURV, bool SUTH, bool INTERIOR>
__device__ __forceinline__ void viscous_node(const DevParams &P, const double *__restrict__ prim, const double *__restrict__ grad,
                                             double *__restrict__ R, int accumulate, const int (&nd)[3], const int (&cls_in)[3]) {
  const Layout &L = P.L;
  const long long at = L.at(nd[0], nd[1], nd[2]);
  const long long sv = L.sv;
  const long long st[3] = {1, L.sy, L.sz};
  constexpr double kD1[5] = {1.0, -8.0, 0.0, 8.0, -1.0}, kD2[5] = {-1.0, 16.0, -30.0, 16.0, -1.0};
  bool act[3];
  int cls[3];
  double s1[3], s2[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    act[k] = L.n[k] > 1;
    cls[k] = INTERIOR ? 0 : cls_in[k];
    s1[k] = CURV ? (1.0 / 12.0) : P.inv12d[k];
    s2[k] = CURV ? (1.0 / 12.0) : P.inv12d2[k];
  }
  auto F = [&](int f, long long off) { return __ldg(prim + f * sv + at + off); };
  auto Gd = [&](int f, int l, long long off) { return __ldg(grad + (f * 3 + l) * sv + at + off); };
  constexpr int NF1 = SUTH ? 5 : 4;
  constexpr int IJ[3][3] = {{0, 1, 2}, {1, 3, 4}, {2, 4, 5}};
  // the residual this kernel adds to: requested first, consumed last
  double rold[4] = {0.0, 0.0, 0.0, 0.0};
  if (accumulate) {
#pragma unroll
    for (int c = 0; c < 4; ++c) rold[c] = R[(c + 1) * sv + at];
  }

  double D[3][3];
  if constexpr (CURV) {
#pragma unroll
    for (int k = 0; k < 3; ++k)
#pragma unroll
      for (int j = 0; j < 3; ++j) D[k][j] = __ldg(P.D[k][j] + at);
  }
  // computational first differences c1[f][k] = delta_k f (stored by gradients_kernel) and physical first derivatives
  double c1[5][3], g1[5][3];
#pragma unroll
  for (int f = 0; f < 5; ++f)
#pragma unroll
    for (int k = 0; k < 3; ++k) c1[f][k] = (f < NF1 && act[k]) ? Gd(f, k, 0) : 0.0;
#pragma unroll
  for (int f = 0; f < 5; ++f)
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      if constexpr (CURV) g1[f][j] = fma(D[0][j], c1[f][0], fma(D[1][j], c1[f][1], D[2][j] * c1[f][2]));
      else g1[f][j] = c1[f][j];
    }

  // second derivatives, one field at a time: lap[f] = sum_j d_jj f;  gdiv[a] = d_a(d_k u_k) = sum_f d_a d_f u_f
  double lap[4], gdiv[3] = {0.0, 0.0, 0.0};
#pragma unroll
  for (int f = 0; f < 4; ++f) {
    double c2[3][3];
#pragma unroll
    for (int k = 0; k < 3; ++k)
#pragma unroll
      for (int l = k; l < 3; ++l) {
        double acc = 0.0;
        // uniform grids only need d_i d_k u_k: mixed terms of velocity component f along (f, other)
        const bool needed = CURV || k == l || (f < 3 && (k == f || l == f));
        if (needed && act[k] && act[l]) {
          const int o = INTERIOR ? -2 : c_off[cls[k]];
          if (k == l) {
#pragma unroll
            for (int m = 0; m < 5; ++m)
              acc = fma((INTERIOR ? kD2[m] : c_d2[cls[k]][m]) * s2[k], F(f, (long long)(o + m) * st[k]), acc);
          } else {
            // delta_k (delta_l f), k < l: the first-difference stencil along k over the stored delta_l f.  Closures: no
            // run-time test for a zero coefficient (a predicate in front of a load keeps it from being hoisted)
#pragma unroll
            for (int m = 0; m < 5; ++m) {
              if (INTERIOR && m == 2) continue;
              acc = fma((INTERIOR ? kD1[m] : c_d1[cls[k]][m]) * s1[k], Gd(f, l, (long long)(o + m) * st[k]), acc);
            }
          }
        }
        c2[k][l] = acc;
        c2[l][k] = acc;
      }
    // physical d_a d_b f for the (a, b) that are used: the diagonal, and (a, f) for the velocity components
    auto g2 = [&](int a_, int b_) {
      if constexpr (!CURV) return c2[a_][b_];
      else {
        double acc = 0.0;
#pragma unroll
        for (int k = 0; k < 3; ++k)
#pragma unroll
          for (int l = 0; l < 3; ++l) acc = fma(D[k][a_] * D[l][b_], c2[k][l], acc);
#pragma unroll
        for (int l = 0; l < 3; ++l) acc = fma(__ldg(P.E[l][IJ[a_][b_]] + at), c1[f][l], acc);
        return acc;
      }
    };
    double dg[3];
#pragma unroll
    for (int a_ = 0; a_ < 3; ++a_) dg[a_] = g2(a_, a_);
    lap[f] = dg[0] + dg[1] + dg[2];
    if (f < 3) {
#pragma unroll
      for (int a_ = 0; a_ < 3; ++a_) gdiv[a_] += (a_ == f) ? dg[f] : g2(a_, f);
    }
  }

  const double vel[3] = {F(0, 0), F(1, 0), F(2, 0)};
  const double mu = SUTH ? F(4, 0) : 1.0;
  const double div = g1[0][0] + g1[1][1] + g1[2][2];
  // M_i = Re d_j tau_ij = mu (lap u_i + d_i(div u)/3) + d_j mu (d_j u_i + d_i u_j) - 2/3 d_i mu div u
  double M[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    double m = mu * fma(gdiv[a], 1.0 / 3.0, lap[a]);
    if constexpr (SUTH) {
      double cross = 0.0;
#pragma unroll
      for (int b = 0; b < 3; ++b) cross = fma(g1[4][b], g1[a][b] + g1[b][a], cross);
      m += cross - (2.0 / 3.0) * g1[4][a] * div;
    }
    M[a] = m;
  }
  // tau_ij d_j u_i (eq. 5) and -d_j q_j (eq. 4)
  double phi = 0.0;
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b) {
      const double s = g1[a][b] + g1[b][a] - (a == b ? (2.0 / 3.0) * div : 0.0);
      phi = fma(s, g1[a][b], phi);
    }
  phi *= mu * P.inv_Re;
  double heat = mu * lap[3];
  if constexpr (SUTH) heat += g1[4][0] * g1[3][0] + g1[4][1] * g1[3][1] + g1[4][2] * g1[3][2];
  heat *= P.cq;

  const double r1 = M[0] * P.inv_Re, r2 = M[1] * P.inv_Re, r3 = M[2] * P.inv_Re;
  const double r4 = fma(vel[0], r1, fma(vel[1], r2, vel[2] * r3)) + phi + heat;
  double *dst = R + sv + at;
  if (!accumulate) R[at] = 0.0;
  dst[0] = rold[0] + r1; dst[sv] = rold[1] + r2; dst[2 * sv] = rold[2] + r3; dst[3 * sv] = rold[3] + r4;
}

#ifndef OSBLI_GV_MINB
#define OSBLI_GV_MINB 3
#endif
template <bool CURV, bool SUTH>
__global__ void __launch_bounds__(128, OSBLI_GV_MINB)
viscous_kernel(const __grid_constant__ DevParams P, const double *__restrict__ prim, const double *__restrict__ grad,
               double *__restrict__ R, int accumulate) {
  const Layout &L = P.L;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= L.n[0]) return;
  const int nd[3] = {i, (int)blockIdx.y, (int)blockIdx.z};
  int cls[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) cls[k] = node_class(L.n[k], nd[k], P.periodic[k]);
  if ((cls[0] | cls[1] | cls[2]) == 0) viscous_node<CURV, SUTH, true>(P, prim, grad, R, accumulate, nd, cls);
  else viscous_node<CURV, SUTH, false>(P, prim, grad, R, accumulate, nd, cls);
}

// ---------------------------------------------------------------------------------------------
// Central convective terms (scheme 4, uniform grids): R = - sum_d delta_d F_d with the 4th-order
// first difference eq. (28) (closures eq. (30)-(33) next to non-periodic boundaries) of the point-wise
// flux vectors.  One thread per node, x fastest: every neighbour access of a warp
// is a contiguous row segment; the 12 neighbours are shared with the adjacent threads / rows through
// L1 and L2.  First kernel of the stage: writes all five components of R.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128)
central_kernel(const __grid_constant__ DevParams P, const double *__restrict__ Q, double *__restrict__ R) {
  const Layout &L = P.L;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= L.n[0]) return;
  const int nd[3] = {i, (int)blockIdx.y, (int)blockIdx.z};
  const long long at = L.at(nd[0], nd[1], nd[2]);
  const long long sv = L.sv;
  const long long st[3] = {1, L.sy, L.sz};
  double acc[5] = {0, 0, 0, 0, 0};
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    if (L.n[d] <= 1) continue;
    double c[5];
    const int o = d1_stencil(L.n[d], nd[d], P.periodic[d], c);
    const double s = P.inv12d[d];
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      if (c[m] == 0.0) continue;
      const long long a = at + (long long)(o + m) * st[d];
      const double r = __ldg(Q + a), mx = __ldg(Q + sv + a), my = __ldg(Q + 2 * sv + a), mz = __ldg(Q + 3 * sv + a);
      const double E = __ldg(Q + 4 * sv + a);
      const double ir = 1.0 / r;
      const double p = P.gm1 * (E - 0.5 * ir * (mx * mx + my * my + mz * mz));
      const double th = (d == 0 ? mx : (d == 1 ? my : mz)) * ir;
      const double w = c[m] * s;
      acc[0] = fma(w, r * th, acc[0]);
      acc[1] = fma(w, mx * th + (d == 0 ? p : 0.0), acc[1]);
      acc[2] = fma(w, my * th + (d == 1 ? p : 0.0), acc[2]);
      acc[3] = fma(w, mz * th + (d == 2 ? p : 0.0), acc[3]);
      acc[4] = fma(w, (E + p) * th, acc[4]);
    }
  }
#pragma unroll
  for (int c = 0; c < 5; ++c) R[c * sv + at] = -acc[c];
}

cudaError_t launch_central(const DevParams &P, const double *Q, double *R, cudaStream_t st) {
  const Layout &L = P.L;
  dim3 grid((L.n[0] + 127) / 128, L.n[1], L.n[2]);
  central_kernel<<<grid, 128, 0, st>>>(P, Q, R);
  return cudaGetLastError();
}

cudaError_t launch_primitives(const DevParams &P, const double *Q, double *prim, cudaStream_t st) {
  const Layout &L = P.L;
  const int NX = L.n[0] + 2 * L.h[0];
  dim3 grid((NX + 255) / 256, L.n[1] + 2 * L.h[1], L.n[2] + 2 * L.h[2]);
  if (P.visc == 2) primitives_kernel<true><<<grid, 256, 0, st>>>(P, Q, prim);
  else primitives_kernel<false><<<grid, 256, 0, st>>>(P, Q, prim);
  return cudaGetLastError();
}

// stored first differences live behind the staged primitive fields in the workspace (osbli_workspace_bytes)
static double *grad_fields(const DevParams &P, const double *prim) {
  return const_cast<double *>(prim) + (long long)(P.visc == 2 ? 5 : 4) * P.L.sv;
}

cudaError_t launch_gradients(const DevParams &P, const double *prim, cudaStream_t st) {
  const Layout &L = P.L;
  const bool curv = P.curvilinear != 0, suth = P.visc == 2;
  double *grad = grad_fields(P, prim);
  int ext[3];
  for (int d = 0; d < 3; ++d) ext[d] = (L.n[d] > 1 && P.periodic[d]) ? 2 : 0;
  const int NX = L.n[0] + 2 * ext[0];
  dim3 grid((NX + 127) / 128, L.n[1] + 2 * ext[1], L.n[2] + 2 * ext[2]);
  if (suth) gradients_kernel<5><<<grid, 128, 0, st>>>(P, prim, grad, curv ? 1 : 0);
  else gradients_kernel<4><<<grid, 128, 0, st>>>(P, prim, grad, curv ? 1 : 0);
  return cudaGetLastError();
}

cudaError_t launch_viscous_assemble(const DevParams &P, const double *prim, double *R, int accumulate, cudaStream_t st) {
  const Layout &L = P.L;
  const bool curv = P.curvilinear != 0, suth = P.visc == 2;
  const double *grad = grad_fields(P, prim);
  const int bx = L.n[0] >= 128 ? 128 : 64;
  dim3 grid((L.n[0] + bx - 1) / bx, L.n[1], L.n[2]);
  if (curv && suth) viscous_kernel<true, true><<<grid, bx, 0, st>>>(P, prim, grad, R, accumulate);
  else if (curv) viscous_kernel<true, false><<<grid, bx, 0, st>>>(P, prim, grad, R, accumulate);
  else if (suth) viscous_kernel<false, true><<<grid, bx, 0, st>>>(P, prim, grad, R, accumulate);
  else viscous_kernel<false, false><<<grid, bx, 0, st>>>(P, prim, grad, R, accumulate);
  return cudaGetLastError();
}

cudaError_t launch_viscous(const DevParams &P, const double *Q, const double *prim, double *R, int accumulate,
                           cudaStream_t st) {
  (void)Q;
  cudaError_t e = launch_gradients(P, prim, st);
  if (e != cudaSuccess) return e;
  return launch_viscous_assemble(P, prim, R, accumulate, st);
}

// =============================================================================================
// Fast path: uniform grid, mu = 1, three active periodic directions (the Taylor-Green cases).
//
// 2.5-D marching: a block owns a 32 x 8 (x,y) tile and walks along z.  The kernel is bound by the
// shared-memory data path (every in-plane stencil value is an LDS), so every in-plane stencil is read
// exactly ONCE, when its plane enters the pipeline (two steps before it becomes the centre plane):
//   * raw plane tiles (36 x 12 x 5 variables) arrive by TMA two steps ahead (4-D tensor map, mbarrier),
//     are turned into u, v, w, T planes in a 2-slot shared-memory ring (the plane being staged and the
//     plane entering);
//   * on entry a thread reads the x- and y-stencils of its node (32 LDS) and forms every in-plane first and
//     second difference at once; what the centre step will need of them waits in registers: z-windows of
//     u, v, w and of S0 = d_x w, S1 = d_y w, S2 = d_x u + d_y v (whose z-differences are the x-z / y-z
//     mixed terms of d_i(div u)), the in-plane parts of the three momentum operators (3-deep delay
//     lines), and 5-deep scatter accumulators of the energy equation's linear + in-plane part;
//   * the x-y mixed differences d_x(d_y u), d_x(d_y v) come from a small exchange buffer: each thread
//     publishes d_y u, d_y v of its node (one warp adds the 2-deep x halo columns) and reads its four
//     x-neighbours one step later -- 8 LDS instead of the 32 of a direct 16-point evaluation.
// 44 LDS.64 per node instead of 84; one barrier per plane; R of the node travels by cp.async into a
// per-thread slot.
// =============================================================================================
#ifndef OSBLI_VCHUNK
#define OSBLI_VCHUNK 32
#endif
#ifndef OSBLI_VMINB
#define OSBLI_VMINB 2
#endif

// Raw planes reach shared memory by TMA: the 36 x 12 tile of all five variables of one plane is one box of a
// 4-D tensor map over the state, loaded by one cp.async.bulk.tensor issued by one thread, completion on an
// mbarrier; rows and columns past the array are zero-filled by the hardware (ragged tiles need no guards).
struct VSmem {
  double tile[2][5][kVPY][kVPX];       // TMA destinations (128-byte aligned: first member), double buffered
  double f[2][4][kVPY][kVPX];          // u, v, w, T: the plane being staged and the plane entering
  double g[2][2][kVY][kVPX];           // d_y u, d_y v of the tile rows incl. the x halo, double buffered
  double r[2][4][kVX * kVY];           // per-thread slots: R of the two nodes in flight (cp.async, issued one step ahead)
  unsigned long long mbar[2];          // one mbarrier per TMA buffer
};

__global__ void __launch_bounds__(kVX * kVY, OSBLI_VMINB)
viscous_tgv_kernel(const __grid_constant__ DevParams P, const double *__restrict__ Q, double *__restrict__ R,
                   int chunk, const __grid_constant__ CUtensorMap tmap) {
  extern __shared__ __align__(128) unsigned char vs_raw[];
  VSmem &S = *reinterpret_cast<VSmem *>(vs_raw);
  const Layout &L = P.L;
  const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * kVX + tx;
  const int x0 = blockIdx.x * kVX, y0 = blockIdx.y * kVY;
  const int z0 = blockIdx.z * chunk, z1 = min(z0 + chunk, L.n[2]);
  const int i = x0 + tx, j = y0 + ty;
  const bool inside = i < L.n[0] && j < L.n[1];
  const long long sv = L.sv;

  // the (up to) two tile points this thread stages per plane
  constexpr int NPT = kVPX * kVPY;                                // 432
  int pi[2], pj[2];
  bool pv[2];
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    const int t = tid + s * (kVX * kVY);
    pv[s] = t < NPT;
    const int yy = pv[s] ? t / kVPX : 0, xx = pv[s] ? t % kVPX : 0;
    pi[s] = xx; pj[s] = yy;
    // clamp to the halo-extended domain: clamped points are never used by live threads
    pv[s] = pv[s] && (x0 + xx - kVH) < L.n[0] + kVH && (y0 + yy - kVH) < L.n[1] + kVH;
  }
  // plane number jj = plane - (z0 - 2) of this block goes through TMA buffer jj & 1; its mbarrier has then
  // completed (jj >> 1) phases before, which fixes the parity to wait for
  auto fetch = [&](int plane) {
    if (tid == 0) {
      const int b = (plane - (z0 - 2)) & 1;
      mbar_expect_tx(&S.mbar[b], kVTileBytes);
      tma_load_4d(&S.tile[b][0][0][0], &tmap, (int)L.xoff + x0 - kVH, L.h[1] + y0 - kVH, L.h[2] + plane, 0, &S.mbar[b]);
    }
  };
  auto stage = [&](int plane) {
    const int slot = (plane + 8) & 1;
    const int jj = plane - (z0 - 2), b = jj & 1;
    mbar_wait(&S.mbar[b], (unsigned)(jj >> 1) & 1u);
#pragma unroll
    for (int s = 0; s < 2; ++s)
      if (pv[s]) {
        const double q0 = S.tile[b][0][pj[s]][pi[s]], q1 = S.tile[b][1][pj[s]][pi[s]], q2 = S.tile[b][2][pj[s]][pi[s]];
        const double q3 = S.tile[b][3][pj[s]][pi[s]], q4 = S.tile[b][4][pj[s]][pi[s]];
        const double ir = fast_rcp(q0);
        const double u = q1 * ir, v = q2 * ir, w = q3 * ir;
        const double p = P.gm1 * (q4 - 0.5 * (q1 * u + q2 * v + q3 * w));
        S.f[slot][0][pj[s]][pi[s]] = u;
        S.f[slot][1][pj[s]][pi[s]] = v;
        S.f[slot][2][pj[s]][pi[s]] = w;
        S.f[slot][3][pj[s]][pi[s]] = P.gM2 * p * ir;
      }
  };
  if (tid == 0) {
    mbar_init(&S.mbar[0], 1);
    mbar_init(&S.mbar[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  const double cx = P.inv12d[0], cy = P.inv12d[1], cz = P.inv12d[2];
  const double cxx = P.inv12d2[0], cyy = P.inv12d2[1], czz = P.inv12d2[2];
  auto d1 = [](double m2, double m1, double p1, double p2, double c) { return c * ((m2 - p2) + 8.0 * (p1 - m1)); };
  auto d2 = [](double m2, double m1, double f0, double p1, double p2, double c) {
    return c * fma(-30.0, f0, fma(16.0, m1 + p1, -(m2 + p2)));
  };
  constexpr double third = 1.0 / 3.0, four3 = 4.0 / 3.0;

  // Register state of this thread's column.  After the shift of step k: windows hold planes k-2..k+2 (slots
  // 0..4), the delay lines planes k..k+2 (slots 0..2), the energy accumulators planes k..k+4.  (Unrolling the plane loop five times so that the windows rotate without
  // register moves was measured: 0.467 -> 0.492 ms, 66 KB of code against a 32 KB instruction cache.)
  double uw[5], vw[5], ww[5], s0w[5], s1w[5], s2w[5];
  double Au[3], Av[3], Aw[3];        // in-plane parts of M_0, M_1, M_2 (incl. the x-y mixed terms, folded one step later)
  double aE[5];                      // cq (T_xx + T_yy + T_zz) + (2 u_x^2 + 2 v_y^2 + (u_y + v_x)^2)/Re, scatter form
#pragma unroll
  for (int m = 0; m < 5; ++m) uw[m] = vw[m] = ww[m] = s0w[m] = s1w[m] = s2w[m] = aE[m] = 0.0;
#pragma unroll
  for (int m = 0; m < 3; ++m) Au[m] = Av[m] = Aw[m] = 0.0;

  // Software pipeline, one barrier per plane: during step k (node k is finished) plane k+3 is staged into
  // the ring slot plane k+1 has left, the raw plane k+4 is fetched, plane k+2 (staged one step earlier)
  // enters, the x-y mixed terms of plane k+1 are folded in, and plane k is completed from registers alone.
  fetch(z0 - 2);
  stage(z0 - 2);
  fetch(z0 - 1);
  __syncthreads();
  const int X = tx + kVH, Y = ty + kVH;
  // the warp that also publishes d_y u, d_y v of the x halo columns: 8 rows x 4 columns
  const int hr = tid >> 2, hc = (tid & 3) < 2 ? (tid & 3) : kVX + (tid & 3);

  constexpr int M2 = 0, M1 = 1, C = 2, P1 = 3, P2 = 4;          // window slots of planes k-2, k-1, k, k+1, k+2
  for (int k = z0 - 4; k < z1; ++k) {
    if (k > z0 - 4) __syncthreads();
    if (k + 3 < z1 + 2) stage(k + 3);
    // R of node k+1 goes to a per-thread shared-memory slot by cp.async, one whole step before it is needed (the
    // arithmetic of a single step does not cover the DRAM latency)
    if (k + 1 >= z0 && k + 1 < z1 && inside) {
      const long long a1 = L.at(i, j, k + 1);
#pragma unroll
      for (int c = 0; c < 4; ++c) cp_async8(&S.r[(k + 1) & 1][c][tid], R + (c + 1) * sv + a1);
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
    if (k + 4 < z1 + 2) fetch(k + 4);                          // raw plane k+4 into the buffer plane k+2 has left
#pragma unroll
    for (int m = 0; m < 4; ++m) {
      uw[m] = uw[m + 1]; vw[m] = vw[m + 1]; ww[m] = ww[m + 1];
      s0w[m] = s0w[m + 1]; s1w[m] = s1w[m + 1]; s2w[m] = s2w[m + 1]; aE[m] = aE[m + 1];
    }
    aE[4] = 0.0;
    Au[0] = Au[1]; Au[1] = Au[2]; Av[0] = Av[1]; Av[1] = Av[2]; Aw[0] = Aw[1]; Aw[1] = Aw[2];
    // ---- plane k+2 enters: every in-plane stencil of this node, read once.  The two planes either side of the
    // chunk only feed z-stencils: they need u, v, w, T, S0, S1, S2 and nothing else (FULL = false).
    auto enter = [&](auto full_tag) {
      constexpr bool FULL = decltype(full_tag)::value;
      const int e = (k + 2 + 8) & 1;
      const double (*F)[kVPY][kVPX] = S.f[e];
      const double u = F[0][Y][X], v = F[1][Y][X], w = F[2][Y][X], T = F[3][Y][X];
      const double uxm2 = F[0][Y][X - 2], uxm1 = F[0][Y][X - 1], uxp1 = F[0][Y][X + 1], uxp2 = F[0][Y][X + 2];
      const double vym2 = F[1][Y - 2][X], vym1 = F[1][Y - 1][X], vyp1 = F[1][Y + 1][X], vyp2 = F[1][Y + 2][X];
      const double wxm2 = F[2][Y][X - 2], wxm1 = F[2][Y][X - 1], wxp1 = F[2][Y][X + 1], wxp2 = F[2][Y][X + 2];
      const double wym2 = F[2][Y - 2][X], wym1 = F[2][Y - 1][X], wyp1 = F[2][Y + 1][X], wyp2 = F[2][Y + 2][X];
      const double u_x = d1(uxm2, uxm1, uxp1, uxp2, cx), v_y = d1(vym2, vym1, vyp1, vyp2, cy);
      uw[P2] = u; vw[P2] = v; ww[P2] = w;
      s0w[P2] = d1(wxm2, wxm1, wxp1, wxp2, cx);
      s1w[P2] = d1(wym2, wym1, wyp1, wyp2, cy);
      s2w[P2] = u_x + v_y;
      // energy equation, everything that is linear in plane k+2 or lives in it: the z-stencil of T scattered to
      // the five planes k..k+4 it feeds (weights -1, 16, -30, 16, -1), plus the in-plane terms
      const double tz = (P.cq * czz) * T;
      aE[0] -= tz; aE[1] = fma(16.0, tz, aE[1]); aE[2] = fma(-30.0, tz, aE[2]); aE[3] = fma(16.0, tz, aE[3]); aE[4] -= tz;
      if constexpr (FULL) {
        const double uym2 = F[0][Y - 2][X], uym1 = F[0][Y - 1][X], uyp1 = F[0][Y + 1][X], uyp2 = F[0][Y + 2][X];
        const double vxm2 = F[1][Y][X - 2], vxm1 = F[1][Y][X - 1], vxp1 = F[1][Y][X + 1], vxp2 = F[1][Y][X + 2];
        const double u_y = d1(uym2, uym1, uyp1, uyp2, cy), v_x = d1(vxm2, vxm1, vxp1, vxp2, cx);
        Au[2] = fma(four3, d2(uxm2, uxm1, u, uxp1, uxp2, cxx), d2(uym2, uym1, u, uyp1, uyp2, cyy));
        Av[2] = fma(four3, d2(vym2, vym1, v, vyp1, vyp2, cyy), d2(vxm2, vxm1, v, vxp1, vxp2, cxx));
        S.g[e][0][ty][X] = u_y;
        S.g[e][1][ty][X] = v_y;
        Aw[2] = d2(wxm2, wxm1, w, wxp1, wxp2, cxx) + d2(wym2, wym1, w, wyp1, wyp2, cyy);
        const double lapT = d2(F[3][Y][X - 2], F[3][Y][X - 1], T, F[3][Y][X + 1], F[3][Y][X + 2], cxx) +
                            d2(F[3][Y - 2][X], F[3][Y - 1][X], T, F[3][Y + 1][X], F[3][Y + 2][X], cyy);
        const double sxy = u_y + v_x;
        aE[2] += fma(P.cq, lapT, P.inv_Re * fma(sxy, sxy, 2.0 * fma(u_x, u_x, v_y * v_y)));
        if (tid < 32) {                                          // x halo columns of the exchange buffer
          const int Yh = hr + kVH;
          S.g[e][0][hr][hc] = d1(F[0][Yh - 2][hc], F[0][Yh - 1][hc], F[0][Yh + 1][hc], F[0][Yh + 2][hc], cy);
          S.g[e][1][hr][hc] = d1(F[1][Yh - 2][hc], F[1][Yh - 1][hc], F[1][Yh + 1][hc], F[1][Yh + 2][hc], cy);
        }
      }
    };
    if (k + 2 >= z0 && k + 2 < z1) enter(std::true_type{});
    else enter(std::false_type{});
    if (k + 1 >= z0 && k + 1 < z1) {
      // ---- x-y mixed terms of plane k+1: d_x of the d_y values published one step ago
      const double (*G)[kVY][kVPX] = S.g[(k + 1 + 8) & 1];
      Au[1] = fma(third, d1(G[1][ty][X - 2], G[1][ty][X - 1], G[1][ty][X + 1], G[1][ty][X + 2], cx), Au[1]);   // + v_xy / 3
      Av[1] = fma(third, d1(G[0][ty][X - 2], G[0][ty][X - 1], G[0][ty][X + 1], G[0][ty][X + 2], cx), Av[1]);   // + u_xy / 3
    }
    if (k < z0 || !inside) continue;

    // ---- plane k is complete: z-direction terms from the register windows
    const double u = uw[C], v = vw[C], w = ww[C];
    const double u_z = d1(uw[M2], uw[M1], uw[P1], uw[P2], cz);
    const double v_z = d1(vw[M2], vw[M1], vw[P1], vw[P2], cz);
    const double w_z = d1(ww[M2], ww[M1], ww[P1], ww[P2], cz);
    const double u_zz = d2(uw[M2], uw[M1], u, uw[P1], uw[P2], czz);
    const double v_zz = d2(vw[M2], vw[M1], v, vw[P1], vw[P2], czz);
    const double w_zz = d2(ww[M2], ww[M1], w, ww[P1], ww[P2], czz);
    const double M0 = Au[0] + fma(third, d1(s0w[M2], s0w[M1], s0w[P1], s0w[P2], cz), u_zz);          // + w_xz / 3
    const double M1v = Av[0] + fma(third, d1(s1w[M2], s1w[M1], s1w[P1], s1w[P2], cz), v_zz);         // + w_yz / 3
    const double M2v = Aw[0] + fma(third, d1(s2w[M2], s2w[M1], s2w[P1], s2w[P2], cz), four3 * w_zz); // + (u_xz + v_yz)/3
    // tau_ij d_j u_i = [2 (u_x^2 + v_y^2 + w_z^2) - 2/3 div^2 + s_xy^2 + s_xz^2 + s_yz^2]/Re; the in-plane part is in aE
    const double div = s2w[C] + w_z;
    const double sxz = u_z + s0w[C], syz = v_z + s1w[C];
    const double phiz = fma(sxz, sxz, fma(syz, syz, fma(2.0 * w_z, w_z, (-2.0 / 3.0) * (div * div))));
    const double r1 = M0 * P.inv_Re, r2 = M1v * P.inv_Re, r3 = M2v * P.inv_Re;
    const double r4 = fma(u, r1, fma(v, r2, w * r3)) + fma(phiz, P.inv_Re, aE[0]);
    asm volatile("cp.async.wait_group 1;" ::: "memory");       // R of node k (issued one step ago) has landed
    const long long at = L.at(i, j, k);
    const double rold[4] = {S.r[k & 1][0][tid], S.r[k & 1][1][tid], S.r[k & 1][2][tid], S.r[k & 1][3][tid]};
    R[sv + at] = rold[0] + r1;
    R[2 * sv + at] = rold[1] + r2;
    R[3 * sv + at] = rold[2] + r3;
    R[4 * sv + at] = rold[3] + r4;
  }
}

bool viscous_fast_path(const DevParams &P) {
  if (P.curvilinear || P.visc != 1) return false;
  for (int d = 0; d < 3; ++d)
    if (P.L.n[d] <= 1 || !P.periodic[d]) return false;
  return true;
}

cudaError_t launch_viscous_fast(const DevParams &P, const double *Q, double *R, TmapCache *cache, cudaStream_t st) {
  const Layout &L = P.L;
  const int chunk = L.n[2] > OSBLI_VCHUNK ? OSBLI_VCHUNK : L.n[2];
  dim3 grid((L.n[0] + kVX - 1) / kVX, (L.n[1] + kVY - 1) / kVY, (L.n[2] + chunk - 1) / chunk);
  const CUtensorMap *map = state_tensor_map(L, Q, cache);
  if (!map) return cudaErrorNotSupported;
  viscous_tgv_kernel<<<grid, dim3(kVX, kVY), sizeof(VSmem), st>>>(P, Q, R, chunk, *map);
  return cudaGetLastError();
}

// Opt-in shared-memory sizes of the kernels of this file, once per device (called by osbli_init).
cudaError_t viscous_set_attributes() {
  return cudaFuncSetAttribute(viscous_tgv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(VSmem));
}

}  // namespace osbli
