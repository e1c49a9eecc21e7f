// osbli_visc.cu -- viscous and heat-flux terms of eq. (2)-(5), discretised with the
// 4th-order central differences of eq. (28)-(29) (eq. (28) with its sign corrected, Q1)
// and the one-sided closures of eq. (30)-(35), next to non-periodic boundaries;
// metric chain rule on curvilinear grids.
//
// Two kernels: (1) point-wise u, v, w, T (, mu) staged once per stage on the halo-extended grid
// (the paper's "store some" idea: keep the few fields every derivative needs,
// recompute the rest); (2) one thread per node assembling all derivatives from those fields and
// adding  d_j tau_ij,  d_j(u_i tau_ij) - d_j q_j  to R.
#include "osbli_kernels.h"

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

template <bool CURV, bool SUTH>
__global__ void __launch_bounds__(128)
viscous_kernel(const __grid_constant__ DevParams P, const double *__restrict__ prim, double *__restrict__ R,
               int accumulate) {
  const Layout &L = P.L;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= L.n[0]) return;
  const int nd[3] = {i, (int)blockIdx.y, (int)blockIdx.z};
  const long long at = L.at(nd[0], nd[1], nd[2]);
  const long long sv = L.sv;
  const long long st[3] = {1, L.sy, L.sz};
  bool act[3];
  double a1[3][5], a2[3][5];
  int o1[3], o2[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    act[k] = L.n[k] > 1;
    o1[k] = d1_stencil(L.n[k], nd[k], P.periodic[k], a1[k]);
    o2[k] = d2_stencil(L.n[k], nd[k], P.periodic[k], a2[k]);
    const double s1 = CURV ? (1.0 / 12.0) : P.inv12d[k];
    const double s2 = CURV ? (1.0 / 12.0) : P.inv12d2[k];
#pragma unroll
    for (int m = 0; m < 5; ++m) { a1[k][m] *= s1; a2[k][m] *= s2; }
  }
  auto F = [&](int f, long long off) { return __ldg(prim + f * sv + at + off); };

  // computational differences: c1[f][k] = delta_k f, c2[f][k][l] = delta_kl f
  constexpr int NF1 = SUTH ? 5 : 4;
  double c1[5][3], c2[4][3][3];
#pragma unroll
  for (int f = 0; f < 5; ++f)
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      double acc = 0.0;
      if (f < NF1 && act[k]) {
#pragma unroll
        for (int m = 0; m < 5; ++m)
          if (a1[k][m] != 0.0) acc = fma(a1[k][m], F(f, (long long)(o1[k] + m) * st[k]), acc);
      }
      c1[f][k] = acc;
    }
#pragma unroll
  for (int f = 0; f < 4; ++f)
#pragma unroll
    for (int k = 0; k < 3; ++k)
#pragma unroll
      for (int l = k; l < 3; ++l) {
        double acc = 0.0;
        // uniform grids only need d_i d_k u_k: mixed terms of velocity component f along (f, other)
        const bool needed = CURV || k == l || (f < 3 && (k == f || l == f));
        if (needed && act[k] && act[l]) {
          if (k == l) {
#pragma unroll
            for (int m = 0; m < 5; ++m) acc = fma(a2[k][m], F(f, (long long)(o2[k] + m) * st[k]), acc);
          } else {
#pragma unroll
            for (int a = 0; a < 5; ++a) {
              if (a1[k][a] == 0.0) continue;
              double in = 0.0;
#pragma unroll
              for (int b = 0; b < 5; ++b)
                if (a1[l][b] != 0.0)
                  in = fma(a1[l][b], F(f, (long long)(o1[k] + a) * st[k] + (long long)(o1[l] + b) * st[l]), in);
              acc = fma(a1[k][a], in, acc);
            }
          }
        }
        c2[f][k][l] = acc;
        c2[f][l][k] = acc;
      }

  // physical derivatives g1[f][j] = d_j f, g2[f][i][j] = d_i d_j f
  double g1[5][3], g2[4][3][3];
  if constexpr (!CURV) {
#pragma unroll
    for (int f = 0; f < 5; ++f)
#pragma unroll
      for (int j = 0; j < 3; ++j) g1[f][j] = c1[f][j];
#pragma unroll
    for (int f = 0; f < 4; ++f)
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) g2[f][a][b] = c2[f][a][b];
  } else {
    constexpr int IJ[3][3] = {{0, 1, 2}, {1, 3, 4}, {2, 4, 5}};
    double D[3][3], E[3][6];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
#pragma unroll
      for (int j = 0; j < 3; ++j) D[k][j] = __ldg(P.D[k][j] + at);
#pragma unroll
      for (int m = 0; m < 6; ++m) E[k][m] = __ldg(P.E[k][m] + at);
    }
#pragma unroll
    for (int f = 0; f < 5; ++f)
#pragma unroll
      for (int j = 0; j < 3; ++j)
        g1[f][j] = fma(D[0][j], c1[f][0], fma(D[1][j], c1[f][1], D[2][j] * c1[f][2]));
#pragma unroll
    for (int f = 0; f < 4; ++f)
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = a; b < 3; ++b) {
          double acc = 0.0;
#pragma unroll
          for (int k = 0; k < 3; ++k)
#pragma unroll
            for (int l = 0; l < 3; ++l) acc = fma(D[k][a] * D[l][b], c2[f][k][l], acc);
#pragma unroll
          for (int l = 0; l < 3; ++l) acc = fma(E[l][IJ[a][b]], c1[f][l], acc);
          g2[f][a][b] = acc;
          g2[f][b][a] = acc;
        }
  }

  const double vel[3] = {F(0, 0), F(1, 0), F(2, 0)};
  const double mu = SUTH ? F(4, 0) : 1.0;
  const double div = g1[0][0] + g1[1][1] + g1[2][2];
  // M_i = Re d_j tau_ij = mu (lap u_i + d_i(div u)/3) + d_j mu (d_j u_i + d_i u_j) - 2/3 d_i mu div u
  double M[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double lap = g2[a][0][0] + g2[a][1][1] + g2[a][2][2];
    const double gdiv = g2[0][a][0] + g2[1][a][1] + g2[2][a][2];
    double m = mu * fma(gdiv, 1.0 / 3.0, lap);
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
  const double lapT = g2[3][0][0] + g2[3][1][1] + g2[3][2][2];
  double heat = mu * lapT;
  if constexpr (SUTH) heat += g1[4][0] * g1[3][0] + g1[4][1] * g1[3][1] + g1[4][2] * g1[3][2];
  heat *= P.cq;

  const double r1 = M[0] * P.inv_Re, r2 = M[1] * P.inv_Re, r3 = M[2] * P.inv_Re;
  const double r4 = fma(vel[0], r1, fma(vel[1], r2, vel[2] * r3)) + phi + heat;
  double *dst = R + sv + at;
  if (accumulate) {
    dst[0] += r1; dst[sv] += r2; dst[2 * sv] += r3; dst[3 * sv] += r4;
  } else {
    R[at] = 0.0; dst[0] = r1; dst[sv] = r2; dst[2 * sv] = r3; dst[3 * sv] = r4;
  }
}

cudaError_t launch_primitives(const DevParams &P, const double *Q, double *prim, cudaStream_t st) {
  const Layout &L = P.L;
  const int NX = L.n[0] + 2 * L.h[0];
  dim3 grid((NX + 255) / 256, L.n[1] + 2 * L.h[1], L.n[2] + 2 * L.h[2]);
  if (P.visc == 2) primitives_kernel<true><<<grid, 256, 0, st>>>(P, Q, prim);
  else primitives_kernel<false><<<grid, 256, 0, st>>>(P, Q, prim);
  return cudaGetLastError();
}

cudaError_t launch_viscous(const DevParams &P, const double *Q, const double *prim, double *R, int accumulate,
                           cudaStream_t st) {
  (void)Q;
  const Layout &L = P.L;
  const int bx = L.n[0] >= 128 ? 128 : 64;
  dim3 grid((L.n[0] + bx - 1) / bx, L.n[1], L.n[2]);
  const bool curv = P.curvilinear != 0, suth = P.visc == 2;
  if (curv && suth) viscous_kernel<true, true><<<grid, bx, 0, st>>>(P, prim, R, accumulate);
  else if (curv) viscous_kernel<true, false><<<grid, bx, 0, st>>>(P, prim, R, accumulate);
  else if (suth) viscous_kernel<false, true><<<grid, bx, 0, st>>>(P, prim, R, accumulate);
  else viscous_kernel<false, false><<<grid, bx, 0, st>>>(P, prim, R, accumulate);
  return cudaGetLastError();
}

}  // namespace osbli
