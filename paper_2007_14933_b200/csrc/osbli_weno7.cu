// osbli_weno7.cu -- 7th-order WENO-Z sweeps (scheme 6; "any arbitrary odd order", eq. (15)-(16), (20),
// (22); used at 7th order in PAPER.md:485-495 and 531-533; Q40): R (-)= (f^_{i+1/2} - f^_{i-1/2}) / Delta_d
// (or / detJ_i) with the characteristic flux reconstruction of PAPER.md:100-111 on the eight-point window i-3..i+4.
//
// A side scheme, written for correctness and not tuned like the 5th/6th-order sweeps of
// osbli_sweep.cu: one thread per node evaluates both of its interface fluxes (each interface twice over the grid),
// eigenvectors are applied as dense 5x5 matrices for a general unit normal (uniform grids: e_d), the stage update is
// the separate rk_update_kernel.  What it shares with the tuned path is the layout, the boundary fills and the
// viscous kernels; the halo depth is 4 (Layout::h).
#include "osbli_kernels.h"

namespace osbli {

namespace {

// WENO-7Z value at the interface between v[3] and v[4], upwind side v[0..3]; D_j = v[j+1] - v[j].
// Candidate r lives on nodes {3-r .. 6-r} and uses D_{3-r}, D_{4-r}, D_{5-r} =: e0, e1, e2; with p = r the position
// of node 3 in the stencil, the cubic's value at the interface (minus v[3]) and its Taylor coefficients at node 3:
//   p = 0: q = (9 e0 - 4 e1 + e2)/12     a1 = (43 e0 - 26 e1 + 7 e2)/24   a2 = (-2 e0 + 3 e1 - e2)/2
//   p = 1: q = (e0 + 6 e1 - e2)/12       a1 = (7 e0 + 22 e1 - 5 e2)/24    a2 = (e1 - e0)/2
//   p = 2: q = (-e0 + 4 e1 + 3 e2)/12    a1 = (-5 e0 + 22 e1 + 7 e2)/24   a2 = (e2 - e1)/2
//   p = 3: q = (3 e0 - 10 e1 + 13 e2)/12 a1 = (7 e0 - 26 e1 + 43 e2)/24   a2 = (e0 - 3 e1 + 2 e2)/2
//   a3 = (e0 - 2 e1 + e2)/6 for all;  beta = a1^2 + 13/3 a2^2 + 3129/80 a3^2 + a1 a3/2   (eq. (16) on a cubic)
// ideal weights (4, 18, 12, 1)/35, tau_7 = |beta_0 - beta_3|, alpha_r = d_r (1 + (tau/(beta_r + eps))^2), eq. (22).
__device__ __forceinline__ double weno7z(const double (&v)[7], double eps) {
  double D[6];
#pragma unroll
  for (int j = 0; j < 6; ++j) D[j] = v[j + 1] - v[j];
  constexpr double cq[4][3] = {{9.0 / 12.0, -4.0 / 12.0, 1.0 / 12.0}, {1.0 / 12.0, 6.0 / 12.0, -1.0 / 12.0},
                               {-1.0 / 12.0, 4.0 / 12.0, 3.0 / 12.0}, {3.0 / 12.0, -10.0 / 12.0, 13.0 / 12.0}};
  constexpr double c1[4][3] = {{43.0 / 24.0, -26.0 / 24.0, 7.0 / 24.0}, {7.0 / 24.0, 22.0 / 24.0, -5.0 / 24.0},
                               {-5.0 / 24.0, 22.0 / 24.0, 7.0 / 24.0}, {7.0 / 24.0, -26.0 / 24.0, 43.0 / 24.0}};
  constexpr double c2[4][3] = {{-1.0, 1.5, -0.5}, {-0.5, 0.5, 0.0}, {0.0, -0.5, 0.5}, {0.5, -1.5, 1.0}};
  constexpr double dw[4] = {4.0 / 35.0, 18.0 / 35.0, 12.0 / 35.0, 1.0 / 35.0};
  double q[4], beta[4];
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    const double e0 = D[3 - r], e1 = D[4 - r], e2 = D[5 - r];
    q[r] = fma(cq[r][0], e0, fma(cq[r][1], e1, cq[r][2] * e2));
    const double a1 = fma(c1[r][0], e0, fma(c1[r][1], e1, c1[r][2] * e2));
    const double a2 = fma(c2[r][0], e0, fma(c2[r][1], e1, c2[r][2] * e2));
    const double a3 = (e0 - 2.0 * e1 + e2) * (1.0 / 6.0);
    beta[r] = fma(a1, a1, fma(13.0 / 3.0 * a2, a2, fma(3129.0 / 80.0 * a3, a3, 0.5 * (a1 * a3))));
  }
  const double tau = fabs(beta[0] - beta[3]);
  double num = 0.0, den = 0.0;
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    const double x = tau / (beta[r] + eps);
    const double al = dw[r] * fma(x, x, 1.0);
    num = fma(al, q[r], num);
    den += al;
  }
  return v[3] + num / den;
}

// f^_{i+1/2} between node `at` and `at + s` (s = stride of DIR), PAPER.md:100-111 steps 1-2.
template <int DIR, bool CURV>
__device__ __forceinline__ void interface_flux7(const DevParams &P, const double *__restrict__ Q, long long at, long long s,
                                                double (&fhat)[5]) {
  const long long sv = P.L.sv;
  double U[8][5], F[8][5], lam[8][3], Kil[2][3];
  // step 1: solution vector, flux and wave speeds at the eight stencil points i-3..i+4
#pragma unroll
  for (int m = 0; m < 8; ++m) {
    const long long pt = at + (long long)(m - 3) * s;
#pragma unroll
    for (int c = 0; c < 5; ++c) U[m][c] = __ldg(Q + c * sv + pt);
    double K[3] = {DIR == 0 ? 1.0 : 0.0, DIR == 1 ? 1.0 : 0.0, DIR == 2 ? 1.0 : 0.0};
    if constexpr (CURV) {
      const double J = __ldg(P.detJ + pt);
#pragma unroll
      for (int a = 0; a < 3; ++a) K[a] = J * __ldg(P.D[DIR][a] + pt);
    }
    if (m == 3 || m == 4) { Kil[m - 3][0] = K[0]; Kil[m - 3][1] = K[1]; Kil[m - 3][2] = K[2]; }
    const double ir = 1.0 / U[m][0];
    const double u = U[m][1] * ir, v = U[m][2] * ir, w = U[m][3] * ir;
    const double p = P.gm1 * (U[m][4] - 0.5 * (U[m][1] * u + U[m][2] * v + U[m][3] * w));
    const double a = sqrt(P.gamma * p * ir);
    const double th = K[0] * u + K[1] * v + K[2] * w;
    const double Kn = CURV ? sqrt(K[0] * K[0] + K[1] * K[1] + K[2] * K[2]) : 1.0;
    F[m][0] = U[m][0] * th;
    F[m][1] = fma(U[m][1], th, p * K[0]);
    F[m][2] = fma(U[m][2], th, p * K[1]);
    F[m][3] = fma(U[m][3], th, p * K[2]);
    F[m][4] = (U[m][4] + p) * th;
    lam[m][0] = fabs(th); lam[m][1] = fabs(th + a * Kn); lam[m][2] = fabs(th - a * Kn);
  }
  // step 2(a): Roe (or simple) average of nodes i, i+1; interface normal from the averaged K
  double n[3] = {DIR == 0 ? 1.0 : 0.0, DIR == 1 ? 1.0 : 0.0, DIR == 2 ? 1.0 : 0.0};
  if constexpr (CURV) {
    const double kx = 0.5 * (Kil[0][0] + Kil[1][0]), ky = 0.5 * (Kil[0][1] + Kil[1][1]), kz = 0.5 * (Kil[0][2] + Kil[1][2]);
    const double ik = 1.0 / sqrt(kx * kx + ky * ky + kz * kz);
    n[0] = kx * ik; n[1] = ky * ik; n[2] = kz * ik;
  }
  double u, v, w, H;
  {
    const double *UL = U[3], *UR = U[4];
    if (P.averaging != 0) {            // U_{i+1/2} = (U_i + U_{i+1})/2
      const double r = 0.5 * (UL[0] + UR[0]), ir = 1.0 / r;
      u = 0.5 * (UL[1] + UR[1]) * ir; v = 0.5 * (UL[2] + UR[2]) * ir; w = 0.5 * (UL[3] + UR[3]) * ir;
      const double E = 0.5 * (UL[4] + UR[4]);
      const double p = P.gm1 * (E - 0.5 * r * (u * u + v * v + w * w));
      H = (E + p) * ir;
    } else {
      const double pL = P.gm1 * (UL[4] - 0.5 * (UL[1] * UL[1] + UL[2] * UL[2] + UL[3] * UL[3]) / UL[0]);
      const double pR = P.gm1 * (UR[4] - 0.5 * (UR[1] * UR[1] + UR[2] * UR[2] + UR[3] * UR[3]) / UR[0]);
      const double sl = sqrt(UL[0]), sr = sqrt(UR[0]), is = 1.0 / (sl + sr);
      u = (UL[1] / sl + UR[1] / sr) * is; v = (UL[2] / sl + UR[2] / sr) * is; w = (UL[3] / sl + UR[3] / sr) * is;
      H = ((UL[4] + pL) / sl + (UR[4] + pR) / sr) * is;
    }
  }
  const double q2 = u * u + v * v + w * w;
  const double a = sqrt(P.gm1 * (H - 0.5 * q2));
  const double th = n[0] * u + n[1] * v + n[2] * w;
  const double b1 = P.gm1 / (a * a), b2 = 0.5 * b1 * q2;
  // step 2(b): left eigenvectors (rows) and right eigenvectors for the unit normal n: fields 0, 1, 2
  // (speed theta): l_k = n_k (1 - b2, b1 u, -b1) + ((m - rho u~) x n)_k; fields 3, 4: theta +- a
  const double Lm[5][5] = {
      {n[0] * (1.0 - b2) - (v * n[2] - w * n[1]), n[0] * b1 * u, n[0] * b1 * v + n[2], n[0] * b1 * w - n[1], -n[0] * b1},
      {n[1] * (1.0 - b2) - (w * n[0] - u * n[2]), n[1] * b1 * u - n[2], n[1] * b1 * v, n[1] * b1 * w + n[0], -n[1] * b1},
      {n[2] * (1.0 - b2) - (u * n[1] - v * n[0]), n[2] * b1 * u + n[1], n[2] * b1 * v - n[0], n[2] * b1 * w, -n[2] * b1},
      {0.5 * (b2 - th / a), 0.5 * (-b1 * u + n[0] / a), 0.5 * (-b1 * v + n[1] / a), 0.5 * (-b1 * w + n[2] / a), 0.5 * b1},
      {0.5 * (b2 + th / a), 0.5 * (-b1 * u - n[0] / a), 0.5 * (-b1 * v - n[1] / a), 0.5 * (-b1 * w - n[2] / a), 0.5 * b1}};
  const double Rm[5][5] = {   // Rm[k][c]: component c of r_k
      {n[0], u * n[0], v * n[0] + n[2], w * n[0] - n[1], 0.5 * q2 * n[0] + v * n[2] - w * n[1]},
      {n[1], u * n[1] - n[2], v * n[1], w * n[1] + n[0], 0.5 * q2 * n[1] + w * n[0] - u * n[2]},
      {n[2], u * n[2] + n[1], v * n[2] - n[0], w * n[2], 0.5 * q2 * n[2] + u * n[1] - v * n[0]},
      {1.0, u + a * n[0], v + a * n[1], w + a * n[2], H + a * th},
      {1.0, u - a * n[0], v - a * n[1], w - a * n[2], H - a * th}};
#pragma unroll
  for (int c = 0; c < 5; ++c) fhat[c] = 0.0;
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    const int lk = k < 3 ? 0 : (k == 3 ? 1 : 2);
    double alpha = 0.0;                                  // step 2(d): max over the stencil points (Q10)
#pragma unroll
    for (int m = 0; m < 8; ++m) alpha = fmax(alpha, lam[m][lk]);
    double gp[8], gm[8];
#pragma unroll
    for (int m = 0; m < 8; ++m) {                        // step 2(c), eq. (13)
      double V = 0.0, G = 0.0;
#pragma unroll
      for (int c = 0; c < 5; ++c) { V = fma(Lm[k][c], U[m][c], V); G = fma(Lm[k][c], F[m][c], G); }
      gp[m] = 0.5 * fma(alpha, V, G);
      gm[m] = 0.5 * fma(-alpha, V, G);
    }
    const double vp[7] = {gp[0], gp[1], gp[2], gp[3], gp[4], gp[5], gp[6]};
    const double vm[7] = {gm[7], gm[6], gm[5], gm[4], gm[3], gm[2], gm[1]};       // mirror image (Q4)
    const double gk = weno7z(vp, P.eps) + weno7z(vm, P.eps);                       // step 2(e)
#pragma unroll
    for (int c = 0; c < 5; ++c) fhat[c] = fma(gk, Rm[k][c], fhat[c]);              // step 2(f)
  }
}

template <int DIR, bool CURV>
__global__ void __launch_bounds__(128)
sweep7_kernel(const __grid_constant__ DevParams P, const double *__restrict__ Q, double *__restrict__ R, int accumulate) {
  const Layout &L = P.L;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= L.n[0]) return;
  const long long at = L.at(i, blockIdx.y, blockIdx.z), s = L.stride(DIR), sv = L.sv;
  double fr[5], fl[5];
  interface_flux7<DIR, CURV>(P, Q, at, s, fr);
  interface_flux7<DIR, CURV>(P, Q, at - s, s, fl);
  double sc = P.inv_delta[DIR];
  if constexpr (CURV) sc = 1.0 / __ldg(P.detJ + at);
#pragma unroll
  for (int c = 0; c < 5; ++c) {
    const double d = (fl[c] - fr[c]) * sc;                  // step 3, eq. (10)
    R[c * sv + at] = accumulate ? R[c * sv + at] + d : d;
  }
}

template <int DIR>
cudaError_t launch7(const DevParams &P, const double *Q, double *R, int accumulate, cudaStream_t st) {
  dim3 grid((P.L.n[0] + 127) / 128, P.L.n[1], P.L.n[2]);
  if (P.curvilinear) sweep7_kernel<DIR, true><<<grid, 128, 0, st>>>(P, Q, R, accumulate);
  else sweep7_kernel<DIR, false><<<grid, 128, 0, st>>>(P, Q, R, accumulate);
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_sweep7(const DevParams &P, int dir, const double *Q, double *R, int accumulate, cudaStream_t st) {
  if (dir == 0) return launch7<0>(P, Q, R, accumulate, st);
  if (dir == 1) return launch7<1>(P, Q, R, accumulate, st);
  return launch7<2>(P, Q, R, accumulate, st);
}

}  // namespace osbli
