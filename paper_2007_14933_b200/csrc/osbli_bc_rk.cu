// osbli_bc_rk.cu -- halo / boundary-plane fill (eq. (40)-(46); 503; 586) and the
// low-storage RK3 stage update (eq. (36)-(37)).
#include "osbli_kernels.h"

namespace osbli {

// One thread per grid line along DIR (transverse range: directions below DIR over their
// halo-extended range, directions above over the interior -- they are filled afterwards), both
// sides.  For DIR = 1, 2 consecutive threads are consecutive x, so accesses are coalesced.
template <int DIR>
__global__ void __launch_bounds__(128)
bc_kernel(const __grid_constant__ DevParams P, double *__restrict__ Q) {
  const Layout &L = P.L;
  constexpr int E1 = (DIR == 0) ? 1 : 0;         // fastest transverse direction
  constexpr int E2 = (DIR == 2) ? 1 : 2;         // slowest transverse direction
  const int lo1 = (E1 < DIR) ? -L.h[E1] : 0, n1 = (E1 < DIR) ? L.n[E1] + 2 * L.h[E1] : L.n[E1];
  const int lo2 = (E2 < DIR) ? -L.h[E2] : 0, n2 = (E2 < DIR) ? L.n[E2] + 2 * L.h[E2] : L.n[E2];
  const int t1 = blockIdx.x * blockDim.x + threadIdx.x;
  const int t2 = blockIdx.y;
  if (t1 >= n1 || t2 >= n2) return;
  int ijk[3];
  ijk[DIR] = 0; ijk[E1] = lo1 + t1; ijk[E2] = lo2 + t2;
  const long long base = L.at(ijk[0], ijk[1], ijk[2]);     // node 0 of this line
  const long long s = L.stride(DIR);
  const long long sv = L.sv;
  const int n = L.n[DIR];
  const int hd = L.h[DIR];                         // halo depth: 3, or 4 for the 7th-order scheme

#pragma unroll
  for (int side = 0; side < 2; ++side) {
    const int type = P.bc[DIR][side];
    const long long wall = base + (side == 0 ? 0 : (long long)(n - 1) * s);   // boundary node
    const long long inw = side == 0 ? s : -s;                                   // one node into the domain
    if (type == 0) {                   // periodic wrap
      for (int m = 1; m <= hd; ++m)
        for (int c = 0; c < 5; ++c) {
          double *q = Q + c * sv;
          if (side == 0) q[base - m * s] = q[base + (long long)(n - m) * s];
          else           q[base + (long long)(n - 1 + m) * s] = q[base + (long long)(m - 1) * s];
        }
    } else if (type == 1) {            // zero-order extrapolation
      for (int c = 0; c < 5; ++c) {
        const double v = Q[c * sv + wall];
        for (int m = 1; m <= hd; ++m) Q[c * sv + wall - m * inw] = v;
      }
    } else if (type == 2) {            // Dirichlet: boundary plane and halos from the frozen state
      for (int m = 0; m <= hd; ++m)
        for (int c = 0; c < 5; ++c) Q[c * sv + wall - m * inw] = __ldg(P.dirichlet + c * sv + wall - m * inw);
    } else {                           // no-slip wall, eq. (40)-(46): isothermal (3) or adiabatic (4)
      auto temperature = [&](long long a) {
        const double r = Q[a], mx = Q[sv + a], my = Q[2 * sv + a], mz = Q[3 * sv + a], E = Q[4 * sv + a];
        const double u = mx / r, v = my / r, w = mz / r;
        return P.gM2 * (P.gm1 * (E - 0.5 * r * (u * u + v * v + w * w))) / r;
      };
      double Tw = P.wall_T[DIR][side];
      if (type == 4)                   // one-sided 4th-order dT/dn = 0 solved for T_w
        Tw = (48.0 * temperature(wall + inw) - 36.0 * temperature(wall + 2 * inw) + 16.0 * temperature(wall + 3 * inw) -
              3.0 * temperature(wall + 4 * inw)) / 25.0;
      const double rw = Q[wall];                             // rho_w floats (continuity)
      Q[sv + wall] = 0.0; Q[2 * sv + wall] = 0.0; Q[3 * sv + wall] = 0.0;   // eq. (40)
      const double Ew = rw * Tw / (P.gM2 * P.gm1);           // eq. (41)
      Q[4 * sv + wall] = Ew;
      const double pw = P.gm1 * Ew;
      double T1;
      {
        const long long a = wall + inw;
        const double r = Q[a], mx = Q[sv + a], my = Q[2 * sv + a], mz = Q[3 * sv + a], E = Q[4 * sv + a];
        const double u = mx / r, v = my / r, w = mz / r;
        const double p = P.gm1 * (E - 0.5 * r * (u * u + v * v + w * w));
        T1 = P.gM2 * p / r;
      }
      for (int m = 1; m <= hd; ++m) {
        const double Tm = (m + 1) * Tw - m * T1;             // eq. (42)
        const double rm = P.gM2 * pw / Tm;                   // eq. (43)
        const long long a = wall + m * inw, g = wall - m * inw;
        const double r = Q[a];
        const double u = Q[sv + a] / r, v = Q[2 * sv + a] / r, w = Q[3 * sv + a] / r;
        Q[g] = rm;
        Q[sv + g] = -rm * u;                                 // eq. (44)-(46): reflected velocity
        Q[2 * sv + g] = -rm * v;
        Q[3 * sv + g] = -rm * w;
        Q[4 * sv + g] = pw / P.gm1 + 0.5 * rm * (u * u + v * v + w * w);
      }
    }
  }
}

// Constant body force per unit volume (the laminar channel of PAPER.md:535-546; Q34).
__global__ void __launch_bounds__(128)
force_kernel(const __grid_constant__ DevParams P, const double *__restrict__ Q, double *__restrict__ R) {
  const Layout &L = P.L;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= L.n[0]) return;
  const long long at = L.at(i, blockIdx.y, blockIdx.z), sv = L.sv;
  const double ir = 1.0 / Q[at];
  double work = 0.0;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    R[(1 + a) * sv + at] += P.force[a];
    work += Q[(1 + a) * sv + at] * ir * P.force[a];
  }
  R[4 * sv + at] += work;
}

cudaError_t launch_force(const DevParams &P, const double *Q, double *R, cudaStream_t st) {
  dim3 grid((P.L.n[0] + 127) / 128, P.L.n[1], P.L.n[2]);
  force_kernel<<<grid, 128, 0, st>>>(P, Q, R);
  return cudaGetLastError();
}

cudaError_t launch_bc(const DevParams &P, int dir, double *Q, cudaStream_t st) {
  const Layout &L = P.L;
  if (L.n[dir] <= 1) return cudaSuccess;
  auto ext = [&](int e) { return (e < dir) ? L.n[e] + 2 * L.h[e] : L.n[e]; };
  if (dir == 0) {
    dim3 grid((ext(1) + 127) / 128, ext(2));
    bc_kernel<0><<<grid, 128, 0, st>>>(P, Q);
  } else if (dir == 1) {
    dim3 grid((ext(0) + 127) / 128, ext(2));
    bc_kernel<1><<<grid, 128, 0, st>>>(P, Q);
  } else {
    dim3 grid((ext(0) + 127) / 128, ext(1));
    bc_kernel<2><<<grid, 128, 0, st>>>(P, Q);
  }
  return cudaGetLastError();
}

// eq. (36)-(37) with the 3-stage coefficients of ref. [23] (Williamson's 2N-storage scheme,
// DESIGN.md Q15): A = (0, -5/9, -153/128), B = (1/3, 15/16, 8/15).
// One thread per pair of x-adjacent interior nodes: 128-bit loads/stores (rows are 128-byte
// aligned and x_offset is even), scalar tail for odd nx.
template <bool FIRST>
__global__ void __launch_bounds__(128)
rk_update_kernel(const __grid_constant__ DevParams P, double A, double B, double dt, double *__restrict__ Q,
                 double *__restrict__ Qtmp, const double *__restrict__ R) {
  const Layout &L = P.L;
  const int i = 2 * (blockIdx.x * blockDim.x + threadIdx.x);
  if (i >= L.n[0]) return;
  const long long at = L.at(i, blockIdx.y, blockIdx.z);
  if (i + 1 < L.n[0]) {
#pragma unroll
    for (int c = 0; c < 5; ++c) {
      const long long o = c * L.sv + at;
      const double2 r = *reinterpret_cast<const double2 *>(R + o);
      double2 d, q = *reinterpret_cast<double2 *>(Q + o);
      if constexpr (FIRST) { d.x = dt * r.x; d.y = dt * r.y; }      // A_0 = 0: dU^(0) is never read
      else {
        d = *reinterpret_cast<double2 *>(Qtmp + o);
        d.x = fma(A, d.x, dt * r.x); d.y = fma(A, d.y, dt * r.y);
      }
      q.x = fma(B, d.x, q.x); q.y = fma(B, d.y, q.y);
      *reinterpret_cast<double2 *>(Qtmp + o) = d;
      *reinterpret_cast<double2 *>(Q + o) = q;
    }
  } else {
#pragma unroll
    for (int c = 0; c < 5; ++c) {
      const long long o = c * L.sv + at;
      double d = dt * R[o];
      if constexpr (!FIRST) d = fma(A, Qtmp[o], d);
      Qtmp[o] = d;
      Q[o] = fma(B, d, Q[o]);
    }
  }
}

// Coefficients of eq. (36)-(37) "from [23]": nstages = 3 -> Williamson's 2N-storage RK3
// (Q15); nstages = 5 -> Carpenter & Kennedy's five-stage 4th-order 2N-storage scheme (Q35).
// form = 1 (nstages = 3 only): the strong-stability-preserving 2N-storage set of ref. [44] (
// DESIGN.md Q39), as published (B_1 to six digits); its A_3 is 0, so the last stage does not read dU.
void rk_coefficients(int nstages, int form, int stage, double *A, double *B) {
  static const double as3[3] = {0.0, -2.915493957701923, 0.0};
  static const double bs3[3] = {0.924574, 0.287713063186749, 0.626538109512740};
  if (nstages == 3 && form == 1) { *A = as3[stage]; *B = bs3[stage]; return; }
  static const double a3[3] = {0.0, -5.0 / 9.0, -153.0 / 128.0};
  static const double b3[3] = {1.0 / 3.0, 15.0 / 16.0, 8.0 / 15.0};
  static const double a5[5] = {0.0, -567301805773.0 / 1357537059087.0, -2404267990393.0 / 2016746695238.0,
                               -3550918686646.0 / 2091501179385.0, -1275806237668.0 / 842570457699.0};
  static const double b5[5] = {1432997174477.0 / 9575080441755.0, 5161836677717.0 / 13612068292357.0,
                               1720146321549.0 / 2090206949498.0, 3134564353537.0 / 4481467310338.0,
                               2277821191437.0 / 14882151754819.0};
  *A = nstages == 5 ? a5[stage] : a3[stage];
  *B = nstages == 5 ? b5[stage] : b3[stage];
}

cudaError_t launch_rk_update(const DevParams &P, int nstages, int stage, double dt, double *Q, double *Qtmp,
                             const double *R, cudaStream_t st) {
  double A, B;
  rk_coefficients(nstages, P.rk3_form, stage, &A, &B);
  const Layout &L = P.L;
  const int pairs = (L.n[0] + 1) / 2;
  dim3 grid((pairs + 127) / 128, L.n[1], L.n[2]);
  if (A == 0.0) rk_update_kernel<true><<<grid, 128, 0, st>>>(P, A, B, dt, Q, Qtmp, R);
  else rk_update_kernel<false><<<grid, 128, 0, st>>>(P, A, B, dt, Q, Qtmp, R);
  return cudaGetLastError();
}

}  // namespace osbli
