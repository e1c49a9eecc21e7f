// osbli_weno7.cu -- 7th-order WENO-Z sweeps (scheme 6; "any arbitrary odd order", eq. (15)-(16), (20),
// (22); used at 7th order in PAPER.md:485-495 and 531-533; Q40): R (-)= (f^_{i+1/2} - f^_{i-1/2}) / Delta_d
// (or / detJ_i) with the characteristic flux reconstruction of PAPER.md:100-111 on the eight-point window i-3..i+4.
//
// A side scheme: a tiled kernel of its own (below), not the register-window march of the
// 5th/6th-order sweeps (an 8-point window of staged points does not fit the register file next to the rest); dense
// eigenvectors for a general unit normal (uniform grids: e_d), the stage update is the separate rk_update_kernel.  What
// it shares with the tuned path is the layout, the boundary fills and the viscous kernels; halo depth 4 (Layout::h).
#include "osbli_flux.cuh"
#include "osbli_kernels.h"

#include <type_traits>

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

// ---------------------------------------------------------------------------------------------
// Tiled kernel.  A block owns NS consecutive nodes of 32 (y, z sweeps: x-neighbouring) or 8 (x sweep) grid lines
// along the sweep direction.  (1) The NS + 8 stencil points of every line are staged once in shared memory as
// (U, p, theta = K.u, c = a |K| [, K]); (2) thread (f, line) computes the ONE interface flux between nodes s0-1+f and
// s0+f, f = 0..NS (PAPER.md:100-111 steps 2(a)-(f)), reading the staged points field by field, and leaves it in shared
// memory; (3) thread (f < NS, line) takes the difference (step 3, eq. (10)) for node s0+f.  Every point's
// thermodynamics is computed (NS+8)/NS times and every flux (NS+1)/NS times.
//   y, z sweeps: threadIdx.x = x lane (coalesced rows), threadIdx.y = f;  NS = 8 (6 on curvilinear grids: 3 more
//   staged doubles per point);   x sweep: threadIdx.x = f (32 interfaces, NS = 31 nodes), threadIdx.y = line of 8.
// W = 8: scheme 6 (WENO-Z7).  W = 6: the 5th/6th-order schemes through the same kernel (OSBLI_CURV_TILED, curvilinear grids).
template <int DIR, bool CURV, int W> struct Tile7 {
  static constexpr int H = W / 2;                                 // window point H-1 = node i, H = node i+1 of interface i+1/2
  static constexpr int NS = DIR == 0 ? 31 : (CURV ? (W == 8 ? 6 : 7) : 8);      // nodes per block along the sweep
  static constexpr int NF = NS + 1, NP = NS + W;                  // interfaces, staged points (s0-H .. s0+NS+H-1)
  static constexpr int NT = DIR == 0 ? 8 : 32;                    // lines per block
  static constexpr int NV = CURV ? 11 : 8;                        // staged doubles per point
  static constexpr int NTHREADS = NF * NT;
  // (p, t) -> index; the fastest index is the one consecutive lanes differ in (no bank conflicts)
  static __device__ __forceinline__ int at(int p, int t) { return DIR == 0 ? t * NP + p : p * NT + t; }
  static __device__ __forceinline__ int fat(int f, int t) { return DIR == 0 ? t * NF + f : f * NT + t; }
};

template <int DIR, bool CURV, int SCHEME>
__global__ void __launch_bounds__((Tile7<DIR, CURV, SCHEME == 6 ? 8 : 6>::NTHREADS), 2)
sweep7_kernel(const __grid_constant__ DevParams P, const double *__restrict__ Q, double *__restrict__ R, int accumulate) {
  constexpr int W = SCHEME == 6 ? 8 : 6;
  using T7 = Tile7<DIR, CURV, W>;
  constexpr int NS = T7::NS, NF = T7::NF, NP = T7::NP, NT = T7::NT, NV = T7::NV, HL = T7::H - 1, HR = T7::H;
  const RecPar rp = make_recpar(P);
  __shared__ double pts[NV][NP * NT];
  __shared__ double flx[5][NF * NT];
  const Layout &L = P.L;
  const long long sv = L.sv, st = L.stride(DIR);
  const int tid = threadIdx.y * blockDim.x + threadIdx.x;
  const int f = DIR == 0 ? threadIdx.x : threadIdx.y;             // interface between nodes s0-1+f and s0+f
  const int t = DIR == 0 ? threadIdx.y : threadIdx.x;             // line within the block
  const int n = L.n[DIR];
  int s0;
  // node 0 of line t (clamped to the last valid line: its results are computed and not stored)
  auto line_base = [&](int tt, bool &valid) -> long long {
    if constexpr (DIR == 0) {
      const int nl = L.n[1] * L.n[2];
      int line = blockIdx.y * NT + tt;
      valid = line < nl;
      line = min(line, nl - 1);
      return L.at(0, line % L.n[1], line / L.n[1]);
    } else {
      int i = blockIdx.x * NT + tt;
      valid = i < L.n[0];
      i = min(i, L.n[0] - 1);
      return DIR == 1 ? L.at(i, 0, blockIdx.y) : L.at(i, blockIdx.y, 0);
    }
  };
  if constexpr (DIR == 0) s0 = blockIdx.x * NS; else s0 = blockIdx.z * NS;

  // (1) stage the points
  for (int e = tid; e < NP * NT; e += T7::NTHREADS) {
    const int pp = DIR == 0 ? e % NP : e / NT, tt = DIR == 0 ? e / NP : e % NT;
    bool valid;
    const long long base = line_base(tt, valid);
    const int node = min(s0 - T7::H + pp, n + T7::H - 1);         // beyond n+H-1 nothing is read by a stored result
    const long long o = base + (long long)node * st;
    const double r = __ldg(Q + o), mx = __ldg(Q + sv + o), my = __ldg(Q + 2 * sv + o), mz = __ldg(Q + 3 * sv + o);
    const double E = __ldg(Q + 4 * sv + o);
    double K[3] = {DIR == 0 ? 1.0 : 0.0, DIR == 1 ? 1.0 : 0.0, DIR == 2 ? 1.0 : 0.0};
    if constexpr (CURV) {
      const double J = __ldg(P.detJ + o);
#pragma unroll
      for (int a = 0; a < 3; ++a) K[a] = J * __ldg(P.D[DIR][a] + o);
    }
    const double ir = 1.0 / r;
    const double u = mx * ir, v = my * ir, w = mz * ir;
    const double p = P.gm1 * (E - 0.5 * (mx * u + my * v + mz * w));
    const double a = sqrt(P.gamma * p * ir);
    const int ix = T7::at(pp, tt);
    pts[0][ix] = r; pts[1][ix] = mx; pts[2][ix] = my; pts[3][ix] = mz; pts[4][ix] = E; pts[5][ix] = p;
    pts[6][ix] = K[0] * u + K[1] * v + K[2] * w;
    pts[7][ix] = CURV ? a * sqrt(K[0] * K[0] + K[1] * K[1] + K[2] * K[2]) : a;
    if constexpr (CURV) { pts[8][ix] = K[0]; pts[9][ix] = K[1]; pts[10][ix] = K[2]; }
  }
  __syncthreads();

  // (2) one interface flux per thread: window point m = staged point f + m (m = HL, HR: nodes s0-1+f, s0+f)
  {
    // read through a volatile pointer: the staged values are fetched again for every field instead of being kept in
    // registers across the five fields (the cached form needs more than 255 registers and spills)
    const volatile double *vp_ = &pts[0][0];
    auto S = [&](int v, int m) { return vp_[v * (NP * NT) + T7::at(f + m, t)]; };
    // step 2(a): Roe (or simple) average of the two nodes next to the interface; interface normal from the averaged K
    double nrm[3] = {DIR == 0 ? 1.0 : 0.0, DIR == 1 ? 1.0 : 0.0, DIR == 2 ? 1.0 : 0.0};
    if constexpr (CURV) {
      const double kx = 0.5 * (S(8, HL) + S(8, HR)), ky = 0.5 * (S(9, HL) + S(9, HR)), kz = 0.5 * (S(10, HL) + S(10, HR));
      const double ik = 1.0 / sqrt(kx * kx + ky * ky + kz * kz);
      nrm[0] = kx * ik; nrm[1] = ky * ik; nrm[2] = kz * ik;
    }
    double u, v, w, H;
    {
      const double rL = S(0, HL), rR = S(0, HR);
      if (P.averaging != 0) {            // U_{i+1/2} = (U_i + U_{i+1})/2
        const double r = 0.5 * (rL + rR), ir = 1.0 / r;
        u = 0.5 * (S(1, HL) + S(1, HR)) * ir; v = 0.5 * (S(2, HL) + S(2, HR)) * ir; w = 0.5 * (S(3, HL) + S(3, HR)) * ir;
        const double E = 0.5 * (S(4, HL) + S(4, HR));
        const double p = P.gm1 * (E - 0.5 * r * (u * u + v * v + w * w));
        H = (E + p) * ir;
      } else {
        const double sl = sqrt(rL), sr = sqrt(rR), is = 1.0 / (sl + sr);
        u = (S(1, HL) / sl + S(1, HR) / sr) * is; v = (S(2, HL) / sl + S(2, HR) / sr) * is; w = (S(3, HL) / sl + S(3, HR) / sr) * is;
        H = ((S(4, HL) + S(5, HL)) / sl + (S(4, HR) + S(5, HR)) / sr) * is;
      }
    }
    const double q2 = u * u + v * v + w * w;
    const double a = sqrt(P.gm1 * (H - 0.5 * q2));
    const double th = nrm[0] * u + nrm[1] * v + nrm[2] * w;
    const double b1 = P.gm1 / (a * a), b2 = 0.5 * b1 * q2, ia = 1.0 / a;
    const double ut[3] = {u, v, w};
    // step 2(d): alpha = max over the eight stencil points of |theta|, |theta + c|, |theta - c| (Q10)
    double al0 = 0.0, alp = 0.0, alm = 0.0;
#pragma unroll
    for (int m = 0; m < W; ++m) {
      const double thm = S(6, m), cm = S(7, m);
      al0 = fmax(al0, fabs(thm)); alp = fmax(alp, fabs(thm + cm)); alm = fmax(alm, fabs(thm - cm));
    }
    double fh[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      // step 2(b): row k of L and column k of R for the unit normal nrm (fields 0-2: speed theta; 3, 4: theta +- a)
      double l[5], rc[5], alpha;
      if (k < 3) {
        constexpr int I1[3] = {1, 2, 0}, I2[3] = {2, 0, 1};
        const int i1 = I1[k], i2 = I2[k];
        // l_k = n_k (1 - b2, b1 u, -b1) + e_k x n acting on (m - rho u~);  r_k = (n_k, u n_k + (n x e_k), q2/2 n_k + (u x n)_k)
        l[0] = nrm[k] * (1.0 - b2) - (ut[i1] * nrm[i2] - ut[i2] * nrm[i1]);
        l[1 + k] = nrm[k] * b1 * ut[k];
        l[1 + i1] = nrm[k] * b1 * ut[i1] + nrm[i2];
        l[1 + i2] = nrm[k] * b1 * ut[i2] - nrm[i1];
        l[4] = -nrm[k] * b1;
        rc[0] = nrm[k];
        rc[1 + k] = ut[k] * nrm[k];
        rc[1 + i1] = ut[i1] * nrm[k] + nrm[i2];
        rc[1 + i2] = ut[i2] * nrm[k] - nrm[i1];
        rc[4] = 0.5 * q2 * nrm[k] + ut[i1] * nrm[i2] - ut[i2] * nrm[i1];
        alpha = al0;
      } else {
        const double sg = k == 3 ? 1.0 : -1.0;
        l[0] = 0.5 * (b2 - sg * th * ia);
#pragma unroll
        for (int c = 0; c < 3; ++c) { l[1 + c] = 0.5 * (-b1 * ut[c] + sg * nrm[c] * ia); rc[1 + c] = ut[c] + sg * a * nrm[c]; }
        l[4] = 0.5 * b1;
        rc[0] = 1.0;
        rc[4] = H + sg * a * th;
        alpha = k == 3 ? alp : alm;
      }
      // step 2(c), eq. (13): g+- = (l.F +- alpha l.U)/2 with F = theta U + p (0, K, theta)
      double gp[W], gm[W];
#pragma unroll
      for (int m = 0; m < W; ++m) {
        const double V = fma(l[0], S(0, m), fma(l[1], S(1, m), fma(l[2], S(2, m), fma(l[3], S(3, m), l[4] * S(4, m)))));
        const double thm = S(6, m);
        double lk;
        if constexpr (CURV) lk = fma(l[1], S(8, m), fma(l[2], S(9, m), fma(l[3], S(10, m), l[4] * thm)));
        else lk = fma(l[4], thm, l[1 + DIR]);
        const double G = fma(thm, V, S(5, m) * lk);
        gp[m] = fma(alpha, V, G);                            // twice the split fluxes
        gm[m] = fma(-alpha, V, G);
      }
      double gk;                                             // twice (g^+ + g^-), step 2(e)
      if constexpr (W == 8) {
        const double vp[7] = {0.5 * gp[0], 0.5 * gp[1], 0.5 * gp[2], 0.5 * gp[3], 0.5 * gp[4], 0.5 * gp[5], 0.5 * gp[6]};
        const double vm[7] = {0.5 * gm[7], 0.5 * gm[6], 0.5 * gm[5], 0.5 * gm[4], 0.5 * gm[3], 0.5 * gm[2], 0.5 * gm[1]};   // mirror image (Q4)
        gk = 2.0 * (weno7z(vp, P.eps) + weno7z(vm, P.eps));
      } else {
        gk = reconstruct_pair<SCHEME>(gp, gm, rp);           // osbli_flux.cuh: data and result carry the factor 2
      }
#pragma unroll
      for (int c = 0; c < 5; ++c) fh[c] = fma(gk, rc[c], fh[c]);                    // step 2(f)
    }
    const int fx = T7::fat(f, t);
#pragma unroll
    for (int c = 0; c < 5; ++c) flx[c][fx] = 0.5 * fh[c];          // the 1/2 of eq. (13)
  }
  __syncthreads();

  // (3) flux difference of node s0 + f, eq. (10)
  bool valid;
  const long long base = line_base(t, valid);
  const int node = s0 + f;
  if (valid && f < NS && node < n) {
    const long long o = base + (long long)node * st;
    double sc = P.inv_delta[DIR];
    if constexpr (CURV) sc = 1.0 / __ldg(P.detJ + o);
    const int f0 = T7::fat(f, t), f1 = T7::fat(f + 1, t);
#pragma unroll
    for (int c = 0; c < 5; ++c) {
      const double d = (flx[c][f0] - flx[c][f1]) * sc;
      R[c * sv + o] = accumulate ? R[c * sv + o] + d : d;
    }
  }
}

template <int DIR, int SCHEME>
cudaError_t launch7(const DevParams &P, const double *Q, double *R, int accumulate, cudaStream_t st) {
  const Layout &L = P.L;
  auto go = [&](auto curv) {
    constexpr bool CURV = decltype(curv)::value;
    using T7 = Tile7<DIR, CURV, SCHEME == 6 ? 8 : 6>;
    dim3 block, grid;
    if constexpr (DIR == 0) {
      block = dim3(T7::NF, T7::NT);
      grid = dim3((L.n[0] + T7::NS - 1) / T7::NS, (L.n[1] * L.n[2] + T7::NT - 1) / T7::NT, 1);
    } else {
      block = dim3(T7::NT, T7::NF);
      grid = dim3((L.n[0] + T7::NT - 1) / T7::NT, DIR == 1 ? L.n[2] : L.n[1], (L.n[DIR] + T7::NS - 1) / T7::NS);
    }
    sweep7_kernel<DIR, CURV, SCHEME><<<grid, block, 0, st>>>(P, Q, R, accumulate);
  };
  if constexpr (SCHEME == 6) {
    if (P.curvilinear) go(std::true_type{}); else go(std::false_type{});
  } else {
    go(std::true_type{});                                    // the 5th/6th-order schemes come here on curvilinear grids only
  }
  return cudaGetLastError();
}

template <int SCHEME>
cudaError_t launch7_dir(const DevParams &P, int dir, const double *Q, double *R, int accumulate, cudaStream_t st) {
  if (dir == 0) return launch7<0, SCHEME>(P, Q, R, accumulate, st);
  if (dir == 1) return launch7<1, SCHEME>(P, Q, R, accumulate, st);
  return launch7<2, SCHEME>(P, Q, R, accumulate, st);
}

}  // namespace

cudaError_t launch_sweep7(const DevParams &P, int dir, const double *Q, double *R, int accumulate, cudaStream_t st) {
  return launch7_dir<6>(P, dir, Q, R, accumulate, st);
}

// The 5th/6th-order schemes on curvilinear grids through the tiled kernel (one flux per thread, points in shared
// memory, no fused stage update): scheme 0 WENO-Z5, 1 TENO5, 2 TENO6, 3 WENO-JS5, 5 WENO-Z3.
cudaError_t launch_sweep_tiled(const DevParams &P, int dir, const double *Q, double *R, int accumulate, cudaStream_t st) {
  if (!P.curvilinear) return cudaErrorInvalidValue;
  switch (P.scheme) {
    case 0: return launch7_dir<0>(P, dir, Q, R, accumulate, st);
    case 1: return launch7_dir<1>(P, dir, Q, R, accumulate, st);
    case 2: return launch7_dir<2>(P, dir, Q, R, accumulate, st);
    case 3: return launch7_dir<3>(P, dir, Q, R, accumulate, st);
    case 5: return launch7_dir<5>(P, dir, Q, R, accumulate, st);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace osbli
