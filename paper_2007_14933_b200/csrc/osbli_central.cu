// osbli_central.cu -- the central ("StoreSome") path for smooth problems in ONE kernel per Runge-Kutta stage
// ("Central schemes are also applied to smooth problems that do not require
// shock-capturing", 625-637: the paper's low-memory algorithm recomputes derivatives instead of storing them;
// here nothing but Q and dU touches HBM):
//
//     R  = - sum_d delta_d F_d  (eq. (28) on the point-wise flux vectors, Q36)
//          + d_j tau_ij, d_j(u_i tau_ij) - d_j q_j  (eq. (2)-(5), 4th-order central, mu = 1)
//     dU = A dU + dt R,   Qout = Q + B dU            (eq. (36)-(37))
//
// for uniform grids with three active periodic directions (the Taylor-Green cases).  Algorithmic traffic: Q in,
// dU in (not in the first stage), dU out, Qout out = 160 (120) bytes per point and stage.
//
// Structure: the 2.5-D marching of the fast viscous kernel (osbli_visc.cu) -- a block owns a 32 x 8 (x,y) tile and
// walks along z; raw plane tiles arrive by TMA; every in-plane stencil is read once when its plane enters, two
// steps before the plane is completed from registers.  Staged per point: u, v, w, T, rho, G = rho E + p.
// The convective fluxes of the eight in-plane neighbours are rebuilt from those (F_x = u (rho, rho u, rho v,
// rho w, G) + p e_x with p = rho T / (gamma M^2)), the four z-neighbours from register windows.  In-plane parts of
// the five residuals wait in 3-deep delay lines / the energy scatter accumulators; Q and dU of the node travel by
// cp.async into per-thread slots one plane ahead.  The periodic images of boundary-near nodes are written too, so
// that no halo fill is needed between stages (as in the fused sweeps).
#include "osbli_kernels.h"
#include "osbli_tma.cuh"

#include <type_traits>

namespace osbli {

#ifndef OSBLI_CCHUNK
#define OSBLI_CCHUNK 64
#endif
#ifndef OSBLI_CY
#define OSBLI_CY 8
#endif
constexpr int kCY = OSBLI_CY, kCPY = kCY + 2 * kVH;              // tile rows of this kernel: 32 x kCY nodes, 36 x (kCY + 4) staged
constexpr unsigned kCTileBytes = 5 * kCPY * kVPX * sizeof(double);

struct CSmem {
  double tile[3][5][kCPY][kVPX];       // TMA destinations (128-byte aligned: first member), fetched two planes ahead
  double f[2][6][kCPY][kVPX];          // u, v, w, T, rho, G: the plane being staged and the plane entering
  double g[2][2][kCY][kVPX];           // d_y u, d_y v of the tile rows incl. the x halo, double buffered
  double q[2][10][kVX * kCY];          // per-thread slots: Q (0-4) and dU (5-9) of the two nodes in flight
  unsigned long long mbar[3];
};

template <bool FIRST>
__global__ void __launch_bounds__(kVX * kCY, 1)
central_fused_kernel(const __grid_constant__ DevParams P, const double *__restrict__ Q, int chunk,
                     const __grid_constant__ CUtensorMap tmap, const RkArgs rk) {
  extern __shared__ __align__(128) unsigned char cs_raw[];
  CSmem &S = *reinterpret_cast<CSmem *>(cs_raw);
  const Layout &L = P.L;
  const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * kVX + tx;
  const int x0 = blockIdx.x * kVX, y0 = blockIdx.y * kCY;
  const int z0 = blockIdx.z * chunk, z1 = min(z0 + chunk, L.n[2]);
  const int i = x0 + tx, j = y0 + ty;
  const bool inside = i < L.n[0] && j < L.n[1];
  const long long sv = L.sv;

  constexpr int NPT = kVPX * kCPY;                                // 432 tile points, up to two per thread
  int pi[2], pj[2];
  bool pv[2];
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    const int t = tid + s * (kVX * kCY);
    pv[s] = t < NPT;
    const int yy = pv[s] ? t / kVPX : 0, xx = pv[s] ? t % kVPX : 0;
    pi[s] = xx; pj[s] = yy;
    pv[s] = pv[s] && (x0 + xx - kVH) < L.n[0] + kVH && (y0 + yy - kVH) < L.n[1] + kVH;
  }
  auto fetch = [&](int plane) {
    if (tid == 0) {
      const int b = (plane - (z0 - 2)) % 3;
      mbar_expect_tx(&S.mbar[b], kCTileBytes);
      tma_load_4d(&S.tile[b][0][0][0], &tmap, (int)L.xoff + x0 - kVH, L.h[1] + y0 - kVH, L.h[2] + plane, 0, &S.mbar[b]);
    }
  };
  auto stage = [&](int plane) {
    const int slot = (plane + 8) & 1;
    const int jj = plane - (z0 - 2), b = jj % 3;               // the mbarrier of buffer b has completed jj / 3 phases before
    mbar_wait(&S.mbar[b], (unsigned)(jj / 3) & 1u);
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
        S.f[slot][4][pj[s]][pi[s]] = q0;
        S.f[slot][5][pj[s]][pi[s]] = q4 + p;
      }
  };
  if (tid == 0) {
    mbar_init(&S.mbar[0], 1);
    mbar_init(&S.mbar[1], 1);
    mbar_init(&S.mbar[2], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  const double cx = P.inv12d[0], cy = P.inv12d[1], cz = P.inv12d[2];
  const double cxx = P.inv12d2[0], cyy = P.inv12d2[1], czz = P.inv12d2[2];
  const double cp = 1.0 / P.gM2;                                  // p = rho T / (gamma M^2)
  auto d1 = [](double m2, double m1, double p1, double p2, double c) { return c * ((m2 - p2) + 8.0 * (p1 - m1)); };
  auto d2 = [](double m2, double m1, double f0, double p1, double p2, double c) {
    return c * fma(-30.0, f0, fma(16.0, m1 + p1, -(m2 + p2)));
  };
  constexpr double third = 1.0 / 3.0, four3 = 4.0 / 3.0;

  // periodic images of this thread's column (bits 0/1: x below 3 / above nx-4; bits 2/3: the same for y)
  const int wrap_mask = (i < kHalo ? 1 : 0) | (i >= L.n[0] - kHalo ? 2 : 0) | (j < kHalo ? 4 : 0) | (j >= L.n[1] - kHalo ? 8 : 0);

  // register state of this thread's column; after the shift of step k: windows = planes k-2..k+2, delay lines =
  // planes k..k+2, energy accumulators = planes k..k+4
  double uw[5], vw[5], ww[5], rw[5], Gw[5], pw[5], s0w[5], s1w[5], s2w[5];
  double B0[3], B1[3], B2[3], B3[3];   // in-plane parts of the residuals of rho, rho u, rho v, rho w
  double aE[5];                        // everything of the energy residual that is linear in one plane or lives in it
#pragma unroll
  for (int m = 0; m < 5; ++m) uw[m] = vw[m] = ww[m] = rw[m] = Gw[m] = pw[m] = s0w[m] = s1w[m] = s2w[m] = aE[m] = 0.0;
#pragma unroll
  for (int m = 0; m < 3; ++m) B0[m] = B1[m] = B2[m] = B3[m] = 0.0;

  fetch(z0 - 2);
  stage(z0 - 2);
  fetch(z0 - 1);
  fetch(z0);
  __syncthreads();
  const int X = tx + kVH, Y = ty + kVH;
  const int hr = tid >> 2, hc = (tid & 3) < 2 ? (tid & 3) : kVX + (tid & 3);

  // flux vector along direction D (0: x, 1: y, 2: z) of a point given by its staged values
  auto flux = [&](auto dtag, double r_, double u_, double v_, double w_, double p_, double G_, double (&f)[5]) {
    constexpr int D = decltype(dtag)::value;
    const double th = D == 0 ? u_ : (D == 1 ? v_ : w_);
    const double rt = r_ * th;
    f[0] = rt;
    f[1] = D == 0 ? fma(rt, u_, p_) : rt * u_;
    f[2] = D == 1 ? fma(rt, v_, p_) : rt * v_;
    f[3] = D == 2 ? fma(rt, w_, p_) : rt * w_;
    f[4] = G_ * th;
  };
  // first difference eq. (28) of the flux vectors of the four neighbours (order -2, -1, +1, +2), added to acc
  auto dflux = [&](auto dtag, const double (&r4)[4], const double (&u4)[4], const double (&v4)[4], const double (&w4)[4],
                   const double (&p4)[4], const double (&G4)[4], double c, double (&acc)[5]) {
    double fm2[5], fm1[5], fp1[5], fp2[5];
    flux(dtag, r4[0], u4[0], v4[0], w4[0], p4[0], G4[0], fm2);
    flux(dtag, r4[1], u4[1], v4[1], w4[1], p4[1], G4[1], fm1);
    flux(dtag, r4[2], u4[2], v4[2], w4[2], p4[2], G4[2], fp1);
    flux(dtag, r4[3], u4[3], v4[3], w4[3], p4[3], G4[3], fp2);
#pragma unroll
    for (int q = 0; q < 5; ++q) acc[q] = fma(c, (fm2[q] - fp2[q]) + 8.0 * (fp1[q] - fm1[q]), acc[q]);
  };

  for (int k = z0 - 4; k < z1; ++k) {
    if (k > z0 - 4) __syncthreads();
    if (k + 3 < z1 + 2) stage(k + 3);
    // Q and dU of node k+1 go to per-thread shared-memory slots by cp.async, one whole step before they are needed
    if (k + 1 >= z0 && k + 1 < z1 && inside) {
      const long long a1 = L.at(i, j, k + 1);
#pragma unroll
      for (int c = 0; c < 5; ++c) cp_async8(&S.q[(k + 1) & 1][c][tid], Q + c * sv + a1);
      if constexpr (!FIRST) {
#pragma unroll
        for (int c = 0; c < 5; ++c) cp_async8(&S.q[(k + 1) & 1][5 + c][tid], rk.Qtmp + c * sv + a1);
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
    if (k + 5 < z1 + 2) fetch(k + 5);                          // raw plane k+5 into the buffer plane k+2 has left
#pragma unroll
    for (int m = 0; m < 4; ++m) {
      uw[m] = uw[m + 1]; vw[m] = vw[m + 1]; ww[m] = ww[m + 1]; rw[m] = rw[m + 1]; Gw[m] = Gw[m + 1]; pw[m] = pw[m + 1];
      s0w[m] = s0w[m + 1]; s1w[m] = s1w[m + 1]; s2w[m] = s2w[m + 1]; aE[m] = aE[m + 1];
    }
    aE[4] = 0.0;
    B0[0] = B0[1]; B0[1] = B0[2]; B1[0] = B1[1]; B1[1] = B1[2]; B2[0] = B2[1]; B2[1] = B2[2]; B3[0] = B3[1]; B3[1] = B3[2];

    // ---- plane k+2 enters.  The two planes either side of the chunk only feed z-stencils (FULL = false).
    auto enter = [&](auto full_tag) {
      constexpr bool FULL = decltype(full_tag)::value;
      const int e = (k + 2 + 8) & 1;
      const double (*F)[kCPY][kVPX] = S.f[e];
      const double u = F[0][Y][X], v = F[1][Y][X], w = F[2][Y][X], T = F[3][Y][X], r = F[4][Y][X], G = F[5][Y][X];
      const double ux[4] = {F[0][Y][X - 2], F[0][Y][X - 1], F[0][Y][X + 1], F[0][Y][X + 2]};
      const double vy[4] = {F[1][Y - 2][X], F[1][Y - 1][X], F[1][Y + 1][X], F[1][Y + 2][X]};
      const double wx[4] = {F[2][Y][X - 2], F[2][Y][X - 1], F[2][Y][X + 1], F[2][Y][X + 2]};
      const double wy[4] = {F[2][Y - 2][X], F[2][Y - 1][X], F[2][Y + 1][X], F[2][Y + 2][X]};
      const double u_x = d1(ux[0], ux[1], ux[2], ux[3], cx), v_y = d1(vy[0], vy[1], vy[2], vy[3], cy);
      uw[4] = u; vw[4] = v; ww[4] = w; rw[4] = r; Gw[4] = G; pw[4] = cp * r * T;
      s0w[4] = d1(wx[0], wx[1], wx[2], wx[3], cx);
      s1w[4] = d1(wy[0], wy[1], wy[2], wy[3], cy);
      s2w[4] = u_x + v_y;
      const double tz = (P.cq * czz) * T;                       // z-stencil of T scattered to the five planes it feeds
      aE[0] -= tz; aE[1] = fma(16.0, tz, aE[1]); aE[2] = fma(-30.0, tz, aE[2]); aE[3] = fma(16.0, tz, aE[3]); aE[4] -= tz;
      if constexpr (FULL) {
        const double uy[4] = {F[0][Y - 2][X], F[0][Y - 1][X], F[0][Y + 1][X], F[0][Y + 2][X]};
        const double vx[4] = {F[1][Y][X - 2], F[1][Y][X - 1], F[1][Y][X + 1], F[1][Y][X + 2]};
        const double Tx[4] = {F[3][Y][X - 2], F[3][Y][X - 1], F[3][Y][X + 1], F[3][Y][X + 2]};
        const double Ty[4] = {F[3][Y - 2][X], F[3][Y - 1][X], F[3][Y + 1][X], F[3][Y + 2][X]};
        const double u_y = d1(uy[0], uy[1], uy[2], uy[3], cy), v_x = d1(vx[0], vx[1], vx[2], vx[3], cx);
        S.g[e][0][ty][X] = u_y;
        S.g[e][1][ty][X] = v_y;
        // viscous in-plane parts (as in viscous_tgv_kernel), already divided by Re
        const double Au = P.inv_Re * fma(four3, d2(ux[0], ux[1], u, ux[2], ux[3], cxx), d2(uy[0], uy[1], u, uy[2], uy[3], cyy));
        const double Av = P.inv_Re * fma(four3, d2(vy[0], vy[1], v, vy[2], vy[3], cyy), d2(vx[0], vx[1], v, vx[2], vx[3], cxx));
        const double Aw = P.inv_Re * (d2(wx[0], wx[1], w, wx[2], wx[3], cxx) + d2(wy[0], wy[1], w, wy[2], wy[3], cyy));
        const double lapT = d2(Tx[0], Tx[1], T, Tx[2], Tx[3], cxx) + d2(Ty[0], Ty[1], T, Ty[2], Ty[3], cyy);
        const double sxy = u_y + v_x;
        double ev = fma(P.cq, lapT, P.inv_Re * fma(sxy, sxy, 2.0 * fma(u_x, u_x, v_y * v_y)));
        ev = fma(u, Au, fma(v, Av, fma(w, Aw, ev)));           // u_i (in-plane part of d_j tau_ij)
        // convective in-plane parts: delta_x F_x + delta_y F_y from the staged values of the eight neighbours
        double cv[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
        {
          const double rx[4] = {F[4][Y][X - 2], F[4][Y][X - 1], F[4][Y][X + 1], F[4][Y][X + 2]};
          const double Gx[4] = {F[5][Y][X - 2], F[5][Y][X - 1], F[5][Y][X + 1], F[5][Y][X + 2]};
          const double px[4] = {cp * rx[0] * Tx[0], cp * rx[1] * Tx[1], cp * rx[2] * Tx[2], cp * rx[3] * Tx[3]};
          dflux(std::integral_constant<int, 0>{}, rx, ux, vx, wx, px, Gx, cx, cv);
        }
        {
          const double ry[4] = {F[4][Y - 2][X], F[4][Y - 1][X], F[4][Y + 1][X], F[4][Y + 2][X]};
          const double Gy[4] = {F[5][Y - 2][X], F[5][Y - 1][X], F[5][Y + 1][X], F[5][Y + 2][X]};
          const double py[4] = {cp * ry[0] * Ty[0], cp * ry[1] * Ty[1], cp * ry[2] * Ty[2], cp * ry[3] * Ty[3]};
          dflux(std::integral_constant<int, 1>{}, ry, uy, vy, wy, py, Gy, cy, cv);
        }
        B0[2] = -cv[0]; B1[2] = Au - cv[1]; B2[2] = Av - cv[2]; B3[2] = Aw - cv[3];
        aE[2] += ev - cv[4];
        if (tid < 4 * kCY) {                                     // x halo columns of the exchange buffer
          const int Yh = hr + kVH;
          S.g[e][0][hr][hc] = d1(F[0][Yh - 2][hc], F[0][Yh - 1][hc], F[0][Yh + 1][hc], F[0][Yh + 2][hc], cy);
          S.g[e][1][hr][hc] = d1(F[1][Yh - 2][hc], F[1][Yh - 1][hc], F[1][Yh + 1][hc], F[1][Yh + 2][hc], cy);
        }
      }
    };
    if (k + 2 >= z0 && k + 2 < z1) enter(std::true_type{});
    else enter(std::false_type{});
    if (k + 1 >= z0 && k + 1 < z1) {
      // ---- x-y mixed terms of plane k+1 (d_x of the d_y values published one step ago), divided by 3 Re
      const double (*Gm)[kCY][kVPX] = S.g[(k + 1 + 8) & 1];
      const double vxy = (third * P.inv_Re) * d1(Gm[1][ty][X - 2], Gm[1][ty][X - 1], Gm[1][ty][X + 1], Gm[1][ty][X + 2], cx);
      const double uxy = (third * P.inv_Re) * d1(Gm[0][ty][X - 2], Gm[0][ty][X - 1], Gm[0][ty][X + 1], Gm[0][ty][X + 2], cx);
      B1[1] += vxy;
      B2[1] += uxy;
      aE[1] = fma(uw[3], vxy, fma(vw[3], uxy, aE[1]));          // their share of u_i d_j tau_ij (u, v of plane k+1)
    }
    if (k < z0 || !inside) continue;

    // ---- plane k is complete
    const double u = uw[2], v = vw[2], w = ww[2];
    const double u_z = d1(uw[0], uw[1], uw[3], uw[4], cz);
    const double v_z = d1(vw[0], vw[1], vw[3], vw[4], cz);
    const double w_z = d1(ww[0], ww[1], ww[3], ww[4], cz);
    const double Mz0 = P.inv_Re * fma(third, d1(s0w[0], s0w[1], s0w[3], s0w[4], cz), d2(uw[0], uw[1], u, uw[3], uw[4], czz));
    const double Mz1 = P.inv_Re * fma(third, d1(s1w[0], s1w[1], s1w[3], s1w[4], cz), d2(vw[0], vw[1], v, vw[3], vw[4], czz));
    const double Mz2 = P.inv_Re * fma(third, d1(s2w[0], s2w[1], s2w[3], s2w[4], cz), four3 * d2(ww[0], ww[1], w, ww[3], ww[4], czz));
    const double div = s2w[2] + w_z;
    const double sxz = u_z + s0w[2], syz = v_z + s1w[2];
    const double phiz = fma(sxz, sxz, fma(syz, syz, fma(2.0 * w_z, w_z, (-2.0 / 3.0) * (div * div))));
    double res[5] = {B0[0], B1[0] + Mz0, B2[0] + Mz1, B3[0] + Mz2,
                     aE[0] + fma(u, Mz0, fma(v, Mz1, fma(w, Mz2, phiz * P.inv_Re)))};
    {
      // - delta_z F_z from the register windows (planes k-2, k-1, k+1, k+2)
      const double r4[4] = {rw[0], rw[1], rw[3], rw[4]}, u4[4] = {uw[0], uw[1], uw[3], uw[4]}, v4[4] = {vw[0], vw[1], vw[3], vw[4]};
      const double w4[4] = {ww[0], ww[1], ww[3], ww[4]}, p4[4] = {pw[0], pw[1], pw[3], pw[4]}, G4[4] = {Gw[0], Gw[1], Gw[3], Gw[4]};
      dflux(std::integral_constant<int, 2>{}, r4, u4, v4, w4, p4, G4, -cz, res);
    }
    // ---- stage update eq. (36)-(37) and the periodic images of the new state
    asm volatile("cp.async.wait_group 1;" ::: "memory");       // Q, dU of node k (issued one step ago) have landed
    const long long at = L.at(i, j, k);
    double qo[5];
#pragma unroll
    for (int c = 0; c < 5; ++c) {
      double d = rk.dt * res[c];
      if constexpr (!FIRST) d = fma(rk.A, S.q[k & 1][5 + c][tid], d);
      rk.Qtmp[c * sv + at] = d;
      qo[c] = fma(rk.B, d, S.q[k & 1][c][tid]);
      rk.Qout[c * sv + at] = qo[c];
    }
    const int sm = (k < kHalo ? 1 : 0) | (k >= L.n[2] - kHalo ? 2 : 0);
    if (wrap_mask | sm)
      wrap_store(rk.Qout + at, sv, wrap_mask | (sm << 4), (long long)L.n[0], (long long)L.n[1] * L.sy, (long long)L.n[2] * L.sz,
                 qo[0], qo[1], qo[2], qo[3], qo[4]);
  }
}

bool central_fused_path(const DevParams &P) { return P.scheme == 4 && viscous_fast_path(P); }

cudaError_t central_set_attributes() {
  cudaError_t e = cudaFuncSetAttribute(central_fused_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(CSmem));
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(central_fused_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(CSmem));
}

cudaError_t launch_central_fused(const DevParams &P, const double *Q, const RkArgs &rk, TmapCache *cache, cudaStream_t st) {
  const Layout &L = P.L;
  // 64 planes per block: 6 warm-up planes per chunk (9 %); at 256^3 1024 blocks = 6.9 waves of one block per SM
  const int chunk = L.n[2] > OSBLI_CCHUNK ? OSBLI_CCHUNK : L.n[2];
  dim3 grid((L.n[0] + kVX - 1) / kVX, (L.n[1] + kCY - 1) / kCY, (L.n[2] + chunk - 1) / chunk);
  const CUtensorMap *map = state_tensor_map(L, Q, cache, kCPY);
  if (!map) return cudaErrorNotSupported;
  if (rk.first) central_fused_kernel<true><<<grid, dim3(kVX, kCY), sizeof(CSmem), st>>>(P, Q, chunk, *map, rk);
  else central_fused_kernel<false><<<grid, dim3(kVX, kCY), sizeof(CSmem), st>>>(P, Q, chunk, *map, rk);
  return cudaGetLastError();
}

}  // namespace osbli
