// osbli_sweep.cu -- per-direction characteristic reconstruction sweeps (PAPER.md:100-111 steps 1-4,
// eq. (10)): R (-)= (f^_{i+1/2} - f^_{i-1/2}) / Delta_d   (or / detJ_i on curvilinear grids).
//
// Design ("marching"): every thread owns one grid line segment along the sweep direction and
// walks along it with a 6-point register window of staged point states.  Each point's
// thermodynamics (step 1) is computed once per sweep, each interface flux (step 2) once, and the
// previous interface flux stays in registers for the difference (step 3) -- no redundant work
// apart from a 5-point warm-up and one extra flux per segment.
//   * y, z sweeps: thread <-> x index, so every global access of a warp is a contiguous row
//     segment (coalesced, 128-byte aligned rows).
//   * x sweep: lane <-> line (32 consecutive (j,k) lines per warp).  Rows are moved in 8-point
//     tiles through warp-private shared memory (a 32 x 8 transpose, padded to stride 9), so global
//     traffic stays in whole 64-byte segments and nothing needs a block-wide barrier.
#include "osbli_flux.cuh"
#include "osbli_kernels.h"

namespace osbli {

// ---------------------------------------------------------------------------------------------
// y / z sweeps
// ---------------------------------------------------------------------------------------------
#ifndef OSBLI_YZ_MINB
#define OSBLI_YZ_MINB 1
#endif
#ifndef OSBLI_X_MINB
#define OSBLI_X_MINB 1
#endif
// RK = 0: R (-)= flux difference.  RK = 1 / 2: this is the last kernel of the stage and also does
// the low-storage Runge-Kutta update eq. (36)-(37) of its nodes (1: first stage, A_0 = 0, dU is not
// read): with R_in the residual accumulated by the earlier kernels of the stage,
//   dU = A dU + dt (R_in - (f^_{q+1/2} - f^_{q-1/2})/Delta),   Qout = Q + B dU,
// evaluated as (A dU + dt R_in) + (dt/Delta)(f^_{q-1/2} - f^_{q+1/2}) so that one value per variable
// waits in registers for the flux.  Q of node q is window slot 2; Qout must not alias Q (other
// blocks still read Q next to the chunk boundaries).  The final residual is not written anywhere.
template <int DIR, int SCHEME, bool CURV, bool ACCUM, int RK>
__global__ void __launch_bounds__(128, CURV ? 1 : OSBLI_YZ_MINB)
sweep_yz_kernel(const __grid_constant__ DevParams P, const double *__restrict__ Q, double *__restrict__ R,
                int chunk, const RkArgs rk) {
  static_assert(DIR == 1 || DIR == 2, "x has its own kernel");
  __shared__ double stg[CURV ? 6 : 8][5][128];   // per-thread slots: R (0-2) and dU (3-5) of nodes n % 3, raw state (6-7) of nodes n & 1
  __shared__ double kring[CURV ? 18 : 1][128];    // curvilinear: K_m of the six window points (KRing)
  KRing<128> KR{&kring[0][threadIdx.x], 0};
  const Layout &Ly = P.L;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= Ly.n[0]) return;
  const int t = blockIdx.y;                      // transverse index: k for the y sweep, j for the z sweep
  const int n = Ly.n[DIR];
  const int s0 = blockIdx.z * chunk;
  const int s1 = min(s0 + chunk, n);
  const long long st = (DIR == 1) ? Ly.sy : Ly.sz;
  const long long line0 = (DIR == 1) ? Ly.at(i, 0, t) : Ly.at(i, t, 0);   // node 0 of this line
  const long long sv = Ly.sv;
  const RecPar rp = make_recpar(P);
  const double inv_d = P.inv_delta[DIR];

  // periodic images of this thread's column: bit 0/1 = x below 3 / above nx-4, bits 2/3 = the same
  // for the transverse index (only used by the fused update with rk.wrap)
  int wrap_mask = 0;
  if constexpr (RK != 0) {
    const int nt_ = Ly.n[DIR == 1 ? 2 : 1];
    wrap_mask = (i < kHalo ? 1 : 0) | (i >= Ly.n[0] - kHalo ? 2 : 0);
    if (nt_ > 1) wrap_mask |= (t < kHalo ? 4 : 0) | (t >= nt_ - kHalo ? 8 : 0);
  }

  Pt<CURV> w[6];
  double rsq[3] = {1.0, 1.0, 1.0};               // 1/sqrt(rho) of window slots 3, 4, 5
  RoeSide rl = {0, 0, 0, 0, 0};
  double prev[5] = {0, 0, 0, 0, 0};

  auto load = [&](int node, double (&q)[5], double (&K)[3]) {
    const long long o = line0 + (long long)node * st;
#pragma unroll
    for (int c = 0; c < 5; ++c) q[c] = __ldg(Q + c * sv + o);
    if constexpr (CURV) {
      const double J = __ldg(P.detJ + o);
      K[0] = J * __ldg(P.D[DIR][0] + o);
      K[1] = J * __ldg(P.D[DIR][1] + o);
      K[2] = J * __ldg(P.D[DIR][2] + o);
    } else {
      K[0] = K[1] = K[2] = 0.0;
    }
  };

  // warm-up: nodes s0-3 .. s0+1 into slots 1..5 (after the first shift they sit in 0..4)
#pragma unroll
  for (int m = 1; m < 6; ++m) {
    double q[5], K[3];
    load(s0 - 4 + m, q, K);
    double rs;
    make_point<DIR, CURV>(P, q[0], q[1], q[2], q[3], q[4], K[0], K[1], K[2], w[m], rs);
    if constexpr (CURV) KR.put(m, K[0], K[1], K[2]);
    if (m >= 3) rsq[m - 3] = rs;
    if (m == 3) rl = roe_side<CURV>(P, w[3], rs);   // node s0-1 = left node of the first interface
  }
  // Asynchronous staging, two iterations ahead (one iteration of flux arithmetic does not keep enough bytes in
  // flight for HBM with 8 warps per SM): R (and dU) of node n travel by cp.async into the per-thread slot n % 3,
  // issued while interface n-2 is computed; in the fused update on uniform grids the raw state of the node that
  // enters the window is staged the same way (slot n & 1), elsewhere it is prefetched into registers.
  constexpr bool kAsyncQ = !CURV && RK != 0;
  constexpr int kGroups = kAsyncQ ? 2 : 1;       // cp.async groups committed per iteration
  auto issue_rd = [&](int node) {                // group 1: R, dU of `node` (empty outside [s0, s1))
    if (node >= s0 && node < s1) {
      const long long o = line0 + (long long)node * st;
      if constexpr (ACCUM) {
#pragma unroll
        for (int c = 0; c < 5; ++c) cp_async8(&stg[node % 3][c][threadIdx.x], R + c * sv + o);
      }
      if constexpr (RK == 2) {
#pragma unroll
        for (int c = 0; c < 5; ++c) cp_async8(&stg[3 + node % 3][c][threadIdx.x], rk.Qtmp + c * sv + o);
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  auto issue_q = [&](int node) {                 // group 2: raw state of `node` (needed up to node s1+2)
    if (node <= s1 + 2) {
      const long long o = line0 + (long long)node * st;
#pragma unroll
      for (int c = 0; c < 5; ++c) cp_async8(&stg[6 + (node & 1)][c][threadIdx.x], Q + c * sv + o);
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  double qn[5], Kn[3] = {0.0, 0.0, 0.0};
  // prologue = what iterations s0-3 and s0-2 would have issued
  issue_rd(s0 - 1);
  if constexpr (kAsyncQ) issue_q(s0 + 2);
  issue_rd(s0);
  if constexpr (kAsyncQ) issue_q(s0 + 3);
  else load(s0 + 2, qn, Kn);                     // prefetched raw state of the next node

  for (int q = s0 - 1; q < s1; ++q) {            // interface q+1/2, between nodes q and q+1
#pragma unroll
    for (int m = 0; m < 5; ++m) w[m] = w[m + 1];
    rsq[0] = rsq[1]; rsq[1] = rsq[2];
    if constexpr (kAsyncQ) {
      asm volatile("cp.async.wait_group 2;" ::: "memory");      // node q+3 has landed (issued two iterations ago)
#pragma unroll
      for (int c = 0; c < 5; ++c) qn[c] = stg[6 + ((q + 3) & 1)][c][threadIdx.x];
    }
    make_point<DIR, CURV>(P, qn[0], qn[1], qn[2], qn[3], qn[4], Kn[0], Kn[1], Kn[2], w[5], rsq[2]);
    if constexpr (CURV) { KR.advance(); KR.put(5, Kn[0], Kn[1], Kn[2]); }
    if constexpr (!kAsyncQ) {
      if (q + 1 < s1) load(q + 4, qn, Kn);       // node (q+1)+3, used by the next interface
    }
    issue_rd(q + 2);
    if constexpr (kAsyncQ) issue_q(q + 5);
    double rold[5] = {0, 0, 0, 0, 0};
    const RoeSide rr = roe_side<CURV>(P, w[3], rsq[0]);
    double f[5];
    if constexpr (CURV) interface_flux_curv<SCHEME>(P, w, KR, rl, rr, rp, f);
    else interface_flux<DIR, SCHEME>(P, w, rl, rr, rp, f);
    rl = rr;
    if (q >= s0) {
      const long long o = line0 + (long long)q * st;
      double sc = inv_d;
      if constexpr (CURV) sc = 1.0 / __ldg(P.detJ + o);
      // R, dU of node q were issued two iterations ago: everything younger may still be in flight
      if constexpr (kGroups == 2) asm volatile("cp.async.wait_group 4;" ::: "memory");
      else asm volatile("cp.async.wait_group 2;" ::: "memory");
      if constexpr (ACCUM) {
#pragma unroll
        for (int c = 0; c < 5; ++c) rold[c] = stg[q % 3][c][threadIdx.x];
      }
      if constexpr (RK != 0) {
        double dold[5] = {0, 0, 0, 0, 0};
        if constexpr (RK == 2) {
#pragma unroll
          for (int c = 0; c < 5; ++c) dold[c] = stg[3 + q % 3][c][threadIdx.x];
        }
#pragma unroll
        for (int c = 0; c < 5; ++c) {
          rold[c] *= rk.dt;
          if constexpr (RK == 2) rold[c] = fma(rk.A, dold[c], rold[c]);
        }
      }
      if constexpr (RK == 0) {
#pragma unroll
        for (int c = 0; c < 5; ++c) R[c * sv + o] = fma(prev[c] - f[c], sc, rold[c]);
      } else {
        const double qc[5] = {w[2].r, w[2].m[0], w[2].m[1], w[2].m[2], w[2].E};   // slot 2 = node q
        double qo[5];
        sc *= rk.dt;
#pragma unroll
        for (int c = 0; c < 5; ++c) {
          const double d = fma(prev[c] - f[c], sc, rold[c]);
          rk.Qtmp[c * sv + o] = d;
          qo[c] = fma(rk.B, d, qc[c]);
          rk.Qout[c * sv + o] = qo[c];
        }
        // All-periodic problems: nodes within 3 of a face also write their periodic images into the
        // halos of Qout (PAPER.md:503 periodic wrap, what osbli_bc would do next), so the next
        // stage starts without a halo-fill pass.  About 7 % of the nodes at 256^3.
        if (rk.wrap) {
          const int sm = (q < kHalo ? 1 : 0) | (q >= n - kHalo ? 2 : 0);
          if ((wrap_mask >> 2) | sm | ((wrap_mask & 3) == 3)) {
            wrap_store(rk.Qout + o, sv, wrap_mask | (sm << 4), (long long)Ly.n[0],
                       (long long)Ly.n[DIR == 1 ? 2 : 1] * ((DIR == 1) ? Ly.sz : Ly.sy), n * st, qo[0], qo[1], qo[2],
                       qo[3], qo[4]);
          } else if (wrap_mask) {      // x image only (two warps of every row at 256^3): plain predicated stores
            const long long oo = o + ((wrap_mask & 1) ? (long long)Ly.n[0] : -(long long)Ly.n[0]);
#pragma unroll
            for (int c = 0; c < 5; ++c) rk.Qout[c * sv + oo] = qo[c];
          }
        }
      }
    }
#pragma unroll
    for (int c = 0; c < 5; ++c) prev[c] = f[c];
  }
}

// ---------------------------------------------------------------------------------------------
// x sweep
// ---------------------------------------------------------------------------------------------
constexpr int kXT = 8;                 // points per transposed tile
constexpr int kXP = kXT + 1;           // padded row stride in shared memory (bank-conflict free)
constexpr int kXWarps = 4;             // warps per block

template <bool CURV> struct XSmem {
  double in[CURV ? 9 : 5][32][kXP];    // staged rows: 5 conservative variables (+ detJ, K_x, K_y, K_z)
  double out[5][32][kXP];              // staged flux differences
  double K[CURV ? 18 : 1][32];         // curvilinear: K_m of the six window points of every lane (KRing)
};

template <int SCHEME, bool CURV>
__global__ void __launch_bounds__(kXWarps * 32, CURV ? 1 : OSBLI_X_MINB)
sweep_x_kernel(const __grid_constant__ DevParams P, const double *__restrict__ Q, double *__restrict__ R,
               int chunk, int accumulate) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const Layout &Ly = P.L;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  XSmem<CURV> &S = reinterpret_cast<XSmem<CURV> *>(smem_raw)[warp];
  const int nlines = Ly.n[1] * Ly.n[2];
  const int line0 = (blockIdx.x * kXWarps + warp) * 32;
  if (line0 >= nlines) return;                                   // whole warp leaves together
  const int line = min(line0 + lane, nlines - 1);                // clamp: idle lanes mirror the last line
  const bool live = (line0 + lane) < nlines;
  const long long row = Ly.at(0, line % Ly.n[1], line / Ly.n[1]);   // node 0 of my line
  const long long sv = Ly.sv;
  const int nx = Ly.n[0];
  const int s0 = blockIdx.y * chunk;                             // chunk is a multiple of kXT
  const int s1 = min(s0 + chunk, nx);
  const RecPar rp = make_recpar(P);
  const double inv_d = P.inv_delta[0];

  // cooperative tile load: 32 rows x 8 points, each instruction moves 4 rows of 64 bytes
  const int lr = lane >> 3, lc = lane & 7;
  auto load_tile = [&](int a) {                                  // points [a, a+8), a multiple of 8
#pragma unroll
    for (int it = 0; it < 8; ++it) {
      const int rr_ = it * 4 + lr;
      const long long ro = __shfl_sync(0xffffffffu, row, rr_) + a + lc;
#pragma unroll
      for (int c = 0; c < 5; ++c) S.in[c][rr_][lc] = __ldg(Q + c * sv + ro);
      if constexpr (CURV) {
        S.in[5][rr_][lc] = __ldg(P.detJ + ro);
        S.in[6][rr_][lc] = __ldg(P.D[0][0] + ro);
        S.in[7][rr_][lc] = __ldg(P.D[0][1] + ro);
        S.in[8][rr_][lc] = __ldg(P.D[0][2] + ro);
      }
    }
  };
  auto store_tile = [&](int a) {                                 // flux differences of points [a, a+8) ∩ [s0, s1)
#pragma unroll
    for (int it = 0; it < 8; ++it) {
      const int rr_ = it * 4 + lr;
      const long long ro = __shfl_sync(0xffffffffu, row, rr_) + a + lc;
      const bool ok = (line0 + rr_ < nlines) && (a + lc < s1);
      if (ok) {
#pragma unroll
        for (int c = 0; c < 5; ++c) {
          double *dst = R + c * sv + ro;
          const double v = S.out[c][rr_][lc];
          *dst = accumulate ? (*dst + v) : v;
        }
      }
    }
  };

  Pt<CURV> w[6];
  KRing<32> KR{&S.K[0][lane], 0};
  if constexpr (CURV) {
#pragma unroll
    for (int m = 0; m < 6; ++m) KR.put(m, 1.0, 0.0, 0.0);        // placeholders until six real points have entered
  }
  double rsq[3] = {1.0, 1.0, 1.0};
  double Jw[4] = {1.0, 1.0, 1.0, 1.0};           // detJ of window slots 2..5 (curvilinear divisor)
  RoeSide rl = {0, 0, 0, 0, 0};
  double prev[5] = {0, 0, 0, 0, 0};
#pragma unroll
  for (int m = 0; m < 6; ++m) { w[m].r = 1.0; w[m].m[0] = w[m].m[1] = w[m].m[2] = 0.0; w[m].E = 1.0; w[m].p = 1.0; w[m].th = 0.0; w[m].c = 1.0; }

  int a_in = ((s0 - 3) >= 0) ? ((s0 - 3) / kXT) * kXT : -kXT;    // tile holding node s0-3 (s0-3 >= -3)
  load_tile(a_in);
  __syncwarp();

  for (int node = s0 - 3; node < s1 + 3; ++node) {               // node entering window slot 5
    if (node >= a_in + kXT) {
      __syncwarp();
      a_in += kXT;
      load_tile(a_in);
      __syncwarp();
    }
    const int col = node - a_in;
#pragma unroll
    for (int m = 0; m < 5; ++m) w[m] = w[m + 1];
    rsq[0] = rsq[1]; rsq[1] = rsq[2];
    Jw[0] = Jw[1]; Jw[1] = Jw[2]; Jw[2] = Jw[3];
    {
      const double r = S.in[0][lane][col], mx = S.in[1][lane][col], my = S.in[2][lane][col];
      const double mz = S.in[3][lane][col], E = S.in[4][lane][col];
      double kx = 0.0, ky = 0.0, kz = 0.0;
      if constexpr (CURV) {
        const double J = S.in[5][lane][col];
        kx = J * S.in[6][lane][col]; ky = J * S.in[7][lane][col]; kz = J * S.in[8][lane][col];
        Jw[3] = J;
      }
      make_point<0, CURV>(P, r, mx, my, mz, E, kx, ky, kz, w[5], rsq[2]);
      if constexpr (CURV) { KR.advance(); KR.put(5, kx, ky, kz); }
    }
    const int q = node - 3;                                      // interface q+1/2 is now computable
    if (q == s0 - 2) rl = roe_side<CURV>(P, w[3], rsq[0]);         // slot 3 holds node s0-1
    if (q < s0 - 1) continue;
    const RoeSide rr = roe_side<CURV>(P, w[3], rsq[0]);
    double f[5];
    if constexpr (CURV) interface_flux_curv<SCHEME>(P, w, KR, rl, rr, rp, f);
    else interface_flux<0, SCHEME>(P, w, rl, rr, rp, f);
    rl = rr;
    if (q >= s0) {
      double sc = inv_d;
      if constexpr (CURV) sc = 1.0 / Jw[0];                      // slot 2 = node q
      const int oc = q & (kXT - 1);
#pragma unroll
      for (int c = 0; c < 5; ++c) S.out[c][lane][oc] = (prev[c] - f[c]) * sc;
      if (oc == kXT - 1 || q == s1 - 1) {
        __syncwarp();
        store_tile(q - oc);
        __syncwarp();
      }
    }
#pragma unroll
    for (int c = 0; c < 5; ++c) prev[c] = f[c];
  }
  (void)live;
}

// ---------------------------------------------------------------------------------------------
// host-side launchers
// ---------------------------------------------------------------------------------------------
template <int SCHEME, bool CURV>
static cudaError_t launch_x(const DevParams &P, const double *Q, double *R, int accumulate, cudaStream_t st) {
  const int nlines = P.L.n[1] * P.L.n[2];
  const int nx = P.L.n[0];
  // segments of 64 nodes (6 warm-up nodes each); small problems (config 4: 2000 lines) take shorter segments until
  // there are at least as many warps as the chip holds resident (148 SMs x 8)
  int chunk = 64;
  while (chunk > 16 && (long long)((nlines + 31) / 32) * ((nx + chunk - 1) / chunk) < 148LL * 8) chunk /= 2;
  if (nx <= chunk) chunk = ((nx + kXT - 1) / kXT) * kXT;
  dim3 grid((nlines + kXWarps * 32 - 1) / (kXWarps * 32), (nx + chunk - 1) / chunk, 1);
  const size_t smem = sizeof(XSmem<CURV>) * kXWarps;
  sweep_x_kernel<SCHEME, CURV><<<grid, kXWarps * 32, smem, st>>>(P, Q, R, chunk, accumulate);
  return cudaGetLastError();
}

template <int DIR, int SCHEME, bool CURV>
static cudaError_t launch_yz(const DevParams &P, const double *Q, double *R, int accumulate, const RkArgs *rk,
                             cudaStream_t st) {
  const int nx = P.L.n[0];
  const int n = P.L.n[DIR];
  const int nt = (DIR == 1) ? P.L.n[2] : P.L.n[1];
  const int bx = nx >= 128 ? 128 : (nx > 64 ? 128 : (nx > 32 ? 64 : 32));
  // segments of 64 nodes (6 warm-up nodes each) where that still leaves >= 4 waves of blocks, else 32
  int chunk = n > 64 ? 32 : n;
  if (n > 64 && (long long)((nx + bx - 1) / bx) * nt * ((n + 63) / 64) >= 4LL * 2 * 148) chunk = 64;
  // small problems: 16-node segments when 32-node ones leave warp slots of the chip (148 SMs x 8 warps) empty
  if (n > 16 && chunk >= 32 && (long long)((nx + bx - 1) / bx) * (bx / 32) * nt * ((n + chunk - 1) / chunk) < 148LL * 8) chunk = 16;
  dim3 grid((nx + bx - 1) / bx, nt, (n + chunk - 1) / chunk);
  const RkArgs none = {0.0, 0.0, 0.0, nullptr, nullptr, 0, 0};
  if (rk) {
    if (!accumulate) return cudaErrorInvalidValue;              // the fused update is never the first kernel
    if (rk->first) sweep_yz_kernel<DIR, SCHEME, CURV, true, 1><<<grid, bx, 0, st>>>(P, Q, R, chunk, *rk);
    else sweep_yz_kernel<DIR, SCHEME, CURV, true, 2><<<grid, bx, 0, st>>>(P, Q, R, chunk, *rk);
  } else if (accumulate) sweep_yz_kernel<DIR, SCHEME, CURV, true, 0><<<grid, bx, 0, st>>>(P, Q, R, chunk, none);
  else sweep_yz_kernel<DIR, SCHEME, CURV, false, 0><<<grid, bx, 0, st>>>(P, Q, R, chunk, none);
  return cudaGetLastError();
}

// Opt-in dynamic shared memory of every x-sweep instantiation, for the current device (osbli_init).
template <int SCHEME, bool CURV>
static cudaError_t set_x_attr() {
  return cudaFuncSetAttribute(sweep_x_kernel<SCHEME, CURV>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)(sizeof(XSmem<CURV>) * kXWarps));
}
cudaError_t sweep_set_attributes() {
  cudaError_t e;
#define OSBLI_ATTR(SCH) \
  if ((e = set_x_attr<SCH, false>()) != cudaSuccess) return e; \
  if ((e = set_x_attr<SCH, true>()) != cudaSuccess) return e;
  OSBLI_ATTR(0) OSBLI_ATTR(1) OSBLI_ATTR(2) OSBLI_ATTR(3) OSBLI_ATTR(5)
#undef OSBLI_ATTR
  return cudaSuccess;
}

cudaError_t launch_sweep(const DevParams &P, int dir, const double *Q, double *R, int accumulate, const RkArgs *rk,
                         cudaStream_t st) {
  const bool curv = P.curvilinear != 0;
  const int sch = P.scheme;
  if (rk && dir == 0) return cudaErrorInvalidValue;             // only the y / z sweeps carry the fused update
#define OSBLI_DISPATCH(SCH, CRV)                                              \
  if (sch == SCH && curv == CRV) {                                            \
    if (dir == 0) return launch_x<SCH, CRV>(P, Q, R, accumulate, st);         \
    if (dir == 1) return launch_yz<1, SCH, CRV>(P, Q, R, accumulate, rk, st); \
    return launch_yz<2, SCH, CRV>(P, Q, R, accumulate, rk, st);               \
  }
  OSBLI_DISPATCH(0, false)
  OSBLI_DISPATCH(1, false)
  OSBLI_DISPATCH(0, true)
  OSBLI_DISPATCH(1, true)
  OSBLI_DISPATCH(2, false)
  OSBLI_DISPATCH(2, true)
  OSBLI_DISPATCH(3, false)
  OSBLI_DISPATCH(3, true)
  OSBLI_DISPATCH(5, false)
  OSBLI_DISPATCH(5, true)
#undef OSBLI_DISPATCH
  return cudaErrorInvalidValue;
}

}  // namespace osbli
