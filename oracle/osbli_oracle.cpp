/* osbli_oracle.cpp -- CPU ORACLE (test infrastructure, NOT product code; see osbli_oracle.h).
 *
 * A plain, slow, step-by-step restatement of the per-RK-stage residual of PAPER.md
 * (arXiv 2007.14933) sections 2.1-2.7 and 3.1.3, in the paper's order and notation:
 *
 *   O1  point-wise thermodynamics              eq. (6)-(7)
 *   O2  characteristic flux reconstruction     steps 1-4
 *       WENO-Z5 / TENO5                        eq. (14)-(26)
 *   O3  viscous + heat-flux terms              eq. (2)-(5),(28)-(35)
 *   O4  low-storage RK3                        eq. (36)-(38)
 *   O5  boundary conditions                    eq. (40)-(46)
 *
 * No blocking, fusion or reordering beyond what those passages state.  Build:
 *   g++ -std=c++17 -O2 -ffp-contract=off -fopenmp -shared -fPIC osbli_oracle.cpp
 */
#include "osbli_oracle.h"

#include <cmath>
#include <cstdlib>
#include <limits>
#include <vector>

namespace {

/* ------------------------------------------------------------------ grid bookkeeping ---- */
struct Grid {
  int n[3], h[3], N[3];
  long total;                                  /* one scalar field                          */
  long idx(int i, int j, int k) const {
    return ((long)(k + h[2]) * N[1] + (j + h[1])) * N[0] + (i + h[0]);
  }
  long stride(int d) const { return d == 0 ? 1 : (d == 1 ? (long)N[0] : (long)N[0] * N[1]); }
  bool active(int d) const { return n[d] > 1; }
};

Grid make_grid(const oracle_params *p) {
  Grid g;
  for (int d = 0; d < 3; ++d) {
    g.n[d] = p->n[d];
    /* ghost points: 3 for the 5th/6th-order stencils, 4 for the 7th-order one (i-3..i+4) */
    g.h[d] = p->n[d] > 1 ? (p->scheme == ORACLE_WENOZ7 ? 4 : 3) : 0;
    g.N[d] = g.n[d] + 2 * g.h[d];
  }
  g.total = (long)g.N[0] * g.N[1] * g.N[2];
  return g;
}

bool periodic(const oracle_params *p, int d) { return p->bc[d][0] == ORACLE_BC_PERIODIC; }

/* ------------------------------------------------------- O1: point-wise thermodynamics -- */
struct Prim { double rho, u, v, w, p, a, H, T, mu; };

/* PAPER.md:63-66 eq. (7): p = (gamma-1)(rhoE - rho u_i u_i / 2) = rho T/(gamma M^2),
 * a = sqrt(gamma p / rho);  PAPER.md:317-318: mu = T^1.5 (1+S)/(T+S), S = SuthT/RefT. */
Prim prim_of(const oracle_params *p, const double *q) {
  Prim s;
  s.rho = q[0];
  s.u = q[1] / q[0];
  s.v = q[2] / q[0];
  s.w = q[3] / q[0];
  s.p = (p->gamma - 1.0) * (q[4] - 0.5 * s.rho * (s.u * s.u + s.v * s.v + s.w * s.w));
  s.a = std::sqrt(p->gamma * s.p / s.rho);
  s.H = (q[4] + s.p) / s.rho;
  s.T = p->gamma * p->Minf * p->Minf * s.p / s.rho;
  if (p->visc == ORACLE_VISC_SUTHERLAND) {
    const double S = p->suth_ratio;
    s.mu = s.T * std::sqrt(s.T) * (1.0 + S) / (s.T + S);
  } else {
    s.mu = 1.0;
  }
  return s;
}

void load_state(const Grid &g, const double *Q, long at, double *q) {
  for (int c = 0; c < 5; ++c) q[c] = Q[c * g.total + at];
}

/* ------------------------------------------------------ WENO-Z5 / TENO5 reconstruction -- */
/* Reconstruct at the interface between c and d; upwind side is a,b,c.
 * Candidates (eq. 14; coefficients by polynomial exactness, Q3):
 *   q_R = (2c+5d-e)/6 on {c,d,e};  q_C = (-b+5c+2d)/6 on {b,c,d};  q_L = (2a-7b+11c)/6 on {a,b,c}
 * ideal weights d_R = 3/10, d_C = 6/10, d_L = 1/10.
 * Smoothness indicators eq. (17)-(19): beta_0 -> R, beta_1 -> C, beta_2 -> L. */
double reconstruct(int scheme, double a, double b, double c, double d, double e,
                   double eps, double ct, double *margin) {
  const double qR = (2.0 * c + 5.0 * d - e) / 6.0;
  const double qC = (-b + 5.0 * c + 2.0 * d) / 6.0;
  const double qL = (2.0 * a - 7.0 * b + 11.0 * c) / 6.0;
  const double dR = 3.0 / 10.0, dC = 6.0 / 10.0, dL = 1.0 / 10.0;

  const double s0 = c - 2.0 * d + e, t0 = 3.0 * c - 4.0 * d + e;
  const double s1 = b - 2.0 * c + d, t1 = b - d;
  const double s2 = a - 2.0 * b + c, t2 = a - 4.0 * b + 3.0 * c;
  const double bR = 13.0 / 12.0 * (s0 * s0) + 0.25 * (t0 * t0);   /* eq. (17) */
  const double bC = 13.0 / 12.0 * (s1 * s1) + 0.25 * (t1 * t1);   /* eq. (18) */
  const double bL = 13.0 / 12.0 * (s2 * s2) + 0.25 * (t2 * t2);   /* eq. (19) */
  const double tau = std::fabs(bR - bL);                          /* eq. (22) text, eq. (26) */

  if (margin) *margin = std::numeric_limits<double>::infinity();

  if (scheme == ORACLE_WENOZ3) {
    /* Third-order WENO-Z (k = 2 in the notation of PAPER.md:147-167): two 2-point candidates
     * q_0 = (c + d)/2 on {c,d}, q_1 = (-b + 3c)/2 on {b,c}; ideal weights 2/3, 1/3 (their combination is the
     * 3rd-order value (-b + 5c + 2d)/6); Jiang-Shu indicators of the linear candidates beta_0 = (d - c)^2,
     * beta_1 = (c - b)^2; tau = |beta_0 - beta_1|; weights eq. (22) (Q37). */
    const double q0 = 0.5 * (c + d), q1 = 0.5 * (-b + 3.0 * c);
    const double be0 = (d - c) * (d - c), be1 = (c - b) * (c - b);
    const double tau3 = std::fabs(be0 - be1);
    const double r0 = tau3 / (be0 + eps), r1 = tau3 / (be1 + eps);
    const double a0 = 2.0 / 3.0 * (1.0 + r0 * r0), a1 = 1.0 / 3.0 * (1.0 + r1 * r1);
    return a0 / (a0 + a1) * q0 + a1 / (a0 + a1) * q1;
  }

  if (scheme == ORACLE_WENOJS5) {
    /* eq. (20)-(21): alpha_r = d_r / (eps + beta_r)^p, p = 2 (eps = 1e-6 there) */
    const double aR = dR / ((eps + bR) * (eps + bR));
    const double aC = dC / ((eps + bC) * (eps + bC));
    const double aL = dL / ((eps + bL) * (eps + bL));
    const double sum = aR + aC + aL;
    return aR / sum * qR + aC / sum * qC + aL / sum * qL;         /* eq. (15), (20) */
  }

  if (scheme == ORACLE_WENOZ5) {
    /* eq. (22): alpha_r = d_r (1 + (tau/(beta_r+eps))^2), omega_r = alpha_r/sum */
    const double rR = tau / (bR + eps), rC = tau / (bC + eps), rL = tau / (bL + eps);
    const double aR = dR * (1.0 + rR * rR);
    const double aC = dC * (1.0 + rC * rC);
    const double aL = dL * (1.0 + rL * rL);
    const double sum = aR + aC + aL;
    const double wR = aR / sum, wC = aC / sum, wL = aL / sum;
    return wR * qR + wC * qC + wL * qL;                           /* eq. (15) */
  }

  /* TENO5: eq. (25) gamma_r = (C + tau/(beta_r+eps))^q, C = 1, q = 6 (x^6 = x^2 x^2 x^2);
   * eq. (24) chi_r = gamma_r / sum; cut-off: delta_r = 0 iff chi_r < C_T; eq. (23). */
  const double xR = 1.0 + tau / (bR + eps);
  const double xC = 1.0 + tau / (bC + eps);
  const double xL = 1.0 + tau / (bL + eps);
  const double xR2 = xR * xR, xC2 = xC * xC, xL2 = xL * xL;
  const double gR = xR2 * xR2 * xR2, gC = xC2 * xC2 * xC2, gL = xL2 * xL2 * xL2;
  const double gsum = gR + gC + gL;
  const double cR = gR / gsum, cC = gC / gsum, cL = gL / gsum;
  const double eR = cR < ct ? 0.0 : 1.0;
  const double eC = cC < ct ? 0.0 : 1.0;
  const double eL = cL < ct ? 0.0 : 1.0;
  if (margin) {
    double m = std::fabs(cR / ct - 1.0);
    m = std::fmin(m, std::fabs(cC / ct - 1.0));
    m = std::fmin(m, std::fabs(cL / ct - 1.0));
    *margin = m;
  }
  const double dsum = dR * eR + dC * eC + dL * eL;
  const double wR = dR * eR / dsum, wC = dC * eC / dsum, wL = dL * eL / dsum;
  return wR * qR + wC * qC + wL * qL;
}

/* ------------------------------------------------------------- TENO6 reconstruction ---- */
/* Sixth-order TENO (OpenSBLI "has both 5th and 6th order TENO schemes"): the three
 * 3-point candidates of eq. (14) plus a 4-point candidate on {c,d,e,f} (K - 2 = 4 stencils, r = 0..3),
 * weights eq. (23)-(25), global indicator eq. (27): tau_6 = |beta_3 - (beta_0 + beta_2 + 4 beta_1)/6|.
 * The paper prints neither d_r nor beta_3 for this scheme (refs [20, 21]); they follow from
 * definitions it does give (Q32):
 *   - q_3 = (3c + 13d - 5e + f)/12: the cubic with cell averages c,d,e,f evaluated at the interface;
 *   - d_r: the weights for which sum_r d_r q_r is the 6th-order value (a-8b+37c+37d-8e+f)/60:
 *     d_0 (R) = 6/20, d_1 (C) = 9/20, d_2 (L) = 1/20, d_3 = 4/20;
 *   - beta_3: the Jiang-Shu indicator [36] of that cubic, sum_l dx^(2l-1) int (d^l p/dx^l)^2 dx over
 *     the cell of c (re-derived symbolically in tests/test_oracle_teno6.py), evaluated as a sum of
 *     products of difference combinations like the printed eq. (17)-(19).
 * beta_0 -> R, beta_1 -> C, beta_2 -> L as in eq. (17)-(19). */
double reconstruct6(double a, double b, double c, double d, double e, double f,
                    double eps, double ct, double *margin, double *indicators = nullptr) {
  const double q[4] = {(2.0 * c + 5.0 * d - e) / 6.0, (-b + 5.0 * c + 2.0 * d) / 6.0,
                       (2.0 * a - 7.0 * b + 11.0 * c) / 6.0, (3.0 * c + 13.0 * d - 5.0 * e + f) / 12.0};
  const double dw[4] = {6.0 / 20.0, 9.0 / 20.0, 1.0 / 20.0, 4.0 / 20.0};
  const double s0 = c - 2.0 * d + e, t0 = 3.0 * c - 4.0 * d + e;
  const double s1 = b - 2.0 * c + d, t1 = b - d;
  const double s2 = a - 2.0 * b + c, t2 = a - 4.0 * b + 3.0 * c;
  double beta[4];
  beta[0] = 13.0 / 12.0 * (s0 * s0) + 0.25 * (t0 * t0);   /* eq. (17) */
  beta[1] = 13.0 / 12.0 * (s1 * s1) + 0.25 * (t1 * t1);   /* eq. (18) */
  beta[2] = 13.0 / 12.0 * (s2 * s2) + 0.25 * (t2 * t2);   /* eq. (19) */
  /* beta_3 in the form of eq. (17)-(19) (which are a_1^2 + 13/3 a_2^2 of the quadratics): with
   * a_1, a_2, a_3 the Taylor coefficients of the cubic at the centre of cell c,
   * beta_3 = a_1^2 + 13/3 a_2^2 + 3129/80 a_3^2 + a_1 a_3 / 2.  Expanded it is the usual
   * (2107 c^2 - 9402 cd + ... + 547 f^2)/240, which loses ~(c/dc)^2 digits to cancellation. */
  const double a1 = (-43.0 * c + 69.0 * d - 33.0 * e + 7.0 * f) / 24.0;
  const double a2 = (2.0 * c - 5.0 * d + 4.0 * e - f) / 2.0;
  const double a3 = (-c + 3.0 * d - 3.0 * e + f) / 6.0;
  beta[3] = a1 * a1 + 13.0 / 3.0 * (a2 * a2) + 3129.0 / 80.0 * (a3 * a3) + 0.5 * (a1 * a3);
  const double tau = std::fabs(beta[3] - (beta[0] + beta[2] + 4.0 * beta[1]) / 6.0);   /* eq. (27) */
  if (indicators) {
    for (int r = 0; r < 4; ++r) indicators[r] = beta[r];
    indicators[4] = tau;
  }
  double g[4], gsum = 0.0;
  for (int r = 0; r < 4; ++r) {
    const double x = 1.0 + tau / (beta[r] + eps);          /* eq. (25), C = 1, q = 6 */
    const double x2 = x * x;
    g[r] = x2 * x2 * x2;
    gsum += g[r];
  }
  double dsum = 0.0, del[4], m = std::numeric_limits<double>::infinity();
  for (int r = 0; r < 4; ++r) {
    const double chi = g[r] / gsum;                        /* eq. (24) */
    del[r] = chi < ct ? 0.0 : 1.0;
    m = std::fmin(m, std::fabs(chi / ct - 1.0));
    dsum += dw[r] * del[r];
  }
  if (margin) *margin = m;
  double v = 0.0;
  for (int r = 0; r < 4; ++r) v += dw[r] * del[r] / dsum * q[r];   /* eq. (23), (15) */
  return v;
}

/* ---------------------------------------------------------- Roe-averaged eigensystem ---- */
/* PAPER.md:104-105, steps 2(a)-(b): "Compute the average U_{i+1/2} state with either simple or Roe
 * averaging."  Roe average (averaging == ORACLE_AVG_ROE): u_j and H with sqrt(rho) weights, a~ from
 * H~ (Q11).  Simple average (ORACLE_AVG_SIMPLE, Q38): the arithmetic mean of the
 * two conservative states, U_{i+1/2} = (U_i + U_{i+1})/2, and u_j, H, a of THAT state.
 * Eigenvectors for a general unit normal n without tangent vectors
 * (Q12); fields ordered 0,1,2 (speed theta), 3 (theta+a), 4 (theta-a). */
void eigensystem(double gamma, int averaging, const double *QL, const double *QR, const double *n,
                 double *L, double *R, double *roe) {
  double u, v, w, H;
  if (averaging == ORACLE_AVG_SIMPLE) {
    double qm[5];
    for (int c = 0; c < 5; ++c) qm[c] = 0.5 * (QL[c] + QR[c]);
    u = qm[1] / qm[0];
    v = qm[2] / qm[0];
    w = qm[3] / qm[0];
    const double pm = (gamma - 1.0) * (qm[4] - 0.5 * qm[0] * (u * u + v * v + w * w));
    H = (qm[4] + pm) / qm[0];
  } else {
    const double rL = QL[0], rR = QR[0];
    const double uL = QL[1] / rL, vL = QL[2] / rL, wL = QL[3] / rL;
    const double uR = QR[1] / rR, vR = QR[2] / rR, wR = QR[3] / rR;
    const double pL = (gamma - 1.0) * (QL[4] - 0.5 * rL * (uL * uL + vL * vL + wL * wL));
    const double pR = (gamma - 1.0) * (QR[4] - 0.5 * rR * (uR * uR + vR * vR + wR * wR));
    const double HL = (QL[4] + pL) / rL, HR = (QR[4] + pR) / rR;
    const double sl = std::sqrt(rL), sr = std::sqrt(rR);
    u = (sl * uL + sr * uR) / (sl + sr);
    v = (sl * vL + sr * vR) / (sl + sr);
    w = (sl * wL + sr * wR) / (sl + sr);
    H = (sl * HL + sr * HR) / (sl + sr);
  }
  const double q2 = u * u + v * v + w * w;
  const double a = std::sqrt((gamma - 1.0) * (H - 0.5 * q2));
  const double nx = n[0], ny = n[1], nz = n[2];
  const double th = nx * u + ny * v + nz * w;
  const double b1 = (gamma - 1.0) / (a * a);
  const double b2 = 0.5 * b1 * q2;
  if (roe) { roe[0] = u; roe[1] = v; roe[2] = w; roe[3] = H; roe[4] = a; }

  /* right eigenvectors r_k = column k of R (R[row*5 + k]) */
  const double r0[5] = {nx, u * nx, v * nx + nz, w * nx - ny, 0.5 * q2 * nx + v * nz - w * ny};
  const double r1[5] = {ny, u * ny - nz, v * ny, w * ny + nx, 0.5 * q2 * ny + w * nx - u * nz};
  const double r2[5] = {nz, u * nz + ny, v * nz - nx, w * nz, 0.5 * q2 * nz + u * ny - v * nx};
  const double r3[5] = {1.0, u + a * nx, v + a * ny, w + a * nz, H + a * th};
  const double r4[5] = {1.0, u - a * nx, v - a * ny, w - a * nz, H - a * th};
  for (int r = 0; r < 5; ++r) {
    R[r * 5 + 0] = r0[r]; R[r * 5 + 1] = r1[r]; R[r * 5 + 2] = r2[r];
    R[r * 5 + 3] = r3[r]; R[r * 5 + 4] = r4[r];
  }
  /* left eigenvectors l_k = row k of L */
  const double l0[5] = {nx * (1.0 - b2) - (v * nz - w * ny), nx * b1 * u, nx * b1 * v + nz, nx * b1 * w - ny, -nx * b1};
  const double l1[5] = {ny * (1.0 - b2) - (w * nx - u * nz), ny * b1 * u - nz, ny * b1 * v, ny * b1 * w + nx, -ny * b1};
  const double l2[5] = {nz * (1.0 - b2) - (u * ny - v * nx), nz * b1 * u + ny, nz * b1 * v - nx, nz * b1 * w, -nz * b1};
  const double l3[5] = {0.5 * (b2 - th / a), 0.5 * (-b1 * u + nx / a), 0.5 * (-b1 * v + ny / a), 0.5 * (-b1 * w + nz / a), 0.5 * b1};
  const double l4[5] = {0.5 * (b2 + th / a), 0.5 * (-b1 * u - nx / a), 0.5 * (-b1 * v - ny / a), 0.5 * (-b1 * w - nz / a), 0.5 * b1};
  for (int c = 0; c < 5; ++c) {
    L[0 * 5 + c] = l0[c]; L[1 * 5 + c] = l1[c]; L[2 * 5 + c] = l2[c];
    L[3 * 5 + c] = l3[c]; L[4 * 5 + c] = l4[c];
  }
}

/* ------------------------------------------- O2: interface flux along one direction ----- */
/* Area-weighted normal K_m of step 1 (Q13, Q24): uniform K = e_d; curvilinear
 * K = J (D_d0, D_d1, D_d2) with point-wise metrics. */
void normal_at(const oracle_params *p, int dir, long at, double *K) {
  if (!p->curvilinear) {
    K[0] = K[1] = K[2] = 0.0;
    K[dir] = 1.0;
  } else {
    const double J = p->detJ[at];
    for (int c = 0; c < 3; ++c) K[c] = J * p->D[dir][c][at];
  }
}

/* ------------------------------------------------------------ WENO-7Z reconstruction ---- */
/* Seventh-order WENO-Z (k = 4 in eq. (15), (20), (22); "any arbitrary odd order", used at 7th order
 * in PAPER.md:485-495 and 531-533).  v[0..6] = nodes i-3..i+3, value at i+1/2.  Candidate r lives on the four
 * nodes {i-r .. i-r+3}, r = 0..3 (r = 0 the most downwind one, as beta_0 of eq. (17)), and is the cubic with those
 * cell averages evaluated at the interface; the ideal weights d_r = (4, 18, 12, 1)/35 [18] combine them to the
 * 7th-order value (-3, 25, -101, 319, 214, -38, 4)/420.  beta_r: eq. (16) on the cubic, written as for TENO6
 * (a_1^2 + 13/3 a_2^2 + 3129/80 a_3^2 + a_1 a_3 / 2 with the Taylor coefficients of the cubic at the centre of
 * cell i).  tau_7 = |beta_0 - beta_3|, "the absolute difference in the smoothness indicators over the full
 * reconstruction stencil" (Q40).  Weights eq. (22). */
double reconstruct7(const double *v, double eps, double *indicators = nullptr) {
  const double m3 = v[0], m2 = v[1], m1 = v[2], c = v[3], p1 = v[4], p2 = v[5], p3 = v[6];
  const double q[4] = {(3.0 * c + 13.0 * p1 - 5.0 * p2 + p3) / 12.0, (-m1 + 7.0 * c + 7.0 * p1 - p2) / 12.0,
                       (m2 - 5.0 * m1 + 13.0 * c + 3.0 * p1) / 12.0, (-3.0 * m3 + 13.0 * m2 - 23.0 * m1 + 25.0 * c) / 12.0};
  const double dw[4] = {4.0 / 35.0, 18.0 / 35.0, 12.0 / 35.0, 1.0 / 35.0};
  /* Taylor coefficients (first, second, third) at the centre of cell i of the four cubics */
  const double a1[4] = {(-43.0 * c + 69.0 * p1 - 33.0 * p2 + 7.0 * p3) / 24.0, (-7.0 * m1 - 15.0 * c + 27.0 * p1 - 5.0 * p2) / 24.0,
                        (5.0 * m2 - 27.0 * m1 + 15.0 * c + 7.0 * p1) / 24.0, (-7.0 * m3 + 33.0 * m2 - 69.0 * m1 + 43.0 * c) / 24.0};
  const double a2[4] = {(2.0 * c - 5.0 * p1 + 4.0 * p2 - p3) / 2.0, (m1 - 2.0 * c + p1) / 2.0, (m1 - 2.0 * c + p1) / 2.0,
                        (-m3 + 4.0 * m2 - 5.0 * m1 + 2.0 * c) / 2.0};
  const double a3[4] = {(-c + 3.0 * p1 - 3.0 * p2 + p3) / 6.0, (-m1 + 3.0 * c - 3.0 * p1 + p2) / 6.0,
                        (-m2 + 3.0 * m1 - 3.0 * c + p1) / 6.0, (-m3 + 3.0 * m2 - 3.0 * m1 + c) / 6.0};
  double beta[4];
  for (int r = 0; r < 4; ++r)
    beta[r] = a1[r] * a1[r] + 13.0 / 3.0 * (a2[r] * a2[r]) + 3129.0 / 80.0 * (a3[r] * a3[r]) + 0.5 * (a1[r] * a3[r]);
  const double tau = std::fabs(beta[0] - beta[3]);
  if (indicators) {
    for (int r = 0; r < 4; ++r) indicators[r] = beta[r];
    indicators[4] = tau;
  }
  double al[4], sum = 0.0;
  for (int r = 0; r < 4; ++r) {
    const double x = tau / (beta[r] + eps);
    al[r] = dw[r] * (1.0 + x * x);                          /* eq. (22) */
    sum += al[r];
  }
  double val = 0.0;
  for (int r = 0; r < 4; ++r) val += al[r] / sum * q[r];    /* eq. (15), (20) */
  return val;
}

/* f^_{i+1/2} between node `at` and `at + stride(dir)`; PAPER.md:100-111 steps 1-2. */
void interface_flux(const oracle_params *p, const Grid &g, const double *Q, int dir, long at,
                    double *fhat, double *margin) {
  const long s = g.stride(dir);
  /* window: nodes i-2..i+3 (six points); the 7th-order scheme: i-3..i+4 (eight); il = window index of node i */
  const int W = p->scheme == ORACLE_WENOZ7 ? 8 : 6, il = W / 2 - 1;
  double U[8][5], F[8][5], lam0[8], lamp[8], lamm[8], K[8][3];

  /* step 1: flux f(U_m), solution vector U_m and wave speeds at the stencil points */
  for (int m = 0; m < W; ++m) {
    const long pt = at + (long)(m - il) * s;
    load_state(g, Q, pt, U[m]);
    const Prim w = prim_of(p, U[m]);
    normal_at(p, dir, pt, K[m]);
    const double th = K[m][0] * w.u + K[m][1] * w.v + K[m][2] * w.w;
    const double Kn = std::sqrt(K[m][0] * K[m][0] + K[m][1] * K[m][1] + K[m][2] * K[m][2]);
    F[m][0] = w.rho * th;
    F[m][1] = U[m][1] * th + w.p * K[m][0];
    F[m][2] = U[m][2] * th + w.p * K[m][1];
    F[m][3] = U[m][3] * th + w.p * K[m][2];
    F[m][4] = (U[m][4] + w.p) * th;
    lam0[m] = th;
    lamp[m] = th + w.a * Kn;
    lamm[m] = th - w.a * Kn;
  }

  /* step 2(a)-(b): Roe average of nodes i, i+1 and its eigensystem; interface normal from
   * the averaged K (uniform: e_d). */
  double nhat[3];
  {
    const double kx = 0.5 * (K[il][0] + K[il + 1][0]);
    const double ky = 0.5 * (K[il][1] + K[il + 1][1]);
    const double kz = 0.5 * (K[il][2] + K[il + 1][2]);
    const double kn = std::sqrt(kx * kx + ky * ky + kz * kz);
    nhat[0] = kx / kn; nhat[1] = ky / kn; nhat[2] = kz / kn;
  }
  double L[25], R[25];
  eigensystem(p->gamma, p->averaging, U[il], U[il + 1], nhat, L, R, nullptr);

  for (int c = 0; c < 5; ++c) fhat[c] = 0.0;
  double mmin = std::numeric_limits<double>::infinity();

  for (int k = 0; k < 5; ++k) {
    /* step 2(c): V_k,m = l_k . U_m, G_k,m = l_k . f_m */
    double V[8], G[8];
    for (int m = 0; m < W; ++m) {
      double sv = 0.0, sg = 0.0;
      for (int c = 0; c < 5; ++c) {
        sv += L[k * 5 + c] * U[m][c];
        sg += L[k * 5 + c] * F[m][c];
      }
      V[m] = sv;
      G[m] = sg;
    }
    /* step 2(d): alpha_k = max over the stencil points of |lambda_k| (Q10) */
    const double *lam = (k < 3) ? lam0 : (k == 3 ? lamp : lamm);
    double alpha = 0.0;
    for (int m = 0; m < W; ++m) alpha = std::fmax(alpha, std::fabs(lam[m]));
    double gp[8], gm[8];
    for (int m = 0; m < W; ++m) {
      gp[m] = 0.5 * (G[m] + alpha * V[m]);          /* eq. (13) */
      gm[m] = 0.5 * (G[m] - alpha * V[m]);
    }
    /* step 2(e): g+ from the left-biased stencil, g- from its mirror image (Q4) */
    double m1, m2;
    double hp, hm;
    if (p->scheme == ORACLE_WENOZ7) {
      double mir[7];
      for (int m = 0; m < 7; ++m) mir[m] = gm[7 - m];
      hp = reconstruct7(gp, p->eps);
      hm = reconstruct7(mir, p->eps);
      m1 = m2 = std::numeric_limits<double>::infinity();
    } else if (p->scheme == ORACLE_TENO6) {
      hp = reconstruct6(gp[0], gp[1], gp[2], gp[3], gp[4], gp[5], p->eps, p->teno_ct, &m1);
      hm = reconstruct6(gm[5], gm[4], gm[3], gm[2], gm[1], gm[0], p->eps, p->teno_ct, &m2);
    } else {
      hp = reconstruct(p->scheme, gp[0], gp[1], gp[2], gp[3], gp[4], p->eps, p->teno_ct, &m1);
      hm = reconstruct(p->scheme, gm[5], gm[4], gm[3], gm[2], gm[1], p->eps, p->teno_ct, &m2);
    }
    mmin = std::fmin(mmin, std::fmin(m1, m2));
    /* step 2(f): back to physical space, f^ += (g^+ + g^-) r_k */
    const double gk = hp + hm;
    for (int c = 0; c < 5; ++c) fhat[c] += gk * R[c * 5 + k];
  }
  if (margin) *margin = mmin;
}

/* ----------------------------------------------- central differences, eq. (28)-(35) ----- */
/* Coefficients (times 12 delta) of the first derivative at node i of a line of n nodes.
 * Interior: eq. (28) with the sign corrected (Q1): (f_-2 - 8 f_-1 + 8 f_+1 - f_+2).
 * Non-periodic ends: eq. (30)-(33).  Returns the offset of the first stencil node. */
int d1_coeffs(int n, int i, bool per, double *c) {
  if (!per && i == 0)      { c[0] = -25; c[1] = 48;  c[2] = -36; c[3] = 16;  c[4] = -3; return 0; }   /* (30) */
  if (!per && i == 1)      { c[0] = -3;  c[1] = -10; c[2] = 18;  c[3] = -6;  c[4] = 1;  return -1; }  /* (31) */
  if (!per && i == n - 2)  { c[0] = -1;  c[1] = 6;   c[2] = -18; c[3] = 10;  c[4] = 3;  return -3; }  /* (32) */
  if (!per && i == n - 1)  { c[0] = 3;   c[1] = -16; c[2] = 36;  c[3] = -48; c[4] = 25; return -4; }  /* (33) */
  c[0] = 1; c[1] = -8; c[2] = 0; c[3] = 8; c[4] = -1;                                                 /* (28) */
  return -2;
}
/* Second derivative: interior eq. (29); ends eq. (34)-(35) and their mirror images. */
int d2_coeffs(int n, int i, bool per, double *c) {
  if (!per && i == 0)      { c[0] = 35; c[1] = -104; c[2] = 114; c[3] = -56;  c[4] = 11; return 0; }  /* (34) */
  if (!per && i == 1)      { c[0] = 11; c[1] = -20;  c[2] = 6;   c[3] = 4;    c[4] = -1; return -1; } /* (35) */
  if (!per && i == n - 2)  { c[0] = -1; c[1] = 4;    c[2] = 6;   c[3] = -20;  c[4] = 11; return -3; }
  if (!per && i == n - 1)  { c[0] = 11; c[1] = -56;  c[2] = 114; c[3] = -104; c[4] = 35; return -4; }
  c[0] = -1; c[1] = 16; c[2] = -30; c[3] = 16; c[4] = -1;                                             /* (29) */
  return -2;
}

double d1_line(const double *f, long s, int n, int i, bool per, double delta) {
  double c[5];
  const int o = d1_coeffs(n, i, per, c);
  double acc = 0.0;
  for (int m = 0; m < 5; ++m) acc += c[m] * f[(long)(i + o + m) * s];
  return acc / (12.0 * delta);
}
double d2_line(const double *f, long s, int n, int i, bool per, double delta) {
  double c[5];
  const int o = d2_coeffs(n, i, per, c);
  double acc = 0.0;
  for (int m = 0; m < 5; ++m) acc += c[m] * f[(long)(i + o + m) * s];
  return acc / (12.0 * delta * delta);
}

/* ------------------------------------------------ O3: viscous and heat-flux terms ------- */
/* Source of primitive values u,v,w,T,mu: either whole-field arrays (full residual) or
 * computed on the fly from Q (sampled residual).  Same function, same bits. */
struct PrimSource {
  const oracle_params *p;
  const Grid *g;
  const double *Q;
  const double *fields;   /* 5 fields u,v,w,T,mu in oracle layout, or NULL */
  double get(int f, long at) const {
    if (fields) return fields[f * g->total + at];
    double q[5];
    load_state(*g, Q, at, q);
    const Prim s = prim_of(p, q);
    switch (f) { case 0: return s.u; case 1: return s.v; case 2: return s.w; case 3: return s.T; default: return s.mu; }
  }
};

struct NodeIdx { int c[3]; };

/* delta_k f at a node (first difference along xi_k) */
double dk(const PrimSource &ps, int f, int k, NodeIdx nd, long at) {
  const Grid &g = *ps.g;
  if (!g.active(k)) return 0.0;
  const bool per = periodic(ps.p, k);
  const double delta = ps.p->curvilinear ? 1.0 : ps.p->delta[k];
  double c[5];
  const int o = d1_coeffs(g.n[k], nd.c[k], per, c);
  const long s = g.stride(k);
  double acc = 0.0;
  for (int m = 0; m < 5; ++m) acc += c[m] * ps.get(f, at + (long)(o + m) * s);
  return acc / (12.0 * delta);
}
/* delta_kk f */
double dkk(const PrimSource &ps, int f, int k, NodeIdx nd, long at) {
  const Grid &g = *ps.g;
  if (!g.active(k)) return 0.0;
  const bool per = periodic(ps.p, k);
  const double delta = ps.p->curvilinear ? 1.0 : ps.p->delta[k];
  double c[5];
  const int o = d2_coeffs(g.n[k], nd.c[k], per, c);
  const long s = g.stride(k);
  double acc = 0.0;
  for (int m = 0; m < 5; ++m) acc += c[m] * ps.get(f, at + (long)(o + m) * s);
  return acc / (12.0 * delta * delta);
}
/* delta_kl f := delta_k (delta_l f), k < l, fixed order of composition */
double dkl(const PrimSource &ps, int f, int k, int l, NodeIdx nd, long at) {
  const Grid &g = *ps.g;
  if (!g.active(k) || !g.active(l)) return 0.0;
  const bool per = periodic(ps.p, k);
  const double delta = ps.p->curvilinear ? 1.0 : ps.p->delta[k];
  double c[5];
  const int o = d1_coeffs(g.n[k], nd.c[k], per, c);
  const long s = g.stride(k);
  double acc = 0.0;
  for (int m = 0; m < 5; ++m) {
    if (c[m] == 0.0) continue;
    NodeIdx sh = nd;
    sh.c[k] += o + m;
    acc += c[m] * dk(ps, f, l, sh, at + (long)(o + m) * s);
  }
  return acc / (12.0 * delta);
}

const int IJ[3][3] = {{0, 1, 2}, {1, 3, 4}, {2, 4, 5}};   /* (i,j) -> index into xx,xy,xz,yy,yz,zz */

/* Adds the viscous + heat-flux contribution at one node to r[5].  PAPER.md:49-57 eq. (2)-(5)
 * expanded by the product rule (Q21); metric chain rule PAPER.md:228 (Q25). */
void viscous_at(const PrimSource &ps, NodeIdx nd, long at, double *r) {
  const oracle_params *p = ps.p;
  /* computational differences of u,v,w,T (f = 0..3) and mu (f = 4) */
  double c1[5][3], c2[4][3][3];
  for (int f = 0; f < 5; ++f)
    for (int k = 0; k < 3; ++k) c1[f][k] = (f == 4 && p->visc != ORACLE_VISC_SUTHERLAND) ? 0.0 : dk(ps, f, k, nd, at);
  for (int f = 0; f < 4; ++f)
    for (int k = 0; k < 3; ++k)
      for (int l = k; l < 3; ++l) {
        const double v = (k == l) ? dkk(ps, f, k, nd, at) : dkl(ps, f, k, l, nd, at);
        c2[f][k][l] = v;
        c2[f][l][k] = v;
      }
  /* physical derivatives: uniform d_j f = delta_j f; curvilinear d_j f = sum_k D_kj delta_k f,
   * d_i d_j f = sum_k sum_l D_ki D_lj delta_kl f + sum_l E_l,ij delta_l f */
  double g1[5][3], g2[4][3][3];
  if (!p->curvilinear) {
    for (int f = 0; f < 5; ++f) for (int j = 0; j < 3; ++j) g1[f][j] = c1[f][j];
    for (int f = 0; f < 4; ++f) for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) g2[f][i][j] = c2[f][i][j];
  } else {
    double D[3][3], E[3][6];
    for (int k = 0; k < 3; ++k) {
      for (int j = 0; j < 3; ++j) D[k][j] = p->D[k][j][at];
      for (int m = 0; m < 6; ++m) E[k][m] = p->E[k][m][at];
    }
    for (int f = 0; f < 5; ++f)
      for (int j = 0; j < 3; ++j) {
        double acc = 0.0;
        for (int k = 0; k < 3; ++k) acc += D[k][j] * c1[f][k];
        g1[f][j] = acc;
      }
    for (int f = 0; f < 4; ++f)
      for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
          double acc = 0.0;
          for (int k = 0; k < 3; ++k)
            for (int l = 0; l < 3; ++l) acc += D[k][i] * D[l][j] * c2[f][k][l];
          for (int l = 0; l < 3; ++l) acc += E[l][IJ[i][j]] * c1[f][l];
          g2[f][i][j] = acc;
        }
  }
  const double vel[3] = {ps.get(0, at), ps.get(1, at), ps.get(2, at)};
  const double mu = ps.get(4, at);
  const double div = g1[0][0] + g1[1][1] + g1[2][2];
  const double *dmu = g1[4];
  const double *dT = g1[3];

  /* M_i = Re * d_j tau_ij */
  double M[3];
  for (int i = 0; i < 3; ++i) {
    const double lap = g2[i][0][0] + g2[i][1][1] + g2[i][2][2];
    const double gdiv = g2[0][i][0] + g2[1][i][1] + g2[2][i][2];        /* d_i (d_k u_k) */
    double cross = 0.0;
    for (int j = 0; j < 3; ++j) cross += dmu[j] * (g1[i][j] + g1[j][i]);
    M[i] = mu * (lap + gdiv / 3.0) + cross - 2.0 / 3.0 * dmu[i] * div;
  }
  /* tau_ij d_j u_i, eq. (5) */
  double phi = 0.0;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      const double tau = mu / p->Re * (g1[i][j] + g1[j][i] - (i == j ? 2.0 / 3.0 * div : 0.0));
      phi += tau * g1[i][j];
    }
  /* -d_j q_j, eq. (4) */
  const double cq = 1.0 / ((p->gamma - 1.0) * p->Minf * p->Minf * p->Pr * p->Re);
  const double lapT = g2[3][0][0] + g2[3][1][1] + g2[3][2][2];
  const double heat = cq * (mu * lapT + (dmu[0] * dT[0] + dmu[1] * dT[1] + dmu[2] * dT[2]));

  r[1] += M[0] / p->Re;
  r[2] += M[1] / p->Re;
  r[3] += M[2] / p->Re;
  r[4] += (vel[0] * M[0] + vel[1] * M[1] + vel[2] * M[2]) / p->Re + phi + heat;
}

void fill_prim_fields(const oracle_params *p, const Grid &g, const double *Q, double *fields) {
#pragma omp parallel for num_threads(p->nthreads) schedule(static)
  for (long at = 0; at < g.total; ++at) {
    double q[5];
    load_state(g, Q, at, q);
    const Prim s = prim_of(p, q);
    fields[0 * g.total + at] = s.u;
    fields[1 * g.total + at] = s.v;
    fields[2 * g.total + at] = s.w;
    fields[3 * g.total + at] = s.T;
    fields[4 * g.total + at] = s.mu;
  }
}

/* ------------------------------------------------- metric terms ---------- */
/* "The metric terms are evaluated by the same central interior and boundary schemes ...
 * computed once at the start of the simulation."  Given node coordinates x_j(xi) on the
 * halo-extended grid (halos hold the periodic continuation where the direction is periodic;
 * they are not read otherwise), compute A_jk = d x_j/d xi_k with delta_k (eq. 28, 30-33, unit
 * computational spacing), J = det A, D = A^-1 (D_kj = d xi_k/d x_j), and
 * E_l,ij = d_i(D_lj) = sum_k D_ki delta_k(D_lj) for i <= j (Q25).  Halo values of
 * D, J, E: periodic wrap, else copy of the boundary plane (Q25).  An inactive
 * direction k has A_jk = delta[k] if j == k else 0. */
void fill_field_halo(const oracle_params *p, const Grid &g, double *f) {
  for (int d = 0; d < 3; ++d) {
    if (!g.active(d)) continue;
    int lo[3], hi[3];
    for (int e = 0; e < 3; ++e) {
      if (e < d) { lo[e] = -g.h[e]; hi[e] = g.n[e] + g.h[e]; }
      else       { lo[e] = 0;       hi[e] = g.n[e]; }
    }
    const long s = g.stride(d);
    const int n = g.n[d];
    const int e1 = (d + 1) % 3, e2 = (d + 2) % 3;
    for (int a = lo[e2]; a < hi[e2]; ++a)
      for (int b = lo[e1]; b < hi[e1]; ++b) {
        int ijk[3];
        ijk[d] = 0; ijk[e1] = b; ijk[e2] = a;
        const long base = g.idx(ijk[0], ijk[1], ijk[2]);
        for (int m = 1; m <= g.h[d]; ++m) {
          if (periodic(p, d)) {
            f[base - (long)m * s] = f[base + (long)(n - m) * s];
            f[base + (long)(n - 1 + m) * s] = f[base + (long)(m - 1) * s];
          } else {
            f[base - (long)m * s] = f[base];
            f[base + (long)(n - 1 + m) * s] = f[base + (long)(n - 1) * s];
          }
        }
      }
  }
}

void metrics_from_coords(const oracle_params *p, const Grid &g, const double *X,
                         double *const *D, double *detJ, double *const *E) {
  const int nt = p->nthreads;
#pragma omp parallel for num_threads(nt) schedule(static)
  for (int k = 0; k < g.n[2]; ++k)
    for (int j = 0; j < g.n[1]; ++j)
      for (int i = 0; i < g.n[0]; ++i) {
        const long at = g.idx(i, j, k);
        const int nd[3] = {i, j, k};
        double A[3][3];
        for (int c = 0; c < 3; ++c)
          for (int d = 0; d < 3; ++d) {
            if (!g.active(d)) { A[c][d] = (c == d) ? p->delta[d] : 0.0; continue; }
            /* base pointer of the line through this node along d, node index nd[d] */
            const double *line = X + c * g.total + at - (long)nd[d] * g.stride(d);
            A[c][d] = d1_line(line, g.stride(d), g.n[d], nd[d], periodic(p, d), 1.0);
          }
        const double det = A[0][0] * (A[1][1] * A[2][2] - A[1][2] * A[2][1])
                         - A[0][1] * (A[1][0] * A[2][2] - A[1][2] * A[2][0])
                         + A[0][2] * (A[1][0] * A[2][1] - A[1][1] * A[2][0]);
        detJ[at] = det;
        /* inverse by cofactors: D[k][j] = cof(A)[j][k] / det */
        D[0 * 3 + 0][at] = (A[1][1] * A[2][2] - A[1][2] * A[2][1]) / det;
        D[0 * 3 + 1][at] = (A[0][2] * A[2][1] - A[0][1] * A[2][2]) / det;
        D[0 * 3 + 2][at] = (A[0][1] * A[1][2] - A[0][2] * A[1][1]) / det;
        D[1 * 3 + 0][at] = (A[1][2] * A[2][0] - A[1][0] * A[2][2]) / det;
        D[1 * 3 + 1][at] = (A[0][0] * A[2][2] - A[0][2] * A[2][0]) / det;
        D[1 * 3 + 2][at] = (A[0][2] * A[1][0] - A[0][0] * A[1][2]) / det;
        D[2 * 3 + 0][at] = (A[1][0] * A[2][1] - A[1][1] * A[2][0]) / det;
        D[2 * 3 + 1][at] = (A[0][1] * A[2][0] - A[0][0] * A[2][1]) / det;
        D[2 * 3 + 2][at] = (A[0][0] * A[1][1] - A[0][1] * A[1][0]) / det;
      }
  for (int m = 0; m < 9; ++m) fill_field_halo(p, g, D[m]);
  fill_field_halo(p, g, detJ);
#pragma omp parallel for num_threads(nt) schedule(static)
  for (int k = 0; k < g.n[2]; ++k)
    for (int j = 0; j < g.n[1]; ++j)
      for (int i = 0; i < g.n[0]; ++i) {
        const long at = g.idx(i, j, k);
        const int nd[3] = {i, j, k};
        for (int l = 0; l < 3; ++l)
          for (int a = 0; a < 3; ++a)
            for (int b = a; b < 3; ++b) {
              double acc = 0.0;                      /* d_a (D_lb) = sum_k D_ka delta_k (D_lb) */
              for (int d = 0; d < 3; ++d) {
                if (!g.active(d)) continue;
                const double *line = D[l * 3 + b] + at - (long)nd[d] * g.stride(d);
                acc += D[d * 3 + a][at] * d1_line(line, g.stride(d), g.n[d], nd[d], periodic(p, d), 1.0);
              }
              E[l * 6 + IJ[a][b]][at] = acc;
            }
      }
  for (int m = 0; m < 18; ++m) fill_field_halo(p, g, E[m]);
}

/* Divisor of eq. (10): Delta_d (uniform) or J_i (curvilinear, unit computational spacing). */
double flux_divisor(const oracle_params *p, int dir, long at) {
  return p->curvilinear ? p->detJ[at] : p->delta[dir];
}

int validate(const oracle_params *p) {
  for (int d = 0; d < 3; ++d) {
    if (p->n[d] < 1) return 1;
    if (p->n[d] > 1 && p->n[d] < 5) return 1;
    if ((p->bc[d][0] == ORACLE_BC_PERIODIC) != (p->bc[d][1] == ORACLE_BC_PERIODIC)) return 1;
  }
  if (p->nthreads < 1) return 1;
  if (p->averaging != ORACLE_AVG_ROE && p->averaging != ORACLE_AVG_SIMPLE) return 1;
  if (p->rk3_form != ORACLE_RK3_WILLIAMSON && p->rk3_form != ORACLE_RK3_SSP) return 1;
  if (p->scheme == ORACLE_CENTRAL4 && p->curvilinear) return 1;   /* central convective terms: uniform grids only */
  return 0;
}

/* -------------------------------------------------------------- O5: boundary fill ------- */
void bc_direction(const oracle_params *p, const Grid &g, double *Q, int d) {
  if (!g.active(d)) return;
  /* transverse ranges: directions below d are taken over their halo-extended range, the
   * ones above d over the interior only (they are filled afterwards) */
  int lo[3], hi[3];
  for (int e = 0; e < 3; ++e) {
    if (e < d) { lo[e] = -g.h[e]; hi[e] = g.n[e] + g.h[e]; }
    else       { lo[e] = 0;       hi[e] = g.n[e]; }
  }
  const long s = g.stride(d);
  const int n = g.n[d];
  const int e1 = (d + 1) % 3, e2 = (d + 2) % 3;
  const double gam = p->gamma, M2 = p->Minf * p->Minf;
  for (int a = lo[e2]; a < hi[e2]; ++a)
    for (int b = lo[e1]; b < hi[e1]; ++b) {
      int ijk[3];
      ijk[d] = 0; ijk[e1] = b; ijk[e2] = a;
      const long base = g.idx(ijk[0], ijk[1], ijk[2]);      /* node 0 of this line */
      for (int side = 0; side < 2; ++side) {
        const int type = p->bc[d][side];
        /* wall: node index of the boundary plane; inw: +1 into the domain */
        const long wall = base + (side == 0 ? 0 : (long)(n - 1) * s);
        const long inw = side == 0 ? s : -s;
        if (type == ORACLE_BC_PERIODIC) {
          for (int m = 1; m <= g.h[d]; ++m)
            for (int c = 0; c < 5; ++c) {
              double *q = Q + c * g.total;
              if (side == 0) q[base - (long)m * s] = q[base + (long)(n - m) * s];
              else           q[base + (long)(n - 1 + m) * s] = q[base + (long)(m - 1) * s];
            }
        } else if (type == ORACLE_BC_EXTRAP0) {
          for (int m = 1; m <= g.h[d]; ++m)
            for (int c = 0; c < 5; ++c) Q[c * g.total + wall - (long)m * inw] = Q[c * g.total + wall];
        } else if (type == ORACLE_BC_DIRICHLET) {
          for (int m = 0; m <= g.h[d]; ++m)
            for (int c = 0; c < 5; ++c)
              Q[c * g.total + wall - (long)m * inw] = p->dirichlet[c * g.total + wall - (long)m * inw];
        } else if (type == ORACLE_BC_WALL_ISOTHERMAL || type == ORACLE_BC_WALL_ADIABATIC) {
          double Tw = p->wall_T[d][side];
          if (type == ORACLE_BC_WALL_ADIABATIC) {
            /* "a one-sided 4th order approximation of dT/dy = 0 is rearranged using the
             * interior points to calculate the unknown wall temperature": eq. (30) set to zero,
             * -25 T_w + 48 T_1 - 36 T_2 + 16 T_3 - 3 T_4 = 0. */
            double T[5];
            for (int m = 1; m <= 4; ++m) {
              double qm[5];
              load_state(g, Q, wall + (long)m * inw, qm);
              T[m] = prim_of(p, qm).T;
            }
            Tw = (48.0 * T[1] - 36.0 * T[2] + 16.0 * T[3] - 3.0 * T[4]) / 25.0;
          }
          /* eq. (40)-(41): no-slip on the boundary plane, wall energy from T_w; rho_w floats */
          const double rw = Q[wall];
          Q[1 * g.total + wall] = 0.0;
          Q[2 * g.total + wall] = 0.0;
          Q[3 * g.total + wall] = 0.0;
          const double Ew = rw * Tw / (M2 * gam * (gam - 1.0));
          Q[4 * g.total + wall] = Ew;
          const double pw = (gam - 1.0) * Ew;
          /* T_1: temperature of the first interior node */
          double q1[5];
          load_state(g, Q, wall + inw, q1);
          const double T1 = prim_of(p, q1).T;
          for (int m = 1; m <= g.h[d]; ++m) {
            const double Tm = (m + 1) * Tw - m * T1;                       /* eq. (42) */
            const double rm = M2 * gam * pw / Tm;                          /* eq. (43) */
            double qi[5];
            load_state(g, Q, wall + (long)m * inw, qi);
            const double ui = qi[1] / qi[0], vi = qi[2] / qi[0], wi = qi[3] / qi[0];
            const long at = wall - (long)m * inw;
            Q[0 * g.total + at] = rm;
            Q[1 * g.total + at] = -rm * ui;                                /* eq. (44) */
            Q[2 * g.total + at] = -rm * vi;                                /* eq. (45) */
            Q[3 * g.total + at] = -rm * wi;                                /* eq. (46) */
            Q[4 * g.total + at] = pw / (gam - 1.0) + 0.5 * rm * (ui * ui + vi * vi + wi * wi);
          }
        }
      }
    }
}

void rhs_full(const oracle_params *p, const Grid &g, const double *Q, double *R, int parts, double *margin) {
  const int nt = p->nthreads;
  /* R starts at 0 on interior nodes */
#pragma omp parallel for num_threads(nt) schedule(static)
  for (int k = 0; k < g.n[2]; ++k)
    for (int j = 0; j < g.n[1]; ++j)
      for (int i = 0; i < g.n[0]; ++i) {
        const long at = g.idx(i, j, k);
        for (int c = 0; c < 5; ++c) R[c * g.total + at] = 0.0;
        if (margin) margin[at] = std::numeric_limits<double>::infinity();
      }

  if (parts & ORACLE_PART_INVISCID) {
    for (int d = 0; d < 3; ++d) {
      if (!g.active(d)) continue;                      /* step 4: repeat for all dimensions */
      const int e1 = (d + 1) % 3, e2 = (d + 2) % 3;
      const int n = g.n[d];
      const long s = g.stride(d);
#pragma omp parallel for num_threads(nt) schedule(static) collapse(2)
      for (int a = 0; a < g.n[e2]; ++a)
        for (int b = 0; b < g.n[e1]; ++b) {
          int ijk[3];
          ijk[d] = 0; ijk[e1] = b; ijk[e2] = a;
          const long base = g.idx(ijk[0], ijk[1], ijk[2]);
          if (p->scheme == ORACLE_CENTRAL4) {
            /* "Central schemes are also applied to smooth problems that do not require shock-capturing"
             * (PAPER.md:198): the convective terms as the 4th-order central difference eq. (28) of the
             * point-wise flux vectors (one-sided closures eq. (30)-(33) next to non-periodic boundaries);
             * uniform grids only (Q36). */
            for (int i = 0; i < n; ++i) {
              double cf[5];
              const int off = d1_coeffs(n, i, p->bc[d][0] == ORACLE_BC_PERIODIC, cf);
              double acc[5] = {0, 0, 0, 0, 0};
              for (int m = 0; m < 5; ++m) {
                if (cf[m] == 0.0) continue;
                double q[5], f[5];
                load_state(g, Q, base + (long)(i + off + m) * s, q);
                const Prim w = prim_of(p, q);
                const double th = d == 0 ? w.u : (d == 1 ? w.v : w.w);
                f[0] = q[0] * th;
                f[1] = q[1] * th + (d == 0 ? w.p : 0.0);
                f[2] = q[2] * th + (d == 1 ? w.p : 0.0);
                f[3] = q[3] * th + (d == 2 ? w.p : 0.0);
                f[4] = (q[4] + w.p) * th;
                for (int c = 0; c < 5; ++c) acc[c] += cf[m] * f[c];
              }
              const long at = base + (long)i * s;
              for (int c = 0; c < 5; ++c) R[c * g.total + at] -= acc[c] / (12.0 * p->delta[d]);
            }
            continue;
          }
          /* step 2: every half node of this line, -1/2 ... n-1/2 */
          std::vector<double> fh((size_t)(n + 1) * 5), mg((size_t)n + 1);
          for (int q = 0; q <= n; ++q)
            interface_flux(p, g, Q, d, base + (long)(q - 1) * s, &fh[(size_t)q * 5], &mg[q]);
          /* step 3: eq. (10) */
          for (int i = 0; i < n; ++i) {
            const long at = base + (long)i * s;
            const double div = flux_divisor(p, d, at);
            for (int c = 0; c < 5; ++c)
              R[c * g.total + at] -= (fh[(size_t)(i + 1) * 5 + c] - fh[(size_t)i * 5 + c]) / div;
            if (margin) margin[at] = std::fmin(margin[at], std::fmin(mg[i], mg[i + 1]));
          }
        }
    }
  }

  if ((parts & ORACLE_PART_VISCOUS) && p->visc != ORACLE_VISC_NONE) {
    std::vector<double> fields((size_t)5 * g.total);
    fill_prim_fields(p, g, Q, fields.data());
    PrimSource ps{p, &g, Q, fields.data()};
#pragma omp parallel for num_threads(nt) schedule(static)
    for (int k = 0; k < g.n[2]; ++k)
      for (int j = 0; j < g.n[1]; ++j)
        for (int i = 0; i < g.n[0]; ++i) {
          const long at = g.idx(i, j, k);
          double r[5] = {0, 0, 0, 0, 0};
          viscous_at(ps, NodeIdx{{i, j, k}}, at, r);
          for (int c = 1; c < 5; ++c) R[c * g.total + at] += r[c];
        }
  }

  /* constant body force (Q34): momentum += f, energy += u . f */
  if ((parts & ORACLE_PART_VISCOUS) && (p->force[0] != 0.0 || p->force[1] != 0.0 || p->force[2] != 0.0)) {
    for (int k = 0; k < g.n[2]; ++k)
      for (int j = 0; j < g.n[1]; ++j)
        for (int i = 0; i < g.n[0]; ++i) {
          const long at = g.idx(i, j, k);
          double q[5];
          load_state(g, Q, at, q);
          double work = 0.0;
          for (int a = 0; a < 3; ++a) {
            R[(1 + a) * g.total + at] += p->force[a];
            work += q[1 + a] / q[0] * p->force[a];
          }
          R[4 * g.total + at] += work;
        }
  }
}

}  // namespace

/* ======================================================================== C entry points */
extern "C" {

double oracle_reconstruct(int32_t scheme, double a, double b, double c, double d, double e,
                          double eps, double teno_ct, double *margin) {
  return reconstruct(scheme, a, b, c, d, e, eps, teno_ct, margin);
}

double oracle_reconstruct6(double a, double b, double c, double d, double e, double f,
                           double eps, double teno_ct, double *margin) {
  return reconstruct6(a, b, c, d, e, f, eps, teno_ct, margin);
}

double oracle_reconstruct7(const double *v7, double eps, double *out5) { return reconstruct7(v7, eps, out5); }
void oracle_teno6_indicators(double a, double b, double c, double d, double e, double f, double *out5) {
  reconstruct6(a, b, c, d, e, f, 1e-16, 1e-6, nullptr, out5);
}

void oracle_eigensystem(double gamma, const double *QL, const double *QR, const double *nhat,
                        double *L, double *R, double *roe) {
  eigensystem(gamma, ORACLE_AVG_ROE, QL, QR, nhat, L, R, roe);
}
void oracle_eigensystem_avg(double gamma, int32_t averaging, const double *QL, const double *QR,
                            const double *nhat, double *L, double *R, double *roe) {
  eigensystem(gamma, averaging, QL, QR, nhat, L, R, roe);
}

double oracle_d1(const double *f, int32_t n, int32_t i, int32_t per, double delta) {
  return d1_line(f, 1, n, i, per != 0, delta);
}
double oracle_d2(const double *f, int32_t n, int32_t i, int32_t per, double delta) {
  return d2_line(f, 1, n, i, per != 0, delta);
}

int32_t oracle_halo(const oracle_params *p, int32_t *h) {
  const Grid g = make_grid(p);
  for (int d = 0; d < 3; ++d) h[d] = g.h[d];
  return 0;
}
int64_t oracle_field_size(const oracle_params *p) { return make_grid(p).total; }

void oracle_interface_flux(const oracle_params *p, const double *Q, int32_t dir,
                           int32_t i, int32_t j, int32_t k, double *fhat, double *margin) {
  const Grid g = make_grid(p);
  interface_flux(p, g, Q, dir, g.idx(i, j, k), fhat, margin);
}

int32_t oracle_bc(const oracle_params *p, double *Q) {
  if (validate(p)) return 1;
  const Grid g = make_grid(p);
  for (int d = 0; d < 3; ++d) bc_direction(p, g, Q, d);
  return 0;
}

int32_t oracle_rhs(const oracle_params *p, const double *Q, double *R, int32_t parts, double *margin) {
  if (validate(p)) return 1;
  const Grid g = make_grid(p);
  rhs_full(p, g, Q, R, parts, margin);
  return 0;
}

int32_t oracle_rhs_points(const oracle_params *p, const double *Q, int32_t parts,
                          int64_t npts, const int32_t *ijk, double *out) {
  if (validate(p)) return 1;
  if (p->scheme == ORACLE_CENTRAL4) return 2;          /* node-by-node evaluation exists for the reconstruction schemes only */
  const Grid g = make_grid(p);
  PrimSource ps{p, &g, Q, nullptr};
#pragma omp parallel for num_threads(p->nthreads) schedule(dynamic, 16)
  for (int64_t t = 0; t < npts; ++t) {
    const int i = ijk[3 * t], j = ijk[3 * t + 1], k = ijk[3 * t + 2];
    const long at = g.idx(i, j, k);
    double r[5] = {0, 0, 0, 0, 0};
    if (parts & ORACLE_PART_INVISCID) {
      for (int d = 0; d < 3; ++d) {
        if (!g.active(d)) continue;
        double fp[5], fm[5];
        interface_flux(p, g, Q, d, at, fp, nullptr);
        interface_flux(p, g, Q, d, at - g.stride(d), fm, nullptr);
        const double div = flux_divisor(p, d, at);
        for (int c = 0; c < 5; ++c) r[c] -= (fp[c] - fm[c]) / div;
      }
    }
    if ((parts & ORACLE_PART_VISCOUS) && p->visc != ORACLE_VISC_NONE) {
      double rv[5] = {0, 0, 0, 0, 0};
      viscous_at(ps, NodeIdx{{i, j, k}}, at, rv);
      for (int c = 1; c < 5; ++c) r[c] += rv[c];
    }
    if (parts & ORACLE_PART_VISCOUS) {
      double q[5];
      load_state(g, Q, at, q);
      for (int a = 0; a < 3; ++a) {
        r[1 + a] += p->force[a];
        r[4] += q[1 + a] / q[0] * p->force[a];
      }
    }
    for (int c = 0; c < 5; ++c) out[5 * t + c] = r[c];
  }
  return 0;
}

int32_t oracle_metrics(const oracle_params *p, const double *coords,
                       double *const *D, double *detJ, double *const *E) {
  if (validate(p)) return 1;
  const Grid g = make_grid(p);
  metrics_from_coords(p, g, coords, D, detJ, E);
  return 0;
}

/* PAPER.md:232-242 eq. (36)-(38); coefficients of the 3-stage scheme of ref. [23]
 * (Williamson's 2N-storage RK3, Q15). */
void oracle_rk3_update(int32_t s, double dt, int64_t count, double *U, double *dU, const double *R) {
  const double A[3] = {0.0, -5.0 / 9.0, -153.0 / 128.0};
  const double B[3] = {1.0 / 3.0, 15.0 / 16.0, 8.0 / 15.0};
  for (int64_t o = 0; o < count; ++o) {
    /* A_0 = 0: dU^(0) is never read, so it need not be initialised */
    const double du = (s == 0 ? 0.0 : A[s] * dU[o]) + dt * R[o];               /* eq. (36) */
    dU[o] = du;
    U[o] = U[o] + B[s] * du;                                                    /* eq. (37) */
  }
}

/* "plus a 3rd order strong-stability-preserving (SSP) version to improve stability for flows containing
 * discontinuities ... [44] for the SSP version of the 3rd order scheme" (used by the
 * problem script at PAPER.md:343).  Same form eq. (36)-(38); the coefficients are not printed: the three-stage
 * 2N-storage TVD scheme of Gottlieb & Shu, as published to six digits in B_1 (Q39).  A_3 = 0: the
 * last stage is a plain Euler increment from U^(2). */
void oracle_rk3ssp_update(int32_t s, double dt, int64_t count, double *U, double *dU, const double *R) {
  const double A[3] = {0.0, -2.915493957701923, 0.0};
  const double B[3] = {0.924574, 0.287713063186749, 0.626538109512740};
  for (int64_t o = 0; o < count; ++o) {
    const double du = (A[s] == 0.0 ? 0.0 : A[s] * dU[o]) + dt * R[o];          /* eq. (36) */
    dU[o] = du;
    U[o] = U[o] + B[s] * du;                                                    /* eq. (37) */
  }
}

/* The 4th-order member of the same low-storage family eq. (36)-(38): "The 3rd and 4th order schemes have
 * three and five sub-stages per iteration respectively. The coefficients A_i and B_i are taken from [23]"
 * (PAPER.md:242): the five-stage 2N-storage scheme of Carpenter & Kennedy (Q35). */
void oracle_rk4_update(int32_t s, double dt, int64_t count, double *U, double *dU, const double *R) {
  const double A[5] = {0.0, -567301805773.0 / 1357537059087.0, -2404267990393.0 / 2016746695238.0,
                       -3550918686646.0 / 2091501179385.0, -1275806237668.0 / 842570457699.0};
  const double B[5] = {1432997174477.0 / 9575080441755.0, 5161836677717.0 / 13612068292357.0,
                       1720146321549.0 / 2090206949498.0, 3134564353537.0 / 4481467310338.0,
                       2277821191437.0 / 14882151754819.0};
  for (int64_t o = 0; o < count; ++o) {
    const double du = (s == 0 ? 0.0 : A[s] * dU[o]) + dt * R[o];               /* eq. (36) */
    dU[o] = du;
    U[o] = U[o] + B[s] * du;                                                    /* eq. (37) */
  }
}

int32_t oracle_rk4_step(const oracle_params *p, double *Q, double *dU, double *R, double dt) {
  if (validate(p)) return 1;
  const Grid g = make_grid(p);
  for (int s = 0; s < 5; ++s) {
    for (int d = 0; d < 3; ++d) bc_direction(p, g, Q, d);
    rhs_full(p, g, Q, R, ORACLE_PART_INVISCID | ORACLE_PART_VISCOUS, nullptr);
#pragma omp parallel for num_threads(p->nthreads) schedule(static)
    for (int k = 0; k < g.n[2]; ++k)
      for (int j = 0; j < g.n[1]; ++j)
        for (int c = 0; c < 5; ++c) {
          const long o = c * g.total + g.idx(0, j, k);
          oracle_rk4_update(s, dt, g.n[0], Q + o, dU + o, R + o);
        }
  }
  for (int d = 0; d < 3; ++d) bc_direction(p, g, Q, d);
  return 0;
}

int32_t oracle_rk3_step(const oracle_params *p, double *Q, double *dU, double *R, double dt) {
  if (validate(p)) return 1;
  const Grid g = make_grid(p);
  for (int s = 0; s < 3; ++s) {
    for (int d = 0; d < 3; ++d) bc_direction(p, g, Q, d);
    rhs_full(p, g, Q, R, ORACLE_PART_INVISCID | ORACLE_PART_VISCOUS, nullptr);
    /* stage update on interior nodes, one x-line at a time */
#pragma omp parallel for num_threads(p->nthreads) schedule(static)
    for (int k = 0; k < g.n[2]; ++k)
      for (int j = 0; j < g.n[1]; ++j)
        for (int c = 0; c < 5; ++c) {
          const long o = c * g.total + g.idx(0, j, k);
          if (p->rk3_form == ORACLE_RK3_SSP) oracle_rk3ssp_update(s, dt, g.n[0], Q + o, dU + o, R + o);
          else                               oracle_rk3_update(s, dt, g.n[0], Q + o, dU + o, R + o);
        }
  }
  for (int d = 0; d < 3; ++d) bc_direction(p, g, Q, d);
  return 0;
}

}  // extern "C"
