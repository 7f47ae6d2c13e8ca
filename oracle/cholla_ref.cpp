// cholla_ref.cpp — ORACLE. TEST INFRASTRUCTURE ONLY.
//
// A plain, slow, obviously-correct CPU implementation of one unsplit CTU time step of the 3-D
// Euler equations (PPMC reconstruction + exact Riemann solver), written from the text of
// arXiv:1410.4194 (Schneider & Robertson, "Cholla").  Citations are `P:L<line>` =
// /root/reference/PAPER.md line, plus the equation; "G<n>/S<n>" are the readings of garbled /
// silent passages listed in DESIGN.md §"Readings".
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// call this.  It shares no code (no headers, helpers, tables, constants) with the CUDA path in
// paper_1410_4194_b200/csrc/ and must never be linked into or called from the product.
//
// Style: whole-grid arrays for every intermediate of the paper's steps 1-5, one
// loop nest per step, no tiling, no fusion, fp64 throughout, built with -ffp-contract=off.
// The optional OpenMP pragma on the outermost loop of each nest does not change any result (the
// step contains no floating-point reduction; min is exact).
//
// Beyond the north_star path (PPMC + exact solver) it holds the paper's other method choices: the Roe solver with the
// HLLE failsafe and the H correction (B.2, App. C), the PLMC, PCM, PPMP and PLMP reconstructions (A.1, A.2, A.4) and
// the analytic boundary of the Noh test, each selected at run time through ref_set_*.
//
// Parity pins: every function below is pinned by tests/test_oracle_*.py (closed forms,
// invariants, special cases, the paper's printed observations); see DESIGN.md §5.  No function here is "parity unpinned".

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <limits>
#include <new>
#include <string>
#include <vector>

namespace {

constexpr double P_FLOOR = 1e-20;       // P:L231 pressure floor
constexpr double P_GUESS_FLOOR = 1e-6;
constexpr double NEWTON_TOL = 1e-8;     // P:L1095 "e.g. 1e-6"; reading S2: 1e-8
constexpr int NEWTON_CAP = 20;          // reading S2

enum { BC_PERIODIC = 1, BC_REFLECTIVE = 2, BC_OUTFLOW = 3, BC_NOH = 4 };   // 4: analytic inflow of the Noh test
enum { SOLVER_EXACT = 0, SOLVER_ROE = 1 };   // the Riemann solver is selectable
enum { RECON_PPMC = 0, RECON_PLMC = 1, RECON_PCM = 2, RECON_PPMP = 3, RECON_PLMP = 4 };   // so is the reconstruction

thread_local std::string g_err;

// ---------------------------------------------------------------------------------------------
// Eq. 6-10: conserved u=[rho, rho*u, rho*v, rho*w, E] <-> primitive w=[rho,u,v,w,p].
// Pressure floor (reading S1: applied in every conserved->primitive conversion).
// ---------------------------------------------------------------------------------------------
void cons_to_prim(double gamma, const double u[5], double w[5]) {
  const double rho = u[0];
  const double vx = u[1] / rho, vy = u[2] / rho, vz = u[3] / rho;
  const double ke = 0.5 * rho * ((vx * vx + vy * vy) + vz * vz);  // Eq. 7
  double p = (gamma - 1.0) * (u[4] - ke);                         // Eq. 6, 8
  if (!(p >= P_FLOOR)) p = (p != p) ? p : P_FLOOR;                // keep NaN visible
  w[0] = rho; w[1] = vx; w[2] = vy; w[3] = vz; w[4] = p;
}

void prim_to_cons(double gamma, const double w[5], double u[5]) {
  const double rho = w[0];
  u[0] = rho;
  u[1] = rho * w[1];
  u[2] = rho * w[2];
  u[3] = rho * w[3];
  u[4] = w[4] / (gamma - 1.0) + 0.5 * rho * ((w[1] * w[1] + w[2] * w[2]) + w[3] * w[3]);
}

// Direction-local ordering (rho, v_n, v_t1, v_t2, p|E) for a sweep along d: cyclic permutation
// (P:L164).  comp(d,m) = index in the global vector of local component m.
inline int comp(int d, int m) {
  if (m == 0 || m == 4) return m;
  return 1 + (d + (m - 1)) % 3;
}
void to_local(int d, const double g[5], double l[5]) { for (int m = 0; m < 5; ++m) l[m] = g[comp(d, m)]; }
void to_global(int d, const double l[5], double g[5]) { for (int m = 0; m < 5; ++m) g[comp(d, m)] = l[m]; }

// ---------------------------------------------------------------------------------------------
// A9 (first row read as G1: 0.5(-rho du/a + dp/a^2)) and A11.
// ---------------------------------------------------------------------------------------------
void char_project(double rho, double a, const double dw[5], double dxi[5]) {
  const double a2 = a * a;
  dxi[0] = 0.5 * (-(rho * dw[1] / a) + dw[4] / a2);
  dxi[1] = dw[0] - dw[4] / a2;
  dxi[2] = dw[2];
  dxi[3] = dw[3];
  dxi[4] = 0.5 * (rho * dw[1] / a + dw[4] / a2);
}
void char_backproject(double rho, double a, const double dxi[5], double dw[5]) {
  dw[0] = dxi[1] + (dxi[0] + dxi[4]);
  dw[1] = (a / rho) * (dxi[4] - dxi[0]);
  dw[2] = dxi[2];
  dw[3] = dxi[3];
  dw[4] = (a * a) * (dxi[0] + dxi[4]);
}

inline double sgn(double x) { return x < 0.0 ? -1.0 : 1.0; }  // A4

// Monotonised-central limiter A10 (called "van Leer" in the text; the formula governs, G7).
inline double limit(double dL, double dR, double dC) {
  if (dL * dR > 0.0) return sgn(dC) * std::min(std::fabs(dC), std::min(2.0 * std::fabs(dL), 2.0 * std::fabs(dR)));
  return 0.0;
}

// Limited slope of cell q from its neighbours (A2 P:L690, A8-A11 P:L722-743), primitive, local order.
void limited_slope(double gamma, const double wm[5], const double w0[5], const double wp[5], double dw[5]) {
  const double rho = w0[0];
  const double a = std::sqrt(gamma * w0[4] / rho);  // Eq. 21 with cell q's own averages
  double dwL[5], dwR[5], dwC[5], xL[5], xR[5], xC[5], x[5];
  for (int m = 0; m < 5; ++m) {
    dwL[m] = w0[m] - wm[m];
    dwR[m] = wp[m] - w0[m];
    dwC[m] = 0.5 * (wp[m] - wm[m]);
  }
  char_project(rho, a, dwL, xL);
  char_project(rho, a, dwR, xR);
  char_project(rho, a, dwC, xC);
  for (int m = 0; m < 5; ++m) x[m] = limit(xL[m], xR[m], xC[m]);
  char_backproject(rho, a, x, dw);
}

// ---------------------------------------------------------------------------------------------
// PPMC for one cell (A.3).  w[s] = primitive cell averages of cells i-2..i+2 (s=0..4),
// local order.  Outputs: WL,WR = monotonised face values (after A23); WLs,WRs = W*_L, W*_R
// after characteristic tracing (A33), all primitive, local order.  dtdx = dt/dx_d.
// ---------------------------------------------------------------------------------------------
void ppmc_cell(double gamma, double dtdx, const double w[5][5], double WL[5], double WR[5],
               double WLs[5], double WRs[5]) {
  double dwm[5], dw0[5], dwp[5];
  limited_slope(gamma, w[0], w[1], w[2], dwm);  // cell i-1
  limited_slope(gamma, w[1], w[2], w[3], dw0);  // cell i
  limited_slope(gamma, w[2], w[3], w[4], dwp);  // cell i+1
  const double* wi = w[2];
  const double* wim = w[1];
  const double* wip = w[3];

  double dwi[5], w6[5];
  for (int m = 0; m < 5; ++m) {
    // A20
    double L = 0.5 * (wi[m] + wim[m]) - (dw0[m] - dwm[m]) / 6.0;
    double R = 0.5 * (wip[m] + wi[m]) - (dwp[m] - dw0[m]) / 6.0;
    // A21
    if ((R - wi[m]) * (wi[m] - L) <= 0.0) { L = wi[m]; R = wi[m]; }
    // A22: both tests on the pair as it stands after A21 (G8)
    const bool fixL = (R - L) * (L - (3.0 * wi[m] - 2.0 * R)) < 0.0;
    const bool fixR = (R - L) * ((3.0 * wi[m] - 2.0 * L) - R) < 0.0;
    const double L0 = L, R0 = R;
    if (fixL) L = 3.0 * wi[m] - 2.0 * R0;
    if (fixR) R = 3.0 * wi[m] - 2.0 * L0;
    // A23
    L = std::max(std::min(wi[m], wim[m]), L);
    L = std::min(std::max(wi[m], wim[m]), L);
    R = std::max(std::min(wi[m], wip[m]), R);
    R = std::min(std::max(wi[m], wip[m]), R);
    WL[m] = L; WR[m] = R;
    dwi[m] = R - L;                              // A24
    w6[m] = 6.0 * (wi[m] - 0.5 * (L + R));       // A26 read as A50 (G2)
  }

  // A8 eigenvalues from the cell averages; A27
  const double rho = wi[0];
  const double a = std::sqrt(gamma * wi[4] / rho);
  const double lm = wi[1] - a, l0 = wi[1], lp = wi[1] + a;
  const double am = dtdx * std::min(lm, 0.0), bm = dtdx * std::max(lm, 0.0);
  const double a0 = dtdx * std::min(l0, 0.0), b0 = dtdx * std::max(l0, 0.0);
  const double ap = dtdx * std::min(lp, 0.0), bp = dtdx * std::max(lp, 0.0);

  // Domain-of-dependence averages under each characteristic (the six forms at P:L1005-1015;
  // A25 P:L837-838 are the m (left) and p (right) members).
  double WLm[5], WL0[5], WLp[5], WRm[5], WR0[5], WRp[5];
  for (int m = 0; m < 5; ++m) {
    WLm[m] = WL[m] - 0.5 * am * (dwi[m] + w6[m] * (1.0 + (2.0 / 3.0) * am));
    WL0[m] = WL[m] - 0.5 * a0 * (dwi[m] + w6[m] * (1.0 + (2.0 / 3.0) * a0));
    WLp[m] = WL[m] - 0.5 * ap * (dwi[m] + w6[m] * (1.0 + (2.0 / 3.0) * ap));
    WRm[m] = WR[m] - 0.5 * bm * (dwi[m] - w6[m] * (1.0 - (2.0 / 3.0) * bm));
    WR0[m] = WR[m] - 0.5 * b0 * (dwi[m] - w6[m] * (1.0 - (2.0 / 3.0) * b0));
    WRp[m] = WR[m] - 0.5 * bp * (dwi[m] - w6[m] * (1.0 - (2.0 / 3.0) * bp));
  }
  // A29, A30, A32 read as differences of those averages (G3).
  double E[5], B[5], C[5], D[5];
  for (int m = 0; m < 5; ++m) {
    E[m] = WL0[m] - WLm[m];
    B[m] = WLp[m] - WLm[m];
    C[m] = WRm[m] - WRp[m];
    D[m] = WR0[m] - WRp[m];
  }
  const double a2 = a * a;
  double sL[5] = {0, 0, 0, 0, 0}, sR[5] = {0, 0, 0, 0, 0};
  if (l0 < 0.0) {  // A28 first term
    sL[0] += E[0] - E[4] / a2;
    sL[2] += E[2];
    sL[3] += E[3];
  }
  if (lp < 0.0) {  // A28 second term
    sL[0] += 0.5 * (rho * B[1] / a + B[4] / a2);
    sL[1] += 0.5 * (B[1] + B[4] / (a * rho));
    sL[4] += 0.5 * (rho * B[1] * a + B[4]);
  }
  if (lm > 0.0) {  // A31 first term
    sR[0] += 0.5 * (-(rho * C[1] / a) + C[4] / a2);
    sR[1] += 0.5 * (C[1] - C[4] / (a * rho));
    sR[4] += 0.5 * (-(rho * C[1] * a) + C[4]);
  }
  if (l0 > 0.0) {  // A31 second term
    sR[0] += D[0] - D[4] / a2;
    sR[2] += D[2];
    sR[3] += D[3];
  }
  for (int m = 0; m < 5; ++m) {  // A33, reference states A25
    WLs[m] = WLm[m] + sL[m];
    WRs[m] = WRp[m] + sR[m];
  }
}

// ---------------------------------------------------------------------------------------------
// PLMC for one cell (A.2): linear reconstruction with the slope limited in the characteristic
// variables (A8-A11, the same limited_slope PPMC uses), faces A12, monotonised A13, slope A14,
// characteristic tracing A15-A19.  A19's second vector lost its last row in the text: the contact term
// has the same shape as A17's first vector, [x, 0, x, x, 0] (reading G10).  Same argument layout as
// ppmc_cell; only w[1..3] (cells i-1, i, i+1) are used.
// ---------------------------------------------------------------------------------------------
void plmc_cell(double gamma, double dtdx, const double w[5][5], double WL[5], double WR[5],
               double WLs[5], double WRs[5]) {
  const double* wi = w[2];
  const double* wim = w[1];
  const double* wip = w[3];
  double dw0[5], dwi[5];
  limited_slope(gamma, wim, wi, wip, dw0);                       // A8-A11
  for (int m = 0; m < 5; ++m) {
    const double LA = wi[m] - 0.5 * dw0[m], RA = wi[m] + 0.5 * dw0[m];              // A12
    const double LB = std::max(std::min(wi[m], wim[m]), LA);                        // A13
    WL[m] = std::min(std::max(wi[m], wim[m]), LB);
    const double RB = std::max(std::min(wi[m], wip[m]), RA);
    WR[m] = std::min(std::max(wi[m], wip[m]), RB);
    dwi[m] = WR[m] - WL[m];                                                         // A14
  }
  const double rho = wi[0], a = std::sqrt(gamma * wi[4] / wi[0]), a2 = a * a;
  const double lm = wi[1] - a, l0 = wi[1], lp = wi[1] + a;                          // A8
  double sL[5] = {0, 0, 0, 0, 0}, sR[5] = {0, 0, 0, 0, 0};
  if (l0 < 0.0) {                                                                   // A17, contact term
    sL[0] += (lm - l0) * (dwi[0] - dwi[4] / a2);
    sL[2] += (lm - l0) * dwi[2];
    sL[3] += (lm - l0) * dwi[3];
  }
  if (lp < 0.0) {                                                                   // A17, right acoustic term
    sL[0] += 0.5 * (lm - lp) * (rho * dwi[1] / a + dwi[4] / a2);
    sL[1] += 0.5 * (lm - lp) * (dwi[1] + dwi[4] / (a * rho));
    sL[4] += 0.5 * (lm - lp) * (rho * dwi[1] * a + dwi[4]);
  }
  if (lm > 0.0) {                                                                   // A19, left acoustic term
    sR[0] += 0.5 * (lp - lm) * (-(rho * dwi[1] / a) + dwi[4] / a2);
    sR[1] += 0.5 * (lp - lm) * (dwi[1] - dwi[4] / (a * rho));
    sR[4] += 0.5 * (lp - lm) * (-(rho * dwi[1] * a) + dwi[4]);
  }
  if (l0 > 0.0) {                                                                   // A19, contact term (G10)
    sR[0] += (lp - l0) * (dwi[0] - dwi[4] / a2);
    sR[2] += (lp - l0) * dwi[2];
    sR[3] += (lp - l0) * dwi[3];
  }
  for (int m = 0; m < 5; ++m) {
    const double WLt = WL[m] - 0.5 * dtdx * std::min(lm, 0.0) * dwi[m];             // A15
    const double WRt = WR[m] - 0.5 * dtdx * std::max(lp, 0.0) * dwi[m];
    WLs[m] = WLt + 0.5 * dtdx * sL[m];                                              // A16
    WRs[m] = WRt + 0.5 * dtdx * sR[m];                                              // A18
  }
}

// PCM (Eq. 25-26): the face values are the cell average; no time evolution.
void pcm_cell(const double w[5][5], double WL[5], double WR[5], double WLs[5], double WRs[5]) {
  for (int m = 0; m < 5; ++m) WL[m] = WR[m] = WLs[m] = WRs[m] = w[2][m];
}

// ---------------------------------------------------------------------------------------------
// PPMP for one cell (A.4): parabolic reconstruction in the PRIMITIVE variables with contact
// steepening, shock flattening, monotonisation and characteristic tracing in Colella & Woodward's form.
// w[s] = primitive cell averages of cells i-3..i+3 (s = 0..6; cell i is w[3]), local order (rho, u_n, v, w, p).
// Readings: G12 A38 requires OPPOSITE curvature on the two sides of a contact; G13 A41's rho_R uses
// rho_{i+1}; G14 A48's third line assigns W_R; G15 A54's chi_L^p is the mirror image of chi_R^m; S19 the
// order in which A43-A45 are evaluated when p_{i+2} = p_{i-2}.
// ---------------------------------------------------------------------------------------------
// A2-A4 per primitive variable.
void prim_limited_slope(const double wm[5], const double w0[5], const double wp[5], double dw[5]) {
  for (int m = 0; m < 5; ++m) dw[m] = limit(w0[m] - wm[m], wp[m] - w0[m], 0.5 * (wp[m] - wm[m]));
}

// A42-A45: the flattening coefficient F~_j of cell j from p_{j-2..j+2} and u_{j-1}, u_{j+1}.
// A44 / A45 are tested first, so the quotient A42 is only formed where its numerator does not vanish (S19).
double flatten_tilde(const double pm2, const double pm1, const double pp1, const double pp2, const double um1,
                     const double up1) {
  if (std::fabs(pp1 - pm1) / std::min(pp1, pm1) < 1.0 / 3.0) return 0.0;   // A44
  if (up1 - um1 > 0.0) return 0.0;                                         // A45
  const double S = (pp1 - pm1) / (pp2 - pm2);                              // A42
  return std::max(0.0, std::min(1.0, 10.0 * (S - 0.75)));                  // A43
}

void ppmp_cell(double gamma, double dtdx, const double w[7][5], double WL[5], double WR[5], double WLs[5],
               double WRs[5]) {
  const double* wim = w[2];
  const double* wi = w[3];
  const double* wip = w[4];
  double dwm[5], dw0[5], dwp[5];
  prim_limited_slope(w[1], w[2], w[3], dwm);   // cell i-1
  prim_limited_slope(w[2], w[3], w[4], dw0);   // cell i
  prim_limited_slope(w[3], w[4], w[5], dwp);   // cell i+1
  // A34
  double L[5], R[5];
  for (int m = 0; m < 5; ++m) {
    L[m] = 0.5 * (wi[m] + wim[m]) - (dw0[m] - dwm[m]) / 6.0;
    R[m] = 0.5 * (wip[m] + wi[m]) - (dwp[m] - dw0[m]) / 6.0;
  }
  // A.4.2 contact steepening of the density faces
  {
    const double rm = wim[0], rp = wip[0], pm = wim[4], pp = wip[4];
    const double jump = std::fabs(rp - rm) / std::min(rp, rm);
    if (jump > 0.01 &&                                                         // A35
        std::fabs(pp - pm) / std::min(pp, pm) < 0.1 * gamma * jump) {          // A36
      // A37 with dx = 1 (dx^2 cancels in A39)
      const double d2m = (w[3][0] - 2.0 * w[2][0] + w[1][0]) / 6.0;            // delta^2 rho_{i-1}
      const double d2p = (w[5][0] - 2.0 * w[4][0] + w[3][0]) / 6.0;            // delta^2 rho_{i+1}
      if (d2m * d2p < 0.0) {                                                   // A38, reading G12
        const double eta_t = -(d2p - d2m) / (rp - rm);                         // A39
        const double eta = std::max(0.0, std::min(20.0 * eta_t - 1.0, 1.0));   // A40
        L[0] = L[0] * (1.0 - eta) + (rm + 0.5 * dwm[0]) * eta;                 // A41
        R[0] = R[0] * (1.0 - eta) + (rp - 0.5 * dwp[0]) * eta;                 // A41, reading G13
      }
    }
  }
  // A.4.3 shock flattening: F~ of cells i-1, i, i+1 along the sweep (normal velocity)
  {
    const double Fm = flatten_tilde(w[0][4], w[1][4], w[3][4], w[4][4], w[1][1], w[3][1]);   // cell i-1
    const double F0 = flatten_tilde(w[1][4], w[2][4], w[4][4], w[5][4], w[2][1], w[4][1]);   // cell i
    const double Fp = flatten_tilde(w[2][4], w[3][4], w[5][4], w[6][4], w[3][1], w[5][1]);   // cell i+1
    const double F = (wip[4] - wim[4] < 0.0) ? std::max(F0, Fp) : std::max(F0, Fm);          // A46
    for (int m = 0; m < 5; ++m) {                                                            // A47
      L[m] = F * wi[m] + (1.0 - F) * L[m];
      R[m] = F * wi[m] + (1.0 - F) * R[m];
    }
  }
  // A.4.4 monotonicity, A48 = A21 + A22 (third line read as W_R, G14; tests on the pair after A21, G8)
  double dwi[5], w6[5];
  for (int m = 0; m < 5; ++m) {
    double l = L[m], r = R[m];
    if ((r - wi[m]) * (wi[m] - l) <= 0.0) { l = wi[m]; r = wi[m]; }
    const bool fixL = (r - l) * (l - (3.0 * wi[m] - 2.0 * r)) < 0.0;
    const bool fixR = (r - l) * ((3.0 * wi[m] - 2.0 * l) - r) < 0.0;
    const double l0 = l, r0 = r;
    if (fixL) l = 3.0 * wi[m] - 2.0 * r0;
    if (fixR) r = 3.0 * wi[m] - 2.0 * l0;
    WL[m] = l; WR[m] = r;
    dwi[m] = r - l;                              // A50
    w6[m] = 6.0 * (wi[m] - 0.5 * (l + r));
  }
  // A49, A51
  const double a = std::sqrt(gamma * wi[4] / wi[0]);
  const double lm = wi[1] - a, l0c = wi[1], lp = wi[1] + a;
  const double am = dtdx * std::min(lm, 0.0), bm = dtdx * std::max(lm, 0.0);
  const double a0 = dtdx * std::min(l0c, 0.0), b0 = dtdx * std::max(l0c, 0.0);
  const double ap = dtdx * std::min(lp, 0.0), bp = dtdx * std::max(lp, 0.0);
  // A52
  double WLm[5], WL0[5], WLp[5], WRm[5], WR0[5], WRp[5];
  for (int m = 0; m < 5; ++m) {
    WLm[m] = WL[m] - 0.5 * am * (dwi[m] + w6[m] * (1.0 + (2.0 / 3.0) * am));
    WL0[m] = WL[m] - 0.5 * a0 * (dwi[m] + w6[m] * (1.0 + (2.0 / 3.0) * a0));
    WLp[m] = WL[m] - 0.5 * ap * (dwi[m] + w6[m] * (1.0 + (2.0 / 3.0) * ap));
    WRm[m] = WR[m] - 0.5 * bm * (dwi[m] - w6[m] * (1.0 - (2.0 / 3.0) * bm));
    WR0[m] = WR[m] - 0.5 * b0 * (dwi[m] - w6[m] * (1.0 - (2.0 / 3.0) * b0));
    WRp[m] = WR[m] - 0.5 * bp * (dwi[m] - w6[m] * (1.0 - (2.0 / 3.0) * bp));
  }
  // A53: sound speeds of the reference states; C = rho a of the reference state
  const double aL = std::sqrt(gamma * WLm[4] / WLm[0]), aR = std::sqrt(gamma * WRp[4] / WRp[0]);
  const double CL = WLm[0] * aL, CR = WRp[0] * aR;
  // A54, chi_L^p read as the mirror image of chi_R^m (G15); A55
  double chiLp = -1.0 / (2.0 * CL) * ((WLm[1] - WLp[1]) - (WLp[4] - WLm[4]) / CL);
  double chiRm = 1.0 / (2.0 * CR) * ((WRp[1] - WRm[1]) - (WRp[4] - WRm[4]) / CR);
  double chiL0 = (WLm[4] - WL0[4]) / (CL * CL) + 1.0 / WLm[0] - 1.0 / WL0[0];
  double chiR0 = (WRp[4] - WR0[4]) / (CR * CR) + 1.0 / WRp[0] - 1.0 / WR0[0];
  if (l0c > 0.0) chiL0 = 0.0;
  if (lp > 0.0) chiLp = 0.0;
  if (lm < 0.0) chiRm = 0.0;
  if (l0c < 0.0) chiR0 = 0.0;
  // A56
  WLs[0] = 1.0 / (1.0 / WLm[0] - chiL0 - chiLp);
  WRs[0] = 1.0 / (1.0 / WRp[0] - chiRm - chiR0);
  WLs[1] = WLm[1] + CL * chiLp;
  WRs[1] = WRp[1] - CR * chiRm;
  WLs[4] = WLm[4] + (CL * CL) * chiLp;
  WRs[4] = WRp[4] + (CR * CR) * chiRm;
  WLs[2] = WL0[2]; WRs[2] = WR0[2];
  WLs[3] = WL0[3]; WRs[3] = WR0[3];
}

// ---------------------------------------------------------------------------------------------
// PLMP for one cell (A.1): linear reconstruction with the slope limited in the primitive variables
// (A1-A4), evolved half a step with the fluxes of its own two face states in conserved form (A6, A7; Eq. 11).
// Uses cells i-1, i, i+1 of the 7-cell argument (w[2..4]).  WLs, WRs come back PRIMITIVE like the others.
// ---------------------------------------------------------------------------------------------
void euler_flux_local(double gamma, const double wv[5], double U[5], double F[5]) {   // Eq. 9, 11 in local order
  prim_to_cons(gamma, wv, U);
  F[0] = U[1];
  F[1] = U[1] * wv[1] + wv[4];
  F[2] = U[1] * wv[2];
  F[3] = U[1] * wv[3];
  F[4] = (U[4] + wv[4]) * wv[1];
}

void plmp_cell(double gamma, double dtdx, const double w[7][5], double WL[5], double WR[5], double WLs[5],
               double WRs[5]) {
  double dw[5];
  prim_limited_slope(w[2], w[3], w[4], dw);
  for (int m = 0; m < 5; ++m) { WL[m] = w[3][m] - 0.5 * dw[m]; WR[m] = w[3][m] + 0.5 * dw[m]; }   // A1
  double UL[5], UR[5], FL[5], FR[5], ULs[5], URs[5];
  euler_flux_local(gamma, WL, UL, FL);
  euler_flux_local(gamma, WR, UR, FR);
  for (int m = 0; m < 5; ++m) {
    ULs[m] = UL[m] + 0.5 * dtdx * (FL[m] - FR[m]);   // A6
    URs[m] = UR[m] + 0.5 * dtdx * (FL[m] - FR[m]);   // A7
  }
  cons_to_prim(gamma, ULs, WLs);
  cons_to_prim(gamma, URs, WRs);
}

// ---------------------------------------------------------------------------------------------
// Exact Riemann solver (B.1).  Inputs: primitive L/R states in local order
// (rho, u_n, v_t1, v_t2, p).  Output: flux in local order (B22) and diagnostics.
// ---------------------------------------------------------------------------------------------
struct RiemannDiag { double pm, um, rho, u, p; int iters; int region; };

// B5, B6
inline void pressure_function(double gamma, double p0, double rhok, double pk, double ak, double& f, double& fp) {
  if (p0 <= pk) {  // rarefaction
    const double pr = p0 / pk;
    f = 2.0 * ak / (gamma - 1.0) * (std::pow(pr, (gamma - 1.0) / (2.0 * gamma)) - 1.0);
    fp = 1.0 / (rhok * ak) * std::pow(pr, -(gamma + 1.0) / (2.0 * gamma));
  } else {  // shock
    const double A = 2.0 / ((gamma + 1.0) * rhok);       // B4
    const double B = (gamma - 1.0) / (gamma + 1.0) * pk;
    const double s = std::sqrt(A / (p0 + B));
    f = (p0 - pk) * s;
    fp = s * (1.0 - (p0 - pk) / (2.0 * (B + p0)));
  }
}

void riemann_exact(double gamma, const double WL[5], const double WR[5], double flux[5], RiemannDiag* diag) {
  const double rL = WL[0], uL = WL[1], pL = std::max(WL[4], P_FLOOR);
  const double rR = WR[0], uR = WR[1], pR = std::max(WR[4], P_FLOOR);
  const double aL = std::sqrt(gamma * pL / rL);  // B1
  const double aR = std::sqrt(gamma * pR / rR);

  // B2
  double pt = 0.5 * (pL + pR) + 0.125 * (uL - uR) * (rL + rR) * (aL + aR);
  if (pt < 0.0) pt = 0.0;
  // B3, B4
  const double gL = std::sqrt((2.0 / ((gamma + 1.0) * rL)) / (pt + (gamma - 1.0) / (gamma + 1.0) * pL));
  const double gR = std::sqrt((2.0 / ((gamma + 1.0) * rR)) / (pt + (gamma - 1.0) / (gamma + 1.0) * pR));
  double p0 = ((gL * pL + gR * pR) - (uR - uL)) / (gL + gR);
  if (p0 < P_GUESS_FLOOR) p0 = P_GUESS_FLOOR;

  // Newton-Raphson B5-B8
  double pm = p0, fL, fR, fpL, fpR;
  int it = 0;
  for (;;) {
    pressure_function(gamma, p0, rL, pL, aL, fL, fpL);
    pressure_function(gamma, p0, rR, pR, aR, fR, fpR);
    pm = p0 - ((fL + fR) + (uR - uL)) / (fpL + fpR);      // B7
    if (pm < P_FLOOR) pm = P_FLOOR;                        // reading S4
    ++it;
    const double delta = 2.0 * std::fabs(pm - p0) / std::fabs(pm + p0);  // B8
    if (!(delta > NEWTON_TOL) || it >= NEWTON_CAP) break;
    p0 = pm;
  }
  // B9 with f_k re-evaluated at the final p^m (reading S3)
  pressure_function(gamma, pm, rL, pL, aL, fL, fpL);
  pressure_function(gamma, pm, rR, pR, aR, fR, fpR);
  const double um = 0.5 * ((uL + uR) + (fR - fL));

  // Sampling at x/t = 0
  const double z = (gamma - 1.0) / (2.0 * gamma);
  const double gm = (gamma - 1.0) / (gamma + 1.0);
  double rho, u, p;
  int region;
  const double* Wk;
  if (um >= 0.0) {
    Wk = WL;
    if (pm <= pL) {  // left rarefaction
      if (uL - aL >= 0.0) { rho = rL; u = uL; p = pL; region = 0; }                      // B10
      else if (um - aL * std::pow(pm / pL, z) < 0.0) {                                  // B11
        rho = rL * std::pow(pm / pL, 1.0 / gamma); u = um; p = pm; region = 1;
      } else {                                                                          // B12
        const double a = 2.0 / (gamma + 1.0) * (aL + 0.5 * (gamma - 1.0) * uL);
        rho = rL * std::pow(a / aL, 2.0 / (gamma - 1.0));
        u = a;
        p = pL * std::pow(a / aL, 2.0 * gamma / (gamma - 1.0));
        region = 2;
      }
    } else {  // left shock
      const double sL = uL - aL * std::sqrt((gamma + 1.0) / (2.0 * gamma) * (pm / pL) + z);  // B13
      if (sL >= 0.0) { rho = rL; u = uL; p = pL; region = 3; }                            // B14
      else { rho = rL * (pm / pL + gm) / (pm / pL * gm + 1.0); u = um; p = pm; region = 4; }  // B15
    }
  } else {
    Wk = WR;
    if (pm <= pR) {  // right rarefaction
      if (uR + aR <= 0.0) { rho = rR; u = uR; p = pR; region = 5; }                      // B16
      else if (um + aR * std::pow(pm / pR, z) >= 0.0) {                                 // B17
        rho = rR * std::pow(pm / pR, 1.0 / gamma); u = um; p = pm; region = 6;
      } else {                                                                          // B18 (G4)
        const double a = 2.0 / (gamma + 1.0) * (aR - 0.5 * (gamma - 1.0) * uR);
        rho = rR * std::pow(a / aR, 2.0 / (gamma - 1.0));
        u = -a;
        p = pR * std::pow(a / aR, 2.0 * gamma / (gamma - 1.0));
        region = 7;
      }
    } else {  // right shock
      const double sR = uR + aR * std::sqrt((gamma + 1.0) / (2.0 * gamma) * (pm / pR) + z);  // B19 (G5)
      if (sR <= 0.0) { rho = rR; u = uR; p = pR; region = 8; }                            // B20
      else { rho = rR * (pm / pR + gm) / (pm / pR * gm + 1.0); u = um; p = pm; region = 9; }  // B21
    }
  }
  // B22; transverse velocities from side k (reading S9)
  const double vt1 = Wk[2], vt2 = Wk[3];
  const double E = p / (gamma - 1.0) + 0.5 * rho * ((u * u + vt1 * vt1) + vt2 * vt2);
  flux[0] = rho * u;
  flux[1] = rho * u * u + p;
  flux[2] = rho * u * vt1;
  flux[3] = rho * u * vt2;
  flux[4] = (E + p) * u;
  if (diag) { diag->pm = pm; diag->um = um; diag->rho = rho; diag->u = u; diag->p = p; diag->iters = it; diag->region = region; }
}

// ---------------------------------------------------------------------------------------------
// Roe solver with the HLLE failsafe (B.2), x-interface form in direction-local order
// (rho, u, v, w, p).  Step by step as printed; B29 read as NEXT-1/G9 in DESIGN.md:
// s1 = C0(u~ - a~) + C3 u~ + C4(u~ + a~), s3 = C0 w~ + C2 + C3 w~ + C4 w~,
// s4 = C0(H~ - u~ a~) + C1 v~ + C2 w~ + 0.5 C3 V~^2 + C4(H~ + u~ a~)
// (the printed "(u~ - u~)", "C3 2~" and "(H~ - u~ u~)" are the eigenvectors of B31-B32 garbled).
// path: 0 = F_L (supersonic to the right), 1 = F_R, 2 = Roe flux, 3 = HLLE flux.
// ---------------------------------------------------------------------------------------------
void flux_eq11(double gamma, const double W[5], double U[5], double F[5]) {   // Eq. 9, 11
  const double rho = W[0], u = W[1], v = W[2], w = W[3], p = W[4];
  const double E = p / (gamma - 1.0) + 0.5 * rho * ((u * u + v * v) + w * w);
  U[0] = rho; U[1] = rho * u; U[2] = rho * v; U[3] = rho * w; U[4] = E;
  F[0] = rho * u;
  F[1] = rho * u * u + p;
  F[2] = rho * u * v;
  F[3] = rho * u * w;
  F[4] = (E + p) * u;
}

void riemann_roe(double gamma, const double WL[5], const double WR[5], double flux[5], int* path, double etaH = 0.0) {
  double UL[5], UR[5], FL[5], FR[5];
  flux_eq11(gamma, WL, UL, FL);
  flux_eq11(gamma, WR, UR, FR);
  // B23
  const double sl = std::sqrt(WL[0]), sr = std::sqrt(WR[0]);
  const double HL = (UL[4] + WL[4]) / WL[0], HR = (UR[4] + WR[4]) / WR[0];
  const double ut = (sl * WL[1] + sr * WR[1]) / (sl + sr);
  const double vt = (sl * WL[2] + sr * WR[2]) / (sl + sr);
  const double wt = (sl * WL[3] + sr * WR[3]) / (sl + sr);
  const double Ht = (sl * HL + sr * HR) / (sl + sr);
  const double V2 = (ut * ut + vt * vt) + wt * wt;
  const double at = std::sqrt((gamma - 1.0) * (Ht - 0.5 * V2));          // B24
  const double lm = ut - at, l0 = ut, lp = ut + at;                        // B25
  if (lm >= 0.0) { for (int m = 0; m < 5; ++m) flux[m] = FL[m]; if (path) *path = 0; return; }
  if (lp <= 0.0) { for (int m = 0; m < 5; ++m) flux[m] = FR[m]; if (path) *path = 1; return; }
  // B26
  double dU[5];
  for (int m = 0; m < 5; ++m) dU[m] = UR[m] - UL[m];
  // B27
  const double Na = 1.0 / (2.0 * at * at), gp = gamma - 1.0, ia2 = 1.0 / (at * at);
  double xi[5];
  xi[0] = dU[0] * Na * (0.5 * gp * V2 + ut * at) - dU[1] * Na * (gp * ut + at) - dU[2] * Na * gp * vt -
          dU[3] * Na * gp * wt + dU[4] * Na * gp;
  xi[1] = -dU[0] * vt + dU[2];
  xi[2] = -dU[0] * wt + dU[3];
  xi[3] = dU[0] * (1.0 - Na * gp * V2) + dU[1] * gp * ut * ia2 + dU[2] * gp * vt * ia2 + dU[3] * gp * wt * ia2 -
          dU[4] * gp * ia2;
  xi[4] = dU[0] * Na * (0.5 * gp * V2 - ut * at) - dU[1] * Na * (gp * ut - at) - dU[2] * Na * gp * vt -
          dU[3] * Na * gp * wt + dU[4] * Na * gp;
  // B28
  // C3: with the H correction |lambda| -> max(|lambda|, eta^H) here and only here (reading S18)
  const double alm = std::max(std::fabs(lm), etaH), al0 = std::max(std::fabs(l0), etaH), alp = std::max(std::fabs(lp), etaH);
  const double C0 = xi[0] * alm, C1 = xi[1] * al0, C2 = xi[2] * al0, C3 = xi[3] * al0, C4 = xi[4] * alp;
  // B29
  double sv[5];
  sv[0] = C0 + C3 + C4;
  sv[1] = C0 * (ut - at) + C3 * ut + C4 * (ut + at);
  sv[2] = C0 * vt + C1 + C3 * vt + C4 * vt;
  sv[3] = C0 * wt + C2 + C3 * wt + C4 * wt;
  sv[4] = C0 * (Ht - ut * at) + C1 * vt + C2 * wt + 0.5 * C3 * V2 + C4 * (Ht + ut * at);
  // B31, B32: intermediate states; negative density or pressure -> HLLE
  bool hlle = false;
  double Um[5];
  Um[0] = UL[0] + xi[0];
  Um[1] = UL[1] + xi[0] * (ut - at);
  Um[2] = UL[2] + xi[0] * vt;
  Um[3] = UL[3] + xi[0] * wt;
  Um[4] = UL[4] + xi[0] * (Ht - ut * at);
  auto pressure = [&](const double* U) { return (gamma - 1.0) * (U[4] - 0.5 * ((U[1] * U[1] + U[2] * U[2]) + U[3] * U[3]) / U[0]); };
  if (l0 > lm) { if (!(Um[0] > 0.0) || !(pressure(Um) > 0.0)) hlle = true; }
  Um[0] += xi[3];
  Um[1] += xi[3] * ut;
  Um[2] += xi[1] + xi[3] * vt;
  Um[3] += xi[2] + xi[3] * wt;
  Um[4] += xi[1] * vt + xi[2] * wt + 0.5 * xi[3] * V2;
  if (lp > l0) { if (!(Um[0] > 0.0) || !(pressure(Um) > 0.0)) hlle = true; }
  if (!hlle) {
    for (int m = 0; m < 5; ++m) flux[m] = 0.5 * ((FL[m] + FR[m]) - sv[m]);   // B30
    if (path) *path = 2;
    return;
  }
  // HLLE (B33-B35)
  const double aL = std::sqrt(gamma * WL[4] / WL[0]), aR = std::sqrt(gamma * WR[4] / WR[0]);
  const double bm = std::min(std::min(lm, WL[1] - aL), 0.0), bp = std::max(std::max(lp, WR[1] + aR), 0.0);
  const double t = (bp + bm) / (bp - bm);
  for (int m = 0; m < 5; ++m) {
    const double fl = FL[m] - bm * UL[m], fr = FR[m] - bp * UR[m];       // B34
    flux[m] = 0.5 * ((fl + fr) + (fl - fr) * t);                          // B35
  }
  if (path) *path = 3;
}

// Riemann problem at an interface normal to d from two conserved states in GLOBAL order.
void riemann_interface(double gamma, int solver, int d, const double UL[5], const double UR[5], double F[5], double etaH = 0.0) {
  double wl[5], wr[5], ll[5], lr[5], fl[5];
  cons_to_prim(gamma, UL, wl);
  cons_to_prim(gamma, UR, wr);
  to_local(d, wl, ll);
  to_local(d, wr, lr);
  if (solver == SOLVER_ROE) riemann_roe(gamma, ll, lr, fl, nullptr, etaH);
  else riemann_exact(gamma, ll, lr, fl, nullptr);
  to_global(d, fl, F);
}

// ---------------------------------------------------------------------------------------------
// Grid context.
// ---------------------------------------------------------------------------------------------
struct Ctx {
  int n[3], g, gd[3], pd[3];
  long np;
  double gamma, dx[3];
  int bc[6];
  bool active[3];
  bool have_state = false;
  int solver = SOLVER_EXACT;
  int recon = RECON_PPMC;
  bool hcorr = false;   // H correction (Appendix C): Roe solver only, second Riemann pass only, needs g >= 4
  double time = 0.0;    // sum of the dt of all steps since set_state / ref_set_time: the t of the Noh boundary
  double noh_rho0 = 1.0, noh_p0 = 1e-6;
  std::vector<double> u;  // [5][np], x fastest
  inline long idx(int i, int j, int k) const {  // real-cell coordinates, ghosts negative / >= n
    return ((long)(k + gd[2]) * pd[1] + (j + gd[1])) * pd[0] + (i + gd[0]);
  }
};

// Ghost fill (readings S6, S7): x over real (y,z); y over the padded x extent; z over
// padded x,y — the ordering that carries edges and corners.
void ghost_fill(Ctx& c) {
  for (int d = 0; d < 3; ++d) {
    if (!c.active[d]) continue;
    int lo[3], hi[3];
    for (int e = 0; e < 3; ++e) {
      if (e < d) { lo[e] = -c.gd[e]; hi[e] = c.n[e] + c.gd[e]; }   // already-filled padded extent
      else if (e > d) { lo[e] = 0; hi[e] = c.n[e]; }               // real cells only
      else { lo[e] = 0; hi[e] = 1; }                               // placeholder for the fill dim
    }
    const int n = c.n[d], g = c.g;
    for (int side = 0; side < 2; ++side) {
      const int bc = c.bc[2 * d + side];
      for (int l = 1; l <= g; ++l) {
        int gi, si;  // ghost index and its source index along d
        if (side == 0) {
          gi = -l;
          si = bc == BC_PERIODIC ? n - l : bc == BC_REFLECTIVE ? l - 1 : 0;
        } else {
          gi = n - 1 + l;
          si = bc == BC_PERIODIC ? l - 1 : bc == BC_REFLECTIVE ? n - l : n - 1;
        }
        if (bc == BC_NOH) {
          // Analytic boundary of the Noh test: rho = rho0 (1 + t/r)^(n-1), |V| = 1 toward the
          // origin, E = p0/(gamma-1) + rho/2, at the centre of the ghost cell; box origin at x = y = z = 0,
          // n = number of active dimensions, r over the active dimensions.
          int nact = 0;
          for (int e = 0; e < 3; ++e) nact += c.active[e] ? 1 : 0;
          int a[3];
          for (a[2] = lo[2]; a[2] < hi[2]; ++a[2])
            for (a[1] = lo[1]; a[1] < hi[1]; ++a[1])
              for (a[0] = lo[0]; a[0] < hi[0]; ++a[0]) {
                int gq[3] = {a[0], a[1], a[2]};
                gq[d] = gi;
                double x[3], r2 = 0.0;
                for (int e = 0; e < 3; ++e) {
                  x[e] = c.active[e] ? (gq[e] + 0.5) * c.dx[e] : 0.0;
                  r2 += x[e] * x[e];
                }
                const double r = std::sqrt(r2);
                const double q1 = 1.0 + c.time / r;
                double rho = c.noh_rho0;
                for (int e = 1; e < nact; ++e) rho *= q1;
                const long ig = c.idx(gq[0], gq[1], gq[2]);
                c.u[0 * c.np + ig] = rho;
                for (int e = 0; e < 3; ++e) c.u[(1 + e) * c.np + ig] = rho * (-(x[e] / r));
                c.u[4 * c.np + ig] = c.noh_p0 / (c.gamma - 1.0) + 0.5 * rho;
              }
          continue;
        }
        int a[3];
        for (a[2] = lo[2]; a[2] < hi[2]; ++a[2])
          for (a[1] = lo[1]; a[1] < hi[1]; ++a[1])
            for (a[0] = lo[0]; a[0] < hi[0]; ++a[0]) {
              int gq[3] = {a[0], a[1], a[2]}, sq[3] = {a[0], a[1], a[2]};
              gq[d] = gi; sq[d] = si;
              const long ig = c.idx(gq[0], gq[1], gq[2]);
              const long is = c.idx(sq[0], sq[1], sq[2]);
              for (int f = 0; f < 5; ++f) {
                double v = c.u[f * c.np + is];
                if (bc == BC_REFLECTIVE && f == 1 + d) v = -v;
                c.u[f * c.np + ig] = v;
              }
            }
      }
    }
  }
}

// Eq. 22 over real cells; returns C0 * min.  NaN if any cell is non-physical.
double compute_dt(const Ctx& c, double cfl) {
  double dtmin = std::numeric_limits<double>::infinity();
  bool bad = false;
  for (int k = 0; k < c.n[2]; ++k)
    for (int j = 0; j < c.n[1]; ++j)
      for (int i = 0; i < c.n[0]; ++i) {
        const long q = c.idx(i, j, k);
        double uc[5], w[5];
        for (int f = 0; f < 5; ++f) uc[f] = c.u[f * c.np + q];
        if (!(uc[0] > 0.0) || !std::isfinite(uc[0]) || !std::isfinite(uc[4])) { bad = true; continue; }
        cons_to_prim(c.gamma, uc, w);
        const double a = std::sqrt(c.gamma * w[4] / w[0]);  // Eq. 21
        for (int d = 0; d < 3; ++d) {
          if (!c.active[d]) continue;
          const double t = c.dx[d] / (std::fabs(w[1 + d]) + a);
          if (!(t == t)) bad = true;
          if (t < dtmin) dtmin = t;
        }
      }
  if (bad) return std::numeric_limits<double>::quiet_NaN();
  return cfl * dtmin;
}

// One CTU step: steps 1-5 on whole-grid arrays, then the ghost fill.
void ctu_step(Ctx& c, double dt) {
  const long np = c.np;
  const double gamma = c.gamma;
  const int g = c.g;
  (void)g;
  // O1: primitives of every padded cell.
  std::vector<double> w(5 * np);
#pragma omp parallel for
  for (long q = 0; q < np; ++q) {
    double uc[5], wc[5];
    for (int f = 0; f < 5; ++f) uc[f] = c.u[f * np + q];
    cons_to_prim(gamma, uc, wc);
    for (int f = 0; f < 5; ++f) w[f * np + q] = wc[f];
  }

  // extents helpers: along the sweep dim [-1, n]; other active dims [-t, n+t) ; inactive [0,1)
  auto range = [&](int e, int ext, int& lo, int& hi) {
    if (!c.active[e]) { lo = 0; hi = 1; } else { lo = -ext; hi = c.n[e] + ext; }
  };
  const long stride[3] = {1, c.pd[0], (long)c.pd[0] * c.pd[1]};

  // With the H correction the second-pass states are also needed one cell further out in the transverse
  // directions (eta of the neighbouring interfaces, C2), hence F* one interface further out along its own
  // direction, hence U* one cell further out: "an extra ghost cell on each side".
  const int X = c.hcorr ? 2 : 1;
  // Step 1: U*_L, U*_R per direction (conserved, global order) — O2.
  std::vector<double> UsL[3], UsR[3], Fs[3], UhL[3], UhR[3], Fh[3], eta[3];
  for (int d = 0; d < 3; ++d) {
    if (!c.active[d]) continue;
    UsL[d].assign(5 * np, 0.0);
    UsR[d].assign(5 * np, 0.0);
    int lo[3], hi[3];
    for (int e = 0; e < 3; ++e) range(e, X, lo[e], hi[e]);
    const double dtdx = dt / c.dx[d];
#pragma omp parallel for collapse(2)
    for (int k = lo[2]; k < hi[2]; ++k)
      for (int j = lo[1]; j < hi[1]; ++j)
        for (int i = lo[0]; i < hi[0]; ++i) {
          const long q = c.idx(i, j, k);
          double ws[5][5], w7[7][5];
          for (int s = 0; s < 5; ++s) {
            const long qs = q + (s - 2) * stride[d];
            double wg[5];
            for (int f = 0; f < 5; ++f) wg[f] = w[f * np + qs];
            to_local(d, wg, ws[s]);
          }
          const bool wide = c.recon == RECON_PPMP || c.recon == RECON_PLMP;   // 7-cell stencil: g >= 4
          if (wide)
            for (int s = 0; s < 7; ++s) {
              if (c.recon == RECON_PLMP && (s < 2 || s > 4)) {   // PLMP reads cells i-1..i+1 only (g = 3 suffices)
                for (int f = 0; f < 5; ++f) w7[s][f] = 0.0;
                continue;
              }
              const long qs = q + (s - 3) * stride[d];
              double wg[5];
              for (int f = 0; f < 5; ++f) wg[f] = w[f * np + qs];
              to_local(d, wg, w7[s]);
            }
          double WL[5], WR[5], WLs[5], WRs[5], gl[5], gr[5], ul[5], ur[5];
          if (c.recon == RECON_PPMP) ppmp_cell(gamma, dtdx, w7, WL, WR, WLs, WRs);
          else if (c.recon == RECON_PLMP) plmp_cell(gamma, dtdx, w7, WL, WR, WLs, WRs);
          else if (c.recon == RECON_PLMC) plmc_cell(gamma, dtdx, ws, WL, WR, WLs, WRs);
          else if (c.recon == RECON_PCM) pcm_cell(ws, WL, WR, WLs, WRs);
          else ppmc_cell(gamma, dtdx, ws, WL, WR, WLs, WRs);
          to_global(d, WLs, gl);
          to_global(d, WRs, gr);
          prim_to_cons(gamma, gl, ul);
          prim_to_cons(gamma, gr, ur);
          for (int f = 0; f < 5; ++f) { UsL[d][f * np + q] = ul[f]; UsR[d][f * np + q] = ur[f]; }
        }
  }
  // Step 2: F*_d at interface c+1/2 stored at cell index c — O3.  L state = right face of cell
  // c, R state = left face of cell c+1.
  for (int d = 0; d < 3; ++d) {
    if (!c.active[d]) continue;
    Fs[d].assign(5 * np, 0.0);
    int lo[3], hi[3];
    for (int e = 0; e < 3; ++e) range(e, X, lo[e], hi[e]);
    hi[d] -= 1;  // interfaces c in [-X, n+X-2]
#pragma omp parallel for collapse(2)
    for (int k = lo[2]; k < hi[2]; ++k)
      for (int j = lo[1]; j < hi[1]; ++j)
        for (int i = lo[0]; i < hi[0]; ++i) {
          const long q = c.idx(i, j, k), qp = q + stride[d];
          double UL[5], UR[5], F[5];
          for (int f = 0; f < 5; ++f) { UL[f] = UsR[d][f * np + q]; UR[f] = UsL[d][f * np + qp]; }
          riemann_interface(gamma, c.solver, d, UL, UR, F);
          for (int f = 0; f < 5; ++f) Fs[d][f * np + q] = F[f];
        }
  }
  // Step 3: transverse half-step, Eq. 23 — O4.
  for (int d = 0; d < 3; ++d) {
    if (!c.active[d]) continue;
    UhL[d].assign(5 * np, 0.0);
    UhR[d].assign(5 * np, 0.0);
    int lo[3], hi[3];
    for (int e = 0; e < 3; ++e) range(e, (e == d || c.hcorr) ? 1 : 0, lo[e], hi[e]);
#pragma omp parallel for collapse(2)
    for (int k = lo[2]; k < hi[2]; ++k)
      for (int j = lo[1]; j < hi[1]; ++j)
        for (int i = lo[0]; i < hi[0]; ++i) {
          const long q = c.idx(i, j, k);
          for (int f = 0; f < 5; ++f) {
            double corr = 0.0;
            for (int t = 1; t <= 2; ++t) {  // cyclic: d+1 then d+2
              const int e = (d + t) % 3;
              if (!c.active[e]) continue;
              corr += 0.5 * (dt / c.dx[e]) * (Fs[e][f * np + q - stride[e]] - Fs[e][f * np + q]);
            }
            UhL[d][f * np + q] = UsL[d][f * np + q] + corr;
            UhR[d][f * np + q] = UsR[d][f * np + q] + corr;
          }
        }
  }
  // Step 3b (H correction, C1 P:L1281): eta = |(u_R + a_R) - (u_L + a_L)| / 2 at every interface from the
  // second-pass input states, normal velocity and sound speed of each side.
  if (c.hcorr) {
    for (int d = 0; d < 3; ++d) {
      if (!c.active[d]) continue;
      eta[d].assign(np, 0.0);
      int lo[3], hi[3];
      for (int e = 0; e < 3; ++e) range(e, 1, lo[e], hi[e]);
      hi[d] -= 1;
#pragma omp parallel for collapse(2)
      for (int k = lo[2]; k < hi[2]; ++k)
        for (int j = lo[1]; j < hi[1]; ++j)
          for (int i = lo[0]; i < hi[0]; ++i) {
            const long q = c.idx(i, j, k), qp = q + stride[d];
            double UL[5], UR[5], wl[5], wr[5];
            for (int f = 0; f < 5; ++f) { UL[f] = UhR[d][f * np + q]; UR[f] = UhL[d][f * np + qp]; }
            cons_to_prim(gamma, UL, wl);
            cons_to_prim(gamma, UR, wr);
            const double aL = std::sqrt(gamma * wl[4] / wl[0]), aR = std::sqrt(gamma * wr[4] / wr[0]);
            eta[d][q] = 0.5 * std::fabs((wr[1 + d] + aR) - (wl[1 + d] + aL));
          }
    }
  }
  // Step 4: CTU fluxes — O5.
  for (int d = 0; d < 3; ++d) {
    if (!c.active[d]) continue;
    Fh[d].assign(5 * np, 0.0);
    int lo[3], hi[3];
    for (int e = 0; e < 3; ++e) range(e, e == d ? 1 : 0, lo[e], hi[e]);
    hi[d] -= 1;
#pragma omp parallel for collapse(2)
    for (int k = lo[2]; k < hi[2]; ++k)
      for (int j = lo[1]; j < hi[1]; ++j)
        for (int i = lo[0]; i < hi[0]; ++i) {
          const long q = c.idx(i, j, k), qp = q + stride[d];
          double UL[5], UR[5], F[5];
          for (int f = 0; f < 5; ++f) { UL[f] = UhR[d][f * np + q]; UR[f] = UhL[d][f * np + qp]; }
          double etaH = 0.0;
          if (c.hcorr) {
            // C2 read with the cells that share the interface (reading G11): the interface's own eta
            // and, for each transverse direction, eta on the two faces of cell c and of cell c+1
            etaH = eta[d][q];
            for (int e = 0; e < 3; ++e) {
              if (e == d || !c.active[e]) continue;
              etaH = std::max(etaH, std::max(std::max(eta[e][q - stride[e]], eta[e][q]),
                                             std::max(eta[e][qp - stride[e]], eta[e][qp])));
            }
          }
          riemann_interface(gamma, c.solver, d, UL, UR, F, etaH);
          for (int f = 0; f < 5; ++f) Fh[d][f * np + q] = F[f];
        }
  }
  // Step 5: conservative update, Eq. 24 on real cells — O6.
#pragma omp parallel for collapse(2)
  for (int k = 0; k < c.n[2]; ++k)
    for (int j = 0; j < c.n[1]; ++j)
      for (int i = 0; i < c.n[0]; ++i) {
        const long q = c.idx(i, j, k);
        for (int f = 0; f < 5; ++f) {
          double v = c.u[f * np + q];
          for (int d = 0; d < 3; ++d) {
            if (!c.active[d]) continue;
            v += (dt / c.dx[d]) * (Fh[d][f * np + q - stride[d]] - Fh[d][f * np + q]);
          }
          c.u[f * np + q] = v;
        }
      }
  c.time += dt;   // the analytic (Noh) boundary is evaluated at t^{n+1}
  ghost_fill(c);  // O7
}

int fail(const char* msg) { g_err = msg; return -1; }

}  // namespace

// =============================================================================================
// C ABI (prefix ref_): mirrors include/ch.h so one Python harness drives both, plus unit-level
// entry points used by the pins.
// =============================================================================================
extern "C" {

const char* ref_last_error(void) { return g_err.c_str(); }

void* ref_init(int nx, int ny, int nz, int nghost, double gamma, const int* bc) {
  if (nx < 1 || ny < 1 || nz < 1) { fail("n < 1"); return nullptr; }
  if (nghost < 3) { fail("nghost < 3"); return nullptr; }
  if (!(gamma > 1.0)) { fail("gamma <= 1"); return nullptr; }
  Ctx* c = new (std::nothrow) Ctx();
  if (!c) { fail("alloc"); return nullptr; }
  c->n[0] = nx; c->n[1] = ny; c->n[2] = nz;
  c->g = nghost; c->gamma = gamma;
  for (int d = 0; d < 3; ++d) {
    c->active[d] = c->n[d] > 1;
    c->gd[d] = c->active[d] ? nghost : 0;
    c->pd[d] = c->n[d] + 2 * c->gd[d];
    c->dx[d] = 1.0 / nx;  // reading S8
    if (c->active[d] && c->n[d] < nghost) { delete c; fail("active dim smaller than nghost"); return nullptr; }
  }
  for (int s = 0; s < 6; ++s) {
    c->bc[s] = bc ? bc[s] : BC_PERIODIC;
    if (c->active[s / 2] && (c->bc[s] < 1 || c->bc[s] > 4)) { delete c; fail("bad bc"); return nullptr; }
  }
  for (int d = 0; d < 3; ++d)
    if (c->active[d] && ((c->bc[2 * d] == BC_PERIODIC) != (c->bc[2 * d + 1] == BC_PERIODIC))) {
      delete c; fail("unpaired periodic"); return nullptr;
    }
  c->np = (long)c->pd[0] * c->pd[1] * c->pd[2];
  c->u.assign(5 * c->np, 0.0);
  return c;
}

int ref_free(void* h) { delete static_cast<Ctx*>(h); return 0; }

int ref_set_spacing(void* h, double dx, double dy, double dz) {
  Ctx* c = static_cast<Ctx*>(h);
  if (!(dx > 0 && dy > 0 && dz > 0)) return fail("spacing <= 0");
  c->dx[0] = dx; c->dx[1] = dy; c->dx[2] = dz;
  return 0;
}

long ref_padded_cells(void* h) { return static_cast<Ctx*>(h)->np; }

// u = [5][nz][ny][nx] real cells only; copies in and fills the ghosts.
int ref_set_state(void* h, const double* u) {
  Ctx* c = static_cast<Ctx*>(h);
  const long n = (long)c->n[0] * c->n[1] * c->n[2];
  for (int f = 0; f < 5; ++f)
    for (int k = 0; k < c->n[2]; ++k)
      for (int j = 0; j < c->n[1]; ++j)
        for (int i = 0; i < c->n[0]; ++i)
          c->u[f * c->np + c->idx(i, j, k)] = u[f * n + ((long)k * c->n[1] + j) * c->n[0] + i];
  c->time = 0.0;
  ghost_fill(*c);
  c->have_state = true;
  return 0;
}

// Noh test boundary: ambient density and pressure of the analytic inflow; ref_set_time sets the t it
// is evaluated at (set_state resets it to 0, every step adds its dt).
int ref_set_noh(void* h, double rho0, double p0) {
  Ctx* c = static_cast<Ctx*>(h);
  if (!(rho0 > 0.0) || !(p0 > 0.0)) return fail("ref_set_noh: rho0, p0 must be positive");
  c->noh_rho0 = rho0; c->noh_p0 = p0;
  return 0;
}
int ref_set_time(void* h, double t) { static_cast<Ctx*>(h)->time = t; return 0; }
double ref_get_time(void* h) { return static_cast<Ctx*>(h)->time; }
int ref_fill_ghosts(void* h) { ghost_fill(*static_cast<Ctx*>(h)); return 0; }

int ref_get_state(void* h, double* u) {
  Ctx* c = static_cast<Ctx*>(h);
  if (!c->have_state) return fail("no state");
  const long n = (long)c->n[0] * c->n[1] * c->n[2];
  for (int f = 0; f < 5; ++f)
    for (int k = 0; k < c->n[2]; ++k)
      for (int j = 0; j < c->n[1]; ++j)
        for (int i = 0; i < c->n[0]; ++i)
          u[f * n + ((long)k * c->n[1] + j) * c->n[0] + i] = c->u[f * c->np + c->idx(i, j, k)];
  return 0;
}

// Padded store [5][pz][py][px] as is (ghosts included, not refilled): used to run the step on a
// sub-box cut out of a larger grid (sampled parity at full size) and to test the ghost fill.
int ref_set_padded(void* h, const double* up) {
  Ctx* c = static_cast<Ctx*>(h);
  std::memcpy(c->u.data(), up, sizeof(double) * 5 * c->np);
  c->have_state = true;
  return 0;
}
int ref_get_padded(void* h, double* up) {
  Ctx* c = static_cast<Ctx*>(h);
  std::memcpy(up, c->u.data(), sizeof(double) * 5 * c->np);
  return 0;
}

double ref_compute_dt(void* h, double cfl) {
  Ctx* c = static_cast<Ctx*>(h);
  if (!c->have_state) { fail("no state"); return std::numeric_limits<double>::quiet_NaN(); }
  return compute_dt(*c, cfl);
}

int ref_step(void* h, double dt) {
  Ctx* c = static_cast<Ctx*>(h);
  if (!c->have_state) return fail("no state");
  if (!(dt > 0.0) || !std::isfinite(dt)) return fail("bad dt");
  if (c->hcorr && c->solver != SOLVER_ROE) return fail("the H correction goes with the Roe solver (P:L1279)");
  ctu_step(*c, dt);
  return 0;
}

// ---- unit-level entry points for the pins (all primitive, direction-local order) -------------
void ref_cons_to_prim(double gamma, const double* u, double* w) { cons_to_prim(gamma, u, w); }
void ref_prim_to_cons(double gamma, const double* w, double* u) { prim_to_cons(gamma, w, u); }
void ref_char_project(double rho, double a, const double* dw, double* dxi) { char_project(rho, a, dw, dxi); }
void ref_char_backproject(double rho, double a, const double* dxi, double* dw) { char_backproject(rho, a, dxi, dw); }
void ref_limited_slope(double gamma, const double* wm, const double* w0, const double* wp, double* dw) {
  limited_slope(gamma, wm, w0, wp, dw);
}
// w = [5 cells][5 comps]; out = [4][5] = WL, WR, W*_L, W*_R
void ref_ppmc_cell(double gamma, double dtdx, const double* w, double* out) {
  double ws[5][5];
  std::memcpy(ws, w, sizeof(ws));
  ppmc_cell(gamma, dtdx, ws, out, out + 5, out + 10, out + 15);
}
// WL, WR primitive; flux[5]; diag[7] = pm, um, rho, u, p, iterations, region
int ref_set_solver(void* h, int solver) {
  if (!h || (solver != SOLVER_EXACT && solver != SOLVER_ROE)) return fail("ref_set_solver: bad argument");
  static_cast<Ctx*>(h)->solver = solver;
  return 0;
}
int ref_set_reconstruction(void* h, int recon) {
  if (!h || recon < RECON_PPMC || recon > RECON_PLMP) return fail("ref_set_reconstruction: bad argument");
  if (recon == RECON_PPMP && static_cast<Ctx*>(h)->g < 4) return fail("ref_set_reconstruction: PPMP needs nghost >= 4 (P:L962)");
  if (recon == RECON_PPMP && static_cast<Ctx*>(h)->hcorr) return fail("ref_set_reconstruction: the H correction goes with PPMC or lower order (P:L565)");
  static_cast<Ctx*>(h)->recon = recon;
  return 0;
}
// w = [7 cells][5 comps] (cells i-3..i+3); out = [4][5] = WL, WR, W*_L, W*_R
void ref_ppmp_cell(double gamma, double dtdx, const double* w, double* out) {
  double ws[7][5];
  std::memcpy(ws, w, sizeof(ws));
  ppmp_cell(gamma, dtdx, ws, out, out + 5, out + 10, out + 15);
}
void ref_plmp_cell(double gamma, double dtdx, const double* w, double* out) {
  double ws[7][5];
  std::memcpy(ws, w, sizeof(ws));
  plmp_cell(gamma, dtdx, ws, out, out + 5, out + 10, out + 15);
}
void ref_plmc_cell(double gamma, double dtdx, const double* w, double* out) {
  double ws[5][5];
  for (int s = 0; s < 5; ++s) for (int m = 0; m < 5; ++m) ws[s][m] = w[s * 5 + m];
  plmc_cell(gamma, dtdx, ws, out, out + 5, out + 10, out + 15);
}
int ref_set_hcorrection(void* h, int on) {
  if (!h) return fail("ref_set_hcorrection: null");
  Ctx& c = *static_cast<Ctx*>(h);
  if (on && c.g < 4) return fail("ref_set_hcorrection: needs nghost >= 4 (P:L1291)");
  if (on && c.recon == RECON_PPMP) return fail("ref_set_hcorrection: only with PPMC or lower-order reconstructions (P:L565)");
  c.hcorr = on != 0;
  return 0;
}
int ref_riemann_roe_eta(double gamma, const double* WL, const double* WR, double etaH, double* flux) {
  int path = -1;
  riemann_roe(gamma, WL, WR, flux, &path, etaH);
  return path;
}
int ref_riemann_roe(double gamma, const double* WL, const double* WR, double* flux) {
  int path = -1;
  riemann_roe(gamma, WL, WR, flux, &path);
  return path;
}
void ref_riemann_exact(double gamma, const double* WL, const double* WR, double* flux, double* diag) {
  RiemannDiag d;
  riemann_exact(gamma, WL, WR, flux, &d);
  if (diag) { diag[0] = d.pm; diag[1] = d.um; diag[2] = d.rho; diag[3] = d.u; diag[4] = d.p; diag[5] = d.iters; diag[6] = d.region; }
}

}  // extern "C"
