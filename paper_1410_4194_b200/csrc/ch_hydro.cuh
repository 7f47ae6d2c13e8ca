// ch_hydro.cuh — per-cell / per-interface device arithmetic of the CTU step (fp64).
//
// Written from the text of arXiv:1410.4194 (citations `P:L<line>` = /root/reference/PAPER.md line);
// "G<n>/S<n>" are the readings of garbled / silent passages listed in DESIGN.md.  This file shares
// nothing with oracle/: it restates the same equations in a form chosen for the B200 FP64 pipe
// (DESIGN.md §4 "Arithmetic restatements"):
//   * reciprocals and reciprocal square roots are MUFU seeds refined by one cubic Newton step in DFMA
//     (<= 2e-16 relative, measured), with no slow-path branches (every operand is a normal positive double);
//   * one rsqrt(gamma p rho) per cell yields a, 1/a, rho/a, 1/a^2, a/rho by multiplication;
//   * (p/p_k)^z is a 13-term binomial series when |p/p_k - 1| <= 1/16 (smooth flow) and
//     exp(z log(.)) otherwise; (p/p_k)^{1/gamma} = pr / (pr^z)^2;
//   * min / max / clamp are compare-selects (no NaN-propagating fmin/fmax emulation);
//   * B9 and the sampling take f_k, (p/p_k)^z at the converged pressure by a first-order update
//     from the last Newton iterate (error O(tol^2) = 1e-16) instead of a fresh evaluation;
//   * the ten-way sampling is folded onto the left wave family by mirroring when u^m < 0;
//   * PPMC's parabola edges are limited through their deviations from the cell average (A21-A23 are clamps of
//     dR = R - w and dL = w - L; A24 and A26 follow without the cancellation of 6[w - (L + R)/2]), sign tests read the
//     high words, and the centred slope's characteristic components are the mean of the one-sided ones.
//
// All functions work in the direction-local ordering (rho, v_n, v_t1, v_t2, p).
#pragma once

#include <math.h>

#define CH_D __device__ __forceinline__

namespace ch {

constexpr double kPFloor = 1e-20;
constexpr double kPGuessFloor = 1e-6;
constexpr double kNewtonTol = 1e-8;     // P:L1095 "e.g. 1e-6"; reading S2
constexpr int kNewtonCap = 20;          // reading S2
constexpr int kPowTerms = 13;           // binomial series length for (1+t)^z, |t| <= kPowRadius
constexpr double kPowRadius = 1.0 / 16.0;
constexpr int kPowTermsShort = 6;       // ... and for |t| <= kPowRadiusShort (truncation C(z,7) t^7 / (z t) < 1e-17)
constexpr double kPowRadiusShort = 1.0 / 512.0;

// gamma-derived constants, computed once on the host in ch_init (fill_gas in ch_kernels.cu).
struct Gas {
  double gamma;
  double gm1;        // gamma - 1
  double inv_gm1;    // 1/(gamma - 1)
  double two_gm1;    // 2/(gamma - 1)
  double z;          // (gamma - 1)/(2 gamma)
  double gm;         // (gamma - 1)/(gamma + 1)
  double c_sh;       // (gamma + 1)/(2 gamma)
  double half_gp1;   // (gamma + 1)/2
  double two_gp1;    // 2/(gamma + 1)
  double half_gm1;   // (gamma - 1)/2
  double bz[kPowTerms];   // binomial coefficients C(z, k), k = 1..13:  (1+t)^z - 1 = sum bz[k-1] t^k
};

// ---- branch-free reciprocal / reciprocal square root / square root ------------------------------
// MUFU seed (measured on B200: relative error <= 2^-19.9 for both) + ONE cubic Newton step in DFMA:
// measured max relative error over 2^30 inputs spanning 2^-80..2^80: 1.1e-16 (rcp), 1.9e-16 (rsqrt).
// Valid for normal positive x, which every operand on this path is (densities, floored pressures,
// sums of positive terms).  No denormal / inf / zero slow path.
CH_D double rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  e = fma(e, e, e);
  return fma(r, e, r);
}

CH_D double rsqrt_pos(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double t = x * y;
  const double e = fma(-t, y, 1.0);
  const double c = fma(e, 0.375, 0.5);
  return fma(c, y * e, y);
}

// sqrt(x) = x * rsqrt(x) with one residual correction.
CH_D double sqrt_pos(double x) {
  const double y = rsqrt_pos(x);
  const double s = x * y;
  const double r = fma(-s, s, x);
  return fma(r, 0.5 * y, s);
}

CH_D double sel_min(double a, double b) { return (a < b) ? a : b; }
CH_D double sel_max(double a, double b) { return (a > b) ? a : b; }

CH_D double floor_p(double p) { return (p < kPFloor) ? kPFloor : p; }  // keeps NaN visible

// Eq. 6-8: conserved (direction-local momenta) -> primitive, pressure floor (S1).
CH_D void cons2prim(const Gas& G, double d, double mn, double mt1, double mt2, double E, double w[5]) {
  const double r = rcp(d);
  const double u = mn * r, v = mt1 * r, ww = mt2 * r;
  // every multiply-add spelled out: the same cell must get the same bits wherever the compiler inlines this
  // (the warm-up of a marching segment and its loop body contract freely otherwise), so that a result does not
  // depend on where a cell sits in a segment, a tile or a sub-domain
  const double ke = __dmul_rn(0.5 * d, fma(ww, ww, fma(v, v, __dmul_rn(u, u))));
  w[0] = d; w[1] = u; w[2] = v; w[3] = ww;
  w[4] = floor_p(__dmul_rn(G.gm1, E - ke));
}

// Eq. 6-8 inverted: primitive -> conserved (direction-local momenta).
CH_D void prim2cons(const Gas& G, const double w[5], double c[5]) {
  c[0] = w[0];
  c[1] = w[0] * w[1];
  c[2] = w[0] * w[2];
  c[3] = w[0] * w[3];
  c[4] = w[4] * G.inv_gm1 + 0.5 * w[0] * ((w[1] * w[1] + w[2] * w[2]) + w[3] * w[3]);
}

// s = 1/(rho a) with a = sqrt(gamma p / rho) (Eq. 21): the one transcendental per cell; everything
// the characteristic projections need follows by multiplication:
//   a = gamma p s,  1/a = rho s,  rho/a = rho^2 s,  1/a^2 = (rho s)^2,  a/rho = a^2 s,  rho a = gamma p rho s.
CH_D double inv_rho_a(const Gas& G, double rho, double p) { return rsqrt_pos(G.gamma * p * rho); }

// Monotonised-central limiter A10 (reading G7: the formula governs).
CH_D double mc_limit(double dL, double dR, double dC) {
  const double m = sel_min(fabs(dC), __dmul_rn(2.0, sel_min(fabs(dL), fabs(dR))));
  return (__dmul_rn(dL, dR) > 0.0) ? copysign(m, dC) : 0.0;
}

// Limited slope of cell q in primitive variables via characteristic variables (A2 P:L690, A9 P:L730
// with row 0 read as G1, A10, A11 P:L741), projected with cell q's own rho, a.  s = inv_rho_a(q).
// Every operation is an explicitly rounded intrinsic: this function is inlined both into the warm-up of a marching
// segment and into its loop body, and a cell's slope must not depend on which of the two computed it (the result of
// a step is then independent of how the sweeps are cut into segments, tiles or sub-domains — tested bitwise).
CH_D void char_project(double ra, double ia2, double d0, double d1, double d2, double d3, double d4, double x[5]) {
  const double t1 = __dmul_rn(ra, d1), t2 = __dmul_rn(d4, ia2);
  x[0] = __dmul_rn(0.5, __dadd_rn(t2, -t1));
  x[1] = __dadd_rn(d0, -t2);
  x[2] = d2;
  x[3] = d3;
  x[4] = __dmul_rn(0.5, __dadd_rn(t1, t2));
}

// The same limiter with the sign test on the high words instead of a product (limited_slope only: PPMP / PLMP keep the
// product form above).  A vanishing one-sided difference needs no test of its own: the minimum is then zero.
CH_D double mc_limit_bits(double dL, double dR, double dC) {
  const double m = sel_min(fabs(dC), __dmul_rn(2.0, sel_min(fabs(dL), fabs(dR))));
  return ((__double2hiint(dL) ^ __double2hiint(dR)) >= 0) ? copysign(m, dC) : 0.0;
}

CH_D void limited_slope(const Gas& G, const double wm[5], const double w0[5], const double wp[5], double s,
                        double dw[5]) {
  const double rho = w0[0];
  const double a = __dmul_rn(__dmul_rn(G.gamma, w0[4]), s);
  const double ia = __dmul_rn(rho, s);
  const double ra = __dmul_rn(rho, ia);     // rho / a
  const double ia2 = __dmul_rn(ia, ia);     // 1 / a^2
  double dl[5], dr[5], xL[5], xR[5], xC[5], x[5];
#pragma unroll
  for (int m = 0; m < 5; ++m) { dl[m] = __dadd_rn(w0[m], -wm[m]); dr[m] = __dadd_rn(wp[m], -w0[m]); }
  char_project(ra, ia2, dl[0], dl[1], dl[2], dl[3], dl[4], xL);
  char_project(ra, ia2, dr[0], dr[1], dr[2], dr[3], dr[4], xR);
  // centred difference (A2): (w_{i+1} - w_{i-1})/2 is the mean of the two one-sided differences and the projection is linear,
  // so its characteristic components are the means of theirs (one rounding apart from projecting it anew)
#pragma unroll
  for (int m = 0; m < 5; ++m) xC[m] = __dmul_rn(0.5, __dadd_rn(xL[m], xR[m]));
#pragma unroll
  for (int m = 0; m < 5; ++m) x[m] = mc_limit_bits(xL[m], xR[m], xC[m]);
  const double s04 = __dadd_rn(x[0], x[4]);
  const double a2 = __dmul_rn(a, a);
  dw[0] = __dadd_rn(x[1], s04);
  dw[1] = __dmul_rn(__dmul_rn(a2, s), __dadd_rn(x[4], -x[0]));   // a / rho
  dw[2] = x[2];
  dw[3] = x[3];
  dw[4] = __dmul_rn(a2, s04);
}

// PPMC for one cell (A.3): parabola edges A20-A23, A24/A26(=A50, G2), characteristic
// tracing A25-A33 (A30/A32 read as G3).  wm,w0,wp = cells i-1,i,i+1; dwm,dw0,dwp their limited
// slopes; s = inv_rho_a(i); dtdx = dt/dx_d.  Outputs W*_L, W*_R (primitive).
// A20: the interpolated value on the interface between a cell (w_lo, slope d_lo) and its upper
// neighbour (w_hi, d_hi).  It is cell lo's W_{R,A} and cell hi's W_{L,A}: the marching kernels compute it once.
CH_D void ppm_interface(const double w_lo[5], const double w_hi[5], const double d_lo[5], const double d_hi[5],
                        double e[5]) {
#pragma unroll
  for (int m = 0; m < 5; ++m) e[m] = fma(d_lo[m] - d_hi[m], 1.0 / 6.0, 0.5 * (w_hi[m] + w_lo[m]));
}

CH_D void ppmc_from_interfaces(const Gas& G, double dtdx, const double wm[5], const double w0[5], const double wp[5],
                               const double LA[5], const double RA[5], double s, double WLs[5], double WRs[5]);

CH_D void ppmc_faces(const Gas& G, double dtdx, const double wm[5], const double w0[5], const double wp[5],
                      const double dwm[5], const double dw0[5], const double dwp[5], double s, double WLs[5],
                      double WRs[5]) {
  double LA[5], RA[5];
  ppm_interface(wm, w0, dwm, dw0, LA);
  ppm_interface(w0, wp, dw0, dwp, RA);
  ppmc_from_interfaces(G, dtdx, wm, w0, wp, LA, RA, s, WLs, WRs);
}

CH_D void ppmc_from_interfaces(const Gas& G, double dtdx, const double wm[5], const double w0[5], const double wp[5],
                               const double LA[5], const double RA[5], double s, double WLs[5], double WRs[5]) {
  double WL[5], WR[5], dwi[5], w6[5];
#pragma unroll
  for (int m = 0; m < 5; ++m) {
    // A20-A24, A26 on the face DEVIATIONS dR = R - w, dL = w - L (round 2): every correction of A21-A23 is a clamp of
    // a deviation, so the faces themselves are formed once, at the end.
    //   A21: an extremum (dR dL <= 0) flattens the cell: both deviations vanish.
    //   A22 (G8): (R - L)[L - (3w - 2R)] < 0 and (R - L)[(3w - 2L) - R] < 0 are (dR + dL)(2dR - dL) < 0 and
    //     (dR + dL)(2dL - dR) < 0, i.e. |dL| > 2|dR| and |dR| > 2|dL| once A21 has made the signs agree; the replaced
    //     faces 3w - 2R, 3w - 2L are the deviations 2dR, 2dL.  At most one fires; ties leave the face alone.
    //   A23: L within [min(w_{i-1}, w), max(w_{i-1}, w)] says dL lies between 0 and tL = w - w_{i-1}:
    //     opposite signs -> 0, |dL| > |tL| -> tL; likewise dR against tR = w_{i+1} - w.  Signs are compared on the high
    //     words (a zero deviation passes either way and stays zero; a zero t is caught by the magnitude test).
    //   A24 R - L = dR + dL; A26 as A50 (G2) 6[w - (L + R)/2] = 3(dL - dR), free of the cancellation.
    const double wi = w0[m];
    const double dR0 = RA[m] - wi, dL0 = wi - LA[m];
    const double tL = wi - wm[m], tR = wp[m] - wi;
    const bool ext = dR0 * dL0 <= 0.0;
    const double dR1 = ext ? 0.0 : dR0, dL1 = ext ? 0.0 : dL0;
    const double dR2 = dR1 + dR1, dL2 = dL1 + dL1;
    const bool fixL = fabs(dL1) > fabs(dR2), fixR = fabs(dR1) > fabs(dL2);
    const double dL3 = fixL ? dR2 : dL1, dR3 = fixR ? dL2 : dR1;
    const bool oppL = (__double2hiint(dL3) ^ __double2hiint(tL)) < 0, oppR = (__double2hiint(dR3) ^ __double2hiint(tR)) < 0;
    const double cL = (fabs(dL3) > fabs(tL)) ? tL : dL3, cR = (fabs(dR3) > fabs(tR)) ? tR : dR3;
    const double dL = oppL ? 0.0 : cL, dR = oppR ? 0.0 : cR;
    WL[m] = wi - dL; WR[m] = wi + dR;
    dwi[m] = dR + dL;
    w6[m] = 3.0 * (dL - dR);
  }
  const double rho = w0[0];
  const double a = G.gamma * w0[4] * s;
  const double ia = rho * s;
  const double ia2 = ia * ia;
  const double ra = rho * ia;        // rho / a
  const double rhoa = rho * a;       // rho * a
  const double lm = w0[1] - a, l0 = w0[1], lp = w0[1] + a;            // A8
  const double am = dtdx * sel_min(lm, 0.0), a0 = dtdx * sel_min(l0, 0.0), ap = dtdx * sel_min(lp, 0.0);  // A27
  const double bm = dtdx * sel_max(lm, 0.0), b0 = dtdx * sel_max(l0, 0.0), bp = dtdx * sel_max(lp, 0.0);
  const double k23 = 2.0 / 3.0;
  // reference states A25: left face under lambda^m, right face under lambda^p
  double WLm[5], WRp[5];
  {
    const double ca = 0.5 * am, cb = 1.0 + k23 * am;
    const double da = 0.5 * bp, db = 1.0 - k23 * bp;
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      WLm[m] = WL[m] - ca * (dwi[m] + w6[m] * cb);
      WRp[m] = WR[m] - da * (dwi[m] - w6[m] * db);
    }
  }
  double sL0 = 0.0, sL1 = 0.0, sL2 = 0.0, sL3 = 0.0, sL4 = 0.0;
  double sR0 = 0.0, sR1 = 0.0, sR2 = 0.0, sR3 = 0.0, sR4 = 0.0;
  if (l0 < 0.0) {   // A28 first term: E = W_L^0 - W_L^m
    const double ca = 0.5 * a0, cb = 1.0 + k23 * a0;
    const double E0 = (WL[0] - ca * (dwi[0] + w6[0] * cb)) - WLm[0];
    const double E2 = (WL[2] - ca * (dwi[2] + w6[2] * cb)) - WLm[2];
    const double E3 = (WL[3] - ca * (dwi[3] + w6[3] * cb)) - WLm[3];
    const double E4 = (WL[4] - ca * (dwi[4] + w6[4] * cb)) - WLm[4];
    sL0 += E0 - E4 * ia2; sL2 += E2; sL3 += E3;
  }
  if (lp < 0.0) {   // A28 second term: B = W_L^p - W_L^m
    const double ca = 0.5 * ap, cb = 1.0 + k23 * ap;
    const double B1 = (WL[1] - ca * (dwi[1] + w6[1] * cb)) - WLm[1];
    const double B4 = (WL[4] - ca * (dwi[4] + w6[4] * cb)) - WLm[4];
    sL0 += 0.5 * (ra * B1 + B4 * ia2);
    sL1 += 0.5 * (B1 + B4 * s);
    sL4 += 0.5 * (rhoa * B1 + B4);
  }
  if (lm > 0.0) {   // A31 first term: C = W_R^m - W_R^p
    const double da = 0.5 * bm, db = 1.0 - k23 * bm;
    const double C1 = (WR[1] - da * (dwi[1] - w6[1] * db)) - WRp[1];
    const double C4 = (WR[4] - da * (dwi[4] - w6[4] * db)) - WRp[4];
    sR0 += 0.5 * (C4 * ia2 - ra * C1);
    sR1 += 0.5 * (C1 - C4 * s);
    sR4 += 0.5 * (C4 - rhoa * C1);
  }
  if (l0 > 0.0) {   // A31 second term: D = W_R^0 - W_R^p
    const double da = 0.5 * b0, db = 1.0 - k23 * b0;
    const double D0 = (WR[0] - da * (dwi[0] - w6[0] * db)) - WRp[0];
    const double D2 = (WR[2] - da * (dwi[2] - w6[2] * db)) - WRp[2];
    const double D3 = (WR[3] - da * (dwi[3] - w6[3] * db)) - WRp[3];
    const double D4 = (WR[4] - da * (dwi[4] - w6[4] * db)) - WRp[4];
    sR0 += D0 - D4 * ia2; sR2 += D2; sR3 += D3;
  }
  WLs[0] = WLm[0] + sL0; WLs[1] = WLm[1] + sL1; WLs[2] = WLm[2] + sL2; WLs[3] = WLm[3] + sL3; WLs[4] = WLm[4] + sL4;  // A33
  WRs[0] = WRp[0] + sR0; WRs[1] = WRp[1] + sR1; WRs[2] = WRp[2] + sR2; WRs[3] = WRp[3] + sR3; WRs[4] = WRp[4] + sR4;
}

// PLMC for one cell (A.2): faces A12 from the limited slope dw0 of this cell, monotonised A13,
// slope A14, characteristic tracing A15-A19 (A19's contact term restored, reading G10).
CH_D void plmc_faces(const Gas& G, double dtdx, const double wm[5], const double w0[5], const double wp[5],
                     const double dw0[5], double s, double WLs[5], double WRs[5]) {
  double WL[5], WR[5], dwi[5];
#pragma unroll
  for (int m = 0; m < 5; ++m) {
    const double wi = w0[m];
    double L = wi - 0.5 * dw0[m], R = wi + 0.5 * dw0[m];               // A12
    {                                                                  // A13
      const bool up = wm[m] < wi;
      const double lo = up ? wm[m] : wi, hi = up ? wi : wm[m];
      L = sel_min(hi, sel_max(lo, L));
    }
    {
      const bool up = wp[m] < wi;
      const double lo = up ? wp[m] : wi, hi = up ? wi : wp[m];
      R = sel_min(hi, sel_max(lo, R));
    }
    WL[m] = L; WR[m] = R; dwi[m] = R - L;                              // A14
  }
  const double rho = w0[0];
  const double a = G.gamma * w0[4] * s;
  const double ia = rho * s, ia2 = ia * ia, ra = rho * ia, rhoa = rho * a;
  const double lm = w0[1] - a, l0 = w0[1], lp = w0[1] + a;            // A8
  const double h = 0.5 * dtdx;
  double sL0 = 0.0, sL1 = 0.0, sL2 = 0.0, sL3 = 0.0, sL4 = 0.0;
  double sR0 = 0.0, sR1 = 0.0, sR2 = 0.0, sR3 = 0.0, sR4 = 0.0;
  if (l0 < 0.0) {   // A17 contact term
    const double c = lm - l0;
    sL0 += c * (dwi[0] - dwi[4] * ia2); sL2 += c * dwi[2]; sL3 += c * dwi[3];
  }
  if (lp < 0.0) {   // A17 right acoustic term
    const double c = 0.5 * (lm - lp);
    sL0 += c * (ra * dwi[1] + dwi[4] * ia2); sL1 += c * (dwi[1] + dwi[4] * s); sL4 += c * (rhoa * dwi[1] + dwi[4]);
  }
  if (lm > 0.0) {   // A19 left acoustic term
    const double c = 0.5 * (lp - lm);
    sR0 += c * (dwi[4] * ia2 - ra * dwi[1]); sR1 += c * (dwi[1] - dwi[4] * s); sR4 += c * (dwi[4] - rhoa * dwi[1]);
  }
  if (l0 > 0.0) {   // A19 contact term
    const double c = lp - l0;
    sR0 += c * (dwi[0] - dwi[4] * ia2); sR2 += c * dwi[2]; sR3 += c * dwi[3];
  }
  const double cl = h * sel_min(lm, 0.0), cr = h * sel_max(lp, 0.0);   // A15
  const double sLv[5] = {sL0, sL1, sL2, sL3, sL4}, sRv[5] = {sR0, sR1, sR2, sR3, sR4};
#pragma unroll
  for (int m = 0; m < 5; ++m) {
    WLs[m] = (WL[m] - cl * dwi[m]) + h * sLv[m];                       // A16
    WRs[m] = (WR[m] - cr * dwi[m]) + h * sRv[m];                       // A18
  }
}

// ---- PPMP and PLMP (A.4 P:L886-1049, A.1 P:L679-717): reconstructions in the primitive variables ----------------
// PPMP switches corrections on at thresholds (A35, A36, A38, A44, A45): a threshold decided differently on two
// machines changes a face by a finite amount, so every quantity a threshold looks at is formed with explicitly
// rounded IEEE operations from primitives that are themselves formed with IEEE division (cons2prim_ieee): the
// decisions are then functions of the conserved state alone.  Everything downstream of a decision is continuous
// and free to contract.
CH_D void cons2prim_ieee(const Gas& G, double d, double mn, double mt1, double mt2, double E, double w[5]) {
  const double u = __ddiv_rn(mn, d), v = __ddiv_rn(mt1, d), ww = __ddiv_rn(mt2, d);
  const double ke = __dmul_rn(__dmul_rn(0.5, d), __dadd_rn(__dadd_rn(__dmul_rn(u, u), __dmul_rn(v, v)), __dmul_rn(ww, ww)));
  w[0] = d; w[1] = u; w[2] = v; w[3] = ww;
  w[4] = floor_p(__dmul_rn(G.gm1, __dadd_rn(E, -ke)));
}

// A2-A4: monotonised-central slope of one primitive variable
CH_D double mc_slope(double wm, double w0, double wp) {
  return mc_limit(w0 - wm, wp - w0, 0.5 * (wp - wm));
}

// A42-A45: F~ of cell j from p_{j-2}, p_{j-1}, p_{j+1}, p_{j+2}, u_{j-1}, u_{j+1}
CH_D double ppmp_flatten_tilde(double pm2, double pm1, double pp1, double pp2, double um1, double up1) {
  const double num = __dadd_rn(pp1, -pm1);
  const double lo = (pp1 < pm1) ? pp1 : pm1;
  if (__ddiv_rn(fabs(num), lo) < (1.0 / 3.0)) return 0.0;     // A44
  if (__dadd_rn(up1, -um1) > 0.0) return 0.0;                 // A45
  const double S = __ddiv_rn(num, __dadd_rn(pp2, -pm2));      // A42 (IEEE: a vanishing denominator gives +-inf)
  const double t = __dmul_rn(10.0, __dadd_rn(S, -0.75));      // A43
  const double c = (t < 1.0) ? t : 1.0;
  return (c > 0.0) ? c : 0.0;
}

// w[s], s = 0..6 = cells i-3..i+3, direction-local order.  Outputs W*_L, W*_R (primitive).
CH_D void ppmp_faces(const Gas& G, double dtdx, const double (&w)[7][5], double WLs[5], double WRs[5]) {
  const double* wim = w[2];
  const double* wi = w[3];
  const double* wip = w[4];
  double L[5], R[5], dm0 = 0.0, dp0 = 0.0;
#pragma unroll
  for (int m = 0; m < 5; ++m) {
    const double dm = mc_slope(w[1][m], w[2][m], w[3][m]);
    const double d0 = mc_slope(w[2][m], w[3][m], w[4][m]);
    const double dp = mc_slope(w[3][m], w[4][m], w[5][m]);
    L[m] = 0.5 * (wi[m] + wim[m]) - (d0 - dm) * (1.0 / 6.0);        // A34
    R[m] = 0.5 * (wip[m] + wi[m]) - (dp - d0) * (1.0 / 6.0);
    if (m == 0) { dm0 = dm; dp0 = dp; }
  }
  {   // A35-A41: contact steepening of the density faces (A38 read as G12, A41 as G13)
    const double rm = wim[0], rp = wip[0], pm = wim[4], pp = wip[4];
    const double drho = __dadd_rn(rp, -rm);
    const double jump = __ddiv_rn(fabs(drho), (rp < rm) ? rp : rm);
    const double pj = __ddiv_rn(fabs(__dadd_rn(pp, -pm)), (pp < pm) ? pp : pm);
    if (jump > 0.01 && pj < __dmul_rn(__dmul_rn(0.1, G.gamma), jump)) {
      const double d2m = __ddiv_rn(__dadd_rn(__dadd_rn(w[3][0], -__dmul_rn(2.0, w[2][0])), w[1][0]), 6.0);
      const double d2p = __ddiv_rn(__dadd_rn(__dadd_rn(w[5][0], -__dmul_rn(2.0, w[4][0])), w[3][0]), 6.0);
      if (__dmul_rn(d2m, d2p) < 0.0) {
        const double et = __ddiv_rn(-__dadd_rn(d2p, -d2m), drho);                 // A39
        double eta = __dadd_rn(__dmul_rn(20.0, et), -1.0);                         // A40
        eta = (eta < 1.0) ? eta : 1.0;
        eta = (eta > 0.0) ? eta : 0.0;
        L[0] = __dadd_rn(__dmul_rn(L[0], __dadd_rn(1.0, -eta)), __dmul_rn(__dadd_rn(rm, __dmul_rn(0.5, dm0)), eta));   // A41
        R[0] = __dadd_rn(__dmul_rn(R[0], __dadd_rn(1.0, -eta)), __dmul_rn(__dadd_rn(rp, -__dmul_rn(0.5, dp0)), eta));
      }
    }
  }
  {   // A42-A47: shock flattening of every variable
    const double Fm = ppmp_flatten_tilde(w[0][4], w[1][4], w[3][4], w[4][4], w[1][1], w[3][1]);
    const double F0 = ppmp_flatten_tilde(w[1][4], w[2][4], w[4][4], w[5][4], w[2][1], w[4][1]);
    const double Fp = ppmp_flatten_tilde(w[2][4], w[3][4], w[5][4], w[6][4], w[3][1], w[5][1]);
    const double Fn = (__dadd_rn(wip[4], -wim[4]) < 0.0) ? Fp : Fm;               // A46
    const double F = (F0 > Fn) ? F0 : Fn;
    const double oneF = __dadd_rn(1.0, -F);
#pragma unroll
    for (int m = 0; m < 5; ++m) {                                                  // A47
      L[m] = __dadd_rn(__dmul_rn(F, wi[m]), __dmul_rn(oneF, L[m]));
      R[m] = __dadd_rn(__dmul_rn(F, wi[m]), __dmul_rn(oneF, R[m]));
    }
  }
  // A48 (= A21 + A22; G8, G14), A50
  double WL[5], WR[5], dwi[5], w6[5];
#pragma unroll
  for (int m = 0; m < 5; ++m) {
    const double c = wi[m];
    double l = L[m], r = R[m];
    double dR = r - c, dL = c - l;
    if (dR * dL <= 0.0) { l = c; r = c; dR = 0.0; dL = 0.0; }
    const double dR2 = dR + dR, dL2 = dL + dL;
    const bool fixL = fabs(dL) > fabs(dR2), fixR = fabs(dR) > fabs(dL2);     // see ppmc_from_interfaces
    if (fixL) l = c - dR2;
    if (fixR) r = c + dL2;
    WL[m] = l; WR[m] = r;
    dwi[m] = r - l;
    w6[m] = 6.0 * (c - 0.5 * (l + r));
  }
  // A49, A51, A52
  const double a = sqrt_pos(G.gamma * wi[4] * rcp(wi[0]));
  const double lm = wi[1] - a, l0 = wi[1], lp = wi[1] + a;
  const double am = dtdx * sel_min(lm, 0.0), a0 = dtdx * sel_min(l0, 0.0), ap = dtdx * sel_min(lp, 0.0);
  const double bm = dtdx * sel_max(lm, 0.0), b0 = dtdx * sel_max(l0, 0.0), bp = dtdx * sel_max(lp, 0.0);
  const double k23 = 2.0 / 3.0;
  double Lm[5], L0[5], Lp[5], Rm[5], R0[5], Rp[5];
#pragma unroll
  for (int m = 0; m < 5; ++m) {
    Lm[m] = WL[m] - 0.5 * am * (dwi[m] + w6[m] * (1.0 + k23 * am));
    L0[m] = WL[m] - 0.5 * a0 * (dwi[m] + w6[m] * (1.0 + k23 * a0));
    Lp[m] = WL[m] - 0.5 * ap * (dwi[m] + w6[m] * (1.0 + k23 * ap));
    Rm[m] = WR[m] - 0.5 * bm * (dwi[m] - w6[m] * (1.0 - k23 * bm));
    R0[m] = WR[m] - 0.5 * b0 * (dwi[m] - w6[m] * (1.0 - k23 * b0));
    Rp[m] = WR[m] - 0.5 * bp * (dwi[m] - w6[m] * (1.0 - k23 * bp));
  }
  // A53-A56 with C = rho a of the reference state; chi_L^p read as G15; 1/C through one rsqrt: 1/(rho a) = rsqrt(gamma p rho)
  const double iCL = inv_rho_a(G, Lm[0], Lm[4]), iCR = inv_rho_a(G, Rp[0], Rp[4]);
  const double CL = G.gamma * Lm[4] * Lm[0] * iCL, CR = G.gamma * Rp[4] * Rp[0] * iCR;      // rho a = gamma p rho / (rho a)
  double chiLp = -0.5 * iCL * ((Lm[1] - Lp[1]) - (Lp[4] - Lm[4]) * iCL);
  double chiRm = 0.5 * iCR * ((Rp[1] - Rm[1]) - (Rp[4] - Rm[4]) * iCR);
  const double tLm = rcp(Lm[0]), tRp = rcp(Rp[0]);
  double chiL0 = (Lm[4] - L0[4]) * (iCL * iCL) + (tLm - rcp(L0[0]));
  double chiR0 = (Rp[4] - R0[4]) * (iCR * iCR) + (tRp - rcp(R0[0]));
  if (l0 > 0.0) chiL0 = 0.0;                       // A55
  if (lp > 0.0) chiLp = 0.0;
  if (lm < 0.0) chiRm = 0.0;
  if (l0 < 0.0) chiR0 = 0.0;
  WLs[0] = rcp((tLm - chiL0) - chiLp);             // A56
  WRs[0] = rcp((tRp - chiRm) - chiR0);
  WLs[1] = Lm[1] + CL * chiLp;
  WRs[1] = Rp[1] - CR * chiRm;
  WLs[4] = Lm[4] + (CL * CL) * chiLp;
  WRs[4] = Rp[4] + (CR * CR) * chiRm;
  WLs[2] = L0[2]; WRs[2] = R0[2];
  WLs[3] = L0[3]; WRs[3] = R0[3];
}

// PLMP (A1-A7): slope limited in the primitive variables, half-step by the cell's own two face fluxes (Eq. 11).
CH_D void plmp_faces(const Gas& G, double dtdx, const double wm[5], const double w0[5], const double wp[5], double WLs[5],
                     double WRs[5]) {
  double WL[5], WR[5];
#pragma unroll
  for (int m = 0; m < 5; ++m) {
    const double h = 0.5 * mc_slope(wm[m], w0[m], wp[m]);
    WL[m] = w0[m] - h; WR[m] = w0[m] + h;                                         // A1
  }
  double UL[5], UR[5];
  prim2cons(G, WL, UL);
  prim2cons(G, WR, UR);
  const double FL[5] = {UL[1], UL[1] * WL[1] + WL[4], UL[1] * WL[2], UL[1] * WL[3], (UL[4] + WL[4]) * WL[1]};
  const double FR[5] = {UR[1], UR[1] * WR[1] + WR[4], UR[1] * WR[2], UR[1] * WR[3], (UR[4] + WR[4]) * WR[1]};
  const double h = 0.5 * dtdx;
  double cl[5], cr[5];
#pragma unroll
  for (int m = 0; m < 5; ++m) {
    const double dF = FL[m] - FR[m];
    cl[m] = UL[m] + h * dF;                                                        // A6
    cr[m] = UR[m] + h * dF;                                                        // A7
  }
  cons2prim(G, cl[0], cl[1], cl[2], cl[3], cl[4], WLs);
  cons2prim(G, cr[0], cr[1], cr[2], cr[3], cr[4], WRs);
}

// The same for a thread that marches along the sweep: `ifc` carries the A20 value of the cell's lower interface
// in and of its upper interface out (PPMC only; the other reconstructions do not use it).
template <int R>
CH_D void recon_faces_march(const Gas& G, double dtdx, const double wm[5], const double w0[5], const double wp[5],
                            const double dw0[5], const double dwp[5], double s, double ifc[5], double WLs[5],
                            double WRs[5]) {
  if (R == 0) {
    double RA[5];
    ppm_interface(w0, wp, dw0, dwp, RA);
    ppmc_from_interfaces(G, dtdx, wm, w0, wp, ifc, RA, s, WLs, WRs);
#pragma unroll
    for (int m = 0; m < 5; ++m) ifc[m] = RA[m];
  } else if (R == 1) {
    plmc_faces(G, dtdx, wm, w0, wp, dw0, s, WLs, WRs);
  } else if (R == 4) {
    plmp_faces(G, dtdx, wm, w0, wp, WLs, WRs);      // its own slope, in the primitive variables (A1-A4)
  } else {
#pragma unroll
    for (int m = 0; m < 5; ++m) { WLs[m] = w0[m]; WRs[m] = w0[m]; }
  }
}

// Reconstruction selection at compile time: 0 PPMC, 1 PLMC, 2 PCM (Eq. 25-26: the cell average).
template <int R>
CH_D void recon_faces(const Gas& G, double dtdx, const double wm[5], const double w0[5], const double wp[5],
                      const double dwm[5], const double dw0[5], const double dwp[5], double s, double WLs[5],
                      double WRs[5]) {
  if (R == 0) ppmc_faces(G, dtdx, wm, w0, wp, dwm, dw0, dwp, s, WLs, WRs);
  else if (R == 1) plmc_faces(G, dtdx, wm, w0, wp, dw0, s, WLs, WRs);
  else if (R == 4) plmp_faces(G, dtdx, wm, w0, wp, WLs, WRs);
  else {
#pragma unroll
    for (int m = 0; m < 5; ++m) { WLs[m] = w0[m]; WRs[m] = w0[m]; }
  }
}

// (1 + t)^z - 1 for |t| <= kPowRadius: 13-term binomial series in Horner form (truncation
// C(z,14) 16^-14 < 1e-18).  Returns the value WITHOUT the leading 1 so that f_k = 2a/(gamma-1) (x-1)
// (B5) does not cancel.
CH_D double powz_m1_series(const Gas& G, double t) {
  if (fabs(t) <= kPowRadiusShort) {     // smooth flow: pressures within 0.2 % of one another, six terms reach 1e-17
    double h = G.bz[kPowTermsShort - 1];
#pragma unroll
    for (int k = kPowTermsShort - 2; k >= 0; --k) h = fma(h, t, G.bz[k]);
    return h * t;
  }
  double h = G.bz[kPowTerms - 1];
#pragma unroll
  for (int k = kPowTerms - 2; k >= 0; --k) h = fma(h, t, G.bz[k]);
  return h * t;
}

// Pressure function f_k, f'_k (B5, B6) for one side at trial pressure p.
//   rk, pk: density and pressure of side k; ak = sound speed; rpk = 1/pk; ick = 1/(rho_k a_k);
//   rp = 1/p.  On the rarefaction branch x returns (p/pk)^z (re-used by the sampler).
// Returns true on the rarefaction branch.
CH_D bool pressure_fn(const Gas& G, double p, double rp, double rk, double pk, double ak, double rpk, double ick,
                      double& f, double& fp, double& x) {
  const bool rare = (p <= pk);
  if (rare) {
    const double t = (p - pk) * rpk;         // p/pk - 1, exact difference first
    double xm1;
    if (fabs(t) <= kPowRadius) xm1 = powz_m1_series(G, t);
    else xm1 = exp(G.z * log(p * rpk)) - 1.0;
    x = xm1 + 1.0;
    f = G.two_gm1 * ak * xm1;
    fp = ick * x * (pk * rp);                // (p/pk)^{-(gamma+1)/(2 gamma)} = pr^z / pr
  } else {         // shock: sqrt(A/(p+B)) = rsqrt((p + B) rho (gamma+1)/2)   (B4)
    const double h = rk * G.half_gp1;
    const double sq = rsqrt_pos((p + G.gm * pk) * h);
    const double dp = p - pk;
    f = dp * sq;
    fp = sq * (1.0 - 0.5 * dp * (sq * sq) * h);   // 1/(B+p) = sq^2 (gamma+1) rho / 2
  }
  return rare;
}

// Exact Riemann solver (B.1): primitive L/R states (direction-local) -> flux B22.
// Newton-Raphson on the star pressure from the two-shock guess B2-B4.  With p0 the last iterate at
// which f_k, f'_k were evaluated and p^m the accepted pressure (|p^m - p0| <= 1e-8 p, B8), B9 needs
// f_k(p^m) (reading S3): taken as f_k(p0) + f'_k(p0)(p^m - p0), whose error f'' (p^m - p0)^2 / 2 is
// below 1e-16 of the wave-speed scale; likewise (p^m/p_k)^z for the sampler.  The sampler branches
// on the wave type found at p0 (the two wave curves have second-order contact at p = p_k, so the
// choice within 1e-8 of the kink moves nothing above 1e-24).  Iterate floored at 1e-20 (S4).  The
// ten-way sampling at x/t = 0 is folded onto the left-wave family by mirroring (u -> -u) when
// u^m < 0; the mirrored tests coincide with B16-B21 except on the measure-zero tie
// um + a_R x = 0, where fan and star state are equal.
CH_D void riemann_exact(const Gas& G, const double WL[5], const double WR[5], double flux[5]) {
  const double rL = WL[0], uL = WL[1], pL = floor_p(WL[4]);
  const double rR = WR[0], uR = WR[1], pR = floor_p(WR[4]);
  const double icL = inv_rho_a(G, rL, pL), icR = inv_rho_a(G, rR, pR);   // 1/(rho a)
  const double gpL = G.gamma * pL, gpR = G.gamma * pR;
  const double aL = gpL * icL, aR = gpR * icR;                           // B1
  const double rpL = G.gamma * rL * (icL * icL);                         // 1/p = gamma rho /(rho a)^2
  const double rpR = G.gamma * rR * (icR * icR);
  const double du = uR - uL;
  // B2
  double pt = 0.5 * (pL + pR) - 0.125 * du * (rL + rR) * (aL + aR);
  pt = (pt < 0.0) ? 0.0 : pt;
  // B3, B4: g_k = sqrt(A_k/(pt + B_k))
  const double gL = rsqrt_pos((pt + G.gm * pL) * rL * G.half_gp1);
  const double gR = rsqrt_pos((pt + G.gm * pR) * rR * G.half_gp1);
  double p0 = ((gL * pL + gR * pR) - du) * rcp(gL + gR);
  p0 = (p0 < kPGuessFloor) ? kPGuessFloor : p0;
  // Newton-Raphson B5-B8
  double pm, rp0, fL, fR, fpL, fpR, xL = 1.0, xR = 1.0;
  bool rareL, rareR;
  int it = 0;
  for (;;) {
    rp0 = rcp(p0);
    rareL = pressure_fn(G, p0, rp0, rL, pL, aL, rpL, icL, fL, fpL, xL);
    rareR = pressure_fn(G, p0, rp0, rR, pR, aR, rpR, icR, fR, fpR, xR);
    pm = p0 - ((fL + fR) + du) * rcp(fpL + fpR);                        // B7
    pm = (pm < kPFloor) ? kPFloor : pm;                                  // S4
    ++it;
    if (!(2.0 * fabs(pm - p0) > kNewtonTol * fabs(pm + p0)) || it >= kNewtonCap) break;   // B8
    p0 = pm;
  }
  const double dp = pm - p0;                                             // S3 by first-order update
  fL = fma(fpL, dp, fL);
  fR = fma(fpR, dp, fR);
  const double um = 0.5 * ((uL + uR) + (fR - fL));                       // B9

  // Sampling at x/t = 0, mirrored onto the left family.
  const bool left = (um >= 0.0);
  const double sg = left ? 1.0 : -1.0;
  const double rk = left ? rL : rR, pk = left ? pL : pR, ak = left ? aL : aR;
  const double uk = sg * (left ? uL : uR), us = sg * um;
  const double rpk = left ? rpL : rpR;
  const bool rare = left ? rareL : rareR;
  double xk = left ? xL : xR;
  xk = fma(G.z * xk * rp0, dp, xk);                                      // (pm/pk)^z from (p0/pk)^z
  const double vt1 = left ? WL[2] : WR[2], vt2 = left ? WL[3] : WR[3];   // S9
  const double pr = pm * rpk;
  double rho, u, p;
  if (rare) {                                                            // rarefaction
    if (uk - ak >= 0.0) { rho = rk; u = uk; p = pk; }                    // B10 / B16
    else if (us - ak * xk < 0.0) { rho = rk * pr * rcp(xk * xk); u = us; p = pm; }   // B11 / B17: pr^{1/gamma} = pr / x^2
    else {                                                               // B12 / B18 (G4)
      const double af = G.two_gp1 * (ak + G.half_gm1 * uk);
      const double q = af * rcp(ak);
      const double y = exp(G.two_gm1 * log(q));                          // (a/a_k)^{2/(gamma-1)}
      rho = rk * y; u = af; p = pk * y * (q * q);                        // exponent 2 gamma/(gamma-1) = 2/(gamma-1) + 2
    }
  } else {                                                               // shock
    const double sk = uk - ak * sqrt_pos(G.c_sh * pr + G.z);             // B13 / B19 (G5)
    if (sk >= 0.0) { rho = rk; u = uk; p = pk; }                         // B14 / B20
    else { rho = rk * (pr + G.gm) * rcp(pr * G.gm + 1.0); u = us; p = pm; } // B15 / B21
  }
  u *= sg;
  // B22
  const double E = p * G.inv_gm1 + 0.5 * rho * ((u * u + vt1 * vt1) + vt2 * vt2);
  const double ru = rho * u;
  flux[0] = ru;
  flux[1] = ru * u + p;
  flux[2] = ru * vt1;
  flux[3] = ru * vt2;
  flux[4] = (E + p) * u;
}

// Roe solver with the HLLE failsafe (B.2): primitive L/R states (direction-local) -> flux.
// B23-B30 with B29 read as in DESIGN.md (G9); the intermediate states B31-B32 are checked for negative
// density or pressure and the HLLE flux B33-B35 substituted if either occurs.  Square roots and quotients
// through the branch-free rsqrt / rcp above.
// Every multiply-add below is spelled out (fma / __dmul_rn / __dadd_rn): the solver is inlined in several places of
// one kernel (the updating warps and the halo warp of the fused second half) and an interface on a tile seam, solved
// once by each, must get the same bits from both (conservation to the bit, results independent of the tiling).
CH_D void riemann_roe(const Gas& G, const double WL[5], const double WR[5], double flux[5], double etaH = 0.0) {
#define M_ __dmul_rn
#define A_ __dadd_rn
  const double rL = WL[0], uL = WL[1], vL = WL[2], wL = WL[3], pL = floor_p(WL[4]);
  const double rR = WR[0], uR = WR[1], vR = WR[2], wR = WR[3], pR = floor_p(WR[4]);
  const double EL = fma(pL, G.inv_gm1, M_(M_(0.5, rL), fma(wL, wL, fma(vL, vL, M_(uL, uL)))));
  const double ER = fma(pR, G.inv_gm1, M_(M_(0.5, rR), fma(wR, wR, fma(vR, vR, M_(uR, uR)))));
  const double UL[5] = {rL, M_(rL, uL), M_(rL, vL), M_(rL, wL), EL}, UR[5] = {rR, M_(rR, uR), M_(rR, vR), M_(rR, wR), ER};
  const double FL[5] = {UL[1], fma(UL[1], uL, pL), M_(UL[1], vL), M_(UL[1], wL), M_(A_(EL, pL), uL)};   // Eq. 11
  const double FR[5] = {UR[1], fma(UR[1], uR, pR), M_(UR[1], vR), M_(UR[1], wR), M_(A_(ER, pR), uR)};
  // B23
  const double isl = rsqrt_pos(rL), isr = rsqrt_pos(rR);
  const double sl = M_(rL, isl), sr = M_(rR, isr);
  const double inv = rcp(A_(sl, sr));
  const double HL = M_(A_(EL, pL), M_(isl, isl)), HR = M_(A_(ER, pR), M_(isr, isr));
  const double ut = M_(fma(sl, uL, M_(sr, uR)), inv), vt = M_(fma(sl, vL, M_(sr, vR)), inv), wt = M_(fma(sl, wL, M_(sr, wR)), inv);
  const double Ht = M_(fma(sl, HL, M_(sr, HR)), inv);
  const double V2 = fma(wt, wt, fma(vt, vt, M_(ut, ut)));
  const double at2 = M_(G.gm1, fma(-0.5, V2, Ht));                         // B24
  const double iat = rsqrt_pos(at2), at = M_(at2, iat);
  const double lm = A_(ut, -at), l0 = ut, lp = A_(ut, at);                 // B25
  if (lm >= 0.0) {
#pragma unroll
    for (int m = 0; m < 5; ++m) flux[m] = FL[m];
    return;
  }
  if (lp <= 0.0) {
#pragma unroll
    for (int m = 0; m < 5; ++m) flux[m] = FR[m];
    return;
  }
  double dU[5];
#pragma unroll
  for (int m = 0; m < 5; ++m) dU[m] = A_(UR[m], -UL[m]);                   // B26
  // B27: acoustic strengths share  q = gamma' (0.5 V2 drho - u dmx - v dmy - w dmz + dE)
  const double ia2 = M_(iat, iat), Na = M_(0.5, ia2);
  const double q = M_(G.gm1, A_(A_(fma(-ut, dU[1], M_(M_(0.5, V2), dU[0])), -fma(vt, dU[2], M_(wt, dU[3]))), dU[4]));
  const double r = M_(at, fma(ut, dU[0], -dU[1]));
  const double xi0 = M_(Na, A_(q, r)), xi4 = M_(Na, A_(q, -r));
  const double xi1 = fma(-vt, dU[0], dU[2]), xi2 = fma(-wt, dU[0], dU[3]);
  const double xi3 = fma(-q, ia2, dU[0]);
  // B28, B29
  // C3: with the H correction |lambda| -> max(|lambda|, eta^H), here and only here (reading S18)
  const double alm = sel_max(fabs(lm), etaH), al0 = sel_max(fabs(l0), etaH), alp = sel_max(fabs(lp), etaH);
  const double C0 = M_(xi0, alm), C1 = M_(xi1, al0), C2 = M_(xi2, al0), C3 = M_(xi3, al0), C4 = M_(xi4, alp);
  const double ua = M_(ut, at), c04 = A_(C0, C4), c043 = A_(c04, C3);
  const double Hm = A_(Ht, -ua), Hp = A_(Ht, ua);
  double sv[5];
  sv[0] = c043;
  sv[1] = fma(C4, lp, fma(C0, lm, M_(C3, ut)));
  sv[2] = fma(c043, vt, C1);
  sv[3] = fma(c043, wt, C2);
  sv[4] = A_(fma(C0, Hm, M_(C4, Hp)), fma(M_(0.5, C3), V2, fma(C1, vt, M_(C2, wt))));
  // B31, B32: intermediate states
  double Um[5] = {A_(UL[0], xi0), fma(xi0, lm, UL[1]), fma(xi0, vt, UL[2]), fma(xi0, wt, UL[3]), fma(xi0, Hm, UL[4])};
  bool hlle = !(Um[0] > 0.0) || !(fma(Um[4], Um[0], -M_(0.5, fma(Um[3], Um[3], fma(Um[2], Um[2], M_(Um[1], Um[1]))))) > 0.0);
  Um[0] = A_(Um[0], xi3); Um[1] = fma(xi3, ut, Um[1]); Um[2] = A_(Um[2], fma(xi3, vt, xi1)); Um[3] = A_(Um[3], fma(xi3, wt, xi2));
  Um[4] = A_(Um[4], fma(M_(0.5, xi3), V2, fma(xi1, vt, M_(xi2, wt))));
  hlle = hlle || !(Um[0] > 0.0) || !(fma(Um[4], Um[0], -M_(0.5, fma(Um[3], Um[3], fma(Um[2], Um[2], M_(Um[1], Um[1]))))) > 0.0);
  if (!hlle) {
#pragma unroll
    for (int m = 0; m < 5; ++m) flux[m] = M_(0.5, A_(A_(FL[m], FR[m]), -sv[m]));   // B30
    return;
  }
  // HLLE (B33-B35)
  const double aL = M_(M_(G.gamma, pL), inv_rho_a(G, rL, pL)), aR = M_(M_(G.gamma, pR), inv_rho_a(G, rR, pR));
  const double bm = sel_min(sel_min(lm, A_(uL, -aL)), 0.0), bp = sel_max(sel_max(lp, A_(uR, aR)), 0.0);
  const double t = M_(A_(bp, bm), rcp(A_(bp, -bm)));
#pragma unroll
  for (int m = 0; m < 5; ++m) {
    const double fl = fma(-bm, UL[m], FL[m]), fr = fma(-bp, UR[m], FR[m]);   // B34
    flux[m] = M_(0.5, fma(A_(fl, -fr), t, A_(fl, fr)));                      // B35
  }
#undef M_
#undef A_
}

// Solver selection at compile time (reconstruction and solver are selectable): 0 exact, 1 Roe + HLLE.
template <int S>
CH_D void riemann(const Gas& G, const double WL[5], const double WR[5], double flux[5]) {
  if (S == 0) riemann_exact(G, WL, WR, flux);
  else riemann_roe(G, WL, WR, flux);
}

// The fused second half solves the same kind of interface in two places (the updating warps and the warp that serves
// the two halo rows of a tile): both solvers spell out their multiply-adds where it matters, so the copies agree bitwise.
template <int S>
CH_D void riemann_tile(const Gas& G, const double WL[5], const double WR[5], double flux[5]) {
  riemann<S>(G, WL, WR, flux);
}

}  // namespace ch
