// ch_kernels.cu — CUDA kernels (sm_100a) and the C ABI of include/ch.h.
//
// One CTU step =
//   k_reset            reset the dt reduction cells
//   k_pass1_x          PPMC + tracing + exact Riemann along x   -> U*_L,U*_R(.,x), F*      (steps 1-2)
//   k_pass1_march<1|2> same along y / z, marching in registers  -> U*_L,U*_R(.,d), G*, H*
//   k_final3d_tma      3-D grids: Eq. 23 transverse correction + second exact Riemann pass + Eq. 24
//   (k_final3d)        update + Eq. 22 reduction of the new state, fused (steps 3-5; F,G,H^{n+1/2} stay on
//                      chip); planes staged by TMA, issued by a lane of the warp that serves the halo rows
//                      (13-row tiles, eleven updating warps; CH_OPT_TMA = 1: a producer warp of its own and
//                      12-row tiles, the form the H-corrected step takes); plain loads where TMA's 16-byte
//                      stride rules do not hold, or with CH_OPT_TMA = 0
//   k_final2d          the same for x-y grids (one plane, no z carry)
//   k_pass2, k_update  the same two halves unfused: 1-D, x-z / y-z grids, the H-corrected step without TMA (+ k_eta)
//   k_eta3d            H correction on 3-D grids: eta of every interface (C1), tiled march; k_final3d_tma<Roe, HC> then takes
//                      C2's maxima from the staged eta planes
//   k_ghost            ghost fill of the new state, analytic (Noh) faces included
//   k_pick_dt          ch_step_cfl: Eq. 22 finished on the device; the step is then replayed as a CUDA graph on small grids
//   k_halo, k_fill_dim block decomposition: halo slabs and the per-direction fill
// Every kernel that reconstructs or solves is a template on the reconstruction (PPMC / PLMC / PCM / PLMP; PPMP has
// pass-1 kernels of its own with the 7-cell stencil: k_pass1_x_ppmp, k_pass1_march_ppmp) and on the Riemann solver
// (exact / Roe + HLLE); the defaults are the paper's PPMC + exact.
// Data layout: struct-of-arrays fp64, x fastest, ghosts included; every kernel maps
// consecutive lanes to consecutive x so loads and stores coalesce.  No operand is reshaped for
// tensor cores: this is a stencil / ALU path.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <mutex>
#include <vector>
#include <new>
#include <string>

#include "../../include/ch.h"
#include "ch_hydro.cuh"

namespace {

using ch::Gas;

struct Geom {
  int n[3];          // real cells
  int g[3];          // ghost layers (0 for an inactive dimension)
  int pd[3];         // padded extents
  int act[3];        // n_d > 1
  long long st[3];   // strides in doubles: 1, px, px*py
  long long np;      // padded cells
};

struct StepArgs {
  Geom geo;
  Gas gas;
  double dtdx[3];    // dt / dx_d
  double dx[3];
  double idx[3];     // 1 / dx_d
  double* u;         // state [5][np]
  double* Fs[3];     // first-pass fluxes F*_d at interface c+1/2 stored at c  [5][np]
  double* UL[3];     // U*_L(c,d): traced state at the left face of cell c     [5][np]
  double* UR[3];     // U*_R(c,d)
  double* Fh[3];     // CTU fluxes F^{n+1/2}_d                                 [5][np]
  double* eta[3];    // H correction: eta of interface c+1/2 along d stored at c      [np]
  const double* dt_dev;   // ch_step_cfl: the time step lives on the device (written by k_pick_dt); else nullptr
  int ext;           // pass-1 reach along the sweep: cells [-ext, n+ext-1]; 1, or 2 with the H correction
  unsigned long long* red;  // [0] = bits of max cell rate (|v_d|+a)/dx_d, [1] = non-physical flag
};

// dt / dx_d of this step: from the kernel arguments (ch_step) or from the device-resident dt (ch_step_cfl), with
// the same correctly rounded division the host does (done once, by k_pick_dt: a division per thread was 3 % of
// k_pass1_x, whose threads live for one cell), so the two ways of stepping agree bitwise
__device__ __forceinline__ void step_dtdx(const StepArgs& A, double out[3]) {
  if (A.dt_dev) {
#pragma unroll
    for (int d = 0; d < 3; ++d) out[d] = A.dt_dev[2 + d];      // k_pick_dt's correctly rounded dt / dx_d
  } else {
#pragma unroll
    for (int d = 0; d < 3; ++d) out[d] = A.dtdx[d];
  }
}

__device__ __forceinline__ double step_dtdx1(const StepArgs& A, int d) {   // one direction only (pass 1)
  return A.dt_dev ? A.dt_dev[2 + d] : A.dtdx[d];
}

// ch_step_cfl on a non-physical state: k_pick_dt leaves dt = NaN; every kernel of the step then returns at once,
// so the last state and its reduction cells (rate, flag) survive and the failure stays visible (ch_last_dt,
// ch_compute_dt) instead of turning the whole grid into NaN.
__device__ __forceinline__ bool step_refused(const StepArgs& A) { return A.dt_dev && !(*A.dt_dev > 0.0); }

// global component index of direction-local component m for a sweep along D (cyclic)
template <int D>
__device__ __forceinline__ constexpr int comp(int m) {
  return (m == 0 || m == 4) ? m : 1 + (D + (m - 1)) % 3;
}

template <int D>
__device__ __forceinline__ void load_prim(const Gas& G, const double* __restrict__ u, long long np, long long q,
                                          double w[5]) {
  const double d = u[q];
  const double mn = u[comp<D>(1) * np + q];
  const double m1 = u[comp<D>(2) * np + q];
  const double m2 = u[comp<D>(3) * np + q];
  const double E = u[4 * np + q];
  ch::cons2prim(G, d, mn, m1, m2, E, w);
}

template <int D>
__device__ __forceinline__ void load_raw(const double* __restrict__ u, long long np, long long q, double r[5]) {
  r[0] = u[q];
  r[1] = u[comp<D>(1) * np + q];
  r[2] = u[comp<D>(2) * np + q];
  r[3] = u[comp<D>(3) * np + q];
  r[4] = u[4 * np + q];
}

// store a direction-local conserved vector into a global-order SoA array
template <int D>
__device__ __forceinline__ void store_local(double* __restrict__ dst, long long np, long long q, const double c[5]) {
  dst[q] = c[0];
  dst[comp<D>(1) * np + q] = c[1];
  dst[comp<D>(2) * np + q] = c[2];
  dst[comp<D>(3) * np + q] = c[3];
  dst[4 * np + q] = c[4];
}

__device__ __forceinline__ void copy5(double dst[5], const double src[5]) {
#pragma unroll
  for (int m = 0; m < 5; ++m) dst[m] = src[m];
}

// ---------------------------------------------------------------------------------------------
// Pass 1 along y or z: each thread owns one (x, transverse) column and marches a segment of `seg`
// interfaces along D with the 5-cell primitive stencil, three limited slopes and the previous
// cell's right-face state in registers.  Every cell's slope and parabola is computed once per
// segment (warm-up: 3 slopes + 1 parabola per segment).
// ---------------------------------------------------------------------------------------------
#ifndef CH_MARCH_T
#define CH_MARCH_T 128   // threads per CTA of the marching kernels
#endif
#ifndef CH_MARCH_MINB
#define CH_MARCH_MINB 3
#endif
#ifndef CH_X_MINB
#define CH_X_MINB 6
#endif
#ifndef CH_P2_T
#define CH_P2_T 128
#endif
#ifndef CH_P2_MINB
#define CH_P2_MINB 1
#endif

template <int D, int S, int R>
__global__ void __launch_bounds__(CH_MARCH_T, CH_MARCH_MINB) k_pass1_march(const StepArgs A, int seg) {
  if (step_refused(A)) return;
  constexpr int T = 3 - D;   // the other transverse dimension (x is the lane dimension)
  const Geom& g = A.geo;
  const Gas& G = A.gas;
  const int ext0 = g.act[0] ? g.n[0] + 2 : 1, lo0 = g.act[0] ? -1 : 0;
  const int extT = g.act[T] ? g.n[T] + 2 : 1, loT = g.act[T] ? -1 : 0;
  const long long col = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (col >= (long long)ext0 * extT) return;
  const int i = lo0 + (int)(col % ext0);
  const int t = loT + (int)(col / ext0);
  const int c0 = -A.ext + (int)blockIdx.y * seg;      // first interface of this segment
  const int nD = g.n[D];
  int c1 = c0 + seg;                                   // one past the last interface
  const int cend = nD + A.ext - 1;                     // last cell whose faces are needed
  const bool last = c1 >= cend;
  if (last) c1 = cend;
  const long long sD = g.st[D];
  const long long np = g.np;
  const long long base = (long long)(i + g.g[0]) + (long long)(t + g.g[T]) * g.st[T] + (long long)g.g[D] * sD;
  const double dtdx = step_dtdx1(A, D);
  const double* __restrict__ u = A.u;

  double wa[5], wb[5], wc[5], wd[5];   // cells c-1, c, c+1, c+2 (rotating)
  double sb[5], sc[5];                 // slopes of c, c+1
  double ifc[5];                       // A20 value on the lower interface of cell c (PPMC)
  double icb, icc;                     // 1/(rho a) of c, c+1
  double pr_prev[5];                   // previous cell's right-face primitive state W*_R
  double raw[5];                       // conserved values of the next cell to enter the stencil (loaded one step ahead)
  {
    double wz[5];
    load_prim<D>(G, u, np, base + (long long)(c0 - 2) * sD, wz);
    load_prim<D>(G, u, np, base + (long long)(c0 - 1) * sD, wa);
    load_prim<D>(G, u, np, base + (long long)(c0)*sD, wb);
    load_prim<D>(G, u, np, base + (long long)(c0 + 1) * sD, wc);
    load_raw<D>(u, np, base + (long long)(c0 + 2) * sD, raw);
    double sa[5];
    ch::limited_slope(G, wz, wa, wb, ch::inv_rho_a(G, wa[0], wa[4]), sa);
    icb = ch::inv_rho_a(G, wb[0], wb[4]);
    ch::limited_slope(G, wa, wb, wc, icb, sb);
    ch::ppm_interface(wa, wb, sa, sb, ifc);
  }
  for (int c = c0; c <= c1; ++c) {
    const long long q = base + (long long)c * sD;
    ch::cons2prim(G, raw[0], raw[1], raw[2], raw[3], raw[4], wd);
    if (c < c1) load_raw<D>(u, np, q + 3 * sD, raw);     // cell c+3 <= n_D+2: inside the padded store
    icc = ch::inv_rho_a(G, wc[0], wc[4]);
    ch::limited_slope(G, wb, wc, wd, icc, sc);
    double WLs[5], WRs[5], cl[5], cr[5];
    ch::recon_faces_march<R>(G, dtdx, wa, wb, wc, sb, sc, icb, ifc, WLs, WRs);
    ch::prim2cons(G, WLs, cl);     // states are kept conserved between stages
    ch::prim2cons(G, WRs, cr);
    if (c < c1 || last) {
      store_local<D>(A.UL[D], np, q, cl);
      store_local<D>(A.UR[D], np, q, cr);
    }
    if (c > c0) {
      double fl[5];
      ch::riemann<S>(G, pr_prev, WLs, fl);      // the solver's first act would be conserved -> primitive
      store_local<D>(A.Fs[D], np, q - sD, fl);
    }
    copy5(pr_prev, WRs);
    copy5(wa, wb); copy5(wb, wc); copy5(wc, wd);
    copy5(sb, sc);
    icb = icc;
  }
}

// The same march for PPMP (A.4): the thread carries the seven primitive cells c-3 .. c+3 its reconstruction reads
// (formed with IEEE operations in the global component order, reading S21), calls the same ppmp_faces the
// x-sweep kernel calls, and solves interface c-1/2 with the previous cell's right face.  y and z; the x sweep is
// k_pass1_x_ppmp.
template <int D, int S>
__global__ void __launch_bounds__(CH_MARCH_T, 2) k_pass1_march_ppmp(const StepArgs A, int seg) {
  if (step_refused(A)) return;
  constexpr int T = 3 - D;
  const Geom& g = A.geo;
  const Gas& G = A.gas;
  const int ext0 = g.act[0] ? g.n[0] + 2 : 1, lo0 = g.act[0] ? -1 : 0;
  const int extT = g.act[T] ? g.n[T] + 2 : 1, loT = g.act[T] ? -1 : 0;
  const long long col = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (col >= (long long)ext0 * extT) return;
  const int i = lo0 + (int)(col % ext0);
  const int t = loT + (int)(col / ext0);
  const int c0 = -1 + (int)blockIdx.y * seg;
  const int nD = g.n[D];
  int c1 = c0 + seg;
  const int cend = nD;
  const bool last = c1 >= cend;
  if (last) c1 = cend;
  const long long sD = g.st[D], np = g.np;
  const long long base = (long long)(i + g.g[0]) + (long long)(t + g.g[T]) * g.st[T] + (long long)g.g[D] * sD;
  const double dtdx = step_dtdx1(A, D);
  const double* __restrict__ u = A.u;
  double w[7][5], pr_prev[5], raw[5];
#pragma unroll
  for (int s = 0; s < 6; ++s) {
    const long long qs = base + (long long)(c0 - 3 + s) * sD;
    double wg[5];
    ch::cons2prim_ieee(G, u[qs], u[np + qs], u[2 * np + qs], u[3 * np + qs], u[4 * np + qs], wg);
#pragma unroll
    for (int m = 0; m < 5; ++m) w[s][m] = wg[comp<D>(m)];
  }
  {
    const long long qs = base + (long long)(c0 + 3) * sD;
#pragma unroll
    for (int f = 0; f < 5; ++f) raw[f] = u[f * np + qs];
  }
  for (int c = c0; c <= c1; ++c) {
    const long long q = base + (long long)c * sD;
    {
      double wg[5];
      ch::cons2prim_ieee(G, raw[0], raw[1], raw[2], raw[3], raw[4], wg);
#pragma unroll
      for (int m = 0; m < 5; ++m) w[6][m] = wg[comp<D>(m)];
    }
    if (c < c1) {                                           // cell c+4 <= n_D+3: inside the padded store (nghost >= 4)
#pragma unroll
      for (int f = 0; f < 5; ++f) raw[f] = u[f * np + q + 4 * sD];
    }
    double WLs[5], WRs[5], cl[5], cr[5];
    ch::ppmp_faces(G, dtdx, w, WLs, WRs);
    ch::prim2cons(G, WLs, cl);
    ch::prim2cons(G, WRs, cr);
    if (c < c1 || last) {
      store_local<D>(A.UL[D], np, q, cl);
      store_local<D>(A.UR[D], np, q, cr);
    }
    if (c > c0) {
      double fl[5];
      ch::riemann<S>(G, pr_prev, WLs, fl);
      store_local<D>(A.Fs[D], np, q - sD, fl);
    }
    copy5(pr_prev, WRs);
#pragma unroll
    for (int s = 0; s < 6; ++s) copy5(w[s], w[s + 1]);
  }
}

// ---------------------------------------------------------------------------------------------
// Pass 1 along x: one thread per padded cell of a flat run of memory (x fastest, rows follow one
// another), neighbours exchanged through shared memory in three stages (primitives -> slopes ->
// left-face states).  A CTA of T threads yields T-5 interfaces; lanes on cells outside the needed
// ranges are masked so garbage row-crossing stencils cost nothing.
// ---------------------------------------------------------------------------------------------
#ifndef CH_X_T
#define CH_X_T 128
#endif
constexpr int kXT = CH_X_T;    // threads per CTA
constexpr int kXOut = kXT - 5; // interfaces produced per CTA

// Coordinates (relative to the first real cell) of padded index q.  Grids below 2^31 padded cells take 32-bit
// divisions: the two 64-bit ones were 5 % of k_pass1_x's issue slots.
__device__ __forceinline__ void padded_coords(const Geom& g, long long q, int& i, int& j, int& k) {
  if (g.np < (1LL << 31)) {
    unsigned r = (unsigned)q;
    const unsigned s2 = (unsigned)g.st[2], s1 = (unsigned)g.st[1];
    const unsigned kk = r / s2; r -= kk * s2;
    const unsigned jj = r / s1;
    i = (int)(r - jj * s1) - g.g[0]; j = (int)jj - g.g[1]; k = (int)kk - g.g[2];
  } else {
    long long r = q;
    k = (int)(r / g.st[2]); r -= (long long)k * g.st[2];
    j = (int)(r / g.st[1]);
    i = (int)(r - (long long)j * g.st[1]);
    i -= g.g[0]; j -= g.g[1]; k -= g.g[2];
  }
}

template <int S, int R>
__global__ void __launch_bounds__(kXT, CH_X_MINB) k_pass1_x(const StepArgs A, long long q_begin, long long q_end) {
  __shared__ double sP[5][kXT];
  __shared__ double sS[5][kXT];
  __shared__ double sL[5][kXT];
  if (step_refused(A)) return;
  const Geom& g = A.geo;
  const double dtdx0 = step_dtdx1(A, 0);
  const Gas& G = A.gas;
  const long long np = g.np;
  const int tid = threadIdx.x;
  const long long q = q_begin + (long long)blockIdx.x * kXOut + tid - 2;
  const bool inb = (q >= 0 && q < np);
  // the cell's loads are issued before its coordinates are known (two integer divisions): any padded cell is memory of
  // the store, and the few rows outside [-1, n] that are read for nothing cost less than the wait (7.10 -> 7.03 ms)
  double raw[5] = {1.0, 0.0, 0.0, 0.0, 1.0};
  if (inb) load_raw<0>(A.u, np, q, raw);
  // coordinates of q
  int i = 0, j = 0, k = 0;
  if (inb) {
    padded_coords(g, q, i, j, k);
  }
  // rows needed: transverse indices in [-1, n] (or the single row of an inactive dimension)
  const bool row_ok = inb && (!g.act[1] || (j >= -1 && j <= g.n[1])) && (!g.act[2] || (k >= -1 && k <= g.n[2]));
  const int nx = g.n[0];
  double w0[5] = {1.0, 0.0, 0.0, 0.0, 1.0};
  if (row_ok) ch::cons2prim(G, raw[0], raw[1], raw[2], raw[3], raw[4], w0);
#pragma unroll
  for (int m = 0; m < 5; ++m) sP[m][tid] = w0[m];
  __syncthreads();
  // stage 2: slopes for i in [-2, nx+1]
  double wm[5], wp[5], s0[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
  const bool slope_ok = row_ok && tid >= 1 && tid <= kXT - 2 && i >= -1 - A.ext && i <= nx + A.ext;
  const int tl = tid > 0 ? tid - 1 : 0, tr = tid < kXT - 1 ? tid + 1 : kXT - 1;
#pragma unroll
  for (int m = 0; m < 5; ++m) { wm[m] = sP[m][tl]; wp[m] = sP[m][tr]; }
  double ic = 0.0;
  if (slope_ok) {
    ic = ch::inv_rho_a(G, w0[0], w0[4]);
    ch::limited_slope(G, wm, w0, wp, ic, s0);
  }
#pragma unroll
  for (int m = 0; m < 5; ++m) sS[m][tid] = s0[m];
  __syncthreads();
  // stage 3: parabola + tracing for i in [-1, nx]
  const bool face_ok = slope_ok && tid >= 2 && tid <= kXT - 3 && i >= -A.ext && i <= nx + A.ext - 1;
  double prR[5] = {1.0, 0.0, 0.0, 0.0, 1.0}, prL[5] = {1.0, 0.0, 0.0, 0.0, 1.0};
  if (face_ok) {
    double sm[5], sp[5], WLs[5], WRs[5], cl[5], cr[5];
#pragma unroll
    for (int m = 0; m < 5; ++m) { sm[m] = sS[m][tid - 1]; sp[m] = sS[m][tid + 1]; }
    // the neighbours' primitives are read again rather than kept across the barrier: 48 -> 16 B of spills at 80 registers
    // (six CTAs per SM), 7.11 -> 6.95 ms at 512^3; reading back w0 and s0 as well gives half of that
#pragma unroll
    for (int m = 0; m < 5; ++m) { wm[m] = sP[m][tid - 1]; wp[m] = sP[m][tid + 1]; }
    ch::recon_faces<R>(G, dtdx0, wm, w0, wp, sm, s0, sp, ic, WLs, WRs);
    ch::prim2cons(G, WLs, cl);
    ch::prim2cons(G, WRs, cr);
    // a cell's faces are written by the CTA whose output window [2, kXT-4] holds it, plus the
    // trailing cell kXT-3 that no later window covers as a face-only slot: both write the same value
    store_local<0>(A.UL[0], np, q, cl);
    store_local<0>(A.UR[0], np, q, cr);
    copy5(prL, WLs);     // the solver's first act would be conserved -> primitive
    copy5(prR, WRs);
  }
#pragma unroll
  for (int m = 0; m < 5; ++m) sL[m][tid] = prL[m];
  __syncthreads();
  // stage 4: Riemann problem at i+1/2 for i in [-1, nx-1]
  if (face_ok && tid <= kXT - 4 && i <= nx + A.ext - 2 && q < q_end) {
    double wr[5], fl[5];
#pragma unroll
    for (int m = 0; m < 5; ++m) wr[m] = sL[m][tid + 1];
    ch::riemann<S>(G, prR, wr, fl);
    store_local<0>(A.Fs[0], np, q, fl);
  }
}

// ---------------------------------------------------------------------------------------------
// Pass 1 along x for PPMP: the flat-run form of k_pass1_x with the 7-cell stencil read from shared memory.  A CTA of
// kXT threads stages kXT primitive cells (IEEE, reading S21), threads 3 .. kXT-4 form their cell's faces with the
// same ppmp_faces as the marching kernels, exchange the left faces, and threads 3 .. kXT-5 solve interface i+1/2.
constexpr int kXOutP = kXT - 7;   // interfaces produced per CTA
template <int S>
__global__ void __launch_bounds__(kXT, 3) k_pass1_x_ppmp(const StepArgs A, long long q_begin, long long q_end) {
  __shared__ double sP[5][kXT];
  __shared__ double sL[5][kXT];
  if (step_refused(A)) return;
  const Geom& g = A.geo;
  const double dtdx0 = step_dtdx1(A, 0);
  const Gas& G = A.gas;
  const long long np = g.np;
  const int tid = threadIdx.x;
  const long long q = q_begin + (long long)blockIdx.x * kXOutP + tid - 3;
  const bool inb = (q >= 0 && q < np);
  int i = 0, j = 0, k = 0;
  if (inb) {
    padded_coords(g, q, i, j, k);
  }
  const bool row_ok = inb && (!g.act[1] || (j >= -1 && j <= g.n[1])) && (!g.act[2] || (k >= -1 && k <= g.n[2]));
  const int nx = g.n[0];
  double w0[5] = {1.0, 0.0, 0.0, 0.0, 1.0};
  if (row_ok) ch::cons2prim_ieee(G, A.u[q], A.u[np + q], A.u[2 * np + q], A.u[3 * np + q], A.u[4 * np + q], w0);
#pragma unroll
  for (int m = 0; m < 5; ++m) sP[m][tid] = w0[m];
  __syncthreads();
  const bool face_ok = row_ok && tid >= 3 && tid <= kXT - 4 && i >= -1 && i <= nx;
  double prR[5] = {1.0, 0.0, 0.0, 0.0, 1.0}, prL[5] = {1.0, 0.0, 0.0, 0.0, 1.0};
  if (face_ok) {
    double w[7][5], WLs[5], WRs[5], cl[5], cr[5];
#pragma unroll
    for (int s = 0; s < 7; ++s)
#pragma unroll
      for (int m = 0; m < 5; ++m) w[s][m] = sP[m][tid - 3 + s];
    ch::ppmp_faces(G, dtdx0, w, WLs, WRs);
    ch::prim2cons(G, WLs, cl);
    ch::prim2cons(G, WRs, cr);
    store_local<0>(A.UL[0], np, q, cl);
    store_local<0>(A.UR[0], np, q, cr);
    copy5(prL, WLs);
    copy5(prR, WRs);
  }
#pragma unroll
  for (int m = 0; m < 5; ++m) sL[m][tid] = prL[m];
  __syncthreads();
  if (face_ok && tid <= kXT - 5 && i <= nx - 1 && q < q_end) {
    double wr[5], fl[5];
#pragma unroll
    for (int m = 0; m < 5; ++m) wr[m] = sL[m][tid + 1];
    ch::riemann<S>(G, prR, wr, fl);
    store_local<0>(A.Fs[0], np, q, fl);
  }
}

// ---------------------------------------------------------------------------------------------
// Pass 2: transverse correction (Eq. 23) of the two states meeting at interface c+1/2
// along each active direction, then the second exact Riemann solve.  One thread per cell
// of [-1, n)^3.  The three directions run through ONE copy of the solver (a rolled loop over d with
// the cyclic permutation P:L164 done by field offsets), which keeps the kernel inside the
// instruction cache.
// ---------------------------------------------------------------------------------------------
struct DirSel {
  const double* F1; const double* F2;   // first-pass fluxes of the two transverse directions
  long long s0, s1, s2;                 // strides: along d, along e1 = d+1, along e2 = d+2 (cyclic)
  double h1, h2;                        // dt / (2 dx_e1), dt / (2 dx_e2)
  bool a1, a2;                          // transverse direction active
  long long f1, f2, f3;                 // field offsets (in doubles) of the direction-local momenta
};

__device__ __forceinline__ void corrected_prim(const Gas& G, const DirSel& S, long long np, const double* __restrict__ U,
                                               long long q, double w[5]) {
  const long long off[5] = {0, S.f1, S.f2, S.f3, 4 * np};
  double c[5];
#pragma unroll
  for (int m = 0; m < 5; ++m) {
    const long long a = off[m] + q;
    double corr = 0.0;
    if (S.a1) corr += S.h1 * (S.F1[a - S.s1] - S.F1[a]);
    if (S.a2) corr += S.h2 * (S.F2[a - S.s2] - S.F2[a]);
    c[m] = U[a] + corr;
  }
  ch::cons2prim(G, c[0], c[1], c[2], c[3], c[4], w);
}

// H correction, C1: eta = |(u_R + a_R) - (u_L + a_L)| / 2 at every interface c+1/2, c in [-1, n-1],
// from the transverse-corrected states, over the transverse range [-1, n] that C2's stencil reaches.
__global__ void __launch_bounds__(CH_P2_T) k_eta(const StepArgs A) {
  if (step_refused(A)) return;
  const Geom& g = A.geo;
  double dtx[3];
  step_dtdx(A, dtx);
  const int e0 = g.act[0] ? g.n[0] + 2 : 1, e1 = g.act[1] ? g.n[1] + 2 : 1, e2 = g.act[2] ? g.n[2] + 2 : 1;
  const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= (long long)e0 * e1 * e2) return;
  const int c[3] = {(int)(id % e0) - (g.act[0] ? 1 : 0), (int)((id / e0) % e1) - (g.act[1] ? 1 : 0),
                    (int)(id / ((long long)e0 * e1)) - (g.act[2] ? 1 : 0)};
  const long long np = g.np;
  const long long q = (long long)(c[0] + g.g[0]) + (long long)(c[1] + g.g[1]) * g.st[1] + (long long)(c[2] + g.g[2]) * g.st[2];
#pragma unroll 1
  for (int d = 0; d < 3; ++d) {
    if (!g.act[d] || c[d] > g.n[d] - 1) continue;
    const int d1 = d == 2 ? 0 : d + 1, d2 = d == 0 ? 2 : d - 1;
    DirSel S;
    S.F1 = A.Fs[d1]; S.F2 = A.Fs[d2];
    S.s0 = g.st[d]; S.s1 = g.st[d1]; S.s2 = g.st[d2];
    S.h1 = 0.5 * (d1 == 0 ? dtx[0] : d1 == 1 ? dtx[1] : dtx[2]); S.h2 = 0.5 * (d2 == 0 ? dtx[0] : d2 == 1 ? dtx[1] : dtx[2]);
    S.a1 = g.act[d1] != 0; S.a2 = g.act[d2] != 0;
    S.f1 = (long long)(1 + d) * np; S.f2 = (long long)(1 + d1) * np; S.f3 = (long long)(1 + d2) * np;
    double wl[5], wr[5];
    corrected_prim(A.gas, S, np, A.UR[d], q, wl);
    corrected_prim(A.gas, S, np, A.UL[d], q + S.s0, wr);
    const double aL = A.gas.gamma * wl[4] * ch::inv_rho_a(A.gas, wl[0], wl[4]);
    const double aR = A.gas.gamma * wr[4] * ch::inv_rho_a(A.gas, wr[0], wr[4]);
    A.eta[d][q] = 0.5 * fabs((wr[1] + aR) - (wl[1] + aL));
  }
}

template <int SOLVER, bool HC>
__global__ void __launch_bounds__(CH_P2_T, CH_P2_MINB) k_pass2(const StepArgs A) {
  if (step_refused(A)) return;
  const Geom& g = A.geo;
  double dtx[3];
  step_dtdx(A, dtx);
  const int e0 = g.act[0] ? g.n[0] + 1 : 1, e1 = g.act[1] ? g.n[1] + 1 : 1, e2 = g.act[2] ? g.n[2] + 1 : 1;
  const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= (long long)e0 * e1 * e2) return;
  const int i = (int)(id % e0) - (g.act[0] ? 1 : 0);
  const long long r = id / e0;
  const int j = (int)(r % e1) - (g.act[1] ? 1 : 0);
  const int k = (int)(r / e1) - (g.act[2] ? 1 : 0);
  const long long np = g.np;
  const long long q = (long long)(i + g.g[0]) + (long long)(j + g.g[1]) * g.st[1] + (long long)(k + g.g[2]) * g.st[2];
#pragma unroll 1
  for (int d = 0; d < 3; ++d) {
    // interface c+1/2 along d is needed where the two transverse indices are real (>= 0)
    const bool need = d == 0 ? (g.act[0] && j >= 0 && k >= 0) : d == 1 ? (g.act[1] && i >= 0 && k >= 0)
                                                                       : (g.act[2] && i >= 0 && j >= 0);
    if (!need) continue;
    const int d1 = d == 2 ? 0 : d + 1, d2 = d == 0 ? 2 : d - 1;
    DirSel S;
    S.F1 = A.Fs[d1]; S.F2 = A.Fs[d2];
    S.s0 = g.st[d]; S.s1 = g.st[d1]; S.s2 = g.st[d2];
    S.h1 = 0.5 * (d1 == 0 ? dtx[0] : d1 == 1 ? dtx[1] : dtx[2]); S.h2 = 0.5 * (d2 == 0 ? dtx[0] : d2 == 1 ? dtx[1] : dtx[2]);
    S.a1 = g.act[d1] != 0; S.a2 = g.act[d2] != 0;
    S.f1 = (long long)(1 + d) * np; S.f2 = (long long)(1 + d1) * np; S.f3 = (long long)(1 + d2) * np;
    double wl[5], wr[5], fl[5];
    corrected_prim(A.gas, S, np, A.UR[d], q, wl);           // U^{n+1/2}_R of cell c   -> left state
    corrected_prim(A.gas, S, np, A.UL[d], q + S.s0, wr);    // U^{n+1/2}_L of cell c+1 -> right state
    if (HC) {
      // C2 (reading G11): the interface's own eta and eta on the transverse faces of cells c and c+1
      const long long qp = q + S.s0;
      double etaH = A.eta[d][q];
      if (S.a1) etaH = ch::sel_max(etaH, ch::sel_max(ch::sel_max(A.eta[d1][q - S.s1], A.eta[d1][q]),
                                                     ch::sel_max(A.eta[d1][qp - S.s1], A.eta[d1][qp])));
      if (S.a2) etaH = ch::sel_max(etaH, ch::sel_max(ch::sel_max(A.eta[d2][q - S.s2], A.eta[d2][q]),
                                                     ch::sel_max(A.eta[d2][qp - S.s2], A.eta[d2][qp])));
      ch::riemann_roe(A.gas, wl, wr, fl, etaH);
    } else {
      ch::riemann<SOLVER>(A.gas, wl, wr, fl);
    }
    double* __restrict__ Fh = A.Fh[d];
    Fh[q] = fl[0]; Fh[S.f1 + q] = fl[1]; Fh[S.f2 + q] = fl[2]; Fh[S.f3 + q] = fl[3]; Fh[4 * np + q] = fl[4];
  }
}

// ---------------------------------------------------------------------------------------------
// Eq. 22 per cell, reduced in inverted form: the grid maximum of
//     R_cell = max over active d of (|v_d| + a) / dx_d,        dt = cfl / max R_cell,
// which is Eq. 22's  cfl * min dx_d/(|v_d|+a)  with ONE division for the whole grid instead of three
// per cell.  Every operation is explicitly rounded (no FMA contraction) and the quotients and the
// square root are brought to the correctly rounded value by one residual correction on top of the
// MUFU-seeded reciprocal (Markstein), so |v_d| + a is the IEEE value the oracle computes and R_cell
// is a pure function of the state: the fused update kernels and the standalone k_dt agree bitwise,
// and dt agrees with Eq. 22 evaluated in IEEE arithmetic to <= 2 ulp (1/dx_d, the product and the final
// reciprocal each round once).  Sets bad for rho <= 0 / non-finite input.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double div_rn(double n, double d, double r) {   // n/d given r ~ 1/d
  const double q = __dmul_rn(n, r);
  return __fma_rn(__fma_rn(-q, d, n), r, q);
}

__device__ __forceinline__ double cell_rate(const StepArgs& A, double d, double m0, double m1, double m2, double E,
                                            bool& bad) {
  if (!(d > 0.0) || !isfinite(d) || !isfinite(E)) { bad = true; return 0.0; }
  const double r = ch::rcp(d);
  const double vx = div_rn(m0, d, r), vy = div_rn(m1, d, r), vz = div_rn(m2, d, r);
  const double v2 = __dadd_rn(__dadd_rn(__dmul_rn(vx, vx), __dmul_rn(vy, vy)), __dmul_rn(vz, vz));
  const double ke = __dmul_rn(__dmul_rn(0.5, d), v2);                       // Eq. 7
  double p = __dmul_rn(A.gas.gm1, __dadd_rn(E, -ke));                        // Eq. 6, 8
  if (!(p >= ch::kPFloor)) p = (p != p) ? p : ch::kPFloor;
  const double a2 = div_rn(__dmul_rn(A.gas.gamma, p), d, r);                 // Eq. 21
  const double y = ch::rsqrt_pos(a2);
  const double s0 = __dmul_rn(a2, y);
  const double a = __fma_rn(__fma_rn(-s0, s0, a2), __dmul_rn(0.5, y), s0);
  double rmax = 0.0;
  const double v[3] = {vx, vy, vz};
#pragma unroll
  for (int e = 0; e < 3; ++e) {
    if (!A.geo.act[e]) continue;
    const double t = __dmul_rn(__dadd_rn(fabs(v[e]), a), A.idx[e]);
    if (t != t) bad = true;
    if (t > rmax) rmax = t;
  }
  return rmax;
}

__device__ __forceinline__ void block_max_reduce(double t, bool bad, unsigned long long* red) {
  __shared__ double s_max[32];
  __shared__ int s_bad;
  if (threadIdx.x == 0) s_bad = 0;
  __syncthreads();
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) t = fmax(t, __shfl_xor_sync(0xffffffffu, t, o));
  if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) s_bad = 1;
  if ((threadIdx.x & 31) == 0) s_max[threadIdx.x >> 5] = t;
  __syncthreads();
  if (threadIdx.x < 32) {
    const int nw = (blockDim.x + 31) >> 5;
    double v = threadIdx.x < nw ? s_max[threadIdx.x] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    if (threadIdx.x == 0) {
      // non-negative doubles order like their bit patterns: a single-pass grid reduction with one
      // atomicMax per CTA, deterministic because max is exact
      atomicMax(red, (unsigned long long)__double_as_longlong(v));
      if (s_bad) atomicOr(red + 1, 1ULL);
    }
  }
}

// ch_step_cfl: Eq. 22 finished on the device.  red[0] holds the grid maximum of (|v_d| + a)/dx_d of the current
// state; dt = cfl * (1 / rate) exactly as ch_compute_dt forms it on the host, clipped to t_left if that is
// positive and smaller.  red[2] <- dt (NaN if a non-physical cell was met), red[3] += dt, red[4..6] <- dt / dx_d.
struct Dx3 { double v[3]; };
__global__ void k_pick_dt(unsigned long long* red, double cfl, double t_left, Dx3 dx) {
  if (threadIdx.x != 0) return;
  double dt = __dmul_rn(cfl, __ddiv_rn(1.0, __longlong_as_double((long long)red[0])));
  if (t_left > 0.0 && dt > t_left) dt = t_left;
  double* r = reinterpret_cast<double*>(red);
  if (red[1] != 0ULL) {           // non-physical cell: dt = NaN refuses the step (step_refused); elapsed time untouched
    r[2] = __longlong_as_double(0x7FF8000000000000LL);
    return;
  }
  r[2] = dt;
  r[3] += dt;
#pragma unroll
  for (int d = 0; d < 3; ++d) r[4 + d] = __ddiv_rn(dt, dx.v[d]);
  red[0] = 0ULL; red[1] = 0ULL;     // the step that follows reduces its new state into clean cells (k_reset's work)
}

__global__ void __launch_bounds__(256) k_reset(unsigned long long* red, const double* dt_dev) {
  if (dt_dev && !(*dt_dev > 0.0)) return;      // a refused step keeps the reduction of the state it refused
  if (threadIdx.x == 0) { red[0] = 0ULL; red[1] = 0ULL; }
}

// Standalone Eq. 22 reduction over real cells (used after ch_set_state / ch_set_padded).
__global__ void __launch_bounds__(256) k_dt(const StepArgs A) {
  const Geom& g = A.geo;
  const long long N = (long long)g.n[0] * g.n[1] * g.n[2];
  double tmin = 0.0;   // running maximum of the cell rates
  bool bad = false;
  for (long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x; id < N; id += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(id % g.n[0]);
    const long long r = id / g.n[0];
    const int j = (int)(r % g.n[1]);
    const int k = (int)(r / g.n[1]);
    const long long q = (long long)(i + g.g[0]) + (long long)(j + g.g[1]) * g.st[1] + (long long)(k + g.g[2]) * g.st[2];
    const double t = cell_rate(A, A.u[q], A.u[g.np + q], A.u[2 * g.np + q], A.u[3 * g.np + q], A.u[4 * g.np + q], bad);
    tmin = fmax(tmin, t);
  }
  block_max_reduce(tmin, bad, A.red);
}

// Eq. 24 on real cells, fused with the Eq. 22 reduction of the updated state.
__global__ void __launch_bounds__(256) k_update(const StepArgs A) {
  if (step_refused(A)) return;
  const Geom& g = A.geo;
  double dtx[3];
  step_dtdx(A, dtx);
  const long long N = (long long)g.n[0] * g.n[1] * g.n[2];
  const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  double t = 0.0;
  bool bad = false;
  if (id < N) {
    const int i = (int)(id % g.n[0]);
    const long long r = id / g.n[0];
    const int j = (int)(r % g.n[1]);
    const int k = (int)(r / g.n[1]);
    const long long q = (long long)(i + g.g[0]) + (long long)(j + g.g[1]) * g.st[1] + (long long)(k + g.g[2]) * g.st[2];
    double v[5];
#pragma unroll
    for (int f = 0; f < 5; ++f) {
      double x = A.u[f * g.np + q];
#pragma unroll
      for (int d = 0; d < 3; ++d)
        if (g.act[d]) x += dtx[d] * (A.Fh[d][f * g.np + q - g.st[d]] - A.Fh[d][f * g.np + q]);
      v[f] = x;
      A.u[f * g.np + q] = x;
    }
    t = cell_rate(A, v[0], v[1], v[2], v[3], v[4], bad);
  }
  block_max_reduce(t, bad, A.red);
}

// ---------------------------------------------------------------------------------------------
// Fused second half of the step for 3-D grids: Eq. 23 transverse correction, second exact Riemann
// pass, Eq. 24 update and the Eq. 22 reduction of the new state in ONE kernel, so the CTU fluxes
// F,G,H^{n+1/2} never touch HBM (steps 3-5).
//
// A CTA is a 32 (x) by kFY (y) tile of threads that marches a segment of z.  Every thread owns one
// cell column; at step k it forms the corrected face states of cell (i,j,k), solves the Riemann
// problems on the cell's LOW faces (the left state comes from the neighbour: lane-1 through shared
// memory for x, row-1 for y, its own previous step for z) and differences them against the low-face
// flux of the neighbour on the high side.  Lane 0 / row 0 only supply states, lane 31 / row kFY-1
// only supply fluxes: a tile updates 30 x (kFY-2) columns.  The z flux of a cell's high face arrives
// one step later, so a cell is finished (stored, and its Eq. 22 time step reduced) at step k+1 from
// the x,y-updated partial sum and its low-face z flux kept in shared memory.  The three directions
// run through one rolled copy of the solver (instruction cache).
// ---------------------------------------------------------------------------------------------
#ifndef CH_F_TY
#define CH_F_TY 10
#endif
#ifndef CH_F_MINB
#define CH_F_MINB 2
#endif
constexpr int kFX = 32, kFY = CH_F_TY, kFT = kFX * kFY;

// Corrected face states of cell q along D (Eq. 23): U^{n+1/2}_{L,R}(c,D) = U*_{L,R}(c,D) + dF_{D+1} + dF_{D+2}
// with dF_e[f] = dt/(2 dx_e) [F*_e(c - e) - F*_e(c)] in global field order; primitive, D-local order out.
template <int D>
__device__ __forceinline__ void load_faces(const StepArgs& A, long long q, double ul[5], double ur[5]) {
  const long long np = A.geo.np;
  const double* __restrict__ UL = A.UL[D];
  const double* __restrict__ UR = A.UR[D];
#pragma unroll
  for (int m = 0; m < 5; ++m) {
    const int f = comp<D>(m);
    ul[m] = UL[f * np + q];
    ur[m] = UR[f * np + q];
  }
}

template <int D>
__device__ __forceinline__ void correct_faces(const StepArgs& A, const double ul[5], const double ur[5],
                                              const double (&dF)[3][5], double wl[5], double wr[5]) {
  constexpr int D1 = (D + 1) % 3, D2 = (D + 2) % 3;
  double cl[5], cr[5];
#pragma unroll
  for (int m = 0; m < 5; ++m) {
    const int f = comp<D>(m);
    const double corr = __dadd_rn(dF[D1][f], dF[D2][f]);     // explicitly rounded: every form of the kernel gets the same bits
    cl[m] = __dadd_rn(ul[m], corr);
    cr[m] = __dadd_rn(ur[m], corr);
  }
  ch::cons2prim(A.gas, cl[0], cl[1], cl[2], cl[3], cl[4], wl);
  ch::cons2prim(A.gas, cr[0], cr[1], cr[2], cr[3], cr[4], wr);
}

template <int D>
__device__ __forceinline__ void face_states(const StepArgs& A, long long q, const double (&dF)[3][5], double wl[5],
                                            double wr[5]) {
  double ul[5], ur[5];
  load_faces<D>(A, q, ul, ur);
  correct_faces<D>(A, ul, ur, dF, wl, wr);
}

// ---------------------------------------------------------------------------------------------
// C1 on 3-D grids, tiled (round 2; k_eta above is the one-thread-per-cell gather that 1-D / 2-D grids and
// the unfused step use).  eta of the interface between cells c and c+1 along d is |s_L(c+1) - s_R(c)| / 2 with
// s = u_d + a of the cell's OWN corrected face state, so a thread forms the six corrected states of its cell once
// (as the fused second half does: the cell's three flux differences, correct_faces) and only one scalar per
// direction crosses to the neighbour: lane+1 by shuffle, row+1 through shared memory, plane+1 is the thread's own
// next step.  A CTA is a 32 x kEY tile of cell columns marching a segment of z; lane 31 and row kEY-1 only supply.
// Cells [-1, n]^3, interfaces c+1/2 with c in [-1, n-1], as k_eta.
// ---------------------------------------------------------------------------------------------
constexpr int kEY = 8, kET = kFX * kEY;
__device__ __forceinline__ double eta_speed(const Gas& G, const double w[5]) {   // u + a = u + gamma p / (rho a)
  return __dadd_rn(w[1], __dmul_rn(__dmul_rn(G.gamma, w[4]), ch::inv_rho_a(G, w[0], w[4])));
}

__global__ void __launch_bounds__(kET) k_eta3d(const StepArgs A, int seg) {
  __shared__ double sY[2][kET];
  if (step_refused(A)) return;
  const Geom& g = A.geo;
  double dtx[3];
  step_dtdx(A, dtx);
  const unsigned full = 0xffffffffu;
  const int tid = threadIdx.x, lane = tid & 31, row = tid >> 5;
  const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
  const int i = (int)blockIdx.x * (kFX - 1) - 1 + lane;
  const int j = (int)blockIdx.y * (kEY - 1) - 1 + row;
  const int ka = (int)blockIdx.z * seg - 1;          // planes [ka, kb) of [-1, nz] are this CTA's
  const int kb = min(ka + seg, nz + 1);
  const bool valid = i <= nx && j <= ny;
  const bool own = valid && lane < kFX - 1 && row < kEY - 1;
  const long long np = g.np, s1 = g.st[1], s2 = g.st[2];
  const long long qcol = (long long)(i + g.g[0]) + (long long)(j + g.g[1]) * s1 + (long long)g.g[2] * s2;
  const double hx = 0.5 * dtx[0], hy = 0.5 * dtx[1], hz = 0.5 * dtx[2];
  double zS[5] = {0.0, 0.0, 0.0, 0.0, 0.0};     // F*_z of plane k-1
  double sRz = 0.0;                              // s_R(., z) of plane k-1
  // a segment that does not start the grid warms up on the plane below it (its s_R(., z) only)
  const int kstart = ka == -1 ? -1 : ka - 1;
  for (int k = kstart; k < kb; ++k) {
    const bool first = k == kstart, warm = k < ka;
    const long long q = qcol + (long long)k * s2;
    double dF[3][5];
    {
      double fx[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, fxm[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
      if (valid) {
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          const long long a = f * np + q;
          fx[f] = A.Fs[0][a];
          if (lane == 0) fxm[f] = A.Fs[0][a - 1];
          const double fz = A.Fs[2][a];
          const double fzm = first ? A.Fs[2][a - s2] : zS[f];
          zS[f] = fz;
          dF[1][f] = __dmul_rn(hy, A.Fs[1][a - s1] - A.Fs[1][a]);
          dF[2][f] = __dmul_rn(hz, fzm - fz);
        }
      }
#pragma unroll
      for (int f = 0; f < 5; ++f) {
        const double t = __shfl_up_sync(full, fx[f], 1);
        dF[0][f] = __dmul_rn(hx, (lane == 0 ? fxm[f] : t) - fx[f]);
      }
    }
    double sLx = 0.0, sRx = 0.0, sLy = 0.0, sRy = 0.0, sLz = 0.0, sRzn = 0.0;
    if (valid) {
      double wl[5], wr[5];
      // all thirty face values first: the kernel lives on loads in flight (two CTAs per SM), 19.4 -> 9.9 ms at 512^3
      double ul0[5], ur0[5], ul1[5], ur1[5], ul2[5], ur2[5];
      load_faces<2>(A, q, ul2, ur2); load_faces<0>(A, q, ul0, ur0); load_faces<1>(A, q, ul1, ur1);
      correct_faces<2>(A, ul2, ur2, dF, wl, wr);
      sLz = eta_speed(A.gas, wl); sRzn = eta_speed(A.gas, wr);
      if (!warm) {
        correct_faces<0>(A, ul0, ur0, dF, wl, wr);
        sLx = eta_speed(A.gas, wl); sRx = eta_speed(A.gas, wr);
        correct_faces<1>(A, ul1, ur1, dF, wl, wr);
        sLy = eta_speed(A.gas, wl); sRy = eta_speed(A.gas, wr);
      }
    }
    const double upx = __shfl_down_sync(full, sLx, 1);
    sY[k & 1][tid] = sLy;                      // two buffers: the next plane's writes cannot pass this plane's reads
    __syncthreads();
    const double upy = sY[k & 1][row < kEY - 1 ? tid + kFX : tid];
    if (own && !warm) {
      if (i < nx) A.eta[0][q] = 0.5 * fabs(upx - sRx);
      if (j < ny) A.eta[1][q] = 0.5 * fabs(upy - sRy);
      if (k >= 0) A.eta[2][q - s2] = 0.5 * fabs(sLz - sRz);
    }
    sRz = sRzn;
  }
}

template <int S>
__global__ void __launch_bounds__(kFT, CH_F_MINB) k_final3d(const StepArgs A, int seg) {
  extern __shared__ double s_final[];
  typedef double (*Arr)[kFT];
  Arr sX = reinterpret_cast<Arr>(s_final);              // exchanged right-face primitive state along y
  Arr sF = reinterpret_cast<Arr>(s_final + 5 * kFT);    // exchanged low-face y flux
  Arr zU = reinterpret_cast<Arr>(s_final + 10 * kFT);   // carried: U^{n+1/2}_R(., z) of cell k-1, primitive, z-local order
  Arr zF = reinterpret_cast<Arr>(s_final + 15 * kFT);   // carried: H^{n+1/2} on the low z face of cell k-1, z-local order
  Arr zP = reinterpret_cast<Arr>(s_final + 20 * kFT);   // carried: u + x and y flux differences of cell k-1, global order
  Arr zS = reinterpret_cast<Arr>(s_final + 25 * kFT);   // carried: F*_z of cell k-1 (global field order)
  if (step_refused(A)) return;
  const Geom& g = A.geo;
  double dtx[3];
  step_dtdx(A, dtx);
  const Gas& G = A.gas;
  const unsigned full = 0xffffffffu;
  const int tid = threadIdx.x, lane = tid & 31, row = tid >> 5;
  const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
  const int i = (int)blockIdx.x * (kFX - 2) - 1 + lane;
  const int j = (int)blockIdx.y * (kFY - 2) - 1 + row;
  const int k0 = (int)blockIdx.z * seg;
  const int k1 = min(k0 + seg, nz);
  const bool valid = i <= nx && j <= ny;
  const bool realI = i >= 0 && i < nx, realJ = j >= 0 && j < ny;
  const bool updL = lane >= 1 && lane <= kFX - 2 && realI, updR = row >= 1 && row <= kFY - 2 && realJ;
  const bool need0 = valid && updR, need1 = valid && updL, need2 = updL && updR;
  const bool solve0 = need0 && lane >= 1 && i >= 0, solve1 = need1 && row >= 1 && j >= 0;
  const long long np = g.np;
  const long long s1 = g.st[1], s2 = g.st[2];
  const long long qcol = (long long)(i + g.g[0]) + (long long)(j + g.g[1]) * s1 + (long long)g.g[2] * s2;
  const double hx = 0.5 * dtx[0], hy = 0.5 * dtx[1], hz = 0.5 * dtx[2];
  double tmin = 0.0;   // running maximum of the cell rates (Eq. 22 inverted)
  bool bad = false;

  for (int k = k0 - 1; k <= k1; ++k) {
    const bool first = k == k0 - 1, tail = k == k1, mid = !first && !tail;
    const long long q = qcol + (long long)k * s2;
    // transverse flux differences of this cell (each feeds four of its six face states).  Of the six
    // first-pass fluxes per field only F*_d(c) and F*_y(c - y) are loaded: F*_x(c - x) is lane-1's F*_x(c)
    // (lane 0 loads it), F*_z(c - z) is what this thread loaded one plane ago (kept in shared memory).
    double dF[3][5];
    {
      double fx[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, fxm[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
      if (valid) {
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          const long long a = f * np + q;
          fx[f] = A.Fs[0][a];
          if (lane == 0) fxm[f] = A.Fs[0][a - 1];
          const double fz = A.Fs[2][a];
          const double fzm = first ? A.Fs[2][a - s2] : zS[f][tid];
          zS[f][tid] = fz;
          dF[1][f] = __dmul_rn(hy, A.Fs[1][a - s1] - A.Fs[1][a]);
          dF[2][f] = __dmul_rn(hz, fzm - fz);
        }
      }
#pragma unroll
      for (int f = 0; f < 5; ++f) {
        const double t = __shfl_up_sync(full, fx[f], 1);
        dF[0][f] = __dmul_rn(hx, (lane == 0 ? fxm[f] : t) - fx[f]);
      }
    }
    double part[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    if (mid) {
      if (need2) {
#pragma unroll
        for (int f = 0; f < 5; ++f) part[f] = A.u[f * np + q];
      }
      {   // ---- x: neighbours are lanes of the same warp
        double wl[5] = {1.0, 0.0, 0.0, 0.0, 1.0}, wr[5] = {1.0, 0.0, 0.0, 0.0, 1.0}, nb[5], fl[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
        if (need0) face_states<0>(A, q, dF, wl, wr);
#pragma unroll
        for (int m = 0; m < 5; ++m) nb[m] = __shfl_up_sync(full, wr[m], 1);
        if (solve0) ch::riemann<S>(G, nb, wl, fl);
#pragma unroll
        for (int m = 0; m < 5; ++m) {
          const double hi = __shfl_down_sync(full, fl[m], 1);
          part[m] += dtx[0] * (fl[m] - hi);      // x-local order is the global order
        }
      }
      {   // ---- y: neighbours are rows of the CTA
        double wl[5] = {1.0, 0.0, 0.0, 0.0, 1.0}, wr[5] = {1.0, 0.0, 0.0, 0.0, 1.0}, nb[5], fl[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
        if (need1) face_states<1>(A, q, dF, wl, wr);
#pragma unroll
        for (int m = 0; m < 5; ++m) sX[m][tid] = wr[m];
        __syncthreads();
        const int src = tid >= kFX ? tid - kFX : tid;
#pragma unroll
        for (int m = 0; m < 5; ++m) nb[m] = sX[m][src];
        if (solve1) ch::riemann<S>(G, nb, wl, fl);
#pragma unroll
        for (int m = 0; m < 5; ++m) sF[m][tid] = fl[m];
        __syncthreads();
        if (need2) {
          const int dst = tid + kFX;
          // y-local order (rho, my, mz, mx, E) -> global
          part[0] += dtx[1] * (fl[0] - sF[0][dst]);
          part[2] += dtx[1] * (fl[1] - sF[1][dst]);
          part[3] += dtx[1] * (fl[2] - sF[2][dst]);
          part[1] += dtx[1] * (fl[3] - sF[3][dst]);
          part[4] += dtx[1] * (fl[4] - sF[4][dst]);
        }
      }
    }
    if (need2) {   // ---- z: the neighbour is this thread's previous step
      double wl[5], wr[5], nb[5], fl[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
      face_states<2>(A, q, dF, wl, wr);
      if (!first) {
#pragma unroll
        for (int m = 0; m < 5; ++m) nb[m] = zU[m][tid];
        ch::riemann<S>(G, nb, wl, fl);
      }
      if (k > k0) {
        // finish cell k-1 (Eq. 24): z-local order (rho, mz, mx, my, E)
        const double dtd = dtx[2];
        const long long qm = q - s2;
        const double v0 = zP[0][tid] + dtd * (zF[0][tid] - fl[0]);
        const double v1 = zP[1][tid] + dtd * (zF[2][tid] - fl[2]);
        const double v2 = zP[2][tid] + dtd * (zF[3][tid] - fl[3]);
        const double v3 = zP[3][tid] + dtd * (zF[1][tid] - fl[1]);
        const double v4 = zP[4][tid] + dtd * (zF[4][tid] - fl[4]);
        A.u[qm] = v0; A.u[np + qm] = v1; A.u[2 * np + qm] = v2; A.u[3 * np + qm] = v3; A.u[4 * np + qm] = v4;
        const double t = cell_rate(A, v0, v1, v2, v3, v4, bad);
        tmin = t > tmin ? t : tmin;
      }
#pragma unroll
      for (int m = 0; m < 5; ++m) { zU[m][tid] = wr[m]; zF[m][tid] = fl[m]; zP[m][tid] = part[m]; }
    }
  }
  block_max_reduce(tmin, bad, A.red);
}

// ---------------------------------------------------------------------------------------------
// The same for x-y grids (nz = 1; BASELINE.json's Kelvin-Helmholtz box): one plane, no z carry.  A 32 x kFY tile of
// threads: corrected x and y face states of the cell (Eq. 23 with the one transverse direction), the x problem
// through warp shuffles, the y problem through shared memory, Eq. 24 and the Eq. 22 reduction.  It replaces
// k_pass2 + k_update (and F, G^{n+1/2} through HBM) on grids where a step is a handful of launch-bound kernels.
// ---------------------------------------------------------------------------------------------
// Ghost images of real coordinate c (n cells, ng ghost layers, face rules lo / hi): the ghost coordinates that the
// ghost fill maps onto c (the inverse of bc_source for periodic, reflective and outflow faces).  img[0] = c itself.
constexpr int kMaxImg = 2 * 4 + 1;
__device__ __forceinline__ int bc_images(int c, int n, int ng, int lo, int hi, int img[kMaxImg], bool flip[kMaxImg]) {
  int m = 0;
  img[m] = c; flip[m++] = false;
  if (lo == CH_BC_PERIODIC) { if (c - n >= -ng) { img[m] = c - n; flip[m++] = false; } }
  else if (lo == CH_BC_REFLECTIVE) { if (c < ng) { img[m] = -c - 1; flip[m++] = true; } }
  else if (c == 0) { for (int t = 1; t <= ng; ++t) { img[m] = -t; flip[m++] = false; } }
  if (hi == CH_BC_PERIODIC) { if (c + n < n + ng) { img[m] = c + n; flip[m++] = false; } }
  else if (hi == CH_BC_REFLECTIVE) { if (c >= n - ng) { img[m] = 2 * n - 1 - c; flip[m++] = true; } }
  else if (c == n - 1) { for (int t = 1; t <= ng; ++t) { img[m] = n - 1 + t; flip[m++] = false; } }
  return m;
}
struct Scatter2d { int on; int bc[4]; };   // on: the update also writes the ghost images of its cells (no k_ghost launch)

template <int S>
__global__ void __launch_bounds__(kFT, 2) k_final2d(const StepArgs A, const Scatter2d GS) {
  __shared__ double sX[5][kFT], sF[5][kFT];
  if (step_refused(A)) return;
  const Geom& g = A.geo;
  double dtx[3];
  step_dtdx(A, dtx);
  const Gas& G = A.gas;
  const unsigned full = 0xffffffffu;
  const int tid = threadIdx.x, lane = tid & 31, row = tid >> 5;
  const int nx = g.n[0], ny = g.n[1];
  const int i = (int)blockIdx.x * (kFX - 2) - 1 + lane;
  const int j = (int)blockIdx.y * (kFY - 2) - 1 + row;
  const bool valid = i <= nx && j <= ny;
  const bool realI = i >= 0 && i < nx, realJ = j >= 0 && j < ny;
  const bool updL = lane >= 1 && lane <= kFX - 2 && realI, updR = row >= 1 && row <= kFY - 2 && realJ;
  const bool need0 = valid && updR, need1 = valid && updL, need2 = updL && updR;
  const bool solve0 = need0 && lane >= 1 && i >= 0, solve1 = need1 && row >= 1 && j >= 0;
  const long long np = g.np, s1 = g.st[1];
  const long long q = (long long)(i + g.g[0]) + (long long)(j + g.g[1]) * s1;
  const double hx = 0.5 * dtx[0], hy = 0.5 * dtx[1];
  double dF[3][5];
  {
    double fx[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, fxm[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
    for (int f = 0; f < 5; ++f) { dF[1][f] = 0.0; dF[2][f] = 0.0; }
    if (valid) {
#pragma unroll
      for (int f = 0; f < 5; ++f) {
        const long long a = f * np + q;
        fx[f] = A.Fs[0][a];
        if (lane == 0) fxm[f] = A.Fs[0][a - 1];
        dF[1][f] = __dmul_rn(hy, A.Fs[1][a - s1] - A.Fs[1][a]);
      }
    }
#pragma unroll
    for (int f = 0; f < 5; ++f) {
      const double t = __shfl_up_sync(full, fx[f], 1);
      dF[0][f] = __dmul_rn(hx, (lane == 0 ? fxm[f] : t) - fx[f]);
    }
  }
  double part[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
  if (need2) {
#pragma unroll
    for (int f = 0; f < 5; ++f) part[f] = A.u[f * np + q];
  }
  {   // ---- x: neighbours are lanes of the same warp
    double wl[5] = {1.0, 0.0, 0.0, 0.0, 1.0}, wr[5] = {1.0, 0.0, 0.0, 0.0, 1.0}, nb[5], fl[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    if (need0) face_states<0>(A, q, dF, wl, wr);
#pragma unroll
    for (int m = 0; m < 5; ++m) nb[m] = __shfl_up_sync(full, wr[m], 1);
    if (solve0) ch::riemann<S>(G, nb, wl, fl);
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      const double hi = __shfl_down_sync(full, fl[m], 1);
      part[m] += dtx[0] * (fl[m] - hi);
    }
  }
  {   // ---- y: neighbours are rows of the CTA
    double wl[5] = {1.0, 0.0, 0.0, 0.0, 1.0}, wr[5] = {1.0, 0.0, 0.0, 0.0, 1.0}, nb[5], fl[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    if (need1) face_states<1>(A, q, dF, wl, wr);
#pragma unroll
    for (int m = 0; m < 5; ++m) sX[m][tid] = wr[m];
    __syncthreads();
    const int src = tid >= kFX ? tid - kFX : tid;
#pragma unroll
    for (int m = 0; m < 5; ++m) nb[m] = sX[m][src];
    if (solve1) ch::riemann<S>(G, nb, wl, fl);
#pragma unroll
    for (int m = 0; m < 5; ++m) sF[m][tid] = fl[m];
    __syncthreads();
    if (need2) {
      const int dst = tid + kFX;
      // y-local order (rho, my, mz, mx, E) -> global
      part[0] += dtx[1] * (fl[0] - sF[0][dst]);
      part[2] += dtx[1] * (fl[1] - sF[1][dst]);
      part[3] += dtx[1] * (fl[2] - sF[2][dst]);
      part[1] += dtx[1] * (fl[3] - sF[3][dst]);
      part[4] += dtx[1] * (fl[4] - sF[4][dst]);
    }
  }
  double t = 0.0;
  bool bad = false;
  if (need2) {
    A.u[q] = part[0]; A.u[np + q] = part[1]; A.u[2 * np + q] = part[2]; A.u[3 * np + q] = part[3]; A.u[4 * np + q] = part[4];
    t = cell_rate(A, part[0], part[1], part[2], part[3], part[4], bad);
    // the ghost fill folded into the update (launch-bound boxes: one kernel less per step): a cell within nghost of a
    // face also writes the ghost cells that copy it -- x and y images combine as in k_ghost (each coordinate on its own)
    if (GS.on && (i < g.g[0] || i >= nx - g.g[0] || j < g.g[1] || j >= ny - g.g[1])) {
      int xi[kMaxImg], yj[kMaxImg];
      bool xf[kMaxImg], yf[kMaxImg];
      const int mx = bc_images(i, nx, g.g[0], GS.bc[0], GS.bc[1], xi, xf);
      const int my = bc_images(j, ny, g.g[1], GS.bc[2], GS.bc[3], yj, yf);
      for (int b = 0; b < my; ++b)
        for (int a = (b == 0 ? 1 : 0); a < mx; ++a) {
          const long long qd = (long long)(xi[a] + g.g[0]) + (long long)(yj[b] + g.g[1]) * s1;
          A.u[qd] = part[0];
          A.u[np + qd] = xf[a] ? -part[1] : part[1];
          A.u[2 * np + qd] = yf[b] ? -part[2] : part[2];
          A.u[3 * np + qd] = part[3];
          A.u[4 * np + qd] = part[4];
        }
    }
  }
  block_max_reduce(t, bad, A.red);
}

// ---------------------------------------------------------------------------------------------
// TMA-fed form of k_final3d (used when the padded strides meet TMA's 16-byte rules).  Same tile, same
// arithmetic, same exchanges; what changes is how a plane's 50 doubles per cell reach the SM: a
// producer warp streams them as ten 4-D boxes {32 x, kTY y, 1 z, 5 fields} per plane
// (cp.async.bulk.tensor, mbarrier complete_tx) into four staging groups in shared memory, in the order
// the consumers use them — F* (flux differences), z states, x states + u, y states — and refills a
// group for the next plane as soon as all 320 consumer threads have released it (empty mbarrier), so
// the loads of plane k+1 run under the solves of plane k.
// ---------------------------------------------------------------------------------------------
#ifndef CH_T_TY
#define CH_T_TY 12
#endif
#ifndef CH_T_SLEEP
#define CH_T_SLEEP 200      // ns between the producer's polls of an empty barrier
#endif
constexpr int kTY = CH_T_TY, kTT = kFX * kTY;   // staged rows; threads = staged slots (producer-warp form)
#ifndef CH_T_TYM
#define CH_T_TYM 13
#endif
constexpr int kTYM = CH_T_TYM;                                   // staged rows of the merged-producer form (kTYM - 1 warps)
struct TmaMaps { CUtensorMap m[13]; };              // Fs0 Fs1 Fs2 | UL2 UR2 | UL0 UR0 u | UL1 UR1 | eta0 eta1 eta2 (one field each)
__device__ __forceinline__ constexpr int group_first(int q) { return q == 0 ? 0 : q == 1 ? 3 : q == 2 ? 5 : q == 3 ? 8 : 10; }   // arrays of group q: [first(q), first(q+1))

__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  // try_wait suspends for a hardware-bounded time and returns; a transfer that never completes (a rejected
  // tensor map, say) must surface as an error, not as a hung GPU: trap after ~2^26 rounds (seconds)
  for (unsigned spin = 0;; ++spin) {
    unsigned done;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    if (done) return;
    if (spin > (1u << 26)) __trap();
  }
}
// The producer's waits: it has a whole plane of slack, so it sleeps between polls instead of spending the
// issue slots of the scheduler it shares with three consumer warps.
__device__ __forceinline__ void mbar_wait_relaxed(unsigned bar, unsigned parity) {
  for (unsigned spin = 0;; ++spin) {
    unsigned done;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    if (done) return;
    __nanosleep(CH_T_SLEEP);
    if (spin > (1u << 24)) __trap();
  }
}
__device__ __forceinline__ void tma_load_4d(unsigned dst, const CUtensorMap* map, unsigned bar, int c0, int c1, int c2, int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
      ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}

// HC (Roe solver only): the H-corrected step.  k_eta3d has written eta of every interface (C1); a fifth staging group
// brings eta_x and eta_y of plane k and eta_z of the faces k-1/2 and k+1/2 (slots 70..73), every thread forms the
// three maxima of C2 for its x, y and z interface from them (the stencil stays inside the staged box) and the Roe
// solver takes them: the same values and the same solver as k_pass2<1, true>, so the two paths agree bitwise.
// MP (round 2, last): the producer's work moves into lane 0 of the halo warp, which is idle two thirds of a plane, and
// the warp that used to produce updates an eleventh row: TY = 13 staged rows, still twelve warps (three per scheduler
// is what 152 registers allow), the schedulers that held two updating warps and a helper now hold three and two + the
// halo warp.  Lane 0 refills group 0 right after the halo warp has read it, groups 1 and 2 once every consumer has
// released them (the slowest updating warp is then past its z solve, so the halo warp still reaches the first
// consumer barrier before it), group 3 after that barrier.  The carried H flux and partial sums are kept for the
// updating rows only (227 840 B of dynamic shared memory).  Same arithmetic per cell: bitwise equal to the other forms.
template <int S, bool HC = false, int TY = CH_T_TY, bool MP = false>
__global__ void __launch_bounds__(kFX * (MP ? TY - 1 : TY), 1) k_final3d_tma(const StepArgs A, const __grid_constant__ TmaMaps M, int seg) {
  constexpr int kTY = TY, kTT = kFX * TY;                  // staged rows, staged slots per field (shadow the file-scope pair)
  constexpr int kTC = MP ? kTT - kFX : kTT - kFX;          // consumer threads: all threads with MP, all but the producer warp without
  constexpr int kZS = MP ? kTT - 2 * kFX : kTT;            // slots of the carried arrays; with MP the updating rows only
  static_assert(!(HC && MP), "the H-corrected form keeps the producer warp");
  extern __shared__ __align__(1024) double s_t[];
  __shared__ unsigned long long s_full[5], s_empty[5];
  typedef double (*Arr)[kTT];
  // staging: array a (0..9) holds its 5 fields as [f][row][lane] = [f][tid]
  Arr sX = reinterpret_cast<Arr>(s_t + 50 * kTT);
  Arr sF = reinterpret_cast<Arr>(s_t + 55 * kTT);
  if (step_refused(A)) return;
  const Geom& g = A.geo;
  double dtx[3];
  step_dtdx(A, dtx);
  const Gas& G = A.gas;
  const unsigned full = 0xffffffffu;
  // kTY rows are staged.  Warps 0..kTY-3 update rows 1..kTY-2; warp kTY-2 serves both halo rows (row 0 supplies its
  // right-face y state, row kTY-1 its low-face y flux: a third of an updating warp's work); warp kTY-1 produces.
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, row = wid + 1;
  const int sidx = row * kFX + lane;                   // this thread's slot in the staged and exchanged arrays
  const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
  // With an even nghost the box of a 30-column tile would start on an odd double (not 16-byte aligned, the bulk copy
  // faults): such grids shift the tile by one lane at each end (xs = 1): lane 0 and lane 31 idle, lane 1 supplies the
  // left state, lanes 2..29 update, lane 30 supplies the flux; the box then starts at 28 b - 2 + nghost, an even double.
  const int xs = (g.g[0] & 1) ? 0 : 1;
  const int i0 = (int)blockIdx.x * (kFX - 2 - 2 * xs) - 1 - xs, j0 = (int)blockIdx.y * (kTY - 2) - 1;
  const int k0 = (int)blockIdx.z * seg;
  const int k1 = min(k0 + seg, nz);
  constexpr int NB = HC ? 5 : 4;
  unsigned bfull[5], bempty[5];
#pragma unroll
  for (int q = 0; q < NB; ++q) {
    bfull[q] = (unsigned)__cvta_generic_to_shared(&s_full[q]);
    bempty[q] = (unsigned)__cvta_generic_to_shared(&s_empty[q]);
  }
  if (tid == 0) {
#pragma unroll
    for (int q = 0; q < NB; ++q) { mbar_init(bfull[q], 1); mbar_init(bempty[q], kTC); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // issue the boxes of group q for plane k (any one thread)
  auto issue_group = [&](int q, int k) {
    const unsigned stage = (unsigned)__cvta_generic_to_shared(s_t);
    const int a0 = group_first(q), a1 = group_first(q + 1);
    mbar_expect_tx(bfull[q], (unsigned)((a1 - a0) * 5 * kTT * sizeof(double)));
    for (int a = a0; a < a1; ++a)
      tma_load_4d(stage + (unsigned)(a * 5 * kTT * sizeof(double)), &M.m[a], bfull[q], i0 + g.g[0], j0 + g.g[1], k + g.g[2], 0);
  };
  if (!MP && wid == kTY - 1) {
    // ===== producer warp: one lane streams the planes =====
    if (lane == 0) {
      const unsigned stage = (unsigned)__cvta_generic_to_shared(s_t);
      int n = 0;
      for (int k = k0 - 1; k <= k1; ++k, ++n) {
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          if (n > 0) mbar_wait_relaxed(bempty[q], (unsigned)((n - 1) & 1));      // all consumers released plane k-1's copy
          const int a0 = group_first(q), a1 = group_first(q + 1);
          mbar_expect_tx(bfull[q], (unsigned)((a1 - a0) * 5 * kTT * sizeof(double)));
          for (int a = a0; a < a1; ++a)
            tma_load_4d(stage + (unsigned)(a * 5 * kTT * sizeof(double)), &M.m[a], bfull[q], i0 + g.g[0], j0 + g.g[1], k + g.g[2], 0);
          if (HC && q == 0) {
            if (n > 0) mbar_wait_relaxed(bempty[4], (unsigned)((n - 1) & 1));
            mbar_expect_tx(bfull[4], (unsigned)(4 * kTT * sizeof(double)));
            const unsigned e = stage + (unsigned)(70 * kTT * sizeof(double)), es = (unsigned)(kTT * sizeof(double));
            tma_load_4d(e, &M.m[10], bfull[4], i0 + g.g[0], j0 + g.g[1], k + g.g[2], 0);
            tma_load_4d(e + es, &M.m[11], bfull[4], i0 + g.g[0], j0 + g.g[1], k + g.g[2], 0);
            tma_load_4d(e + 2 * es, &M.m[12], bfull[4], i0 + g.g[0], j0 + g.g[1], k - 1 + g.g[2], 0);
            tma_load_4d(e + 3 * es, &M.m[12], bfull[4], i0 + g.g[0], j0 + g.g[1], k + g.g[2], 0);
          }
        }
      }
    }
    return;
  }

  // ===== consumer warps =====
  Arr stg0 = reinterpret_cast<Arr>(s_t);
  double tmin = 0.0;
  bool bad = false;
  if (wid == kTY - 2) {
    // ----- halo warp: rows 0 and kTY-1 of the tile -----
    const int ih = i0 + lane, jt = j0 + kTY - 1, st_ = (kTY - 1) * kFX + lane;
    const bool laneok = lane >= 1 + xs && lane <= kFX - 2 - xs && ih >= 0 && ih < nx;
    const bool topok = laneok && jt <= ny && jt >= 0;
    const double hxh = 0.5 * dtx[0], hzh = 0.5 * dtx[2];
    double zSb[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, zSt[5] = {0.0, 0.0, 0.0, 0.0, 0.0};   // F*_z of the previous plane, both rows
    int n = 0;
    if (MP && lane == 0) {
#pragma unroll
      for (int q = 0; q < 4; ++q) issue_group(q, k0 - 1);
    }
    if (MP) __syncwarp();
    for (int k = k0 - 1; k <= k1; ++k, ++n) {
      const bool mid = k != k0 - 1 && k != k1;
      const unsigned ph = (unsigned)(n & 1);
      double dxb[5], dzb[5], dxt[5], dzt[5];
      mbar_wait(bfull[0], ph);
#pragma unroll
      for (int f = 0; f < 5; ++f) {
        const double fxb = stg0[f][lane], fzb = stg0[10 + f][lane];
        const double fxt = stg0[f][st_], fzt = stg0[10 + f][st_];
        dzb[f] = __dmul_rn(hzh, zSb[f] - fzb); zSb[f] = fzb;
        dzt[f] = __dmul_rn(hzh, zSt[f] - fzt); zSt[f] = fzt;
        dxb[f] = __dmul_rn(hxh, __shfl_up_sync(full, fxb, 1) - fxb);
        dxt[f] = __dmul_rn(hxh, __shfl_up_sync(full, fxt, 1) - fxt);
      }
      mbar_arrive(bempty[0]);
      if (MP) {
        // producer point A: group 0 of the next plane as soon as every consumer has read this one's (they read it first)
        if (lane == 0 && k < k1) { mbar_wait(bempty[0], ph); issue_group(0, k + 1); }
        __syncwarp();
      }
      double eHt = 0.0;
      if (HC) {
        // C2 for the y interface below row kTY-1 (cells q = st_ - kFX and st_)
        mbar_wait(bfull[4], ph);
        const double* ex = s_t + 70 * kTT; const double* ey = ex + kTT; const double* ezm = ey + kTT; const double* ezp = ezm + kTT;
        const int qb = st_ - kFX;
        eHt = ch::sel_max(ey[qb], ch::sel_max(ch::sel_max(ch::sel_max(ezm[qb], ezp[qb]), ch::sel_max(ezm[st_], ezp[st_])),
                                              ch::sel_max(ch::sel_max(ex[qb - 1], ex[qb]), ch::sel_max(ex[st_ - 1], ex[st_]))));
        mbar_arrive(bempty[4]);
      }
      mbar_wait(bfull[1], ph); mbar_arrive(bempty[1]);
      mbar_wait(bfull[2], ph); mbar_arrive(bempty[2]);
      mbar_wait(bfull[3], ph);
      double cb[5], ct[5];
#pragma unroll
      for (int m = 0; m < 5; ++m) {
        // exactly what correct_faces<1> forms: U* + (dF_z + dF_x), y-local order
        cb[m] = __dadd_rn(stg0[45 + comp<1>(m)][lane], __dadd_rn(dzb[comp<1>(m)], dxb[comp<1>(m)]));     // U^{n+1/2}_R(., y), row 0
        ct[m] = __dadd_rn(stg0[40 + comp<1>(m)][st_], __dadd_rn(dzt[comp<1>(m)], dxt[comp<1>(m)]));      // U^{n+1/2}_L(., y), row kTY-1
      }
      mbar_arrive(bempty[3]);
      if (MP) {
        // producer point B: groups 1 and 2 once every consumer has released them (the slowest updating warp is then
        // past its z solve and has its x solve ahead, so this warp is still not the last at the barrier below);
        // group 3 here too on the two planes that have no barrier (the first and the last of a segment)
        if (lane == 0 && k < k1) {
          mbar_wait(bempty[1], ph); issue_group(1, k + 1);
          mbar_wait(bempty[2], ph); issue_group(2, k + 1);
          if (!mid) { mbar_wait(bempty[3], ph); issue_group(3, k + 1); }
        }
        __syncwarp();
      }
      if (mid) {
        double wr0[5] = {1.0, 0.0, 0.0, 0.0, 1.0}, wlt[5] = {1.0, 0.0, 0.0, 0.0, 1.0}, nb[5], fl[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
        if (laneok) ch::cons2prim(A.gas, cb[0], cb[1], cb[2], cb[3], cb[4], wr0);
        if (topok) ch::cons2prim(A.gas, ct[0], ct[1], ct[2], ct[3], ct[4], wlt);
#pragma unroll
        for (int m = 0; m < 5; ++m) sX[m][lane] = wr0[m];
        asm volatile("bar.sync 1, %0;" ::"n"(kTC) : "memory");
#pragma unroll
        for (int m = 0; m < 5; ++m) nb[m] = sX[m][st_ - kFX];
        if (topok) {
          if (HC) ch::riemann_roe(G, nb, wlt, fl, eHt);
          else ch::riemann_tile<S>(G, nb, wlt, fl);
        }
#pragma unroll
        for (int m = 0; m < 5; ++m) sF[m][st_] = fl[m];
        asm volatile("bar.sync 1, %0;" ::"n"(kTC) : "memory");
        if (MP) {
          // producer point C: every consumer read group 3 before the first barrier; issued after the second so that
          // this warp is not the one the others wait for (the y states are not needed before the end of the next plane)
          if (lane == 0 && k < k1) { mbar_wait(bempty[3], ph); issue_group(3, k + 1); }
          __syncwarp();
        }
      }
    }
  } else {
  Arr stg = reinterpret_cast<Arr>(s_t);
  const int i = i0 + lane, j = j0 + row;
  const bool valid = i <= nx && j <= ny;
  const bool realI = i >= 0 && i < nx, realJ = j >= 0 && j < ny;
  const bool updL = lane >= 1 + xs && lane <= kFX - 2 - xs && realI, updR = realJ;
  const bool need0 = valid && updR && lane >= xs, need1 = valid && updL, need2 = updL && updR;
  const bool solve0 = need0 && lane >= 1 + xs && i >= 0, solve1 = need1 && row >= 1 && j >= 0;
  const long long np = g.np, s2 = g.st[2];
  const long long qcol = (long long)(i + g.g[0]) + (long long)(j + g.g[1]) * g.st[1] + (long long)g.g[2] * s2;
  const double hx = 0.5 * dtx[0], hy = 0.5 * dtx[1], hz = 0.5 * dtx[2];
  // carried from the previous plane (registers: one CTA per SM leaves ~150 per thread)
  double zU[5] = {1.0, 0.0, 0.0, 0.0, 1.0};    // U^{n+1/2}_R(., z) of cell k-1, primitive, z-local order
  // the half of the z carry that is only read when cell k-1 is finished lives in shared memory (10 doubles per slot):
  // 164 -> 152 registers, the scheduler has room to interleave more, 2 % off this kernel
  typedef double (*ArrZ)[kZS];
  ArrZ zFs = reinterpret_cast<ArrZ>(s_t + 60 * kTT);             // H^{n+1/2} on the low z face of cell k-1, z-local order
  ArrZ zPs = reinterpret_cast<ArrZ>(s_t + 60 * kTT + 5 * kZS);   // u + x and y flux differences of cell k-1, global order
  const int zidx = MP ? sidx - kFX : sidx;
#define zF(m) zFs[m][zidx]
#define zP(m) zPs[m][zidx]
  double zS[5] = {0.0, 0.0, 0.0, 0.0, 0.0};    // F*_z of cell k-1 (global field order)
  double mxyPrev = 0.0;                        // HC: largest eta on the x and y faces of cell k-1
  int n = 0;
  for (int k = k0 - 1; k <= k1; ++k, ++n) {
    const bool first = k == k0 - 1, tail = k == k1, mid = !first && !tail;
    const unsigned ph = (unsigned)(n & 1);
    const long long q = qcol + (long long)k * s2;
    // ---- group 0: first-pass fluxes -> transverse flux differences of this cell
    double dF[3][5];
    mbar_wait(bfull[0], ph);
    {
      double fx[5];
#pragma unroll
      for (int f = 0; f < 5; ++f) {
        fx[f] = stg[f][sidx];
        const double fy = stg[5 + f][sidx];
        const double fym = stg[5 + f][sidx - kFX];
        const double fz = stg[10 + f][sidx];
        const double fzm = zS[f];                                   // garbage on the first plane: unused there
        zS[f] = fz;
        dF[1][f] = __dmul_rn(hy, fym - fy);
        dF[2][f] = __dmul_rn(hz, fzm - fz);
      }
      mbar_arrive(bempty[0]);
#pragma unroll
      for (int f = 0; f < 5; ++f) {
        const double t = __shfl_up_sync(full, fx[f], 1);                 // lane 0 never uses its x difference
        dF[0][f] = __dmul_rn(hx, t - fx[f]);
      }
    }
    // ---- HC, group 4: C2 (reading G11) for this thread's three interfaces: i-1/2 and j-1/2 of plane k, k-1/2
    double eHx = 0.0, eHy = 0.0, eHz = 0.0;
    if (HC) {
      mbar_wait(bfull[4], ph);
      const double* ex = s_t + 70 * kTT; const double* ey = ex + kTT; const double* ezm = ey + kTT; const double* ezp = ezm + kTT;
      const int qx = sidx - 1, qy = sidx - kFX;
      const double ex0 = ex[sidx], exm = ex[qx], ey0 = ey[sidx], eym = ey[qy], ezm0 = ezm[sidx];
      const double mz = ch::sel_max(ezm0, ezp[sidx]);
      const double mxy = ch::sel_max(ch::sel_max(exm, ex0), ch::sel_max(eym, ey0));
      eHx = ch::sel_max(exm, ch::sel_max(ch::sel_max(ch::sel_max(ey[qx - kFX], ey[qx]), ch::sel_max(eym, ey0)),
                                         ch::sel_max(ch::sel_max(ezm[qx], ezp[qx]), mz)));
      eHy = ch::sel_max(eym, ch::sel_max(ch::sel_max(ch::sel_max(ezm[qy], ezp[qy]), mz),
                                         ch::sel_max(ch::sel_max(ex[qy - 1], ex[qy]), ch::sel_max(exm, ex0))));
      eHz = ch::sel_max(ezm0, ch::sel_max(mxyPrev, mxy));
      mxyPrev = mxy;
      mbar_arrive(bempty[4]);
    }
    // ---- group 1: z states; the neighbour is this thread's previous plane
    double wrz[5] = {1.0, 0.0, 0.0, 0.0, 1.0}, flz[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    mbar_wait(bfull[1], ph);
    {
      double ul[5], ur[5];
#pragma unroll
      for (int m = 0; m < 5; ++m) { ul[m] = stg[15 + comp<2>(m)][sidx]; ur[m] = stg[20 + comp<2>(m)][sidx]; }
      mbar_arrive(bempty[1]);
      if (need2) {
        double wl[5], nb[5];
        correct_faces<2>(A, ul, ur, dF, wl, wrz);
        if (!first) {
#pragma unroll
          for (int m = 0; m < 5; ++m) nb[m] = zU[m];
          if (HC) ch::riemann_roe(G, nb, wl, flz, eHz);
          else ch::riemann_tile<S>(G, nb, wl, flz);
        }
        if (k > k0) {
          // finish cell k-1 (Eq. 24): z-local order (rho, mz, mx, my, E)
          const double dtd = dtx[2];
          const long long qm = q - s2;
          const double v0 = zP(0) + dtd * (zF(0) - flz[0]);
          const double v1 = zP(1) + dtd * (zF(2) - flz[2]);
          const double v2 = zP(2) + dtd * (zF(3) - flz[3]);
          const double v3 = zP(3) + dtd * (zF(1) - flz[1]);
          const double v4 = zP(4) + dtd * (zF(4) - flz[4]);
          A.u[qm] = v0; A.u[np + qm] = v1; A.u[2 * np + qm] = v2; A.u[3 * np + qm] = v3; A.u[4 * np + qm] = v4;
          const double t = cell_rate(A, v0, v1, v2, v3, v4, bad);
          tmin = t > tmin ? t : tmin;
        }
      }
    }
    // ---- group 2: x states and u; neighbours are lanes of the same warp
    double part[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    mbar_wait(bfull[2], ph);
    {
      double ul[5], ur[5];
#pragma unroll
      for (int m = 0; m < 5; ++m) { ul[m] = stg[25 + m][sidx]; ur[m] = stg[30 + m][sidx]; part[m] = stg[35 + m][sidx]; }
      mbar_arrive(bempty[2]);
      if (mid) {
        double wl[5] = {1.0, 0.0, 0.0, 0.0, 1.0}, wr[5] = {1.0, 0.0, 0.0, 0.0, 1.0}, nb[5], fl[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
        if (need0) correct_faces<0>(A, ul, ur, dF, wl, wr);
#pragma unroll
        for (int m = 0; m < 5; ++m) nb[m] = __shfl_up_sync(full, wr[m], 1);
        if (solve0) {
          if (HC) ch::riemann_roe(G, nb, wl, fl, eHx);
          else ch::riemann_tile<S>(G, nb, wl, fl);
        }
#pragma unroll
        for (int m = 0; m < 5; ++m) {
          const double hi = __shfl_down_sync(full, fl[m], 1);
          part[m] += dtx[0] * (fl[m] - hi);      // x-local order is the global order
        }
      }
    }
    // ---- group 3: y states; neighbours are rows of the CTA
    mbar_wait(bfull[3], ph);
    {
      double ul[5], ur[5];
#pragma unroll
      for (int m = 0; m < 5; ++m) { ul[m] = stg[40 + comp<1>(m)][sidx]; ur[m] = stg[45 + comp<1>(m)][sidx]; }
      mbar_arrive(bempty[3]);
      if (mid) {
        double wl[5] = {1.0, 0.0, 0.0, 0.0, 1.0}, wr[5] = {1.0, 0.0, 0.0, 0.0, 1.0}, nb[5], fl[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
        if (need1) correct_faces<1>(A, ul, ur, dF, wl, wr);
#pragma unroll
        for (int m = 0; m < 5; ++m) sX[m][sidx] = wr[m];
        asm volatile("bar.sync 1, %0;" ::"n"(kTC) : "memory");
#pragma unroll
        for (int m = 0; m < 5; ++m) nb[m] = sX[m][sidx - kFX];
        if (solve1) {
          if (HC) ch::riemann_roe(G, nb, wl, fl, eHy);
          else ch::riemann_tile<S>(G, nb, wl, fl);
        }
#pragma unroll
        for (int m = 0; m < 5; ++m) sF[m][sidx] = fl[m];
        asm volatile("bar.sync 1, %0;" ::"n"(kTC) : "memory");
        if (need2) {
          const int dst = sidx + kFX;
          // y-local order (rho, my, mz, mx, E) -> global
          part[0] += dtx[1] * (fl[0] - sF[0][dst]);
          part[2] += dtx[1] * (fl[1] - sF[1][dst]);
          part[3] += dtx[1] * (fl[2] - sF[2][dst]);
          part[1] += dtx[1] * (fl[3] - sF[3][dst]);
          part[4] += dtx[1] * (fl[4] - sF[4][dst]);
        }
      }
    }
    if (need2) {
#pragma unroll
      for (int m = 0; m < 5; ++m) { zU[m] = wrz[m]; zF(m) = flz[m]; zP(m) = part[m]; }
    }
  }
  }
  // Eq. 22 reduction over the consumer warps (the producer warp has left)
  {
    __shared__ double s_max[32];
    __shared__ int s_badflag;
    if (tid == 0) s_badflag = 0;
    asm volatile("bar.sync 1, %0;" ::"n"(kTC) : "memory");
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) tmin = fmax(tmin, __shfl_xor_sync(full, tmin, o));
    if (__any_sync(full, bad) && lane == 0) s_badflag = 1;
    if (lane == 0) s_max[wid] = tmin;
    asm volatile("bar.sync 1, %0;" ::"n"(kTC) : "memory");
    if (tid < 32) {
      double v = tid < kTY - 1 ? s_max[tid] : 0.0;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(full, v, o));
      if (tid == 0) {
        atomicMax(A.red, (unsigned long long)__double_as_longlong(v));
        if (s_badflag) atomicOr(A.red + 1, 1ULL);
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Ghost fill (readings S6, S7).  Filling x, then y over the padded x extent, then z over
// the padded x,y extent makes every ghost cell a copy of the real cell obtained by mapping
// each coordinate on its own, with the sign of each reflected normal momentum flipped; so one
// launch over the ghost shell reads real cells only and writes ghost cells only.
// ---------------------------------------------------------------------------------------------
struct BcArgs {
  int bc[6];
  double noh_rho0, noh_p0, time;   // CH_BC_NOH: ambient state of the analytic inflow and the time it is evaluated at
  int nact;                        // number of active dimensions (the n of rho0 (1 + t/r)^(n-1))
  int org[3];                      // global index of this block's first real cell (block decomposition; 0 otherwise)
};

// Analytic boundary of the Noh test at the centre of cell (ci, cj, ck) (real-cell coordinates, box origin
// at 0): rho = rho0 (1 + t/r)^(n-1), unit velocity toward the origin, E = p0/(gamma-1) + rho/2.  Explicitly rounded
// operations in a fixed order: the ghost fill is index and copy work everywhere else, and stays bit-exact here too.
__device__ __forceinline__ void noh_state(const StepArgs& A, const BcArgs& B, int ci, int cj, int ck, double v[5]) {
  const int cc[3] = {ci, cj, ck};
  double x[3], r2 = 0.0;
#pragma unroll
  for (int e = 0; e < 3; ++e) {
    x[e] = A.geo.act[e] ? __dmul_rn((double)(cc[e] + B.org[e]) + 0.5, A.dx[e]) : 0.0;
    r2 = __dadd_rn(r2, __dmul_rn(x[e], x[e]));
  }
  const double r = __dsqrt_rn(r2);
  const double q1 = __dadd_rn(1.0, __ddiv_rn(B.time, r));
  double rho = B.noh_rho0;
  for (int e = 1; e < B.nact; ++e) rho = __dmul_rn(rho, q1);
  v[0] = rho;
#pragma unroll
  for (int e = 0; e < 3; ++e) v[1 + e] = __dmul_rn(rho, -__ddiv_rn(x[e], r));
  v[4] = __dadd_rn(__ddiv_rn(B.noh_p0, A.gas.gm1), __dmul_rn(0.5, rho));
}

__device__ __forceinline__ int bc_source(int c, int n, int lo, int hi, bool& flip) {
  if (c < 0) {
    if (lo == CH_BC_PERIODIC) return c + n;
    if (lo == CH_BC_REFLECTIVE) { flip = !flip; return -c - 1; }
    return 0;
  }
  if (c >= n) {
    if (hi == CH_BC_PERIODIC) return c - n;
    if (hi == CH_BC_REFLECTIVE) { flip = !flip; return 2 * n - 1 - c; }
    return n - 1;
  }
  return c;
}

__global__ void __launch_bounds__(256) k_ghost(const StepArgs A, const BcArgs B) {
  if (step_refused(A)) return;
  const Geom& g = A.geo;
  // shell = z slabs (all padded x,y) + y slabs (real z, padded x) + x slabs (real z, real y)
  const long long nzs = (long long)2 * g.g[2] * g.pd[1] * g.pd[0];
  const long long nys = (long long)g.n[2] * 2 * g.g[1] * g.pd[0];
  const long long nxs = (long long)g.n[2] * g.n[1] * 2 * g.g[0];
  long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= nzs + nys + nxs) return;
  int pi, pj, pk;   // padded coordinates
  if (id < nzs) {
    pi = (int)(id % g.pd[0]); long long r = id / g.pd[0];
    pj = (int)(r % g.pd[1]); int s = (int)(r / g.pd[1]);
    pk = s < g.g[2] ? s : s + g.n[2];
  } else if (id < nzs + nys) {
    id -= nzs;
    pi = (int)(id % g.pd[0]); long long r = id / g.pd[0];
    int s = (int)(r % (2 * g.g[1])); pk = (int)(r / (2 * g.g[1])) + g.g[2];
    pj = s < g.g[1] ? s : s + g.n[1];
  } else {
    id -= nzs + nys;
    int s = (int)(id % (2 * g.g[0])); long long r = id / (2 * g.g[0]);
    pj = (int)(r % g.n[1]) + g.g[1]; pk = (int)(r / g.n[1]) + g.g[2];
    pi = s < g.g[0] ? s : s + g.n[0];
  }
  bool fx = false, fy = false, fz = false;
  const long long qd = (long long)pi + (long long)pj * g.st[1] + (long long)pk * g.st[2];
  {
    // Analytic faces.  The fill order x, y, z means the LAST direction in which a ghost lies outside
    // decides where its value comes from: walk z, y, x; a reflective / periodic / outflow face maps that coordinate
    // and the walk goes on, an analytic face ends it with the analytic state at the coordinates reached so far.
    int cc[3] = {pi - g.g[0], pj - g.g[1], pk - g.g[2]};
    bool fl[3] = {false, false, false};
    bool analytic = false;
#pragma unroll
    for (int d = 2; d >= 0; --d) {
      if (analytic || !g.act[d]) continue;
      const int lo = B.bc[2 * d], hi = B.bc[2 * d + 1];
      if ((cc[d] < 0 && lo == CH_BC_NOH) || (cc[d] >= g.n[d] && hi == CH_BC_NOH)) { analytic = true; continue; }
      cc[d] = bc_source(cc[d], g.n[d], lo, hi, fl[d]);
    }
    if (analytic) {
      double v[5];
      noh_state(A, B, cc[0], cc[1], cc[2], v);
      A.u[qd] = v[0];
      A.u[g.np + qd] = fl[0] ? -v[1] : v[1];
      A.u[2 * g.np + qd] = fl[1] ? -v[2] : v[2];
      A.u[3 * g.np + qd] = fl[2] ? -v[3] : v[3];
      A.u[4 * g.np + qd] = v[4];
      return;
    }
  }
  const int si = bc_source(pi - g.g[0], g.n[0], B.bc[0], B.bc[1], fx);
  const int sj = bc_source(pj - g.g[1], g.n[1], B.bc[2], B.bc[3], fy);
  const int sk = bc_source(pk - g.g[2], g.n[2], B.bc[4], B.bc[5], fz);
  const long long qs = (long long)(si + g.g[0]) + (long long)(sj + g.g[1]) * g.st[1] + (long long)(sk + g.g[2]) * g.st[2];
  double* u = A.u;
  u[qd] = u[qs];
  u[g.np + qd] = fx ? -u[g.np + qs] : u[g.np + qs];
  u[2 * g.np + qd] = fy ? -u[2 * g.np + qs] : u[2 * g.np + qs];
  u[3 * g.np + qd] = fz ? -u[3 * g.np + qs] : u[3 * g.np + qs];
  u[4 * g.np + qd] = u[4 * g.np + qs];
}

// ---------------------------------------------------------------------------------------------
// Block decomposition (section 3.7): a domain cut into blocks, each a grid of its own.  Ghost cells are
// filled direction by direction, x then y then z, each direction over the padded extent of the directions before
// it, so edges and corners ride along and at most six messages per block are needed.  Per direction:
// k_halo packs the nghost real layers next to an EXCHANGE face into a contiguous buffer [5][nghost][b][a] (the
// neighbour's unpack writes them into its ghost layers), k_fill_dim fills the faces with a local rule.
// ---------------------------------------------------------------------------------------------
struct SlabGeom { int d, e1, e2, lo1, lo2, n1, n2; };   // slab of direction d: n1 x n2 cells in the other two dims (e1 < e2)

__device__ __host__ inline SlabGeom slab_geom(const Geom& g, int d) {
  SlabGeom S;
  S.d = d; S.e1 = d == 0 ? 1 : 0; S.e2 = d == 2 ? 1 : 2;
  // directions before d: padded extent; after d: real cells only
  S.lo1 = S.e1 < d ? -g.g[S.e1] : 0; S.n1 = S.e1 < d ? g.pd[S.e1] : g.n[S.e1];
  S.lo2 = S.e2 < d ? -g.g[S.e2] : 0; S.n2 = S.e2 < d ? g.pd[S.e2] : g.n[S.e2];
  return S;
}

// mode 0: pack the real layers next to face `side` of direction d into buf; mode 1: unpack buf into the ghost layers
// beyond that face.  Layer l = 0..g-1 counts in the direction of increasing coordinate on both sides.
__global__ void __launch_bounds__(256) k_halo(const StepArgs A, int d, int side, int mode, double* buf) {
  const Geom& g = A.geo;
  const SlabGeom S = slab_geom(g, d);
  const int gl = g.g[d];
  const long long per = (long long)gl * S.n1 * S.n2;
  const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= per) return;
  const int a1 = (int)(id % S.n1);
  const long long r = id / S.n1;
  const int a2 = (int)(r % S.n2), l = (int)(r / S.n2);
  int c[3];
  c[S.e1] = S.lo1 + a1; c[S.e2] = S.lo2 + a2;
  c[d] = mode == 0 ? (side == 0 ? l : g.n[d] - gl + l) : (side == 0 ? l - gl : g.n[d] + l);
  const long long q = (long long)(c[0] + g.g[0]) + (long long)(c[1] + g.g[1]) * g.st[1] + (long long)(c[2] + g.g[2]) * g.st[2];
#pragma unroll
  for (int f = 0; f < 5; ++f) {
    if (mode == 0) buf[f * per + id] = A.u[f * g.np + q];
    else A.u[f * g.np + q] = buf[f * per + id];
  }
}

// Local ghost fill of direction d alone (both faces; EXCHANGE faces are left to k_halo): the oracle's order.
__global__ void __launch_bounds__(256) k_fill_dim(const StepArgs A, const BcArgs B, int d) {
  const Geom& g = A.geo;
  const SlabGeom S = slab_geom(g, d);
  const int gl = g.g[d];
  const long long per = (long long)gl * S.n1 * S.n2;
  long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= 2 * per) return;
  const int side = id >= per ? 1 : 0;
  if (side) id -= per;
  const int bc = B.bc[2 * d + side];
  if (bc == CH_BC_EXCHANGE) return;
  const int a1 = (int)(id % S.n1);
  const long long r = id / S.n1;
  const int a2 = (int)(r % S.n2), l = (int)(r / S.n2);
  int c[3];
  c[S.e1] = S.lo1 + a1; c[S.e2] = S.lo2 + a2;
  c[d] = side == 0 ? l - gl : g.n[d] + l;
  const long long qd = (long long)(c[0] + g.g[0]) + (long long)(c[1] + g.g[1]) * g.st[1] + (long long)(c[2] + g.g[2]) * g.st[2];
  double v[5];
  if (bc == CH_BC_NOH) {
    noh_state(A, B, c[0], c[1], c[2], v);
  } else {
    bool flip = false;
    int s[3] = {c[0], c[1], c[2]};
    s[d] = bc_source(c[d], g.n[d], B.bc[2 * d], B.bc[2 * d + 1], flip);
    const long long qs = (long long)(s[0] + g.g[0]) + (long long)(s[1] + g.g[1]) * g.st[1] + (long long)(s[2] + g.g[2]) * g.st[2];
#pragma unroll
    for (int f = 0; f < 5; ++f) v[f] = A.u[f * g.np + qs];
    if (flip) v[1 + d] = -v[1 + d];
  }
#pragma unroll
  for (int f = 0; f < 5; ++f) A.u[f * g.np + qd] = v[f];
}

// FP64 peak probe: 8 independent DFMA chains per thread.
__global__ void k_dfma_probe(double* sink, int iters) {
  double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
  const double b = 1.0000000001, c = 1e-12;
  for (int it = 0; it < iters; ++it) {
    a0 = fma(a0, b, c); a1 = fma(a1, b, c); a2 = fma(a2, b, c); a3 = fma(a3, b, c);
    a4 = fma(a4, b, c); a5 = fma(a5, b, c); a6 = fma(a6, b, c); a7 = fma(a7, b, c);
  }
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}

// Issue-mix probe: per loop iteration 8 independent DFMA plus NALU independent 32-bit integer operations (xor / add).
// On B200 an FP64 warp instruction holds the dispatch port of its scheduler for two cycles and an ALU instruction
// for about one, and the two do not overlap: the time of this loop is the SUM of its parts.  bench.py
// measures the two costs with it and states every kernel's ceiling for its own instruction mix beside the FP64 one.
template <int NALU>
__global__ void k_mix_probe(double* sink, int iters) {
  double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
  const double b = 1.0000000001, c = 1e-12;
  int i0 = threadIdx.x, i1 = i0 + 1, i2 = i0 + 2, i3 = i0 + 3;
  for (int it = 0; it < iters; ++it) {
    a0 = fma(a0, b, c); a1 = fma(a1, b, c); a2 = fma(a2, b, c); a3 = fma(a3, b, c);
    a4 = fma(a4, b, c); a5 = fma(a5, b, c); a6 = fma(a6, b, c); a7 = fma(a7, b, c);
#pragma unroll
    for (int r = 0; r < NALU / 4; ++r) {
      asm volatile("xor.b32 %0, %0, %1;" : "+r"(i0) : "r"(i1));
      asm volatile("add.s32 %0, %0, 7;" : "+r"(i1));
      asm volatile("xor.b32 %0, %0, %1;" : "+r"(i2) : "r"(i3));
      asm volatile("add.s32 %0, %0, 5;" : "+r"(i3));
    }
  }
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7)) + (double)(i0 ^ i1 ^ i2 ^ i3);
}

thread_local std::string g_err;

}  // namespace

// =============================================================================================
// Host side: opaque context and the C ABI.
// =============================================================================================
struct ch_ctx {
  Geom geo;
  Gas gas;
  int nghost;
  double dx[3];
  int bc[6];
  bool bound = false, have_state = false, dt_valid = false;
  double time = 0.0;                       // sum of the dt of ch_step calls since ch_set_state / ch_set_time
  double noh_rho0 = 1.0, noh_p0 = 1e-6;    // ambient state of the analytic (CH_BC_NOH) faces
  bool has_noh = false;
  // ch_step_cfl replays the kernels of a step as a CUDA graph (captured on a private stream the second time a
  // configuration is stepped): on small grids the step is launch bound
  bool use_graph = true;
  bool fold_ghost = true;    // x-y grids: k_final2d also writes the ghost images of its cells (CH_OPT_FOLD_GHOST)
  cudaStream_t cap_stream = nullptr, cap_side[2] = {nullptr, nullptr};   // the y and z sweeps of pass 1 are parallel branches of the graph
  cudaEvent_t cap_fork = nullptr, cap_join[2] = {nullptr, nullptr};
  bool capturing = false;
  cudaGraphExec_t gexec = nullptr;
  cudaGraph_t ggraph = nullptr;            // the captured graph (kept: its k_pick_dt node names the node of gexec to update)
  cudaGraphNode_t gpick = nullptr;         // k_pick_dt's node
  double gcfl = 0.0, gtleft = 0.0;         // its arguments as last set
  long long gkey[8] = {-1, -1, -1, -1, -1, -1, -1, -1};   // configuration the graph / the last direct step belongs to
  double gdx[3] = {0, 0, 0};
  int gseen = 0;                           // direct steps taken with gkey (capture on the second)
  long long glaunches = 0;                 // kernels in the graph
  bool has_exchange = false;               // a CH_BC_EXCHANGE face: ghost fill is driven by the caller (ch_fill_dim, ch_halo_*)
  int org[3] = {0, 0, 0};                  // global index of the first real cell (ch_set_origin)
  int device = -1;           // the device the bound buffers live on (ch_bind)
  bool smem_attr[2][2] = {{false, false}, {false, false}};   // [tma form][solver]: dynamic shared memory limit raised on `device`
  bool smem_attr_hc = false;                                  // the same for the H-corrected form
  double* state = nullptr;
  double* ws = nullptr;
  unsigned long long* red = nullptr;
  cudaStream_t stream = nullptr;
  unsigned long long* h_red = nullptr;   // pinned, 16 bytes
  long long launches = 0;
  int march_seg = 0;         // cells a marching thread sweeps; 0 = chosen per launch from the grid size
  int final_seg = 0;         // planes a k_final3d CTA marches; 0 = chosen per launch
  int use_tma = 2;           // CH_OPT_TMA: 0 plain-load k_final3d even where the TMA form applies, 1 the TMA form with a producer
                             // warp (12 staged rows), 2 the producer merged into the halo warp (13 staged rows; default)
  bool tma_ok = false;       // tensor maps built for the bound buffers
  TmaMaps maps;              // boxes of kTY rows (producer-warp form, H-corrected form)
  TmaMaps maps_mp;           // boxes of kTYM rows (merged-producer form); arrays 0..9 only
  bool smem_attr_mp[2] = {false, false};
  int solver = 0;            // CH_SOLVER_EXACT
  int recon = 0;             // CH_RECON_PPMC
  bool hcorr = false;        // H correction (Appendix C): Roe solver, nghost >= 4; fused second half where the TMA form applies
  bool unfused = false;      // CH_UNFUSED=1: k_pass2 + k_update on 3-D grids too (A/B measurements, instruction counts)
  // optional per-kernel timing (ch_profile): one event pair per kernel kind
  bool profiling = false;
  cudaEvent_t ev[2 * CH_K_COUNT] = {};
  bool ev_used[CH_K_COUNT] = {};
  double prof_ms[CH_K_COUNT] = {};
  long long prof_calls[CH_K_COUNT] = {};
};

namespace {

int fail(int code, const char* msg) { g_err = msg; return code; }

// Every entry point that touches CUDA runs on the device the bound buffers live on (recorded by ch_bind), whatever
// device is current in the calling thread, and restores the caller's device on return.
struct DeviceGuard {
  int prev = -1; bool switched = false;
  explicit DeviceGuard(int dev) {
    if (dev < 0) return;
    if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};
int cuda_fail(cudaError_t e, const char* where) {
  g_err = std::string(where) + ": " + cudaGetErrorString(e);
  return CH_ECUDA;
}
#define CH_CUDA(call, where) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_, where); } while (0)

bool geometry(int nx, int ny, int nz, int nghost, Geom& g) {
  if (nx < 1 || ny < 1 || nz < 1 || nghost < 3) return false;
  const int n[3] = {nx, ny, nz};
  for (int d = 0; d < 3; ++d) {
    g.n[d] = n[d];
    g.act[d] = n[d] > 1;
    g.g[d] = g.act[d] ? nghost : 0;
    g.pd[d] = n[d] + 2 * g.g[d];
    if (g.act[d] && n[d] < nghost) return false;
  }
  g.st[0] = 1; g.st[1] = g.pd[0]; g.st[2] = (long long)g.pd[0] * g.pd[1];
  g.np = g.st[2] * g.pd[2];
  return true;
}

StepArgs make_args(const ch_ctx* c, double dt) {
  StepArgs A;
  A.geo = c->geo; A.gas = c->gas;
  for (int d = 0; d < 3; ++d) { A.dx[d] = c->dx[d]; A.idx[d] = 1.0 / c->dx[d]; A.dtdx[d] = dt / c->dx[d]; }
  A.u = c->state;
  const long long blk = 5 * c->geo.np;
  for (int d = 0; d < 3; ++d) {
    A.Fs[d] = c->ws + (long long)(0 + d) * blk;
    A.UL[d] = c->ws + (long long)(3 + d) * blk;
    A.UR[d] = c->ws + (long long)(6 + d) * blk;
    A.Fh[d] = c->ws + (long long)(9 + d) * blk;
  }
  for (int d = 0; d < 3; ++d) A.eta[d] = c->ws + (long long)12 * blk + (long long)d * c->geo.np;
  A.ext = c->hcorr ? 2 : 1;
  A.dt_dev = nullptr;
  A.red = c->red;
  return A;
}

const char* const kKernelNames[CH_K_COUNT] = {"k_reset", "k_pass1_x", "k_pass1_march<y>", "k_pass1_march<z>",
                                              "k_pass2", "k_update", "k_ghost", "k_dt", "k_final3d", "k_eta", "k_pick_dt"};

// event brackets around one launch when profiling is on (no-ops otherwise)
struct Bracket {
  ch_ctx* c; int kind;
  Bracket(ch_ctx* c_, int kind_) : c(c_), kind(kind_) {
    if (c->profiling) { cudaEventRecord(c->ev[2 * kind], c->stream); }
  }
  ~Bracket() {
    ++c->launches;
    if (c->profiling) { cudaEventRecord(c->ev[2 * kind + 1], c->stream); c->ev_used[kind] = true; }
  }
};

int profile_collect(ch_ctx* c) {
  if (!c->profiling) return CH_OK;
  CH_CUDA(cudaStreamSynchronize(c->stream), "profile sync");
  for (int k = 0; k < CH_K_COUNT; ++k) {
    if (!c->ev_used[k]) continue;
    float ms = 0.f;
    CH_CUDA(cudaEventElapsedTime(&ms, c->ev[2 * k], c->ev[2 * k + 1]), "cudaEventElapsedTime");
    c->prof_ms[k] += ms; ++c->prof_calls[k]; c->ev_used[k] = false;
  }
  return CH_OK;
}

int launch_ghost(ch_ctx* c, const StepArgs& A) {
  const Geom& g = c->geo;
  const long long shell = (long long)2 * g.g[2] * g.pd[1] * g.pd[0] + (long long)g.n[2] * 2 * g.g[1] * g.pd[0] +
                          (long long)g.n[2] * g.n[1] * 2 * g.g[0];
  if (shell == 0) return CH_OK;
  BcArgs B; for (int s = 0; s < 6; ++s) B.bc[s] = c->bc[s];
  B.noh_rho0 = c->noh_rho0; B.noh_p0 = c->noh_p0; B.time = c->time;
  B.nact = g.act[0] + g.act[1] + g.act[2];
  for (int d = 0; d < 3; ++d) B.org[d] = c->org[d];
  { Bracket b(c, CH_K_GHOST); k_ghost<<<(unsigned)((shell + 255) / 256), 256, 0, c->stream>>>(A, B); }
  CH_CUDA(cudaGetLastError(), "k_ghost");
  return CH_OK;
}

int copy_real(ch_ctx* c, double* user, bool to_device) {
  const Geom& g = c->geo;
  const size_t N = (size_t)g.n[0] * g.n[1] * g.n[2];
  for (int f = 0; f < 5; ++f) {
    cudaMemcpy3DParms p;
    std::memset(&p, 0, sizeof(p));
    cudaPitchedPtr up = make_cudaPitchedPtr(user + f * N, (size_t)g.n[0] * 8, (size_t)g.n[0] * 8, (size_t)g.n[1]);
    cudaPitchedPtr sp = make_cudaPitchedPtr(c->state + (size_t)f * g.np, (size_t)g.pd[0] * 8, (size_t)g.pd[0] * 8, (size_t)g.pd[1]);
    cudaPos origin = make_cudaPos(0, 0, 0);
    cudaPos ghost = make_cudaPos((size_t)g.g[0] * 8, (size_t)g.g[1], (size_t)g.g[2]);
    if (to_device) { p.srcPtr = up; p.srcPos = origin; p.dstPtr = sp; p.dstPos = ghost; }
    else { p.srcPtr = sp; p.srcPos = ghost; p.dstPtr = up; p.dstPos = origin; }
    p.extent = make_cudaExtent((size_t)g.n[0] * 8, (size_t)g.n[1], (size_t)g.n[2]);
    p.kind = cudaMemcpyDefault;
    CH_CUDA(cudaMemcpy3DAsync(&p, c->stream), "cudaMemcpy3DAsync");
  }
  return CH_OK;
}

// Tensor maps of the ten arrays k_final3d_tma streams: each is [5][pz][py][px] fp64, box {32, kTY, 1, 5}.
// TMA wants 16-byte aligned base addresses and strides: px and np even.  Returns false (plain-load kernel is
// used instead) when that does not hold or the driver entry point is missing.
bool build_tma_maps(ch_ctx* c) {
  const Geom& g = c->geo;
  if (!(g.act[0] && g.act[1] && g.act[2])) return false;
  if ((g.pd[0] & 1) || (g.np & 1)) return false;
  // (a tile's box must start on an even double: with an even nghost the kernel shifts its tiles, see tma_pitch_x)
  typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                               const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
      qres != cudaDriverEntryPointSuccess) {
    cudaGetLastError();
    return false;
  }
  EncodeFn encode = reinterpret_cast<EncodeFn>(fn);
  const long long blk = 5 * g.np;
  double* Fs[3]; double* UL[3]; double* UR[3];
  for (int d = 0; d < 3; ++d) { Fs[d] = c->ws + (long long)d * blk; UL[d] = c->ws + (long long)(3 + d) * blk; UR[d] = c->ws + (long long)(6 + d) * blk; }
  double* arr[10] = {Fs[0], Fs[1], Fs[2], UL[2], UR[2], UL[0], UR[0], c->state, UL[1], UR[1]};
  const cuuint64_t dims[4] = {(cuuint64_t)g.pd[0], (cuuint64_t)g.pd[1], (cuuint64_t)g.pd[2], 5};
  const cuuint64_t strides[3] = {(cuuint64_t)g.pd[0] * 8, (cuuint64_t)g.st[2] * 8, (cuuint64_t)g.np * 8};
  const cuuint32_t box[4] = {(cuuint32_t)kFX, (cuuint32_t)kTY, 1, 5};
  const cuuint32_t box_mp[4] = {(cuuint32_t)kFX, (cuuint32_t)kTYM, 1, 5};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  for (int a = 0; a < 10; ++a) {
    if ((uintptr_t)arr[a] & 15) return false;
    if (encode(&c->maps.m[a], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, arr[a], dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return false;
    if (encode(&c->maps_mp.m[a], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, arr[a], dims, strides, box_mp, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return false;
  }
  // eta_x, eta_y, eta_z of the H-corrected step: one field each
  const cuuint64_t edims[4] = {(cuuint64_t)g.pd[0], (cuuint64_t)g.pd[1], (cuuint64_t)g.pd[2], 1};
  const cuuint32_t ebox[4] = {(cuuint32_t)kFX, (cuuint32_t)kTY, 1, 1};
  for (int d = 0; d < 3; ++d) {
    double* e = c->ws + (long long)12 * blk + (long long)d * g.np;
    if ((uintptr_t)e & 15) return false;
    if (encode(&c->maps.m[10 + d], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, e, edims, strides, ebox, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return false;
  }
  return true;
}

// Updated columns per tile of k_final3d_tma: 30 with an odd nghost, 28 with an even one (the box must start on an
// even double: 16-byte alignment of the bulk tensor copy).
int tma_pitch_x(const Geom& g) { return (g.g[0] & 1) ? kFX - 2 : kFX - 4; }
// Updated rows per tile of the fused second half: the merged-producer TMA form (not the H-corrected step), the
// producer-warp TMA form, the plain-load form.
int final_rows(const ch_ctx* c) {
  if (!(c->tma_ok && c->use_tma)) return kFY - 2;
  return (c->use_tma == 2 && !c->hcorr) ? kTYM - 2 : kTY - 2;
}

// x-y grids whose four faces are periodic, reflective or outflow: the update kernel writes the ghost cells itself.
bool scatter2d(const ch_ctx* c) {
  if (!c->fold_ghost || c->has_exchange || c->has_noh || c->nghost > 4) return false;
  for (int f = 0; f < 4; ++f)
    if (c->bc[f] != CH_BC_PERIODIC && c->bc[f] != CH_BC_REFLECTIVE && c->bc[f] != CH_BC_OUTFLOW) return false;
  return true;
}

// Interfaces a thread of the marching pass-1 kernel sweeps along d: enough segments to fill the chip on small grids
// (a segment costs ~1.5 cells of warm-up), 64 on large ones; CH_OPT_MARCH_SEG overrides.
int march_segment(const ch_ctx* c, int d) {
  const Geom& g = c->geo;
  if (c->march_seg) return c->march_seg;
  const int T = 3 - d;
  const long long cols = (long long)(g.act[0] ? g.n[0] + 2 : 1) * (g.act[T] ? g.n[T] + 2 : 1);
  const long long want = cols * (g.n[d] + 1) / (148LL * 1024);
  int seg = 4;
  while (seg < 64 && seg * 2 <= want) seg *= 2;
  return seg;
}

// Planes a CTA of the fused second half marches (8, 16, 32 or 64); CH_OPT_FINAL_SEG overrides.
int final_segment(const ch_ctx* c) {
  const Geom& g = c->geo;
  if (c->final_seg) return c->final_seg;
  const bool tma = c->tma_ok && c->use_tma;
  const int px = tma ? tma_pitch_x(g) : kFX - 2;
  const int rows = final_rows(c);
  const long long tiles = (long long)((g.n[0] + px - 1) / px) * ((g.n[1] + rows - 1) / rows);
  // a CTA costs its planes plus about three of start-up (two light planes and the fill of the staging ring), and CTAs
  // run in waves of one per SM (two for the plain-load form): among the segments that leave at least four waves of
  // CTAs (work that is not uniform -- a blast wave in a corner of the box -- needs them to balance: Sedov 128^3 loses
  // 8 % with one wave of 64-plane CTAs where the uniform sweep gains 2 %) the one with the smallest
  // waves x (planes + 3), which reproduces the measured order at 64^3 ... 512^3 (profiles/r02_experiments.md)
  const long long per_wave = tma ? 148 : 296;
  int best = 8;
  long long best_cost = -1;
  for (int seg = 8; seg <= 64; seg *= 2) {
    const long long ctas = tiles * ((g.n[2] + seg - 1) / seg);
    if (seg > 8 && ctas < 4 * per_wave) break;
    const long long cost = ((ctas + per_wave - 1) / per_wave) * ((seg < g.n[2] ? seg : g.n[2]) + 3);
    if (best_cost < 0 || cost <= best_cost) { best = seg; best_cost = cost; }
  }
  return best;
}

}  // namespace

extern "C" {

const char* ch_last_error(void) { return g_err.c_str(); }

ch_ctx* ch_init(int nx, int ny, int nz, int nghost, double gamma, const int* bc) {
  Geom g;
  if (nx < 1 || ny < 1 || nz < 1) { fail(CH_EINVAL, "ch_init: n < 1"); return nullptr; }
  if (nghost < 3) { fail(CH_EINVAL, "ch_init: nghost < 3"); return nullptr; }
  if (!(gamma > 1.0) || !std::isfinite(gamma)) { fail(CH_EINVAL, "ch_init: gamma <= 1"); return nullptr; }
  if (!geometry(nx, ny, nz, nghost, g)) { fail(CH_EINVAL, "ch_init: active dimension smaller than nghost"); return nullptr; }
  ch_ctx* c = new (std::nothrow) ch_ctx();
  if (!c) { fail(CH_EINVAL, "ch_init: out of host memory"); return nullptr; }
  c->geo = g;
  c->nghost = nghost;
  for (int s = 0; s < 6; ++s) {
    c->bc[s] = bc ? bc[s] : CH_BC_PERIODIC;
    if (g.act[s / 2] && (c->bc[s] < 1 || c->bc[s] > 5)) { delete c; fail(CH_EINVAL, "ch_init: bad boundary code"); return nullptr; }
    if (g.act[s / 2] && c->bc[s] == CH_BC_NOH) c->has_noh = true;
    if (g.act[s / 2] && c->bc[s] == CH_BC_EXCHANGE) c->has_exchange = true;
  }
  for (int d = 0; d < 3; ++d) {
    if (g.act[d] && ((c->bc[2 * d] == CH_BC_PERIODIC) != (c->bc[2 * d + 1] == CH_BC_PERIODIC))) {
      delete c; fail(CH_EINVAL, "ch_init: unpaired periodic faces"); return nullptr;
    }
    c->dx[d] = 1.0 / nx;   // reading S8
  }
  Gas& G = c->gas;
  G.gamma = gamma; G.gm1 = gamma - 1.0; G.inv_gm1 = 1.0 / (gamma - 1.0); G.two_gm1 = 2.0 / (gamma - 1.0);
  G.z = (gamma - 1.0) / (2.0 * gamma); G.gm = (gamma - 1.0) / (gamma + 1.0); G.c_sh = (gamma + 1.0) / (2.0 * gamma);
  G.half_gp1 = 0.5 * (gamma + 1.0); G.two_gp1 = 2.0 / (gamma + 1.0); G.half_gm1 = 0.5 * (gamma - 1.0);
  {
    // binomial coefficients C(z,k) = C(z,k-1) (z-k+1)/k of the (1+t)^z series (ch_hydro.cuh)
    const long double zl = ((long double)gamma - 1.0L) / (2.0L * (long double)gamma);
    long double b = 1.0L;
    for (int k = 1; k <= ch::kPowTerms; ++k) { b *= (zl - (long double)(k - 1)) / (long double)k; G.bz[k - 1] = (double)b; }
  }
  return c;
}

static void drop_graph(ch_ctx* c) {
  if (c->gexec) { cudaGraphExecDestroy(c->gexec); c->gexec = nullptr; }
  if (c->ggraph) { cudaGraphDestroy(c->ggraph); c->ggraph = nullptr; }
  c->gpick = nullptr;
  c->gseen = 0;
  c->gkey[0] = -1;
}

int ch_free(ch_ctx* c) {
  if (!c) return CH_OK;
  DeviceGuard guard(c->device);
  drop_graph(c);
  if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
  for (int i = 0; i < 2; ++i) {
    if (c->cap_side[i]) cudaStreamDestroy(c->cap_side[i]);
    if (c->cap_join[i]) cudaEventDestroy(c->cap_join[i]);
  }
  if (c->cap_fork) cudaEventDestroy(c->cap_fork);
  if (c->h_red) cudaFreeHost(c->h_red);
  for (int k = 0; k < 2 * CH_K_COUNT; ++k) if (c->ev[k]) cudaEventDestroy(c->ev[k]);
  delete c;
  return CH_OK;
}

int ch_set_spacing(ch_ctx* c, double dx, double dy, double dz) {
  if (!c) return fail(CH_EINVAL, "ch_set_spacing: null context");
  if (!(dx > 0 && dy > 0 && dz > 0) || !std::isfinite(dx) || !std::isfinite(dy) || !std::isfinite(dz))
    return fail(CH_EINVAL, "ch_set_spacing: spacing <= 0");
  c->dx[0] = dx; c->dx[1] = dy; c->dx[2] = dz;
  c->dt_valid = false;
  return CH_OK;
}

long long ch_padded_cells(const ch_ctx* c) { return c ? c->geo.np : 0; }

size_t ch_workspace_bytes(int nx, int ny, int nz, int nghost) {
  Geom g;
  if (!geometry(nx, ny, nz, nghost, g)) return 0;
  return ((size_t)12 * 5 + 3) * (size_t)g.np * sizeof(double);
}

int ch_bind(ch_ctx* c, const ch_buffers* b, void* stream) {
  if (!c || !b) return fail(CH_EINVAL, "ch_bind: null argument");
  if (!b->state || !b->workspace || !b->reduce) return fail(CH_EINVAL, "ch_bind: null buffer");
  if (b->workspace_bytes < ((size_t)12 * 5 + 3) * (size_t)c->geo.np * sizeof(double))
    return fail(CH_EINVAL, "ch_bind: workspace too small");
  if (((uintptr_t)b->state & 7) || ((uintptr_t)b->workspace & 7) || ((uintptr_t)b->reduce & 7))
    return fail(CH_EINVAL, "ch_bind: misaligned buffer");
  {
    cudaPointerAttributes pa;
    if (cudaPointerGetAttributes(&pa, b->state) != cudaSuccess || pa.type != cudaMemoryTypeDevice) {
      cudaGetLastError();
      return fail(CH_EINVAL, "ch_bind: state is not a device pointer");
    }
    if (pa.device != c->device) { c->smem_attr[0][0] = c->smem_attr[0][1] = c->smem_attr[1][0] = c->smem_attr[1][1] = c->smem_attr_hc = false; }
    c->device = pa.device;
  }
  DeviceGuard guard(c->device);
  c->state = b->state;
  c->ws = static_cast<double*>(b->workspace);
  c->red = static_cast<unsigned long long*>(b->reduce);
  c->stream = static_cast<cudaStream_t>(stream);
  if (!c->h_red) CH_CUDA(cudaHostAlloc((void**)&c->h_red, 16, cudaHostAllocDefault), "cudaHostAlloc");
  c->bound = true; c->have_state = false; c->dt_valid = false;
  drop_graph(c);                           // a captured step holds the old buffers' addresses
  CH_CUDA(cudaMemsetAsync(c->red, 0, 64, c->stream), "ch_bind: clearing the reduction cells");
  c->tma_ok = build_tma_maps(c);
  return CH_OK;
}

int ch_set_state(ch_ctx* c, const double* u) {
  if (!c || !u) return fail(CH_EINVAL, "ch_set_state: null argument");
  if (!c->bound) return fail(CH_ESTATE, "ch_set_state: no buffers bound");
  DeviceGuard guard(c->device);
  int rc = copy_real(c, const_cast<double*>(u), true);
  if (rc) return rc;
  c->time = 0.0;
  StepArgs A = make_args(c, 1.0);
  rc = c->has_exchange ? CH_OK : launch_ghost(c, A);
  if (rc) return rc;
  c->have_state = true; c->dt_valid = false;
  return CH_OK;
}

int ch_get_state(ch_ctx* c, double* u) {
  if (!c || !u) return fail(CH_EINVAL, "ch_get_state: null argument");
  if (!c->have_state) return fail(CH_ESTATE, "ch_get_state: no state set");
  DeviceGuard guard(c->device);
  int rc = copy_real(c, u, false);
  if (rc) return rc;
  CH_CUDA(cudaStreamSynchronize(c->stream), "ch_get_state sync");
  return CH_OK;
}

int ch_set_padded(ch_ctx* c, const double* up) {
  if (!c || !up) return fail(CH_EINVAL, "ch_set_padded: null argument");
  if (!c->bound) return fail(CH_ESTATE, "ch_set_padded: no buffers bound");
  DeviceGuard guard(c->device);
  CH_CUDA(cudaMemcpyAsync(c->state, up, (size_t)5 * c->geo.np * 8, cudaMemcpyDefault, c->stream), "ch_set_padded");
  c->have_state = true; c->dt_valid = false;
  return CH_OK;
}

int ch_get_padded(ch_ctx* c, double* up) {
  if (!c || !up) return fail(CH_EINVAL, "ch_get_padded: null argument");
  if (!c->have_state) return fail(CH_ESTATE, "ch_get_padded: no state set");
  DeviceGuard guard(c->device);
  CH_CUDA(cudaMemcpyAsync(up, c->state, (size_t)5 * c->geo.np * 8, cudaMemcpyDefault, c->stream), "ch_get_padded");
  CH_CUDA(cudaStreamSynchronize(c->stream), "ch_get_padded sync");
  return CH_OK;
}

double ch_compute_dt(ch_ctx* c, double cfl) {
  const double nan = std::numeric_limits<double>::quiet_NaN();
  if (!c) { fail(CH_EINVAL, "ch_compute_dt: null context"); return nan; }
  if (!c->have_state) { fail(CH_ESTATE, "ch_compute_dt: no state set"); return nan; }
  if (!(cfl > 0.0) || !(cfl <= 1.0)) { fail(CH_EINVAL, "ch_compute_dt: cfl not in (0,1]"); return nan; }
  DeviceGuard guard(c->device);
  if (!c->dt_valid) {
    StepArgs A = make_args(c, 1.0);
    { Bracket b(c, CH_K_RESET); k_reset<<<1, 32, 0, c->stream>>>(c->red, nullptr); }
    const long long N = (long long)c->geo.n[0] * c->geo.n[1] * c->geo.n[2];
    long long blocks = (N + 255) / 256;
    if (blocks > 148 * 8) blocks = 148 * 8;
    { Bracket b(c, CH_K_DT); k_dt<<<(unsigned)blocks, 256, 0, c->stream>>>(A); }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { cuda_fail(e, "k_dt"); return nan; }
    if (profile_collect(c) != CH_OK) return nan;
    c->dt_valid = true;
  }
  cudaError_t e = cudaMemcpyAsync(c->h_red, c->red, 16, cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) { cuda_fail(e, "ch_compute_dt read-back"); return nan; }
  if (c->h_red[1] != 0ULL) { fail(CH_ENONPHYS, "ch_compute_dt: non-physical cell (rho <= 0 or non-finite)"); return nan; }
  double rate;                                  // grid maximum of (|v_d| + a) / dx_d
  std::memcpy(&rate, &c->h_red[0], 8);
  return cfl * (1.0 / rate);
}

}  // extern "C"

namespace {

// One CTU step with Riemann solver S (0 exact, 1 Roe + HLLE) compiled into every kernel that solves.
template <int S, int R>
int step_impl(ch_ctx* c, double dt, bool devdt) {
  if (!c) return fail(CH_EINVAL, "ch_step: null context");
  if (!c->have_state) return fail(CH_ESTATE, "ch_step: no state set");
  if (!devdt && (!(dt > 0.0) || !std::isfinite(dt))) return fail(CH_EINVAL, "ch_step: dt <= 0 or non-finite");
  const Geom& g = c->geo;
  StepArgs A = make_args(c, devdt ? 1.0 : dt);
  if (devdt) A.dt_dev = reinterpret_cast<const double*>(c->red) + 2;     // written by k_pick_dt just before
  cudaStream_t st = c->stream;
  if (!devdt) { Bracket b(c, CH_K_RESET); k_reset<<<1, 32, 0, st>>>(c->red, nullptr); }   // ch_step_cfl: k_pick_dt has done it
  // pass 1
  if constexpr (R == 3) {
    // PPMP: kernels of its own (7-cell stencil, IEEE primitives), the same shapes as the PPMC ones
    for (int d = 0; d < 3; ++d) {
      if (!g.act[d]) continue;
      Bracket b(c, d == 0 ? CH_K_PASS1_X : d == 1 ? CH_K_PASS1_Y : CH_K_PASS1_Z);
      if (d == 0) {
        const int j0 = g.act[1] ? g.g[1] - 1 : 0, k0 = g.act[2] ? g.g[2] - 1 : 0;
        const int j1 = g.act[1] ? g.g[1] + g.n[1] : 0, k1 = g.act[2] ? g.g[2] + g.n[2] : 0;
        const long long qb = (long long)j0 * g.st[1] + (long long)k0 * g.st[2];
        const long long qe = (long long)j1 * g.st[1] + (long long)k1 * g.st[2] + g.pd[0];
        const long long nbx = (qe - qb + kXOutP - 1) / kXOutP;
        k_pass1_x_ppmp<S><<<(unsigned)nbx, kXT, 0, st>>>(A, qb, qe);
      } else {
        const int T = 3 - d;
        const long long cols = (long long)(g.act[0] ? g.n[0] + 2 : 1) * (g.act[T] ? g.n[T] + 2 : 1);
        const int seg = march_segment(c, d);
        dim3 grid((unsigned)((cols + CH_MARCH_T - 1) / CH_MARCH_T), (unsigned)((g.n[d] + 1 + seg - 1) / seg));
        if (d == 1) k_pass1_march_ppmp<1, S><<<grid, CH_MARCH_T, 0, st>>>(A, seg);
        else k_pass1_march_ppmp<2, S><<<grid, CH_MARCH_T, 0, st>>>(A, seg);
      }
    }
  } else {
  // The three sweeps of pass 1 are independent (each reads u, writes its own arrays).  While a step is being captured
  // into a graph (launch-bound grids only) the y and z sweeps go to side streams: parallel branches of the graph.
  const bool fork = c->capturing && c->cap_side[0] && c->cap_side[1];
  if (fork) {
    cudaEventRecord(c->cap_fork, st);
    cudaStreamWaitEvent(c->cap_side[0], c->cap_fork, 0);
    cudaStreamWaitEvent(c->cap_side[1], c->cap_fork, 0);
  }
  if (g.act[0]) {
    // flat run of padded cells from the first needed row to the last: rows j,k in [-1, n]
    const int j0 = g.act[1] ? g.g[1] - 1 : 0, k0 = g.act[2] ? g.g[2] - 1 : 0;
    const int j1 = g.act[1] ? g.g[1] + g.n[1] : 0, k1 = g.act[2] ? g.g[2] + g.n[2] : 0;
    const long long qb = (long long)j0 * g.st[1] + (long long)k0 * g.st[2];
    const long long qe = (long long)j1 * g.st[1] + (long long)k1 * g.st[2] + g.pd[0];
    const long long nb = (qe - qb + kXOut - 1) / kXOut;
    Bracket b(c, CH_K_PASS1_X);
    k_pass1_x<S, R><<<(unsigned)nb, kXT, 0, st>>>(A, qb, qe);
  }
  for (int d = 1; d < 3; ++d) {
    if (!g.act[d]) continue;
    const int T = 3 - d;
    const long long cols = (long long)(g.act[0] ? g.n[0] + 2 : 1) * (g.act[T] ? g.n[T] + 2 : 1);
    // enough segments to fill the chip on small grids (a segment costs ~1.5 cells of warm-up), 64 on large ones
    const int seg = march_segment(c, d);
    dim3 grid((unsigned)((cols + CH_MARCH_T - 1) / CH_MARCH_T), (unsigned)((g.n[d] + 2 * A.ext - 1 + seg - 1) / seg));
    Bracket b(c, d == 1 ? CH_K_PASS1_Y : CH_K_PASS1_Z);
    cudaStream_t sd = fork ? c->cap_side[d - 1] : st;
    if (d == 1) k_pass1_march<1, S, R><<<grid, CH_MARCH_T, 0, sd>>>(A, seg);
    else k_pass1_march<2, S, R><<<grid, CH_MARCH_T, 0, sd>>>(A, seg);
  }
  if (fork) {
    for (int i = 0; i < 2; ++i) {
      cudaEventRecord(c->cap_join[i], c->cap_side[i]);
      cudaStreamWaitEvent(st, c->cap_join[i], 0);
    }
  }
  }
  CH_CUDA(cudaGetLastError(), "pass 1");
  bool folded_ghost = false;
  const bool three_d = g.act[0] && g.act[1] && g.act[2];
  if (three_d && !c->unfused && c->hcorr && c->tma_ok && c->use_tma) {
    // H-corrected step, fused: eta of every interface (C1), then the fused second half with C2's maxima taken from the
    // staged eta planes (the plain-load kernel has no such form: without TMA the step stays unfused, below)
    {
      const int nseg = (g.n[2] + 2 + 63) / 64, eseg = (g.n[2] + 2 + nseg - 1) / nseg;
      dim3 egrid((unsigned)((g.n[0] + 2 + kFX - 2) / (kFX - 1)), (unsigned)((g.n[1] + 2 + kEY - 2) / (kEY - 1)), (unsigned)nseg);
      Bracket b(c, CH_K_ETA);
      k_eta3d<<<egrid, kET, 0, st>>>(A, eseg);
    }
    const int seg = final_segment(c);
    const size_t tsmem = (size_t)74 * kTT * sizeof(double);     // + eta_x, eta_y and two planes of eta_z
    if (!c->smem_attr_hc) {
      CH_CUDA(cudaFuncSetAttribute(k_final3d_tma<1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tsmem), "k_final3d_tma<HC> smem attribute");
      c->smem_attr_hc = true;
    }
    const int pitch = tma_pitch_x(g);
    dim3 tgrid((unsigned)((g.n[0] + pitch - 1) / pitch), (unsigned)((g.n[1] + kTY - 3) / (kTY - 2)), (unsigned)((g.n[2] + seg - 1) / seg));
    Bracket b(c, CH_K_FINAL);
    k_final3d_tma<1, true><<<tgrid, kTT, tsmem, st>>>(A, c->maps, seg);
  } else if (three_d && !c->unfused && !c->hcorr) {
    const int seg = final_segment(c);
    dim3 grid((unsigned)((g.n[0] + kFX - 3) / (kFX - 2)), (unsigned)((g.n[1] + kFY - 3) / (kFY - 2)),
              (unsigned)((g.n[2] + seg - 1) / seg));
    if (c->tma_ok && c->use_tma == 2) {
      // merged producer: kTYM staged rows, the carried arrays for the updating rows only
      const size_t tsmem = ((size_t)60 * kFX * kTYM + (size_t)10 * kFX * (kTYM - 2)) * sizeof(double);
      if (!c->smem_attr_mp[S]) {
        CH_CUDA(cudaFuncSetAttribute(k_final3d_tma<S, false, kTYM, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tsmem), "k_final3d_tma<MP> smem attribute");
        c->smem_attr_mp[S] = true;
      }
      const int pitch = tma_pitch_x(g);
      dim3 tgrid((unsigned)((g.n[0] + pitch - 1) / pitch), (unsigned)((g.n[1] + kTYM - 3) / (kTYM - 2)),
                 (unsigned)((g.n[2] + seg - 1) / seg));
      Bracket b(c, CH_K_FINAL);
      k_final3d_tma<S, false, kTYM, true><<<tgrid, kFX * (kTYM - 1), tsmem, st>>>(A, c->maps_mp, seg);
    } else if (c->tma_ok && c->use_tma) {
      const size_t tsmem = (size_t)70 * kTT * sizeof(double);   // 50 staged + 10 exchanged + 10 carried doubles per slot
      if (!c->smem_attr[1][S]) {
        CH_CUDA(cudaFuncSetAttribute(k_final3d_tma<S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tsmem), "k_final3d_tma smem attribute");
        c->smem_attr[1][S] = true;
      }
      const int pitch = tma_pitch_x(g);
      dim3 tgrid((unsigned)((g.n[0] + pitch - 1) / pitch), (unsigned)((g.n[1] + kTY - 3) / (kTY - 2)),
                 (unsigned)((g.n[2] + seg - 1) / seg));
      Bracket b(c, CH_K_FINAL);
      k_final3d_tma<S><<<tgrid, kTT, tsmem, st>>>(A, c->maps, seg);
    } else {
    const size_t smem = (size_t)30 * kFT * sizeof(double);
    if (!c->smem_attr[0][S]) {
      CH_CUDA(cudaFuncSetAttribute(k_final3d<S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), "k_final3d smem attribute");
      c->smem_attr[0][S] = true;
    }
    Bracket b(c, CH_K_FINAL);
    k_final3d<S><<<grid, kFT, smem, st>>>(A, seg);
    }
  } else if (g.act[0] && g.act[1] && !g.act[2] && !c->unfused && !c->hcorr) {
    dim3 grid((unsigned)((g.n[0] + kFX - 3) / (kFX - 2)), (unsigned)((g.n[1] + kFY - 3) / (kFY - 2)), 1);
    Bracket b(c, CH_K_FINAL);
    Scatter2d GS;
    GS.on = scatter2d(c) ? 1 : 0;
    for (int f = 0; f < 4; ++f) GS.bc[f] = c->bc[f];
    k_final2d<S><<<grid, kFT, 0, st>>>(A, GS);
    folded_ghost = GS.on != 0;
  } else {
    {
      const long long cells = (long long)(g.act[0] ? g.n[0] + 1 : 1) * (g.act[1] ? g.n[1] + 1 : 1) * (g.act[2] ? g.n[2] + 1 : 1);
      if (c->hcorr) {
        const long long ecells = (long long)(g.act[0] ? g.n[0] + 2 : 1) * (g.act[1] ? g.n[1] + 2 : 1) * (g.act[2] ? g.n[2] + 2 : 1);
        Bracket b(c, CH_K_ETA);
        k_eta<<<(unsigned)((ecells + CH_P2_T - 1) / CH_P2_T), CH_P2_T, 0, st>>>(A);
      }
      Bracket b(c, CH_K_PASS2);
      if (c->hcorr) k_pass2<1, true><<<(unsigned)((cells + CH_P2_T - 1) / CH_P2_T), CH_P2_T, 0, st>>>(A);
      else k_pass2<S, false><<<(unsigned)((cells + CH_P2_T - 1) / CH_P2_T), CH_P2_T, 0, st>>>(A);
    }
    {
      const long long N = (long long)g.n[0] * g.n[1] * g.n[2];
      Bracket b(c, CH_K_UPDATE);
      k_update<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(A);
    }
}
  CH_CUDA(cudaGetLastError(), "pass 2 / update");
  if (!devdt) c->time += dt;     // analytic faces are evaluated at t^{n+1}
  // a block of a decomposed domain: its ghosts are filled by the caller, direction by direction
  int rc = (c->has_exchange || folded_ghost) ? CH_OK : launch_ghost(c, A);
  if (rc) return rc;
  c->dt_valid = true;
  return profile_collect(c);
}

}  // namespace

extern "C" {

static int step_dispatch(ch_ctx* c, double dt, bool devdt) {
  DeviceGuard guard(c->device);
  const bool roe = c->solver == CH_SOLVER_ROE;
  if (c->hcorr && !roe) return fail(CH_ESTATE, "ch_step: the H correction goes with the Roe solver (ch_set_solver)");
  switch (c->recon) {
    case CH_RECON_PLMC: return roe ? step_impl<1, 1>(c, dt, devdt) : step_impl<0, 1>(c, dt, devdt);
    case CH_RECON_PCM: return roe ? step_impl<1, 2>(c, dt, devdt) : step_impl<0, 2>(c, dt, devdt);
    case CH_RECON_PPMP: return roe ? step_impl<1, 3>(c, dt, devdt) : step_impl<0, 3>(c, dt, devdt);
    case CH_RECON_PLMP: return roe ? step_impl<1, 4>(c, dt, devdt) : step_impl<0, 4>(c, dt, devdt);
    default: return roe ? step_impl<1, 0>(c, dt, devdt) : step_impl<0, 0>(c, dt, devdt);
  }
}

int ch_step(ch_ctx* c, double dt) {
  if (!c) return fail(CH_EINVAL, "ch_step: null context");
  return step_dispatch(c, dt, false);
}

int ch_step_cfl(ch_ctx* c, double cfl, double t_left) {
  if (!c) return fail(CH_EINVAL, "ch_step_cfl: null context");
  if (!c->have_state) return fail(CH_ESTATE, "ch_step_cfl: no state set");
  if (!(cfl > 0.0) || !(cfl <= 1.0)) return fail(CH_EINVAL, "ch_step_cfl: cfl not in (0,1]");
  if (t_left != t_left) return fail(CH_EINVAL, "ch_step_cfl: t_left is NaN");
  if (c->has_exchange) return fail(CH_ESTATE, "ch_step_cfl: a block of a decomposed domain needs the global minimum of dt: use ch_compute_dt + ch_step");
  if (c->has_noh) return fail(CH_ESTATE, "ch_step_cfl: an analytic (CH_BC_NOH) face needs the time on the host: use ch_compute_dt + ch_step");
  DeviceGuard guard(c->device);
  Dx3 dx3;
  for (int d = 0; d < 3; ++d) dx3.v[d] = c->dx[d];
  if (!c->dt_valid) {
    StepArgs A = make_args(c, 1.0);
    { Bracket b(c, CH_K_RESET); k_reset<<<1, 32, 0, c->stream>>>(c->red, nullptr); }
    const long long N = (long long)c->geo.n[0] * c->geo.n[1] * c->geo.n[2];
    long long blocks = (N + 255) / 256;
    if (blocks > 148 * 8) blocks = 148 * 8;
    { Bracket b(c, CH_K_DT); k_dt<<<(unsigned)blocks, 256, 0, c->stream>>>(A); }
    c->dt_valid = true;
  }
  // launch-bound grids only: from ~256^3 up a step is tens of milliseconds of kernels and the replay measured
  // 1-3 % slower than plain launches (384^3: 15.9 against 15.4 ms)
  const long long ncell = (long long)c->geo.n[0] * c->geo.n[1] * c->geo.n[2];
  const bool graphs = c->use_graph && !c->profiling && ncell <= (1LL << 24);
  // The step reads dt from device memory; k_pick_dt's two arguments are the only per-step ones: one graph per
  // configuration, k_pick_dt its first node, its arguments updated in place when they change.  First step with a
  // configuration: direct (sets kernel attributes); second: captured on the private stream; from then on one
  // cudaGraphLaunch on the caller's stream.
  if (graphs) {
    const long long key[8] = {c->solver, c->recon, c->hcorr, c->unfused, c->use_tma, c->march_seg, c->final_seg, 1};
    bool same = true;
    for (int i = 0; i < 8; ++i) same = same && key[i] == c->gkey[i];
    for (int d = 0; d < 3; ++d) same = same && c->gdx[d] == c->dx[d];
    if (!same) {
      drop_graph(c);
      for (int i = 0; i < 8; ++i) c->gkey[i] = key[i];
      for (int d = 0; d < 3; ++d) c->gdx[d] = c->dx[d];
    }
    if (c->gexec) {
      if (cfl != c->gcfl || t_left != c->gtleft) {
        void* args[4] = {(void*)&c->red, (void*)&cfl, (void*)&t_left, (void*)&dx3};
        cudaKernelNodeParams kp = {};
        kp.func = (void*)k_pick_dt;
        kp.gridDim = dim3(1); kp.blockDim = dim3(32); kp.sharedMemBytes = 0; kp.kernelParams = args; kp.extra = nullptr;
        CH_CUDA(cudaGraphExecKernelNodeSetParams(c->gexec, c->gpick, &kp), "cudaGraphExecKernelNodeSetParams");
        c->gcfl = cfl; c->gtleft = t_left;
      }
      CH_CUDA(cudaGraphLaunch(c->gexec, c->stream), "cudaGraphLaunch");
      c->launches += c->glaunches;
      c->dt_valid = true;
      return CH_OK;
    }
  }
  if (!graphs || c->gseen++ == 0) {
    { Bracket b(c, CH_K_PICK_DT); k_pick_dt<<<1, 32, 0, c->stream>>>(c->red, cfl, t_left, dx3); }
    CH_CUDA(cudaGetLastError(), "k_pick_dt");
    return step_dispatch(c, 0.0, true);
  }
  if (!c->cap_stream) {
    CH_CUDA(cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking), "cudaStreamCreate");
    for (int i = 0; i < 2; ++i) {
      CH_CUDA(cudaStreamCreateWithFlags(&c->cap_side[i], cudaStreamNonBlocking), "cudaStreamCreate");
      CH_CUDA(cudaEventCreateWithFlags(&c->cap_join[i], cudaEventDisableTiming), "cudaEventCreate");
    }
    CH_CUDA(cudaEventCreateWithFlags(&c->cap_fork, cudaEventDisableTiming), "cudaEventCreate");
  }
  cudaStream_t user = c->stream;
  const long long before = c->launches;
  cudaGraph_t graph = nullptr;
  CH_CUDA(cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal), "cudaStreamBeginCapture");
  c->stream = c->cap_stream;
  c->capturing = true;
  { Bracket b(c, CH_K_PICK_DT); k_pick_dt<<<1, 32, 0, c->stream>>>(c->red, cfl, t_left, dx3); }
  const int rc = step_dispatch(c, 0.0, true);
  c->capturing = false;
  c->stream = user;
  cudaError_t e = cudaStreamEndCapture(c->cap_stream, &graph);
  c->glaunches = c->launches - before;
  c->launches = before;
  // k_pick_dt's node
  cudaGraphNode_t pick = nullptr;
  if (rc == CH_OK && e == cudaSuccess && graph) {
    size_t nn = 0;
    cudaGraphGetNodes(graph, nullptr, &nn);
    std::vector<cudaGraphNode_t> nodes(nn);
    if (nn) cudaGraphGetNodes(graph, nodes.data(), &nn);
    for (size_t i = 0; i < nn && !pick; ++i) {
      cudaGraphNodeType ty;
      if (cudaGraphNodeGetType(nodes[i], &ty) != cudaSuccess || ty != cudaGraphNodeTypeKernel) continue;
      cudaKernelNodeParams kp;
      if (cudaGraphKernelNodeGetParams(nodes[i], &kp) == cudaSuccess && kp.func == (void*)k_pick_dt) pick = nodes[i];
    }
  }
  if (rc != CH_OK || e != cudaSuccess || !graph || !pick) {
    if (graph) cudaGraphDestroy(graph);
    cudaGetLastError();
    c->use_graph = false;                  // fall back to direct launches for this context
    { Bracket b(c, CH_K_PICK_DT); k_pick_dt<<<1, 32, 0, c->stream>>>(c->red, cfl, t_left, dx3); }
    return step_dispatch(c, 0.0, true);
  }
  e = cudaGraphInstantiate(&c->gexec, graph, 0);
  if (e != cudaSuccess) {
    cudaGraphDestroy(graph);
    c->gexec = nullptr; cudaGetLastError(); c->use_graph = false;
    { Bracket b(c, CH_K_PICK_DT); k_pick_dt<<<1, 32, 0, c->stream>>>(c->red, cfl, t_left, dx3); }
    return step_dispatch(c, 0.0, true);
  }
  c->ggraph = graph; c->gpick = pick; c->gcfl = cfl; c->gtleft = t_left;
  CH_CUDA(cudaGraphLaunch(c->gexec, c->stream), "cudaGraphLaunch");
  c->launches += c->glaunches;
  c->dt_valid = true;
  return CH_OK;
}

double ch_last_dt(ch_ctx* c) {
  const double nan = std::numeric_limits<double>::quiet_NaN();
  if (!c || !c->bound) { fail(CH_ESTATE, "ch_last_dt: no buffers bound"); return nan; }
  DeviceGuard guard(c->device);
  cudaError_t e = cudaMemcpyAsync(c->h_red, c->red + 2, 16, cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) { cuda_fail(e, "ch_last_dt read-back"); return nan; }
  double dt;
  std::memcpy(&dt, &c->h_red[0], 8);
  if (dt != dt) fail(CH_ENONPHYS, "ch_last_dt: non-physical cell (rho <= 0 or non-finite) met by ch_step_cfl");
  return dt;
}

double ch_elapsed(ch_ctx* c) {
  const double nan = std::numeric_limits<double>::quiet_NaN();
  if (!c || !c->bound) { fail(CH_ESTATE, "ch_elapsed: no buffers bound"); return nan; }
  DeviceGuard guard(c->device);
  cudaError_t e = cudaMemcpyAsync(c->h_red, c->red + 2, 16, cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) { cuda_fail(e, "ch_elapsed read-back"); return nan; }
  double t;
  std::memcpy(&t, &c->h_red[1], 8);
  return t;
}

int ch_set_hcorrection(ch_ctx* c, int on) {
  if (!c) return fail(CH_EINVAL, "ch_set_hcorrection: null context");
  if (on && c->nghost < 4) return fail(CH_EINVAL, "ch_set_hcorrection: needs nghost >= 4 (P:L1291)");
  if (on && c->recon >= CH_RECON_PPMP) return fail(CH_EINVAL, "ch_set_hcorrection: only with PPMC, PLMC or PCM (P:L565)");
  c->hcorr = on != 0;
  return CH_OK;
}

int ch_set_reconstruction(ch_ctx* c, int recon) {
  if (!c) return fail(CH_EINVAL, "ch_set_reconstruction: null context");
  if (recon < CH_RECON_PPMC || recon > CH_RECON_PLMP) return fail(CH_EINVAL, "ch_set_reconstruction: unknown reconstruction");
  if (recon == CH_RECON_PPMP && c->nghost < 4) return fail(CH_EINVAL, "ch_set_reconstruction: PPMP needs nghost >= 4 (P:L962)");
  if (recon >= CH_RECON_PPMP && c->hcorr) return fail(CH_EINVAL, "ch_set_reconstruction: the H correction goes with PPMC, PLMC or PCM (P:L565)");
  c->recon = recon;
  return CH_OK;
}

int ch_tiling(const ch_ctx* c, int* out) {
  if (!c || !out) return fail(CH_EINVAL, "ch_tiling: null argument");
  const Geom& g = c->geo;
  const bool three_d = g.act[0] && g.act[1] && g.act[2];
  const bool tma = three_d && c->tma_ok && c->use_tma && !c->unfused;
  out[0] = kXOut;                          // interfaces per CTA of k_pass1_x (flat run of padded cells)
  out[1] = CH_MARCH_T;                     // columns per CTA of the marching kernels
  out[2] = march_segment(c, 1);            // interfaces a marching thread sweeps along y
  out[3] = march_segment(c, 2);            // ... along z
  out[4] = three_d ? (tma ? tma_pitch_x(g) : kFX - 2) : 0;   // updated columns per tile of the fused second half along x
  out[5] = three_d ? (c->unfused ? kFY - 2 : final_rows(c)) : 0;   // ... along y
  out[6] = three_d ? final_segment(c) : 0; // planes a CTA of the fused second half marches
  out[7] = tma ? 1 : 0;
  return CH_OK;
}

int ch_set_noh(ch_ctx* c, double rho0, double p0) {
  if (!c) return fail(CH_EINVAL, "ch_set_noh: null context");
  if (!(rho0 > 0.0) || !(p0 > 0.0) || !std::isfinite(rho0) || !std::isfinite(p0)) return fail(CH_EINVAL, "ch_set_noh: rho0, p0 must be positive");
  c->noh_rho0 = rho0; c->noh_p0 = p0;
  return CH_OK;
}

int ch_set_time(ch_ctx* c, double t) {
  if (!c) return fail(CH_EINVAL, "ch_set_time: null context");
  if (!std::isfinite(t)) return fail(CH_EINVAL, "ch_set_time: t is not finite");
  c->time = t;
  return CH_OK;
}

double ch_get_time(const ch_ctx* c) { return c ? c->time : std::numeric_limits<double>::quiet_NaN(); }

int ch_fill_ghosts(ch_ctx* c) {
  if (!c) return fail(CH_EINVAL, "ch_fill_ghosts: null context");
  if (!c->have_state) return fail(CH_ESTATE, "ch_fill_ghosts: no state set");
  if (c->has_exchange) return fail(CH_ESTATE, "ch_fill_ghosts: a block of a decomposed domain is filled direction by direction (ch_halo_*, ch_fill_dim)");
  DeviceGuard guard(c->device);
  StepArgs A = make_args(c, 1.0);
  return launch_ghost(c, A);
}

int ch_set_origin(ch_ctx* c, int i0, int j0, int k0) {
  if (!c) return fail(CH_EINVAL, "ch_set_origin: null context");
  c->org[0] = i0; c->org[1] = j0; c->org[2] = k0;
  return CH_OK;
}

long long ch_halo_cells(const ch_ctx* c, int d) {
  if (!c || d < 0 || d > 2 || !c->geo.act[d]) return 0;
  const SlabGeom S = slab_geom(c->geo, d);
  return (long long)c->geo.g[d] * S.n1 * S.n2;
}

static int halo_launch(ch_ctx* c, int face, int mode, double* buf, const char* who) {
  if (!c || !buf) return fail(CH_EINVAL, "ch_halo_pack / ch_halo_unpack: null argument");
  if (face < 0 || face > 5 || !c->geo.act[face / 2]) return fail(CH_EINVAL, "ch_halo_pack / ch_halo_unpack: no such face");
  if (!c->have_state) return fail(CH_ESTATE, "ch_halo_pack / ch_halo_unpack: no state set");
  DeviceGuard guard(c->device);
  StepArgs A = make_args(c, 1.0);
  const long long per = ch_halo_cells(c, face / 2);
  { Bracket b(c, CH_K_GHOST); k_halo<<<(unsigned)((per + 255) / 256), 256, 0, c->stream>>>(A, face / 2, face & 1, mode, buf); }
  CH_CUDA(cudaGetLastError(), who);
  if (mode == 1) c->dt_valid = c->dt_valid;   // ghosts do not enter Eq. 22
  return CH_OK;
}

int ch_halo_pack(ch_ctx* c, int face, double* buf) { return halo_launch(c, face, 0, buf, "ch_halo_pack"); }
int ch_halo_unpack(ch_ctx* c, int face, const double* buf) { return halo_launch(c, face, 1, const_cast<double*>(buf), "ch_halo_unpack"); }

int ch_fill_dim(ch_ctx* c, int d) {
  if (!c) return fail(CH_EINVAL, "ch_fill_dim: null context");
  if (d < 0 || d > 2) return fail(CH_EINVAL, "ch_fill_dim: no such direction");
  if (!c->have_state) return fail(CH_ESTATE, "ch_fill_dim: no state set");
  if (!c->geo.act[d]) return CH_OK;
  DeviceGuard guard(c->device);
  StepArgs A = make_args(c, 1.0);
  BcArgs B; for (int s = 0; s < 6; ++s) B.bc[s] = c->bc[s];
  B.noh_rho0 = c->noh_rho0; B.noh_p0 = c->noh_p0; B.time = c->time;
  B.nact = c->geo.act[0] + c->geo.act[1] + c->geo.act[2];
  for (int e = 0; e < 3; ++e) B.org[e] = c->org[e];
  const long long per = ch_halo_cells(c, d);
  { Bracket b(c, CH_K_GHOST); k_fill_dim<<<(unsigned)((2 * per + 255) / 256), 256, 0, c->stream>>>(A, B, d); }
  CH_CUDA(cudaGetLastError(), "k_fill_dim");
  return CH_OK;
}

int ch_set_option(ch_ctx* c, int option, int value) {
  if (!c) return fail(CH_EINVAL, "ch_set_option: null context");
  switch (option) {
    case CH_OPT_MARCH_SEG:
      if (value != 0 && value < 4) return fail(CH_EINVAL, "ch_set_option: march segment < 4");
      c->march_seg = value; return CH_OK;
    case CH_OPT_FINAL_SEG:
      if (value != 0 && value < 4) return fail(CH_EINVAL, "ch_set_option: final segment < 4");
      c->final_seg = value; return CH_OK;
    case CH_OPT_TMA:
      if (value < 0 || value > 2) return fail(CH_EINVAL, "ch_set_option: CH_OPT_TMA takes 0 (plain loads), 1 (producer warp) or 2 (merged producer)");
      c->use_tma = value; return CH_OK;
    case CH_OPT_UNFUSED: c->unfused = value != 0; return CH_OK;
    case CH_OPT_GRAPH: c->use_graph = value != 0; if (!c->use_graph) drop_graph(c); return CH_OK;
    case CH_OPT_FOLD_GHOST: c->fold_ghost = value != 0; drop_graph(c); return CH_OK;
    default: return fail(CH_EINVAL, "ch_set_option: unknown option");
  }
}

int ch_set_solver(ch_ctx* c, int solver) {
  if (!c) return fail(CH_EINVAL, "ch_set_solver: null context");
  if (solver != CH_SOLVER_EXACT && solver != CH_SOLVER_ROE) return fail(CH_EINVAL, "ch_set_solver: unknown solver");
  c->solver = solver;
  return CH_OK;
}

int ch_sync(ch_ctx* c) {
  if (!c) return fail(CH_EINVAL, "ch_sync: null context");
  DeviceGuard guard(c->device);
  CH_CUDA(cudaStreamSynchronize(c->stream), "ch_sync");
  return CH_OK;
}

long long ch_kernel_launches(const ch_ctx* c) { return c ? c->launches : 0; }

int ch_profile(ch_ctx* c, int enable) {
  if (!c) return fail(CH_EINVAL, "ch_profile: null context");
  DeviceGuard guard(c->device);
  if (enable && !c->ev[0]) {
    for (int k = 0; k < 2 * CH_K_COUNT; ++k) CH_CUDA(cudaEventCreate(&c->ev[k]), "cudaEventCreate");
  }
  c->profiling = enable != 0;
  for (int k = 0; k < CH_K_COUNT; ++k) { c->prof_ms[k] = 0.0; c->prof_calls[k] = 0; c->ev_used[k] = false; }
  return CH_OK;
}

int ch_profile_read(const ch_ctx* c, double* ms, long long* calls) {
  if (!c || !ms || !calls) return fail(CH_EINVAL, "ch_profile_read: null argument");
  for (int k = 0; k < CH_K_COUNT; ++k) { ms[k] = c->prof_ms[k]; calls[k] = c->prof_calls[k]; }
  return CH_OK;
}

const char* ch_kernel_name(int kind) { return (kind >= 0 && kind < CH_K_COUNT) ? kKernelNames[kind] : ""; }

double ch_issue_mix_probe(double* sink, int n_alu, int blocks, int threads, int iters, void* stream) {
  if (!sink || blocks < 1 || threads < 1 || threads > 1024 || iters < 1 || (n_alu != 0 && n_alu != 16 && n_alu != 32)) {
    fail(CH_EINVAL, "ch_issue_mix_probe: bad argument (n_alu is 0, 16 or 32)"); return -1.0;
  }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  int dev = -1;
  {
    cudaPointerAttributes pa;
    if (cudaPointerGetAttributes(&pa, sink) == cudaSuccess && pa.type == cudaMemoryTypeDevice) dev = pa.device;
    else cudaGetLastError();
  }
  DeviceGuard guard(dev);
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) { fail(CH_ECUDA, "event create"); return -1.0; }
  for (int rep = 0; rep < 2; ++rep) {      // the first launch warms up
    if (rep == 1) cudaEventRecord(e0, st);
    if (n_alu == 0) k_mix_probe<0><<<blocks, threads, 0, st>>>(sink, iters);
    else if (n_alu == 16) k_mix_probe<16><<<blocks, threads, 0, st>>>(sink, iters);
    else k_mix_probe<32><<<blocks, threads, 0, st>>>(sink, iters);
  }
  cudaEventRecord(e1, st);
  cudaError_t e = cudaEventSynchronize(e1);
  float ms = -1.f;
  if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  if (e != cudaSuccess) { cuda_fail(e, "ch_issue_mix_probe"); return -1.0; }
  return (double)ms;
}

double ch_fp64_peak_probe(double* sink, int blocks, int threads, int iters, void* stream) {
  if (!sink || blocks < 1 || threads < 1 || threads > 1024 || iters < 1) { fail(CH_EINVAL, "ch_fp64_peak_probe: bad argument"); return -1.0; }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  int dev = -1;
  {
    cudaPointerAttributes pa;
    if (cudaPointerGetAttributes(&pa, sink) == cudaSuccess && pa.type == cudaMemoryTypeDevice) dev = pa.device;
    else cudaGetLastError();
  }
  DeviceGuard guard(dev);
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) { fail(CH_ECUDA, "event create"); return -1.0; }
  k_dfma_probe<<<blocks, threads, 0, st>>>(sink, iters);   // warm-up
  cudaEventRecord(e0, st);
  k_dfma_probe<<<blocks, threads, 0, st>>>(sink, iters);
  cudaEventRecord(e1, st);
  cudaError_t e = cudaEventSynchronize(e1);
  float ms = -1.f;
  if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  if (e != cudaSuccess) { cuda_fail(e, "ch_fp64_peak_probe"); return -1.0; }
  return (double)ms;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// ch_dt_noalloc: Eq. 22 for callers that cannot allocate (code under CUDA graph capture, tight serving
// loops, harnesses that forbid cudaMalloc).  A variant of k_dt: the same cell_rate per cell, but the grid reduction
// goes through per-CTA partial maxima kept in a FILE-SCOPE device array instead of the reduction cells of a bound
// workspace, and a second one-CTA kernel finishes dt = cfl / max on the device.  No context, no workspace, no
// cudaMalloc / cudaFree / cudaHostAlloc: the caller passes the padded state (input) and one double (output).
//   scratch: g_na_scratch, 32 header cells + 65536 partial maxima = 524 544 B, held by every GPU that loads the
//   library until exit; one partial per CTA of 256 cells => at most kNaMaxCells = 16 777 216 real cells (256^3).
// In host code the NAME g_na_scratch is a host-side stand-in, not a device address: the address each device gave
// the array is asked once per device, with that device current, through cudaGetSymbolAddress, and that is what the
// kernels get.  Every call shares the array and it keeps the last call's contents: the non-physical flag is cleared
// at the start of each call (the partials a call reads it has written itself); two calls that overlap on the GPU
// (different streams, no ordering) race on it.
// ---------------------------------------------------------------------------------------------
namespace {

constexpr int kNaThreads = 256;
constexpr int kNaBlocks = 65536;                                        // partial maxima the scratch holds
constexpr int kNaHeader = 32;                                           // [0] non-physical flag; rest unused (alignment)
constexpr long long kNaMaxCells = (long long)kNaBlocks * kNaThreads;    // 16 777 216 real cells
constexpr int kNaMaxDevices = 64;

static __device__ __align__(256) unsigned long long g_na_scratch[kNaHeader + kNaBlocks];

// one CTA per 256 real cells: its maximum of (|v_d| + a) / dx_d -> scratch[kNaHeader + blockIdx.x]
__global__ void __launch_bounds__(kNaThreads) k_dt_partials(const StepArgs A, unsigned long long* __restrict__ scratch) {
  __shared__ double s_max[kNaThreads / 32];
  __shared__ int s_bad;
  const Geom& g = A.geo;
  const long long N = (long long)g.n[0] * g.n[1] * g.n[2];
  const long long id = (long long)blockIdx.x * kNaThreads + threadIdx.x;
  if (threadIdx.x == 0) s_bad = 0;
  __syncthreads();
  double t = 0.0;
  bool bad = false;
  if (id < N) {
    const int i = (int)(id % g.n[0]);
    const long long r = id / g.n[0];
    const int j = (int)(r % g.n[1]);
    const int k = (int)(r / g.n[1]);
    const long long q = (long long)(i + g.g[0]) + (long long)(j + g.g[1]) * g.st[1] + (long long)(k + g.g[2]) * g.st[2];
    t = cell_rate(A, A.u[q], A.u[g.np + q], A.u[2 * g.np + q], A.u[3 * g.np + q], A.u[4 * g.np + q], bad);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) t = fmax(t, __shfl_xor_sync(0xffffffffu, t, o));
  if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) s_bad = 1;
  if ((threadIdx.x & 31) == 0) s_max[threadIdx.x >> 5] = t;
  __syncthreads();
  if (threadIdx.x == 0) {
    double v = s_max[0];
#pragma unroll
    for (int w = 1; w < kNaThreads / 32; ++w) v = fmax(v, s_max[w]);
    scratch[kNaHeader + blockIdx.x] = (unsigned long long)__double_as_longlong(v);
    if (s_bad) atomicOr(scratch, 1ULL);
  }
}

// one CTA: maximum of the partials, dt = cfl * (1 / max) rounded as ch_compute_dt rounds it on the host;
// NaN if a non-physical cell (rho <= 0 or non-finite) was met
__global__ void __launch_bounds__(1024) k_dt_finish(const unsigned long long* __restrict__ scratch, int nblocks, double cfl,
                                                    double* __restrict__ dt_out) {
  __shared__ double s_max[32];
  double v = 0.0;
  for (int b = threadIdx.x; b < nblocks; b += blockDim.x) v = fmax(v, __longlong_as_double((long long)scratch[kNaHeader + b]));
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  if ((threadIdx.x & 31) == 0) s_max[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) v = fmax(v, s_max[w]);
    dt_out[0] = scratch[0] != 0ULL ? __longlong_as_double(0x7FF8000000000000LL) : __dmul_rn(cfl, __ddiv_rn(1.0, v));
  }
}

std::mutex g_na_mutex;
unsigned long long* g_na_ptr[kNaMaxDevices] = {};     // device address of g_na_scratch, per device (nullptr: not asked yet)

// the device address of the scratch array on `dev` (which must be current)
int na_scratch(int dev, unsigned long long** out) {
  if (dev < 0 || dev >= kNaMaxDevices) return fail(CH_EINVAL, "ch_dt_noalloc: device index beyond 63");
  std::lock_guard<std::mutex> lock(g_na_mutex);
  if (!g_na_ptr[dev]) {
    unsigned long long* p = nullptr;
    CH_CUDA(cudaGetSymbolAddress((void**)&p, g_na_scratch), "cudaGetSymbolAddress(g_na_scratch)");
    if (!p) return fail(CH_ECUDA, "ch_dt_noalloc: cudaGetSymbolAddress returned a null address");
    g_na_ptr[dev] = p;
  }
  *out = g_na_ptr[dev];
  return CH_OK;
}

}  // namespace

extern "C" {

long long ch_noalloc_max_cells(void) { return kNaMaxCells; }

int ch_noalloc_setup(void) {
  int dev = -1;
  CH_CUDA(cudaGetDevice(&dev), "cudaGetDevice");
  unsigned long long* p = nullptr;
  return na_scratch(dev, &p);
}

int ch_dt_noalloc(const double* u_padded, int nx, int ny, int nz, int nghost, double gamma, double dx, double dy, double dz,
                  double cfl, double* dt_out, void* stream) {
  if (!u_padded || !dt_out) return fail(CH_EINVAL, "ch_dt_noalloc: null pointer");
  if (!(gamma > 1.0) || !std::isfinite(gamma)) return fail(CH_EINVAL, "ch_dt_noalloc: gamma must be > 1");
  if (!(cfl > 0.0) || !(cfl <= 1.0)) return fail(CH_EINVAL, "ch_dt_noalloc: cfl not in (0,1]");
  if (!(dx > 0.0) || !(dy > 0.0) || !(dz > 0.0) || !std::isfinite(dx) || !std::isfinite(dy) || !std::isfinite(dz))
    return fail(CH_EINVAL, "ch_dt_noalloc: cell widths must be positive");
  StepArgs A = {};
  if (!geometry(nx, ny, nz, nghost, A.geo)) return fail(CH_EINVAL, "ch_dt_noalloc: bad grid (n >= 1, nghost >= 3, active n >= nghost)");
  const long long N = (long long)nx * ny * nz;
  if (N > kNaMaxCells)
    return fail(CH_EINVAL, "ch_dt_noalloc: more than 16777216 real cells (256^3): the static scratch holds one partial maximum "
                           "per 256 cells, 65536 of them; use ch_compute_dt with a bound workspace for larger grids");
  cudaPointerAttributes pa, pb;
  if (cudaPointerGetAttributes(&pa, u_padded) != cudaSuccess || pa.type != cudaMemoryTypeDevice ||
      cudaPointerGetAttributes(&pb, dt_out) != cudaSuccess || pb.type != cudaMemoryTypeDevice || pa.device != pb.device) {
    cudaGetLastError();
    return fail(CH_EINVAL, "ch_dt_noalloc: u_padded and dt_out must be device memory of one GPU");
  }
  DeviceGuard guard(pa.device);
  unsigned long long* scratch = nullptr;
  int rc = na_scratch(pa.device, &scratch);
  if (rc != CH_OK) return rc;
  A.gas.gamma = gamma; A.gas.gm1 = gamma - 1.0;                  // all cell_rate reads of the gas
  const double w[3] = {dx, dy, dz};
  for (int d = 0; d < 3; ++d) { A.dx[d] = w[d]; A.idx[d] = 1.0 / w[d]; A.dtdx[d] = 0.0; }
  A.u = const_cast<double*>(u_padded);                           // read only
  A.ext = 1;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int nblocks = (int)((N + kNaThreads - 1) / kNaThreads);
  CH_CUDA(cudaMemsetAsync(scratch, 0, sizeof(unsigned long long), st), "ch_dt_noalloc: clearing the flag");   // must start at zero
  k_dt_partials<<<(unsigned)nblocks, kNaThreads, 0, st>>>(A, scratch);
  k_dt_finish<<<1, 1024, 0, st>>>(scratch, nblocks, cfl, dt_out);
  CH_CUDA(cudaGetLastError(), "ch_dt_noalloc kernels");
  return CH_OK;
}

}  // extern "C"
