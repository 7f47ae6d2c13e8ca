"""Pins of the oracle's PPMC reconstruction + characteristic tracing (oracle/cholla_ref.cpp:
char_project, char_backproject, limited_slope, ppmc_cell) against the
mathematics, not against a retyped copy of its formulas:

* A9/A11 must be the left/right eigenvectors of the primitive-variable matrix A(w) of Eq. 15-16
  (P:L85-93): L R = I and R diag(lambda) L = A, with A and lambda from numpy.linalg.eig — pins
  the garbled first row of A9 (reading G1);
* the limiter (A10) on monotone / extremum / linear data;
* A20 on linear data and on smooth data (the classical 7/12, -1/12 interpolant);
* monotonicity (A21-A23) as properties;
* characteristic tracing (A25-A33): the traced state must equal the reference average plus the
  eigen-projections (numeric eigenvectors) of differences of EXACT averages of the cell's
  parabola over each wave's domain of dependence (numerical quadrature) — pins G2, G3;
* dt = 0 gives W* = W;  mirror symmetry is bitwise.
"""
import numpy as np
import pytest

GAMMA = 5.0 / 3.0


def A_matrix(w, gamma):
    """Quasi-linear matrix of the 1-D Euler equations in primitive variables (Eq. 15) with
    two passively advected transverse velocities."""
    rho, u, _, _, p = w
    A = np.diag([u] * 5).astype(float)
    A[0, 1] = rho
    A[1, 4] = 1.0 / rho
    A[4, 1] = gamma * p
    return A


def oracle_LR(ref, rho, a):
    L = np.array([ref.char_project(rho, a, e) for e in np.eye(5)]).T      # L[:, j] = project(e_j)
    R = np.array([ref.char_backproject(rho, a, e) for e in np.eye(5)]).T
    return L, R


def test_A9_A11_are_eigenvectors_of_A(ref):
    rng = np.random.default_rng(0)
    for _ in range(50):
        w = np.array([rng.uniform(0.1, 3), rng.normal(), rng.normal(), rng.normal(), rng.uniform(0.1, 3)])
        a = np.sqrt(GAMMA * w[4] / w[0])
        L, R = oracle_LR(ref, w[0], a)
        assert np.allclose(L @ R, np.eye(5), atol=1e-14)                  # A11 o A9 = identity
        lam = np.diag([w[1] - a, w[1], w[1], w[1], w[1] + a])             # A8
        A = A_matrix(w, GAMMA)
        assert np.allclose(R @ lam @ L, A, atol=1e-13)
        ev = np.sort(np.linalg.eigvals(A).real)
        assert np.allclose(ev, np.sort(np.diag(lam)), atol=1e-7)   # triple eigenvalue: eig() is ~sqrt(eps) there


def test_roundtrip_identity_random(ref):
    rng = np.random.default_rng(1)
    for _ in range(200):
        rho, a = rng.uniform(0.01, 10), rng.uniform(0.01, 10)
        dw = rng.normal(size=5)
        back = ref.char_backproject(rho, a, ref.char_project(rho, a, dw))
        assert np.allclose(back, dw, rtol=0, atol=8e-16 * (1 + np.abs(dw).max() * max(1, rho * a, 1 / (rho * a), a * a, 1 / (a * a))))


def test_limiter_properties(ref):
    rng = np.random.default_rng(2)
    w0 = np.array([1.0, 0.3, -0.2, 0.1, 0.8])
    # linear data: slope = the centred difference for every component
    b = np.array([0.01, 0.02, -0.03, 0.015, 0.005])
    dw = ref.limited_slope(GAMMA, w0 - b, w0, w0 + b)
    assert np.allclose(dw, b, rtol=1e-13)
    # a strict extremum in every characteristic field -> zero slope
    d = np.array([0.05, 0.0, 0.02, -0.01, 0.0])
    dw = ref.limited_slope(GAMMA, w0 - d, w0, w0 - d)
    assert np.all(dw == 0.0)
    # transverse velocities are their own characteristic fields: classical MC limiter
    for _ in range(100):
        vm, v0, vp = rng.normal(size=3)
        wm, wc, wp = w0.copy(), w0.copy(), w0.copy()
        wm[2], wc[2], wp[2] = vm, v0, vp
        dL, dR, dC = v0 - vm, vp - v0, 0.5 * (vp - vm)
        want = 0.0 if dL * dR <= 0 else np.sign(dC) * min(abs(dC), 2 * abs(dL), 2 * abs(dR))
        assert ref.limited_slope(GAMMA, wm, wc, wp)[2] == pytest.approx(want, abs=1e-16)


def stencil(fn):
    return np.array([fn(s) for s in (-2, -1, 0, 1, 2)], dtype=float)


def test_ppmc_linear_data_is_exact(ref):
    base = np.array([1.0, 0.3, -0.2, 0.1, 0.8])
    b = np.array([0.01, 0.02, -0.03, 0.015, 0.005])
    WL, WR, WLs, WRs = ref.ppmc_cell(GAMMA, 0.0, stencil(lambda s: base + b * s))
    assert np.allclose(WL, base - 0.5 * b, rtol=1e-14) and np.allclose(WR, base + 0.5 * b, rtol=1e-14)
    assert np.array_equal(WLs, WL) and np.array_equal(WRs, WR)           # dt = 0: no evolution


def test_ppmc_smooth_data_is_the_classical_fourth_order_interpolant(ref):
    """Where the limiters are inactive A20 = 7/12 (w_i + w_{i+1}) - 1/12 (w_{i-1} + w_{i+2})."""
    base = np.array([1.0, 0.3, -0.2, 0.1, 0.8])
    amp = np.array([0.02, 0.01, 0.015, -0.01, 0.01])
    f = lambda s: base + amp * np.sin(0.3 * s + 0.4)                      # monotone over the stencil
    w = stencil(f)
    WL, WR, _, _ = ref.ppmc_cell(GAMMA, 0.0, w)
    # the 7/12,-1/12 form needs w_{i+2} for W_R and w_{i-2} for W_L: both are in the stencil
    assert np.allclose(WR, 7 / 12 * (w[2] + w[3]) - 1 / 12 * (w[1] + w[4]), atol=1e-15)
    assert np.allclose(WL, 7 / 12 * (w[1] + w[2]) - 1 / 12 * (w[0] + w[3]), atol=1e-15)


def test_ppmc_monotonicity_properties(ref):
    rng = np.random.default_rng(5)
    for _ in range(500):
        w = rng.normal(size=(5, 5)) * 0.3
        w[:, 0] = rng.uniform(0.2, 3, 5)
        w[:, 4] = rng.uniform(0.2, 3, 5)
        WL, WR, _, _ = ref.ppmc_cell(GAMMA, 0.0, w)
        wi, wm, wp = w[2], w[1], w[3]
        assert np.all(WL >= np.minimum(wi, wm)) and np.all(WL <= np.maximum(wi, wm))   # A23
        assert np.all(WR >= np.minimum(wi, wp)) and np.all(WR <= np.maximum(wi, wp))


def test_ppmc_no_overshoot_on_monotone_steep_data(ref):
    """Transverse velocities are their own characteristic fields, so for them A20-A23 act
    on a scalar: for monotone data of any steepness the limited parabola must have no interior
    extremum (CW84's condition |w6| <= |W_R - W_L|, which A21/A22 enforce)."""
    rng = np.random.default_rng(6)
    hit = 0
    for _ in range(500):
        w = np.tile(np.array([1.0, 0.2, 0.0, 0.0, 0.9]), (5, 1))
        inc = rng.uniform(0, 1, 4) ** 4                      # a few large jumps, many small ones
        w[:, 2] = np.concatenate([[0.0], np.cumsum(inc)])
        w[:, 3] = -w[:, 2][::-1]
        WL, WR, _, _ = ref.ppmc_cell(GAMMA, 0.0, w)
        for c in (2, 3):
            d = WR[c] - WL[c]
            w6 = 6 * (w[2, c] - 0.5 * (WL[c] + WR[c]))
            tol = 1e-13 * (1.0 + np.abs(w[:, c]).max())       # w6 is a difference of O(1) numbers
            assert abs(w6) <= abs(d) + tol
            hit += abs(abs(w6) - abs(d)) < tol and abs(d) > 1e3 * tol
    assert hit > 20                                          # A22 really fired in some cases


def parabola_avg(WL, WR, wi, x0, x1, npts=8):
    """Exact average over [x0,x1] (cell coordinate xi in [0,1]) of the unique parabola with face
    values WL, WR and cell mean wi — by Gauss-Legendre quadrature of the Lagrange-form quadratic
    (no use of the w6 closed forms the oracle uses)."""
    if x1 == x0:
        return WL if x0 == 0.0 else WR
    # q(xi) = c0 + c1 xi + c2 xi^2 with q(0)=WL, q(1)=WR, int_0^1 q = wi
    c0 = WL
    c2 = 3.0 * (WL + WR) - 6.0 * wi
    c1 = WR - WL - c2
    xs, ws = np.polynomial.legendre.leggauss(npts)
    xm = 0.5 * (x0 + x1) + 0.5 * (x1 - x0) * xs
    return sum(wgt * (c0 + c1 * x + c2 * x * x) for x, wgt in zip(xm, ws)) / 2.0


def numeric_projectors(w, gamma):
    """Spectral projectors P_minus, P_0, P_plus of A(w) from numpy's eigen-decomposition."""
    A = A_matrix(w, gamma)
    lam, V = np.linalg.eig(A)
    lam = lam.real; V = V.real
    a = np.sqrt(gamma * w[4] / w[0])
    # P_minus, P_plus from the simple eigenvalues; P_0 = I - P_minus - P_plus
    P = {}
    for name, target in (("m", w[1] - a), ("p", w[1] + a)):
        k = int(np.argmin(np.abs(lam - target)))
        r = V[:, k]
        lamT, VT = np.linalg.eig(A.T)
        kk = int(np.argmin(np.abs(lamT.real - target)))
        l = VT[:, kk].real
        P[name] = np.outer(r, l) / (l @ r)
    P["0"] = np.eye(5) - P["m"] - P["p"]
    return P, (w[1] - a, w[1], w[1] + a)


@pytest.mark.parametrize("mach", [-2.5, -0.6, 0.0, 0.4, 3.0])
def test_characteristic_tracing_equals_projected_parabola_averages(ref, mach):
    rng = np.random.default_rng(int(10 * mach) + 100)
    for _ in range(40):
        base = np.array([rng.uniform(0.5, 2), 0.0, rng.normal(), rng.normal(), rng.uniform(0.5, 2)])
        a0 = np.sqrt(GAMMA * base[4] / base[0])
        base[1] = mach * a0
        slope = rng.normal(size=5) * 0.02
        curv = rng.normal(size=5) * 0.004
        w = stencil(lambda s: base + slope * s + curv * s * s)
        dtdx = rng.uniform(0.05, 0.45) / (abs(base[1]) + a0)
        WL, WR, WLs, WRs = ref.ppmc_cell(GAMMA, dtdx, w)
        wi = w[2]
        P, (lm, l0, lp) = numeric_projectors(wi, GAMMA)
        lam = {"m": lm, "0": l0, "p": lp}
        # left face: domain of dependence of wave n is [0, -lambda_n dt/dx] if lambda_n < 0
        avgL = {n: np.array([parabola_avg(WL[c], WR[c], wi[c], 0.0, max(-lam[n], 0.0) * dtdx) for c in range(5)]) for n in lam}
        wantL = avgL["m"].copy()
        for n in ("0", "p"):
            if lam[n] < 0:
                wantL += P[n] @ (avgL[n] - avgL["m"])
        # right face: [1 - lambda_n dt/dx, 1] if lambda_n > 0
        avgR = {n: np.array([parabola_avg(WL[c], WR[c], wi[c], 1.0 - max(lam[n], 0.0) * dtdx, 1.0) for c in range(5)]) for n in lam}
        wantR = avgR["p"].copy()
        for n in ("m", "0"):
            if lam[n] > 0:
                wantR += P[n] @ (avgR[n] - avgR["p"])
        assert np.allclose(WLs, wantL, rtol=0, atol=2e-14), (WLs - wantL)
        assert np.allclose(WRs, wantR, rtol=0, atol=2e-14), (WRs - wantR)


def test_tracing_of_a_pure_entropy_wave_is_upwind_advection(ref):
    """u, p uniform, rho smooth: the exact solution is advection at speed u.  The traced right
    face state (u>0) must be the parabola's average over the slab that crosses the face."""
    u0, p0 = 0.7, 1.0
    rho = lambda s: 1.0 + 0.05 * s + 0.004 * s * s
    w = stencil(lambda s: np.array([rho(s), u0, 0.0, 0.0, p0]))
    dtdx = 0.3
    WL, WR, WLs, WRs = ref.ppmc_cell(GAMMA, dtdx, w)
    want = parabola_avg(WL[0], WR[0], w[2][0], 1.0 - u0 * dtdx, 1.0)
    assert abs(WRs[0] - want) < 1e-15 and WRs[1] == pytest.approx(u0, abs=1e-15) and WRs[4] == pytest.approx(p0, abs=1e-15)
    # left face: contact moves away (u>0) — density there sees no contact contribution: stays the
    # reference average under lambda^m, with its acoustic part only; u,p uniform => W*_L rho equals
    # the lambda^m average minus nothing
    a0 = np.sqrt(GAMMA * p0 / w[2][0])
    wantL = parabola_avg(WL[0], WR[0], w[2][0], 0.0, max(-(u0 - a0), 0) * dtdx)
    assert abs(WLs[0] - wantL) < 1e-15


def test_mirror_symmetry_is_bitwise(ref):
    rng = np.random.default_rng(9)
    flip = np.array([1.0, -1.0, 1.0, 1.0, 1.0])
    for _ in range(300):
        w = rng.normal(size=(5, 5)) * 0.3
        w[:, 0] = rng.uniform(0.2, 3, 5)
        w[:, 4] = rng.uniform(0.2, 3, 5)
        dtdx = rng.uniform(0, 0.3)
        WL, WR, WLs, WRs = ref.ppmc_cell(GAMMA, dtdx, w)
        wm = (w * flip)[::-1].copy()
        ML, MR, MLs, MRs = ref.ppmc_cell(GAMMA, dtdx, wm)
        assert np.array_equal(ML, WR * flip) and np.array_equal(MR, WL * flip)
        assert np.array_equal(MLs, WRs * flip) and np.array_equal(MRs, WLs * flip)


def test_cons_prim_roundtrip_and_floor(ref):
    rng = np.random.default_rng(4)
    for _ in range(100):
        w = np.array([rng.uniform(0.1, 3), rng.normal(), rng.normal(), rng.normal(), rng.uniform(0.1, 3)])
        u = ref.prim_to_cons(GAMMA, w)
        # Eq. 6-9 written out independently
        E = w[4] / (GAMMA - 1) + 0.5 * w[0] * (w[1] ** 2 + w[2] ** 2 + w[3] ** 2)
        assert np.allclose(u, [w[0], w[0] * w[1], w[0] * w[2], w[0] * w[3], E], rtol=1e-15)
        assert np.allclose(ref.cons_to_prim(GAMMA, u), w, rtol=1e-13)
    # negative internal energy -> pressure floor 1e-20
    assert ref.cons_to_prim(GAMMA, [1.0, 1.0, 0, 0, 0.1])[4] == 1e-20
