"""Pins of the oracle's PPMP and PLMP reconstructions (oracle/cholla_ref.cpp: ppmp_cell, plmp_cell; A.4 P:L886-1049,
A.1 P:L679-717) against what the paper prints and the mathematics fixes:

* A34 on linear data reproduces it, on smooth data it is the classical fourth-order interpolant (7/12, -1/12);
* contact steepening A35-A41: a density step carried by one cell (values worked out by hand from the paper's
  formulas) is rebuilt as the full jump inside that cell; the same step with a pressure jump (A36) or with too
  small a jump (A35) is NOT steepened; this separates reading G12 (A38: opposite curvature) from the printed sign;
* shock flattening A42-A47: a hand-made pressure jump in a compressing flow gives F = 1 (faces = cell average for
  every variable), the same jump in an expanding flow (A45) or a weak one (A44) gives F = 0;
* A48 keeps every parabola monotone; mirror symmetry (catches A41's rho_{i-1} typo, A48's third line, the sign
  pattern of A54: readings G13-G15);
* characteristic tracing A49-A56 equals, to first order in the amplitude, the spectral projection (numpy
  eigen-decomposition) of the parabola's averages over each characteristic's domain of dependence; the residual
  is quadratic in the amplitude (the 1/rho form and the reference-state sound speeds are a different linearisation);
* scheme level: second-order convergence, uniform states, conservation, 1-D in 3-D bitwise, and the paper's own
  observation that PPMP resolves the Sod contact over two zones where PPMC needs three to four.
"""
import math

import numpy as np
import pytest

from paper_1410_4194_b200 import workloads as wl
from paper_1410_4194_b200.driver import run
from tests.test_oracle_ppmc import GAMMA, numeric_projectors

PPMC, PPMP, PLMP = 0, 3, 4


def stencil7(fn):
    return np.array([fn(s) for s in (-3, -2, -1, 0, 1, 2, 3)], dtype=float)


def test_ppmp_linear_and_smooth_data(ref):
    base = np.array([1.0, 0.3, -0.2, 0.1, 0.8])
    b = np.array([0.01, 0.02, -0.03, 0.015, 0.005])
    WL, WR, WLs, WRs = ref.ppmp_cell(GAMMA, 0.0, stencil7(lambda s: base + b * s))
    assert np.allclose(WL, base - 0.5 * b, rtol=1e-14) and np.allclose(WR, base + 0.5 * b, rtol=1e-14)
    assert np.allclose(WLs, WL, rtol=1e-14) and np.allclose(WRs, WR, rtol=1e-14)         # dt = 0: W* = W
    # smooth monotone data, inactive limiter: A34 = 7/12 (w_i + w_{i+1}) - 1/12 (w_{i-1} + w_{i+2})
    f = lambda s: base * (1.0 + 0.02 * s + 0.001 * s * s)
    w = stencil7(f)
    WL, WR, _, _ = ref.ppmp_cell(GAMMA, 0.0, w)
    assert np.allclose(WR, 7.0 / 12.0 * (w[3] + w[4]) - 1.0 / 12.0 * (w[2] + w[5]), rtol=1e-13)
    assert np.allclose(WL, 7.0 / 12.0 * (w[2] + w[3]) - 1.0 / 12.0 * (w[1] + w[4]), rtol=1e-13)


def contact(rho, p=(1,) * 7, u=(0.3,) * 7):
    w = np.zeros((7, 5))
    w[:, 0] = rho; w[:, 1] = u; w[:, 4] = p
    return w


def test_contact_steepening_by_hand(ref):
    """rho = 1,1,1,[1.5],2,2,2 at uniform p: A35 jump 1 > 0.01; A36 0 < 0.1 gamma; A37 d2rho_{i-1} = +0.5/6,
    d2rho_{i+1} = -0.5/6 (opposite curvature: a contact, G12); A39 eta~ = (1/6)/1; A40 eta = min(20/6 - 1, 1) = 1;
    the limited slopes of cells i-1 and i+1 vanish (one-sided differences are 0), so A41 gives rho_L = rho_{i-1} = 1
    and rho_R = rho_{i+1} = 2 (G13): the cell carries the whole jump, and A48 leaves that pair alone."""
    WL, WR, _, _ = ref.ppmp_cell(GAMMA, 0.0, contact([1, 1, 1, 1.5, 2, 2, 2]))
    assert WL[0] == 1.0 and WR[0] == 2.0
    assert WL[4] == 1.0 and WR[4] == 1.0 and WL[1] == 0.3
    # unsteepened A34 value for the same data: 1/2 (1.5 + 1) - (0.5 - 0)/6
    plain = (0.5 * 2.5 - 0.5 / 6.0, 0.5 * 3.5 + 0.5 / 6.0)
    # A36: with a pressure jump of the same relative size it is a shock-like profile, not a contact
    WL, WR, _, _ = ref.ppmp_cell(GAMMA, 0.0, contact([1, 1, 1, 1.5, 2, 2, 2], p=[1, 1, 1, 1.5, 2, 2, 2],
                                        u=[0, 0, 0, 0.1, 0.2, 0.2, 0.2]))      # expanding: A45 keeps the flattening out
    assert abs(WL[0] - plain[0]) < 1e-15 and abs(WR[0] - plain[1]) < 1e-15
    # A35: the same shape at 0.5 % amplitude is noise
    WL, WR, _, _ = ref.ppmp_cell(GAMMA, 0.0, contact(1.0 + 0.005 * (np.array([1, 1, 1, 1.5, 2, 2, 2]) - 1.0)))
    assert abs(WL[0] - (1.0 + 0.005 * (plain[0] - 1.0))) < 1e-15
    # a falling contact is the mirror image
    WL, WR, _, _ = ref.ppmp_cell(GAMMA, 0.0, contact([2, 2, 2, 1.5, 1, 1, 1]))
    assert WL[0] == 2.0 and WR[0] == 1.0
    # partial steepening: eta~ = 0.075 -> eta = 0.5, by hand: rho = 1, 1, 1.05+..., smooth ramp
    rho = np.array([1.0, 1.0, 1.3, 1.5, 1.7, 2.0, 2.0])
    d2m = (rho[3] - 2 * rho[2] + rho[1]) / 6.0
    d2p = (rho[5] - 2 * rho[4] + rho[3]) / 6.0
    assert d2m * d2p < 0
    WL, WR, _, _ = ref.ppmp_cell(GAMMA, 0.0, contact(rho))
    assert WL[0] < WR[0] and rho[2] <= WL[0] and WR[0] <= rho[4]


def test_shock_flattening_by_hand(ref):
    """p = 1,1,1,[5],10,10,10 with u falling 2 -> 0 (compression): for cell i, A42 S = (10 - 1)/(10 - 1) = 1,
    A43 F~ = min(1, 10 (1 - 0.75)) = 1, A44 9/1 > 1/3, A45 u_{i+1} - u_{i-1} = -2 < 0, so F = 1 and A47 returns the
    cell average for EVERY variable.  The same pressures in an expanding flow (A45) are not flattened, and a 20 %
    pressure step (A44) is not either."""
    rho = [1, 1, 1, 1.2, 1.5, 1.5, 1.5]
    w = contact(rho, p=[1, 1, 1, 5, 10, 10, 10], u=[2, 2, 2, 1, 0, 0, 0])
    WL, WR, _, _ = ref.ppmp_cell(GAMMA, 0.0, w)
    assert np.array_equal(WL, w[3]) and np.array_equal(WR, w[3])
    w2 = contact(rho, p=[1, 1, 1, 5, 10, 10, 10], u=[0, 0, 0, 1, 2, 2, 2])
    WL, WR, _, _ = ref.ppmp_cell(GAMMA, 0.0, w2)
    assert WL[4] < 5.0 < WR[4] and WL[1] < 1.0 < WR[1]
    w3 = contact(rho, p=[1, 1, 1, 1.1, 1.2, 1.2, 1.2], u=[2, 2, 2, 1, 0, 0, 0])
    WL, WR, _, _ = ref.ppmp_cell(GAMMA, 0.0, w3)
    assert WL[4] < 1.1 < WR[4]
    # A46: the first post-shock cell has S = 5/9 itself (F~_i = 0) but p_{i+1} - p_{i-1} > 0 hands it F~_{i-1} = 1
    w4 = contact([1, 1, 1.2, 1.5, 1.5, 1.5, 1.5], p=[1, 1, 5, 10, 10, 10, 10], u=[2, 2, 1, 0, 0, 0, 0])
    WL, WR, _, _ = ref.ppmp_cell(GAMMA, 0.0, w4)      # cell i is the first post-shock cell; F~_{i-1} = 1, dp > 0
    assert np.array_equal(WL, w4[3]) and np.array_equal(WR, w4[3])
    # uniform pressure: 0/0 in A42 never reaches the result (S19)
    WL, WR, _, _ = ref.ppmp_cell(GAMMA, 0.0, contact([1, 1.1, 1.2, 1.3, 1.4, 1.5, 1.6], u=[2, 2, 2, 1, 0, 0, 0]))
    assert np.all(np.isfinite(WL)) and np.all(np.isfinite(WR))


def test_monotone_parabolas_and_mirror_symmetry(ref):
    rng = np.random.default_rng(11)
    flip = np.array([1, -1, 1, 1, 1.0])
    for _ in range(300):
        w = rng.uniform(0.3, 2.0, size=(7, 5)); w[:, 1] = rng.normal(size=7) * 0.7
        WL, WR, WLs, WRs = ref.ppmp_cell(GAMMA, 0.2, w)
        wi = w[3]
        for c in range(5):
            # A48: no interior extremum: the parabola's extremum abscissa lies outside (0, 1)
            d, w6 = WR[c] - WL[c], 6.0 * (wi[c] - 0.5 * (WL[c] + WR[c]))
            assert (WR[c] - wi[c]) * (wi[c] - WL[c]) >= 0.0
            assert abs(w6) <= abs(d) * (1 + 1e-12)
        ML, MR, MLs, MRs = ref.ppmp_cell(GAMMA, 0.2, w[::-1] * flip)
        assert np.allclose(MR * flip, WL, rtol=0, atol=1e-14) and np.allclose(ML * flip, WR, rtol=0, atol=1e-14)
        assert np.allclose(MRs * flip, WLs, rtol=0, atol=1e-13) and np.allclose(MLs * flip, WRs, rtol=0, atol=1e-13)
        ML, MR, MLs, MRs = ref.plmp_cell(GAMMA, 0.2, w[::-1] * flip)
        PL, PR, PLs, PRs = ref.plmp_cell(GAMMA, 0.2, w)
        assert np.allclose(MRs * flip, PLs, rtol=0, atol=1e-13) and np.allclose(MLs * flip, PRs, rtol=0, atol=1e-13)


def projected_parabola_states(WL, WR, wi, dtdx, gamma):
    """What characteristic tracing means (Colella & Woodward 1984): the average of the parabola over the domain of
    dependence of the fastest approaching wave, corrected wave by wave with the spectral projectors of A(w_i)."""
    P, (lm, l0, lp) = numeric_projectors(wi, gamma)
    lam = {"m": lm, "0": l0, "p": lp}
    d, w6 = WR - WL, 6.0 * (wi - 0.5 * (WL + WR))

    def mean(x0, x1):           # mean of WL + x (d + w6 (1 - x)) over [x0, x1]
        if x1 == x0:
            return WL + x0 * (d + w6 * (1 - x0))
        F = lambda x: WL * x + d * x * x / 2 + w6 * (x * x / 2 - x ** 3 / 3)
        return (F(x1) - F(x0)) / (x1 - x0)
    avgL = {n: mean(0.0, max(-lam[n], 0.0) * dtdx) for n in lam}
    wantL = avgL["m"].copy()
    for n in ("0", "p"):
        if lam[n] < 0:
            wantL += P[n] @ (avgL[n] - avgL["m"])
    avgR = {n: mean(1.0 - max(lam[n], 0.0) * dtdx, 1.0) for n in lam}
    wantR = avgR["p"].copy()
    for n in ("m", "0"):
        if lam[n] > 0:
            wantR += P[n] @ (avgR[n] - avgR["p"])
    return wantL, wantR


@pytest.mark.parametrize("mach", [-2.5, -0.6, -0.05, 0.4, 3.0])
def test_ppmp_tracing_is_the_projected_parabola_average_to_first_order(ref, mach):
    """A49-A56 against the spectral projection of the parabola's averages.  PPMP linearises about the reference
    state and in 1/rho, so the two differ at second order in the amplitude eps of the variation across the cell:
    the difference must fall by ~4 when eps is halved, and be tiny in absolute terms.  A wrong sign or a swapped
    term in A54-A56 (reading G15) leaves a first-order difference.  Density, normal velocity and pressure are
    compared on both faces; the transverse velocities only on the face the contact wave approaches — on the other
    face A56 takes v^0, which A51 leaves at the un-evolved face value, and that is checked as such."""
    rng = np.random.default_rng(int(10 * mach) + 300)
    for _ in range(25):
        base = np.array([rng.uniform(0.5, 2), 0.0, rng.normal(), rng.normal(), rng.uniform(0.5, 2)])
        a0 = np.sqrt(GAMMA * base[4] / base[0])
        base[1] = mach * a0
        shape1, shape2 = rng.normal(size=5), rng.normal(size=5)
        dtdx = rng.uniform(0.1, 0.45) / (abs(base[1]) + a0)
        errs = []
        for eps in (4e-3, 2e-3, 1e-3):
            w = stencil7(lambda s: base * (1.0 + eps * (shape1 * s + 0.2 * shape2 * s * s)))
            WL, WR, WLs, WRs = ref.ppmp_cell(GAMMA, dtdx, w)
            wantL, wantR = projected_parabola_states(WL, WR, w[3], dtdx, GAMMA)
            nvp = [0, 1, 4]
            e = max(np.max(np.abs(WLs - wantL)[nvp]), np.max(np.abs(WRs - wantR)[nvp]))
            if base[1] < 0:
                e = max(e, np.max(np.abs(WLs - wantL)[2:4]))
                assert np.array_equal(WRs[2:4], WR[2:4])
            else:
                e = max(e, np.max(np.abs(WRs - wantR)[2:4]))
                assert np.array_equal(WLs[2:4], WL[2:4])
            errs.append(e)
        assert errs[0] < 2e-4 and errs[2] < 2e-5, errs
        assert errs[0] < 1e-12 or errs[0] / errs[2] > 9.0, errs     # second order in eps (16 ideally), or exact


def wave_error(ref, n, recon):
    w = wl.linear_wave(n)
    G = ref.RefGrid(*w.shape, 4, w.gamma, w.bc)
    G.set_reconstruction(recon)
    run(G, w)
    return float(np.mean(np.abs(G.get_state() - w.u)))


@pytest.mark.parametrize("recon", [PPMP, PLMP])
def test_second_order_convergence(ref, recon):
    e = [wave_error(ref, n, recon) for n in (32, 64, 128)]
    assert math.log(e[0] / e[2]) / math.log(4.0) > 1.8, e


@pytest.mark.parametrize("recon", [PPMP, PLMP])
def test_uniform_state_conservation_and_embedding(ref, recon):
    u = wl.conserved(0.7, 0.3, -0.45, 0.21, 1.9, 1.4).reshape(5, 1, 1, 1) * np.ones((5, 6, 7, 8))
    G = ref.RefGrid(8, 7, 6, 4, 1.4, (1,) * 6)
    G.set_reconstruction(recon)
    G.set_state(u)
    G.step(G.compute_dt(0.4))
    assert np.array_equal(G.get_state(), u)
    w = wl.sweep(shape=(16, 12, 10))
    G = ref.RefGrid(*w.shape, 4, w.gamma, w.bc)
    G.set_reconstruction(recon)
    G.set_state(w.u)
    for _ in range(3):
        G.step(G.compute_dt(w.cfl))
    u1 = G.get_state()
    for f in range(5):
        assert abs(math.fsum(u1[f].ravel()) - math.fsum(w.u[f].ravel())) <= 1e-13 * (math.fsum(np.abs(w.u[f]).ravel()) + w.u[0].size)
    # a 1-D problem along y in a 3-D box equals the 1-D run bitwise (cyclic permutation of the velocities)
    s1 = wl.sod(48)
    G1 = ref.RefGrid(48, 1, 1, 4, s1.gamma, s1.bc); G1.set_reconstruction(recon); G1.set_state(s1.u)
    s3 = wl.sod(48, axis=1, n_other=5)
    G3 = ref.RefGrid(*s3.shape, 4, s3.gamma, s3.bc); G3.set_reconstruction(recon); G3.set_state(s3.u)
    G3.set_spacing(1.0 / 48, 1.0 / 48, 1.0 / 48)
    for _ in range(5):
        dt = G1.compute_dt(0.4)
        G1.step(dt); G3.step(dt)
    a, b = G1.get_state(), G3.get_state()
    assert np.array_equal(b[0, 2, :, 3], a[0, 0, 0, :]) and np.array_equal(b[2, 2, :, 3], a[1, 0, 0, :])
    assert np.array_equal(b[4, 0, :, 1], a[4, 0, 0, :])


def contact_width(ref, recon, n=100):
    s = wl.sod(n)
    G = ref.RefGrid(n, 1, 1, 4, s.gamma, s.bc)
    G.set_reconstruction(recon)
    run(G, s)
    rho = G.get_state()[0, 0, 0]
    x = (np.arange(n) + 0.5) / n
    lo, hi = 0.265573711705307, 0.426319428178495            # rho*_R, rho*_L (tests/golden/riemann_star_states.txt)
    frac = (rho - lo) / (hi - lo)
    return int(np.sum((x > 0.6) & (x < 0.8) & (frac > 0.05) & (frac < 0.95))), rho


def test_sod_contact_is_two_zones_with_ppmp_and_wider_with_ppmc(ref):
    """"the contact discontinuity is resolved over just two zones using PPMP, and over three to four zones
    using PPMC" (100 cells, t = 0.2).  With the printed sign of A38 the steepening never acts on a contact and PPMP
    gives three zones like PPMC (observed; reading G12)."""
    wp, rho = contact_width(ref, PPMP)
    wc, _ = contact_width(ref, PPMC)
    assert wp == 2, wp
    assert 3 <= wc <= 4, wc
    # and the solution is still the Sod solution: shock at 0.850, plateau densities
    x = (np.arange(100) + 0.5) / 100
    assert abs(rho[(x > 0.72) & (x < 0.82)].mean() - 0.265573711705307) < 5e-3
    assert abs(rho[(x > 0.55) & (x < 0.65)].mean() - 0.426319428178495) < 5e-3


def test_ppmp_and_hcorrection_exclude_each_other_and_ppmp_needs_four_ghosts(ref):
    G = ref.RefGrid(8, 8, 1, 3, 1.4, (1,) * 6)
    with pytest.raises(ValueError):
        G.set_reconstruction(PPMP)                               # 7-cell stencil
    G.set_reconstruction(PLMP)                                   # 3-cell stencil
    G = ref.RefGrid(8, 8, 1, 4, 1.4, (1,) * 6)
    G.set_solver(1); G.set_hcorrection(True)
    with pytest.raises(ValueError):
        G.set_reconstruction(PPMP)
    G.set_hcorrection(False); G.set_reconstruction(PPMP)
    with pytest.raises(ValueError):
        G.set_hcorrection(True)


def test_plmp_pure_advection_closed_form(ref):
    """A1-A7 on a density ramp carried by a uniform flow (u, p constant): F(U_L) - F(U_R) = -u (U_R - U_L) for every
    conserved component, so A6 / A7 give rho*_L = rho_L - (dt/2dx) u drho, rho*_R = rho_R - (dt/2dx) u drho with
    drho = rho_R - rho_L the limited slope, and velocity and pressure stay put: the exact half-step solution of
    linear advection at the two faces."""
    rng = np.random.default_rng(5)
    for _ in range(50):
        u, v, wv, p = rng.normal(), rng.normal(), rng.normal(), rng.uniform(0.5, 2.0)
        r0, b = rng.uniform(1.0, 2.0), rng.uniform(-0.1, 0.1)
        w = stencil7(lambda s: np.array([r0 + b * s, u, v, wv, p]))
        dtdx = rng.uniform(0.05, 0.4)
        WL, WR, WLs, WRs = ref.plmp_cell(GAMMA, dtdx, w)
        assert np.allclose(WL, [r0 - 0.5 * b, u, v, wv, p], rtol=1e-14) and np.allclose(WR, [r0 + 0.5 * b, u, v, wv, p], rtol=1e-14)
        shift = 0.5 * dtdx * u * b
        assert np.allclose(WLs, [r0 - 0.5 * b - shift, u, v, wv, p], rtol=1e-13, atol=1e-14)
        assert np.allclose(WRs, [r0 + 0.5 * b - shift, u, v, wv, p], rtol=1e-13, atol=1e-14)
