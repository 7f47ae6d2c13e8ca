"""Pins of the oracle's Roe solver with the HLLE failsafe (oracle/cholla_ref.cpp: riemann_roe; B.2,
P:L1166-1273) against what the mathematics fixes — not against a retyped copy of B23-B35:

* Roe's property U: an isolated discontinuity that satisfies the Rankine-Hugoniot conditions (a contact, a
  shear wave, an exact shock taken from tests/golden/riemann_star_states.txt) is upwinded exactly — the flux
  is F(W) of the upstream side (catches any wrong eigenvector / wave strength, incl. the garbled B29);
* consistency F(W, W) = Eq. 11; supersonic states return F_L / F_R; mirror symmetry; passive transverse shear;
* HLLE: the symmetric strong rarefaction (123 problem) fails Roe's positivity check and the HLL flux of a
  symmetric problem has the closed form (0, p - rho |u| a, 0, 0, 0);
* scheme level: Sod with the Roe solver converges to the exact solution, the 123 problem stays positive
  (P:L475-479), a sound wave converges at second order.
"""
import math
import os

import numpy as np
import pytest

from paper_1410_4194_b200 import workloads as wl
from paper_1410_4194_b200.driver import run

G = 1.4


def eq11(W, gamma=G):
    rho, u, v, w, p = W
    E = p / (gamma - 1) + 0.5 * rho * (u * u + v * v + w * w)
    return np.array([rho * u, rho * u * u + p, rho * u * v, rho * u * w, (E + p) * u])


def test_identical_states_give_eq11(ref):
    for W in ([1.3, 0.4, -0.2, 0.7, 2.1], [0.5, -0.9, 0.3, 0.0, 0.7], [2.0, 0.0, 0.0, 0.0, 1.0]):
        f, path = ref.riemann_roe(G, W, W)
        assert path in ("roe", "F_L", "F_R")
        assert np.allclose(f, eq11(W), rtol=0, atol=4e-16 * np.max(np.abs(eq11(W))) + 1e-16)


@pytest.mark.parametrize("u", [0.35, -0.35, 0.0])
def test_isolated_contact_and_shear_are_upwinded_exactly(ref, u):
    WL = [2.0, u, 0.3, -0.1, 1.5]
    WR = [0.7, u, -0.4, 0.6, 1.5]          # same normal velocity and pressure: a contact + shear, speed u
    f, path = ref.riemann_roe(G, WL, WR)
    assert path == "roe"
    want = eq11(WL) if u > 0 else eq11(WR) if u < 0 else None
    if want is None:                        # stationary: both sides carry the same flux (0, p, 0, 0, 0)
        assert np.allclose(f, [0, 1.5, 0, 0, 0], atol=1e-15)
    else:
        assert np.allclose(f, want, rtol=0, atol=2e-15)


def golden_star():
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "riemann_star_states.txt")
    out = {}
    for line in open(here):
        if line.strip() and not line.startswith("#"):
            r = line.split()
            out[r[0]] = [float(x) for x in r[1:]]
    return out


@pytest.mark.parametrize("case", ["sod", "strong_shock"])
def test_isolated_exact_shock_is_upwinded_exactly(ref, case):
    rL, uL, pL, rR, uR, pR, gamma, ps, us, rsl, rsr = golden_star()[case]
    # right-going shock between the right star state and the right state; speed from mass conservation
    S = (rsr * us - rR * uR) / (rsr - rR)
    for shift, upstream in ((0.0, "L"), (-(S + 0.3), "R")):      # second frame: the shock moves to the left
        WL = [rsr, us + shift, 0.2, -0.1, ps]
        WR = [rR, uR + shift, 0.2, -0.1, pR]
        f, path = ref.riemann_roe(gamma, WL, WR)
        want = eq11(WL, gamma) if upstream == "L" else eq11(WR, gamma)
        assert path in ("roe", "F_L", "F_R")
        assert np.allclose(f, want, rtol=0, atol=1e-12 * np.max(np.abs(want)))


def test_supersonic_states_return_the_upstream_flux(ref):
    WL, WR = [1.0, 3.0, 0.1, 0.0, 1.0], [0.9, 2.8, 0.0, 0.1, 0.8]
    f, path = ref.riemann_roe(G, WL, WR)
    assert path == "F_L" and np.array_equal(f, ref.riemann_roe(G, WL, WL)[0])
    WL2, WR2 = [c * s for c, s in zip(WR, (1, -1, 1, 1, 1))], [c * s for c, s in zip(WL, (1, -1, 1, 1, 1))]
    f2, path2 = ref.riemann_roe(G, WL2, WR2)
    assert path2 == "F_R" and np.allclose(f2, eq11(WR2))


def test_mirror_symmetry(ref):
    rng = np.random.default_rng(5)
    for _ in range(200):
        WL = [rng.uniform(0.2, 3), rng.normal(0, 0.8), rng.normal(), rng.normal(), rng.uniform(0.2, 3)]
        WR = [rng.uniform(0.2, 3), rng.normal(0, 0.8), rng.normal(), rng.normal(), rng.uniform(0.2, 3)]
        f, p1 = ref.riemann_roe(G, WL, WR)
        m = lambda W: [W[0], -W[1], W[2], W[3], W[4]]
        fm, p2 = ref.riemann_roe(G, m(WR), m(WL))
        scale = np.max(np.abs(f)) + 1.0
        assert np.allclose(fm * np.array([-1, 1, -1, -1, -1]), f, rtol=0, atol=1e-13 * scale)


def test_symmetric_rarefaction_falls_back_to_hlle_closed_form(ref):
    rho, u, p = 1.0, 2.0, 0.4                                  # Einfeldt 123 (reading S14)
    f, path = ref.riemann_roe(G, [rho, -u, 0, 0, p], [rho, u, 0, 0, p])
    assert path == "hlle"
    a = math.sqrt(G * p / rho)
    assert np.allclose(f, [0.0, p - rho * u * a, 0.0, 0.0, 0.0], rtol=0, atol=1e-15)


def l1_density_error_sod(ref, n, solver):
    w = wl.sod(n)
    Gd = ref.RefGrid(*w.shape, 3, w.gamma, w.bc)
    Gd.set_solver(solver)
    run(Gd, w)
    rho = Gd.get_state()[0, 0, 0]
    # exact solution sampled at cell centres through the oracle's exact solver in shifted frames
    x = (np.arange(n) + 0.5) / n
    exact = np.empty(n)
    for i, xi in enumerate((x - 0.5) / 0.2):
        _, d = ref.riemann_exact(w.gamma, [1.0, -xi, 0, 0, 1.0], [0.125, -xi, 0, 0, 0.1])
        exact[i] = d["rho"]
    return float(np.mean(np.abs(rho - exact)))


def test_sod_with_roe_converges_to_the_exact_solution(ref):
    e = [l1_density_error_sod(ref, n, 1) for n in (64, 128, 256)]
    assert e[0] > e[1] > e[2] and e[2] < 0.004
    assert abs(e[1] - l1_density_error_sod(ref, 128, 0)) < 0.3 * e[1]     # same scheme, two consistent solvers


def test_123_problem_stays_positive_with_roe_and_hlle(ref):
    w = wl.riemann_tube(128, (1.0, -2.0, 0.4), (1.0, 2.0, 0.4), gamma=1.4, t_end=0.15)
    Gd = ref.RefGrid(*w.shape, 3, w.gamma, w.bc)
    Gd.set_solver(1)
    run(Gd, w)
    u = Gd.get_state()
    assert np.all(np.isfinite(u)) and np.all(u[0] > 0)
    p = (w.gamma - 1) * (u[4] - 0.5 * u[1] ** 2 / u[0])
    assert np.all(p > 0)
    assert np.allclose(u[0, 0, 0], u[0, 0, 0, ::-1], rtol=1e-12)          # mirror-symmetric problem


def test_second_order_convergence_with_roe(ref):
    errs = []
    for n in (32, 64, 128):
        w = wl.linear_wave(n)
        Gd = ref.RefGrid(*w.shape, 3, w.gamma, w.bc)
        Gd.set_solver(1)
        run(Gd, w)
        errs.append(float(np.mean(np.abs(Gd.get_state() - w.u))))
    order = math.log(errs[0] / errs[2]) / math.log(4.0)
    assert order > 1.8, (errs, order)
