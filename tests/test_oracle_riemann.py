"""Pins of the oracle's exact Riemann solver (oracle/cholla_ref.cpp: riemann_exact)
against what the physics fixes — NOT against a retyped copy of its own formulas:

* star states from the Rankine-Hugoniot jump conditions in conservation form (Eq. 11)
  and the isentropic simple-wave invariants, solved at 30 digits with mpmath;
* the two-rarefaction closed form (123 problem) and the two-shock quadratic;
* published 5-digit star values for the Sod problem (Toro 2009, Table 4.3, test 1);
* invariants of the sampled state in each of the ten regions, continuity of the
  flux across every region boundary, mirror symmetry, identical-state flux = Eq. 11.
"""
import math

import mpmath as mp
import numpy as np
import pytest

mp.mp.dps = 30

SOD = ((1.0, 0.0, 1.0), (0.125, 0.0, 0.1), 1.4)
STRONG = ((10.0, 0.0, 100.0), (1.0, 0.0, 1.0), 1.4)
E123 = ((1.0, -2.0, 0.4), (1.0, 2.0, 0.4), 1.4)              # P:L473-479, reading S14


def W(s, vt=(0.0, 0.0)):
    return [s[0], s[1], vt[0], vt[1], s[2]]


def star_from_physics(left, right, gamma, guess):
    """Left rarefaction + right shock: 5 equations (3 RH in conservation form, entropy, Riemann invariant)."""
    rL, uL, pL = [mp.mpf(x) for x in left]
    rR, uR, pR = [mp.mpf(x) for x in right]
    g = mp.mpf(gamma)
    ER = pR / (g - 1) + rR * uR ** 2 / 2
    aL = mp.sqrt(g * pL / rL)

    def eqs(p, u, rsl, rsr, S):
        Es = p / (g - 1) + rsr * u ** 2 / 2
        return [rsr * (u - S) - rR * (uR - S),
                rsr * u * (u - S) + p - (rR * uR * (uR - S) + pR),
                Es * (u - S) + p * u - (ER * (uR - S) + pR * uR),
                p / rsl ** g - pL / rL ** g,
                u + 2 * mp.sqrt(g * p / rsl) / (g - 1) - (uL + 2 * aL / (g - 1))]
    sol = mp.findroot(eqs, guess, tol=1e-25, maxsteps=100)
    return [float(x) for x in sol]


def test_sod_star_state_from_jump_conditions(ref):
    left, right, gamma = SOD
    p, u, rsl, rsr, S = star_from_physics(left, right, gamma, (0.30313, 0.92745, 0.42632, 0.26557, 1.7522))
    # published 5-digit values (Toro 2009, Table 4.3 test 1)
    assert abs(p - 0.30313) < 1e-5 and abs(u - 0.92745) < 1e-5
    assert abs(rsl - 0.42632) < 1e-5 and abs(rsr - 0.26557) < 1e-5
    _, d = ref.riemann_exact(gamma, W(left), W(right))
    assert abs(d["pm"] - p) <= 1e-12 * p
    assert abs(d["um"] - u) <= 1e-12 * u
    # x/t = 0 lies between the rarefaction tail and the contact: left star density
    assert d["region"] == 1 and abs(d["rho"] - rsl) <= 1e-12 * rsl
    # wave positions the paper quotes at t = 0.2: contact ~0.7, shock ~0.85
    assert abs(0.5 + 0.2 * u - 0.7) < 0.02 and abs(0.5 + 0.2 * S - 0.85) < 0.005


def test_strong_shock_star_state(ref):
    left, right, gamma = STRONG
    p, u, rsl, rsr, S = star_from_physics(left, right, gamma, (19.9, 3.85, 3.16, 4.65, 4.9))
    _, d = ref.riemann_exact(gamma, W(left), W(right))
    assert abs(d["pm"] - p) <= 1e-12 * p and abs(d["um"] - u) <= 1e-12 * u
    # contact position at t=0.07 — the paper reads "x = 0.75" off its figure
    assert abs(0.5 + 0.07 * u - 0.75) < 0.03
    # sampled right of the contact in a frame moving between contact and shock: post-shock density
    xi = 0.5 * (u + S)
    WL, WR = W(left), W(right)
    WL[1] -= xi; WR[1] -= xi
    _, d2 = ref.riemann_exact(gamma, WL, WR)
    assert d2["region"] == 9 and abs(d2["rho"] - rsr) <= 1e-12 * rsr


def test_123_two_rarefaction_closed_form(ref):
    left, right, gamma = E123
    z = (gamma - 1) / (2 * gamma)
    aL = math.sqrt(gamma * left[2] / left[0]); aR = math.sqrt(gamma * right[2] / right[0])
    du = right[1] - left[1]
    p = ((aL + aR - 0.5 * (gamma - 1) * du) / (aL / left[2] ** z + aR / right[2] ** z)) ** (1 / z)
    _, d = ref.riemann_exact(gamma, W(left), W(right))
    assert abs(d["pm"] - p) <= 1e-10 * p            # Newton started from the 1e-6 floor
    assert d["um"] == 0.0                           # symmetric form of B9 -> exactly zero
    assert abs(d["rho"] - left[0] * (p / left[2]) ** (1 / gamma)) <= 1e-10 * d["rho"]
    assert d["iters"] < 20


@pytest.mark.parametrize("u0", [0.1, 1.0, 10.0])
def test_symmetric_collision_two_shock_quadratic(ref, u0):
    gamma, rho, pk = 5.0 / 3.0, 1.3, 0.7
    # (p-pk)^2 A = u0^2 (p+B) with A=2/((g+1)rho), B=(g-1)/(g+1) pk  [two equal shocks, u*=0]
    A = 2 / ((gamma + 1) * rho); B = (gamma - 1) / (gamma + 1) * pk
    # A p^2 - (2 A pk + u0^2) p + (A pk^2 - u0^2 B) = 0, larger root
    b = -(2 * A * pk + u0 * u0); c = A * pk * pk - u0 * u0 * B
    p = (-b + math.sqrt(b * b - 4 * A * c)) / (2 * A)
    f, d = ref.riemann_exact(gamma, [rho, u0, 0.2, -0.3, pk], [rho, -u0, 0.2, -0.3, pk])
    assert abs(d["pm"] - p) <= 1e-12 * p and d["um"] == 0.0
    assert f[0] == 0.0 and abs(f[1] - p) <= 1e-12 * p and f[4] == 0.0


def euler_flux(gamma, w):
    rho, u, v, ww, p = w
    E = p / (gamma - 1) + 0.5 * rho * (u * u + v * v + ww * ww)
    return np.array([rho * u, rho * u * u + p, rho * u * v, rho * u * ww, (E + p) * u])


def test_identical_states_give_eq11_flux(ref):
    rng = np.random.default_rng(7)
    for _ in range(200):
        w = [rng.uniform(0.1, 5), rng.normal() * 2, rng.normal(), rng.normal(), rng.uniform(0.1, 5)]
        f, d = ref.riemann_exact(1.4, w, w)
        F = euler_flux(1.4, w)
        assert np.all(np.abs(f - F) <= 4e-15 * np.maximum(np.abs(F), np.abs(F).max()))
        assert abs(d["pm"] - w[4]) <= 1e-14 * w[4]


def random_states(rng, n, gamma):
    for _ in range(n):
        yield ([rng.uniform(0.05, 4), rng.normal() * 1.5, rng.normal(), rng.normal(), rng.uniform(0.05, 4)],
               [rng.uniform(0.05, 4), rng.normal() * 1.5, rng.normal(), rng.normal(), rng.uniform(0.05, 4)])


@pytest.mark.parametrize("gamma", [1.4, 5.0 / 3.0])
def test_star_state_satisfies_wave_relations(ref, gamma):
    """For random data: each side's star state obeys RH (shock) or the isentropic invariants
    (rarefaction) between the data state and (pm, um) — checked in conservation form."""
    rng = np.random.default_rng(11)
    for WL, WR in random_states(rng, 300, gamma):
        if 2 * (math.sqrt(gamma * WL[4] / WL[0]) + math.sqrt(gamma * WR[4] / WR[0])) / (gamma - 1) <= WR[1] - WL[1]:
            continue  # vacuum generation (reading S5): not handled
        _, d = ref.riemann_exact(gamma, WL, WR)
        pm, um = d["pm"], d["um"]
        for Wk, sign in ((WL, -1.0), (WR, +1.0)):
            rk, uk, pk = Wk[0], Wk[1], Wk[4]
            ak = math.sqrt(gamma * pk / rk)
            if pm > pk:   # shock: mass flux j from momentum RH, then energy RH must close
                gm = (gamma - 1) / (gamma + 1)
                rs = rk * (pm / pk + gm) / (gm * pm / pk + 1)       # density from the Hugoniot
                S = (rs * um - rk * uk) / (rs - rk)                 # mass RH
                mom = rs * um * (um - S) + pm - (rk * uk * (uk - S) + pk)
                Es = pm / (gamma - 1) + 0.5 * rs * um * um; Ek = pk / (gamma - 1) + 0.5 * rk * uk * uk
                en = Es * (um - S) + pm * um - (Ek * (uk - S) + pk * uk)
                scale = rk * ak * ak + pm
                assert abs(mom) <= 1e-9 * scale, (WL, WR, mom)
                assert abs(en) <= 1e-9 * scale * (abs(uk) + ak + abs(S)), (WL, WR, en)
            else:         # rarefaction: entropy and the invariant u + 2a/(g-1) (left) / u - 2a/(g-1) (right)
                rs = rk * (pm / pk) ** (1 / gamma)
                as_ = math.sqrt(gamma * pm / rs)
                inv = (um - sign * 2 * as_ / (gamma - 1)) - (uk - sign * 2 * ak / (gamma - 1))
                assert abs(inv) <= 1e-9 * (ak + abs(uk)), (WL, WR, inv)


def test_sampled_state_invariants_in_each_region(ref):
    """Scan the frame velocity so x/t=0 visits all ten regions of one Riemann fan; check what each
    region must satisfy: data states verbatim; fans: u -/+ a = x/t, entropy, Riemann invariant."""
    gamma = 1.4
    seen = set()
    for base in (W(SOD[0]), W(SOD[1])), (W(SOD[1]), W(SOD[0])), (W(E123[0]), W(E123[1])), \
                ([1.0, 2.0, 0, 0, 1.0], [1.0, -2.0, 0, 0, 1.0]):
        for xi in np.linspace(-4.0, 4.0, 801):
            WL = list(base[0]); WR = list(base[1])
            WL[1] -= xi; WR[1] -= xi
            _, d = ref.riemann_exact(gamma, WL, WR)
            r = d["region"]; seen.add(r)
            Wk = WL if r < 5 else WR
            sign = -1.0 if r < 5 else 1.0
            ak = math.sqrt(gamma * Wk[4] / Wk[0])
            if r in (0, 3, 5, 8):
                assert (d["rho"], d["u"], d["p"]) == (Wk[0], Wk[1], Wk[4])
            elif r in (2, 7):
                a = math.sqrt(gamma * d["p"] / d["rho"])
                assert abs(d["u"] + sign * a) <= 1e-13 * ak                       # characteristic through x/t=0
                assert abs(d["p"] / d["rho"] ** gamma - Wk[4] / Wk[0] ** gamma) <= 1e-12 * Wk[4] / Wk[0] ** gamma
                inv = (d["u"] - sign * 2 * a / (gamma - 1)) - (Wk[1] - sign * 2 * ak / (gamma - 1))
                assert abs(inv) <= 1e-12 * (ak + abs(Wk[1]))
            else:
                assert d["u"] == d["um"] and d["p"] == d["pm"]
                if r in (1, 6):
                    assert abs(d["p"] / d["rho"] ** gamma - Wk[4] / Wk[0] ** gamma) <= 1e-12 * Wk[4] / Wk[0] ** gamma
    assert seen == set(range(10)), seen


def test_flux_is_continuous_across_region_boundaries(ref):
    """The Godunov flux in the lab frame, F(xi) - xi*U(xi), is a continuous function of the frame
    velocity xi (RH across shocks/contact, smoothness across fan edges).  A wrong branch formula
    (e.g. the printed B18, reading G4) shows up as a jump."""
    gamma = 1.4
    for base in (W(SOD[0], (0.3, -0.2)), W(SOD[1], (-0.1, 0.4))), (W(SOD[1], (0.3, -0.2)), W(SOD[0], (-0.1, 0.4))), \
                (W(E123[0]), W(E123[1])), ([1.0, 2.0, 0.1, 0, 1.0], [1.5, -2.0, -0.2, 0, 0.8]):
        xis = np.linspace(-4.0, 4.0, 16001)
        prev = None
        for xi in xis:
            WL = list(base[0]); WR = list(base[1])
            WL[1] -= xi; WR[1] -= xi
            f, d = ref.riemann_exact(gamma, WL, WR)
            if prev is not None:
                # in the moving frame the flux at the frame origin changes by O(dxi) only
                assert np.all(np.abs(f - prev) <= 40 * (xis[1] - xis[0]) * (1 + np.abs(f))), (xi, f, prev, d)
            prev = f


def test_mirror_symmetry_is_bitwise(ref):
    rng = np.random.default_rng(3)
    for WL, WR in random_states(rng, 300, 1.4):
        f1, d1 = ref.riemann_exact(1.4, WL, WR)
        ML = [WR[0], -WR[1], WR[2], WR[3], WR[4]]
        MR = [WL[0], -WL[1], WL[2], WL[3], WL[4]]
        f2, d2 = ref.riemann_exact(1.4, ML, MR)
        if d1["um"] == 0.0:
            continue
        assert d1["pm"] == d2["pm"] and d1["um"] == -d2["um"]
        assert np.array_equal(f1 * np.array([-1, 1, -1, -1, -1]), f2)


def test_galilean_transverse_passive(ref):
    """Transverse velocities are passively advected: they come from the upwind side."""
    f, d = ref.riemann_exact(1.4, W(SOD[0], (3.0, -7.0)), W(SOD[1], (11.0, 13.0)))
    assert d["um"] > 0 and f[2] == f[0] * 3.0 and f[3] == f[0] * -7.0
    f, d = ref.riemann_exact(1.4, W(SOD[1], (3.0, -7.0)), W(SOD[0], (11.0, 13.0)))
    assert d["um"] < 0 and f[2] == f[0] * 11.0 and f[3] == f[0] * 13.0


def test_pressure_floor_and_guess_floor(ref):
    # negative input pressure is floored to 1e-20, the solver still returns finite fluxes
    f, d = ref.riemann_exact(1.4, [1.0, 0.0, 0, 0, -5.0], [1.0, 0.0, 0, 0, -5.0])
    assert np.all(np.isfinite(f)) and d["pm"] > 0
