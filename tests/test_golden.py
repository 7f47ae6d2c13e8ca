"""Fixtures under tests/golden/ against the oracle (`-m "not gpu"`).

riemann_star_states.txt — written by tests/golden/make_star_states.py (40-digit mpmath solve of the
jump conditions; calls neither oracle/ nor the CUDA path).  paper_printed_values.txt — numbers the
paper prints for its worked examples, each with its citation.
"""
import os

import numpy as np

from paper_1410_4194_b200 import workloads as wl
from paper_1410_4194_b200.driver import run

HERE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def rows(name):
    with open(os.path.join(HERE, name)) as f:
        return [l.split() for l in f if l.strip() and not l.startswith("#")]


def test_star_states_match_the_40_digit_solution(ref):
    for r in rows("riemann_star_states.txt"):
        name, (rL, uL, pL, rR, uR, pR, gamma, p, u, rsl, rsr) = r[0], [float(x) for x in r[1:12]]
        _, d = ref.riemann_exact(gamma, [rL, uL, 0.0, 0.0, pL], [rR, uR, 0.0, 0.0, pR])
        tol = 1e-10 if name == "einfeldt_123" else 1e-12      # 123: Newton climbs from the 1e-6 guess floor
        assert abs(d["pm"] - p) <= tol * p, name
        assert abs(d["um"] - u) <= tol * max(abs(u), 1.0), name


def test_paper_printed_wave_positions(ref):
    vals = {r[0]: (float(r[1]), float(r[2])) for r in rows("paper_printed_values.txt")}
    # Sod at t = 0.2 on BASELINE.json's 128 cells: locate contact and shock in the oracle's density profile
    w = wl.sod(128)
    G = ref.RefGrid(*w.shape, 3, w.gamma, w.bc)
    run(G, w)
    rho = G.get_state()[0, 0, 0]
    x = (np.arange(128) + 0.5) / 128
    star = {r[0]: [float(v) for v in r[8:12]] for r in rows("riemann_star_states.txt")}["sod"]
    rsl, rsr = star[2], star[3]
    contact = x[np.argmin(np.abs(rho - 0.5 * (rsl + rsr)) + 10.0 * (x < 0.55))]     # mid-value between the star densities
    shock = x[np.argmin(np.abs(rho - 0.5 * (rsr + 0.125)) + 10.0 * (x < 0.75))]
    v, tol = vals["sod_contact_x_t0.2"]
    assert abs(contact - v) <= tol + 1.0 / 128
    v, tol = vals["sod_shock_x_t0.2"]
    assert abs(shock - v) <= tol + 1.0 / 128


def test_paper_printed_ppmp_contact_and_noh_densities(ref):
    """P:L465 (two zones with PPMP, three to four with PPMC) and P:L561 (rho = 16 ahead of, 64 behind the Noh shock;
    2-D stand-in for the CPU suite: 4 and 16, the same closed form (1 + t/r)^(n-1) and 4^n)."""
    vals = {r[0]: (float(r[1]), float(r[2])) for r in rows("paper_printed_values.txt")}
    from tests.test_oracle_ppmp import contact_width
    wp, _ = contact_width(ref, 3)
    wc, _ = contact_width(ref, 0)
    assert abs(wp - vals["sod_contact_zones_ppmp"][0]) <= vals["sod_contact_zones_ppmp"][1]
    assert abs(wc - vals["sod_contact_zones_ppmc"][0]) <= vals["sod_contact_zones_ppmc"][1]
    # the 3-D numbers are (1 + 3)^2 and 4^3: check that the printed values ARE the closed form the tests gate against
    assert vals["noh_preshock_density_3d"][0] == (1.0 + 3.0) ** 2 and vals["noh_postshock_density_3d"][0] == 4.0 ** 3
