"""Writes tests/golden/riemann_star_states.txt: star states of three shock-tube problems the paper runs
(P:L447-451 Sod with BASELINE.json's rho_R = 0.125; P:L467 strong shock; P:L473 Einfeldt 123), solved at
40 digits from the physics — the Rankine-Hugoniot jump conditions in conservation form (Eq. 11),
isentropy and the Riemann invariant across a rarefaction — with mpmath.  Calls neither oracle/ nor the
CUDA path.  Run from the repo root:  python tests/golden/make_star_states.py
"""
import os

import mpmath as mp

mp.mp.dps = 40
G = mp.mpf("1.4")


def f_side(p, rho, pk):
    """Velocity change across the wave connecting state k to pressure p (exact gas dynamics)."""
    a = mp.sqrt(G * pk / rho)
    if p <= pk:   # isentropic rarefaction: Riemann invariant u +- 2a/(gamma-1), p/rho^gamma constant
        return 2 * a / (G - 1) * ((p / pk) ** ((G - 1) / (2 * G)) - 1)
    # shock: from the three jump conditions, mass flux^2 = (p - pk) / (1/rho - 1/rho*)
    rs = rho * ((G + 1) * p + (G - 1) * pk) / ((G - 1) * p + (G + 1) * pk)
    return mp.sqrt((p - pk) * (1 / rho - 1 / rs))


def star(left, right):
    rL, uL, pL = [mp.mpf(x) for x in left]
    rR, uR, pR = [mp.mpf(x) for x in right]
    p = mp.findroot(lambda p: f_side(p, rL, pL) + f_side(p, rR, pR) + (uR - uL), (mp.mpf("1e-8"), max(pL, pR) * 50),
                    solver="anderson", tol=mp.mpf("1e-35"), maxsteps=400)
    u = (uL + uR + f_side(p, rR, pR) - f_side(p, rL, pL)) / 2

    def dens(rho, pk):
        if p <= pk:
            return rho * (p / pk) ** (1 / G)
        return rho * ((G + 1) * p + (G - 1) * pk) / ((G - 1) * p + (G + 1) * pk)
    return p, u, dens(rL, pL), dens(rR, pR)


CASES = [("sod", ("1", "0", "1"), ("0.125", "0", "0.1"), "P:L447-451, BASELINE.json config 1 (reading S12)"),
         ("strong_shock", ("10", "0", "100"), ("1", "0", "1"), "P:L467-471"),
         ("einfeldt_123", ("1", "-2", "0.4"), ("1", "2", "0.4"), "P:L473-479 (reading S14)")]

if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "riemann_star_states.txt")
    with open(out, "w") as f:
        f.write("# name rhoL uL pL rhoR uR pR gamma | p* u* rho*L rho*R   (40-digit solve of the jump conditions; make_star_states.py)\n")
        for name, L, R, cite in CASES:
            p, u, rl, rr = star(L, R)
            f.write(f"# {cite}\n")
            f.write(" ".join([name, *L, *R, "1.4"] + [mp.nstr(x, 20) for x in (p, u, rl, rr)]) + "\n")
    print(open(out).read())
