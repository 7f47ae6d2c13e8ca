"""Pins of the oracle's PLMC and PCM reconstructions (oracle/cholla_ref.cpp: plmc_cell, pcm_cell; A.2
P:L719-793, Eq. 25-26) against what the mathematics fixes:

* PLMC on linear data reproduces it; faces are bounded by the neighbouring cell averages (A13);
* the traced states A15-A19 equal, wave by wave, the spectral projection (numpy eigen-decomposition of the
  primitive Jacobian, not the paper's closed forms) of the averages of the LINEAR profile over each
  characteristic's domain of dependence — this is what catches the lost last row of A19 (reading G10);
* dt = 0 leaves the faces untouched; a pure entropy wave is advected upwind; mirror symmetry;
* scheme level: second-order convergence of a sound wave with PLMC, first order with PCM, uniform
  states and conservation with both, Sod converging with both.
"""
import math

import numpy as np
import pytest

from paper_1410_4194_b200 import workloads as wl
from paper_1410_4194_b200.driver import run
from tests.test_oracle_ppmc import GAMMA, numeric_projectors, stencil

PLMC, PCM = 1, 2


def test_plmc_linear_data_is_exact_and_bounded(ref):
    rng = np.random.default_rng(3)
    for _ in range(100):
        base = np.array([rng.uniform(0.5, 2), rng.normal(), rng.normal(), rng.normal(), rng.uniform(0.5, 2)])
        b = rng.normal(size=5) * 0.01
        w = stencil(lambda s: base + b * s)
        WL, WR, WLs, WRs = ref.plmc_cell(GAMMA, 0.0, w)
        assert np.allclose(WL, w[2] - 0.5 * b, atol=1e-15) and np.allclose(WR, w[2] + 0.5 * b, atol=1e-15)
        assert np.array_equal(WLs, WL) and np.array_equal(WRs, WR)          # dt = 0: no evolution
    for _ in range(300):                                                    # rough data: A13 bounds
        w = rng.uniform(0.2, 3.0, size=(5, 5))
        WL, WR, _, _ = ref.plmc_cell(GAMMA, 0.0, w)
        for c in range(5):
            assert min(w[1, c], w[2, c]) - 1e-15 <= WL[c] <= max(w[1, c], w[2, c]) + 1e-15
            assert min(w[3, c], w[2, c]) - 1e-15 <= WR[c] <= max(w[3, c], w[2, c]) + 1e-15


@pytest.mark.parametrize("mach", [-2.5, -0.6, 0.0, 0.4, 3.0])
def test_plmc_tracing_equals_projected_linear_averages(ref, mach):
    rng = np.random.default_rng(int(10 * mach) + 200)
    for _ in range(40):
        base = np.array([rng.uniform(0.5, 2), 0.0, rng.normal(), rng.normal(), rng.uniform(0.5, 2)])
        a0 = np.sqrt(GAMMA * base[4] / base[0])
        base[1] = mach * a0
        slope = rng.normal(size=5) * 0.02
        w = stencil(lambda s: base + slope * s + 0.003 * rng.normal(size=5) * s * s)
        dtdx = rng.uniform(0.05, 0.45) / (abs(base[1]) + a0)
        WL, WR, WLs, WRs = ref.plmc_cell(GAMMA, dtdx, w)
        wi = w[2]
        P, (lm, l0, lp) = numeric_projectors(wi, GAMMA)
        lam = {"m": lm, "0": l0, "p": lp}
        lin = lambda x0, x1: WL + 0.5 * (x0 + x1) * (WR - WL)            # mean of the linear profile over [x0, x1]
        avgL = {n: lin(0.0, max(-lam[n], 0.0) * dtdx) for n in lam}
        wantL = avgL["m"].copy()
        for n in ("0", "p"):
            if lam[n] < 0:
                wantL += P[n] @ (avgL[n] - avgL["m"])
        avgR = {n: lin(1.0 - max(lam[n], 0.0) * dtdx, 1.0) for n in lam}
        wantR = avgR["p"].copy()
        for n in ("m", "0"):
            if lam[n] > 0:
                wantR += P[n] @ (avgR[n] - avgR["p"])
        assert np.allclose(WLs, wantL, rtol=0, atol=2e-14), (WLs - wantL)
        assert np.allclose(WRs, wantR, rtol=0, atol=2e-14), (WRs - wantR)


def test_plmc_mirror_symmetry(ref):
    rng = np.random.default_rng(9)
    flip = np.array([1, -1, 1, 1, 1.0])
    for _ in range(100):
        w = rng.uniform(0.3, 2.0, size=(5, 5)); w[:, 1] = rng.normal(size=5) * 0.5
        WL, WR, WLs, WRs = ref.plmc_cell(GAMMA, 0.3, w)
        ML, MR, MLs, MRs = ref.plmc_cell(GAMMA, 0.3, w[::-1] * flip)
        assert np.allclose(MR * flip, WL, atol=1e-14) and np.allclose(ML * flip, WR, atol=1e-14)
        assert np.allclose(MRs * flip, WLs, atol=1e-14) and np.allclose(MLs * flip, WRs, atol=1e-14)


def wave_error(ref, n, recon):
    w = wl.linear_wave(n)
    G = ref.RefGrid(*w.shape, 3, w.gamma, w.bc)
    G.set_reconstruction(recon)
    run(G, w)
    return float(np.mean(np.abs(G.get_state() - w.u)))


def test_convergence_orders(ref):
    e = [wave_error(ref, n, PLMC) for n in (32, 64, 128)]
    assert math.log(e[0] / e[2]) / math.log(4.0) > 1.8, e             # second order
    e = [wave_error(ref, n, PCM) for n in (32, 64, 128)]
    order = math.log(e[0] / e[2]) / math.log(4.0)
    assert 0.7 < order < 1.3, (e, order)                               # first order


@pytest.mark.parametrize("recon", [PLMC, PCM])
def test_uniform_state_conservation_and_sod(ref, recon):
    u = wl.conserved(0.7, 0.3, -0.45, 0.21, 1.9, 1.4).reshape(5, 1, 1, 1) * np.ones((5, 6, 7, 8))
    G = ref.RefGrid(8, 7, 6, 3, 1.4, (1,) * 6)
    G.set_reconstruction(recon)
    G.set_state(u)
    G.step(G.compute_dt(0.4))
    assert np.array_equal(G.get_state(), u)
    w = wl.sweep(shape=(16, 12, 10))
    G = ref.RefGrid(*w.shape, 3, w.gamma, w.bc)
    G.set_reconstruction(recon)
    G.set_state(w.u)
    for _ in range(3):
        G.step(G.compute_dt(w.cfl))
    u1 = G.get_state()
    for f in range(5):
        assert abs(math.fsum(u1[f].ravel()) - math.fsum(w.u[f].ravel())) <= 1e-13 * (math.fsum(np.abs(w.u[f]).ravel()) + w.u[0].size)
    # Sod: both converge towards the exact density profile, PCM more slowly than PLMC
    errs = []
    for n in (64, 256):
        ws = wl.sod(n)
        Gs = ref.RefGrid(*ws.shape, 3, ws.gamma, ws.bc)
        Gs.set_reconstruction(recon)
        run(Gs, ws)
        rho = Gs.get_state()[0, 0, 0]
        exact = np.empty(n)
        for i, xi in enumerate(((np.arange(n) + 0.5) / n - 0.5) / 0.2):
            _, d = ref.riemann_exact(ws.gamma, [1.0, -xi, 0, 0, 1.0], [0.125, -xi, 0, 0, 0.1])
            exact[i] = d["rho"]
        errs.append(float(np.mean(np.abs(rho - exact))))
    assert errs[1] < 0.6 * errs[0]
