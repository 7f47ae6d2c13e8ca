"""Pins of the oracle's analytic (custom) boundary and of the Noh strong-shock test (section 4.3.1):

* the ghost cells of a face with code NOH hold rho0 (1 + t/r)^(n-1), unit velocity toward the origin and
  E = p0/(gamma - 1) + rho/2 at their own centres (closed form, numpy), in 1, 2 and 3 active dimensions, mixed with
  reflective inner faces, edges and corners included;
* the test itself, run as the paper runs it (octant, reflecting inner faces, analytic outer faces, Roe solver with
  the H correction, four ghost layers): the reflected shock sits at r = t/3, the gas behind it has rho = 4^n
  (16 in 2-D, 64 in 3-D) and the gas ahead of it follows rho0 (1 + t/r)^(n-1).
"""
import numpy as np
import pytest

from paper_1410_4194_b200 import workloads as wl
from paper_1410_4194_b200.driver import run

GAMMA = 5.0 / 3.0


@pytest.mark.parametrize("shape", [(12, 1, 1), (10, 8, 1), (7, 6, 5), (1, 9, 8)])
def test_noh_ghost_cells_hold_the_analytic_solution(ref, shape):
    w = wl.noh(shape=shape)
    g = 4
    G = ref.RefGrid(*shape, g, w.gamma, w.bc)
    G.set_noh(1.0, 1e-6)
    G.set_state(w.u)
    G.set_time(0.37)
    G.fill_ghosts()
    up = G.get_padded()
    nx, ny, nz = shape
    dx = 1.0 / nx
    act = [n > 1 for n in (nx, ny, nz)]
    nd = sum(act)
    coords = [((np.arange(n + 2 * g) - g + 0.5) * dx if a else np.zeros(1)) for n, a in zip((nx, ny, nz), act)]
    X, Y, Z = np.meshgrid(*coords, indexing="ij")
    X, Y, Z = (a.transpose(2, 1, 0) for a in (X, Y, Z))
    outer = np.zeros(X.shape, bool)
    for a, n, c in zip(act, (nx, ny, nz), (X, Y, Z)):
        if a:
            outer |= c > n * dx
    r = np.sqrt(X ** 2 + Y ** 2 + Z ** 2)
    rho = (1.0 + 0.37 / r) ** (nd - 1)
    assert outer.any()
    assert np.allclose(up[0][outer], rho[outer], rtol=1e-14)
    for f, c in ((1, X), (2, Y), (3, Z)):
        assert np.allclose(up[f][outer], (rho * (-c / r))[outer], rtol=1e-14, atol=1e-15)
    assert np.allclose(up[4][outer], (1e-6 / (GAMMA - 1) + 0.5 * rho)[outer], rtol=1e-14)
    # inner ghosts (not beyond any analytic face): mirror images with the normal momentum negated
    if act[0]:
        assert np.array_equal(up[0][:, :, g - 1], up[0][:, :, g]) and np.array_equal(up[1][:, :, g - 1], -up[1][:, :, g])


def run_noh(ref, n, dims, t_end):
    w = wl.noh(n=n, dims=dims, t_end=t_end)
    G = ref.RefGrid(*w.shape, 4, w.gamma, w.bc)
    G.set_solver(1)
    G.set_hcorrection(True)
    G.set_noh(1.0, 1e-6)
    run(G, w)
    return G.get_state(), w


def radius(shape):
    nx = shape[0]
    c = [((np.arange(n) + 0.5) / nx if n > 1 else np.zeros(1)) for n in shape]
    X, Y, Z = np.meshgrid(*c, indexing="ij")
    return np.sqrt(X ** 2 + Y ** 2 + Z ** 2).transpose(2, 1, 0)


def test_noh_2d_shock_position_and_densities(ref):
    t = 1.2
    u, w = run_noh(ref, 64, 2, t)
    r, rho = radius(w.shape), u[0]
    post = (r > 0.12) & (r < 0.30)                       # behind the shock at t/3 = 0.4, away from the wall-heated origin
    assert abs(rho[post].mean() - 16.0) < 0.5 and rho[post].min() > 14.5 and rho[post].max() < 17.5
    pre = (r > 0.5) & (r < 0.95)
    assert np.max(np.abs(rho[pre] / (1.0 + t / r[pre]) - 1.0)) < 0.03
    # shock radius: where the azimuthally averaged density falls through the mean of 16 and the pre-shock value 4
    bins = np.linspace(0.2, 0.6, 41)
    prof = np.array([rho[(r >= a) & (r < b)].mean() for a, b in zip(bins[:-1], bins[1:])])
    rc = 0.5 * (bins[1:] + bins[:-1])
    r_shock = rc[np.max(np.nonzero(prof > 10.0)[0])]
    assert abs(r_shock - t / 3.0) < 2.5 / 64, r_shock
    # symmetric about the diagonal, to rounding
    assert np.allclose(rho[0], rho[0].T, rtol=1e-6)


def test_noh_3d_coarse(ref):
    t = 0.9
    u, w = run_noh(ref, 24, 3, t)
    r, rho = radius(w.shape), u[0]
    post = (r > 0.12) & (r < 0.22)
    assert 50.0 < rho[post].mean() < 66.0                # 64 analytically; 24^3 is coarse (shock 7 cells from the origin)
    pre = (r > 0.45) & (r < 0.9)
    assert np.max(np.abs(rho[pre] / (1.0 + t / r[pre]) ** 2 - 1.0)) < 0.05
    assert np.all(np.isfinite(u)) and rho.min() > 0
