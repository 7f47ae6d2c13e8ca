"""Pins of the oracle's H correction (oracle/cholla_ref.cpp; Appendix C):

* C3 on one interface: with eta^H above every |lambda| the Roe dissipation sum_k xi_k |lambda_k| r_k becomes
  eta^H (U_R - U_L) (the right eigenvectors resolve the jump), i.e. the flux is the local Lax-Friedrichs closed
  form F = (F_L + F_R)/2 - eta^H (U_R - U_L)/2; eta^H = 0 is the plain Roe flux, bitwise;
* a planar problem has eta = 0 on every transverse interface, so the 1-D run is reproduced bitwise inside a
  3-D box, and differs from the uncorrected run only through the interface's own eta;
* C2 gathers the transverse eta the same way for every direction: transposing / cyclically permuting the axes
  of the data permutes the result; WHICH cells it gathers from (reading G11: the two cells that share the interface)
  is pinned by test_c2_gathers_from_the_two_cells_that_share_the_interface;
* C1 itself is pinned quantitatively: with PCM the whole H-corrected step is written out by hand from the
  unit-level Roe solver — a 1-D two-state problem, a 2-D shear layer whose x-interfaces get their eta^H from a
  transverse jump only, and random 2-D states — and the same hand-written step with the 1/2 dropped, with u - a
  for u + a, or with eta taken from the states before the transverse correction misses the oracle by far more
  than the gate (each of those mutations of cholla_ref.cpp was checked to fail these tests);
* uniform states, conservation; the correction adds dissipation: a grid-aligned Mach-10 shock with odd-even
  noise ends with smaller transverse density variation than without it (the carbuncle's seed).
"""
import math

import numpy as np
import pytest

from paper_1410_4194_b200 import workloads as wl
from paper_1410_4194_b200.driver import run

G = 1.4
P, R, O = wl.PERIODIC, wl.REFLECTIVE, wl.OUTFLOW


def eq11_and_u(W, gamma=G):
    rho, u, v, w, p = W
    E = p / (gamma - 1) + 0.5 * rho * (u * u + v * v + w * w)
    return np.array([rho * u, rho * u * u + p, rho * u * v, rho * u * w, (E + p) * u]), np.array([rho, rho * u, rho * v, rho * w, E])


def test_c3_large_eta_is_local_lax_friedrichs_and_zero_eta_is_roe(ref):
    rng = np.random.default_rng(4)
    for _ in range(100):
        WL = [rng.uniform(0.5, 2), rng.normal(0, 0.3), rng.normal(), rng.normal(), rng.uniform(0.5, 2)]
        WR = [WL[0] * rng.uniform(0.8, 1.25), WL[1] + rng.normal(0, 0.1), rng.normal(), rng.normal(), WL[4] * rng.uniform(0.8, 1.25)]
        f0, path0 = ref.riemann_roe(G, WL, WR)
        fz, pathz = ref.riemann_roe_eta(G, WL, WR, 0.0)
        assert np.array_equal(f0, fz) and path0 == pathz
        if path0 != "roe":
            continue
        eta = 10.0
        f, path = ref.riemann_roe_eta(G, WL, WR, eta)
        FL, UL = eq11_and_u(WL); FR, UR = eq11_and_u(WR)
        assert path == "roe"
        assert np.allclose(f, 0.5 * (FL + FR) - 0.5 * eta * (UR - UL), rtol=0, atol=1e-12)


def grid(ref, w, hc, g=4):
    Gd = ref.RefGrid(*w.shape, g, w.gamma, w.bc)
    Gd.set_solver(1)
    Gd.set_hcorrection(hc)
    return Gd


def test_needs_four_ghosts_and_the_roe_solver(ref):
    w = wl.sod(32)
    Gd = ref.RefGrid(*w.shape, 3, w.gamma, w.bc)
    with pytest.raises(ValueError):
        Gd.set_hcorrection(True)
    Gd = ref.RefGrid(*w.shape, 4, w.gamma, w.bc)
    Gd.set_hcorrection(True)
    Gd.set_state(w.u)
    with pytest.raises(ValueError):
        Gd.step(1e-4)                       # exact solver selected


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_planar_problem_in_3d_equals_the_1d_run_bitwise(ref, axis):
    n, m = 32, 5
    one = wl.sod(n)
    G1 = grid(ref, one, True)
    dts = []
    run(G1, one, max_steps=10, record_dts=dts)
    u1 = G1.get_state()[:, 0, 0, :]
    shape = [m, m, m]; shape[axis] = n
    u3 = np.zeros((5, shape[2], shape[1], shape[0]))
    idx = [None, None, None]; idx[2 - axis] = slice(None)
    for f_src, f_dst in ((0, 0), (1, 1 + axis), (4, 4)):
        u3[f_dst] = one.u[:, 0, 0, :][f_src][tuple(idx)]
    bc = tuple(O if d == axis else P for d in range(3) for _ in range(2))
    G3 = ref.RefGrid(*shape, 4, one.gamma, bc)
    G3.set_solver(1); G3.set_hcorrection(True)
    G3.set_spacing(1.0 / n, 1.0 / n, 1.0 / n)
    G3.set_state(u3)
    for dt in dts:
        G3.step(dt)
    out = G3.get_state()
    for f_src, f_dst in ((0, 0), (1, 1 + axis), (4, 4)):
        assert np.array_equal(out[f_dst], u1[f_src][tuple(idx)] * np.ones_like(out[0]))
    # and the correction is not a no-op in 1-D: the interface's own eta enters
    G0 = grid(ref, one, False)
    run(G0, one, dts=dts)
    assert not np.array_equal(G0.get_state()[:, 0, 0, :], u1)


def test_transposition_symmetry_pins_the_per_direction_indexing_of_c2(ref):
    """Swapping the x and y axes of the data (and the velocity components) swaps the result: eta of the
    transverse interfaces is gathered the same way for x-, y- and z-interfaces.  (C1 as printed,
    |(u_R + a_R) - (u_L + a_L)|/2, is not mirror symmetric, so mirror images are NOT a property of this
    scheme; which cells C2 gathers from — reading G11 — is pinned by the test at the end of this file.)"""
    w = wl.rough_random(20, 20, 1, seed=8, decades=0.3, mach=0.8, bc=(P,) * 6)
    Gd = grid(ref, w, True)
    Gd.set_state(w.u)
    dt = 0.5 * Gd.compute_dt(w.cfl)
    Gd.step(dt)
    a = Gd.get_state()
    ut = np.ascontiguousarray(np.swapaxes(w.u, 2, 3))[[0, 2, 1, 3, 4]]       # transpose, swap rho*vx <-> rho*vy
    Gt = grid(ref, w, True)
    Gt.set_state(np.ascontiguousarray(ut))
    Gt.step(dt)
    b = np.swapaxes(Gt.get_state(), 2, 3)[[0, 2, 1, 3, 4]]
    assert np.allclose(a, b, rtol=0, atol=1e-13 * np.abs(a).max())
    G0 = grid(ref, w, False)
    G0.set_state(w.u); G0.step(dt)
    assert np.abs(G0.get_state() - a).max() > 1e-6                   # the correction acts on this problem
    # 3-D: cyclic permutation x -> y -> z -> x
    w3 = wl.rough_random(12, 12, 12, seed=9, decades=0.3, mach=0.8, bc=(P,) * 6)
    G3 = grid(ref, w3, True); G3.set_state(w3.u)
    dt = 0.5 * G3.compute_dt(w3.cfl)
    G3.step(dt)
    a = G3.get_state()
    # new[x', y', z'] = old[z', x', y'] with (vx', vy', vz') = (vz, vx, vy): array axes (f, z, y, x)
    up = np.ascontiguousarray(np.transpose(w3.u, (0, 2, 3, 1)))[[0, 3, 1, 2, 4]]
    Gp = grid(ref, w3, True); Gp.set_state(np.ascontiguousarray(up)); Gp.step(dt)
    b = np.transpose(Gp.get_state()[[0, 2, 3, 1, 4]], (0, 3, 1, 2))
    assert np.allclose(a, b, rtol=0, atol=1e-13 * np.abs(a).max())


def test_uniform_state_and_conservation(ref):
    u = wl.conserved(0.7, 0.3, -0.45, 0.21, 1.9, 1.4).reshape(5, 1, 1, 1) * np.ones((5, 6, 7, 8))
    Gd = ref.RefGrid(8, 7, 6, 4, 1.4, (P,) * 6)
    Gd.set_solver(1); Gd.set_hcorrection(True)
    Gd.set_state(u)
    Gd.step(Gd.compute_dt(0.4))
    assert np.array_equal(Gd.get_state(), u)
    w = wl.sweep(shape=(16, 12, 10))
    Gd = grid(ref, w, True)
    Gd.set_state(w.u)
    for _ in range(3):
        Gd.step(Gd.compute_dt(w.cfl))
    u1 = Gd.get_state()
    for f in range(5):
        assert abs(math.fsum(u1[f].ravel()) - math.fsum(w.u[f].ravel())) <= 1e-13 * (math.fsum(np.abs(w.u[f]).ravel()) + w.u[0].size)


def test_adds_crossflow_dissipation_at_a_grid_aligned_shock(ref):
    """Quirk-type odd-even test: a planar Mach-10 shock moving along x through a 2-D duct whose centre-line
    density carries an odd-even perturbation.  The transverse (y) variation of the post-shock density is the
    carbuncle's seed; with the H correction it must be smaller than without."""
    nx, ny, gamma, M = 96, 12, 1.4, 10.0
    rho0, p0 = 1.0, 1.0
    a0 = math.sqrt(gamma * p0 / rho0)
    r = (gamma + 1) * M * M / ((gamma - 1) * M * M + 2)              # Rankine-Hugoniot
    p1 = p0 * (2 * gamma * M * M - (gamma - 1)) / (gamma + 1)
    u1 = M * a0 * (1 - 1 / r)
    x = (np.arange(nx) + 0.5) / nx
    rho = np.where(x < 0.1, rho0 * r, rho0)[None, None, :] * np.ones((1, ny, nx))
    vx = np.where(x < 0.1, u1, 0.0)[None, None, :] * np.ones((1, ny, nx))
    p = np.where(x < 0.1, p1, p0)[None, None, :] * np.ones((1, ny, nx))
    rho[0, ny // 2, :] *= 1.0 + 1e-3 * (-1.0) ** np.arange(nx)       # odd-even noise on the centre line
    u = wl.conserved(rho, vx, 0.0, 0.0, p, gamma)
    res = {}
    for hc in (False, True):
        Gd = ref.RefGrid(nx, ny, 1, 4, gamma, (O, O, P, P, P, P))
        Gd.set_solver(1); Gd.set_hcorrection(hc)
        Gd.set_state(u)
        t = 0.0
        while t < 0.04:
            dt = Gd.compute_dt(0.4)
            Gd.step(dt); t += dt
        d = Gd.get_state()[0, 0]
        assert np.all(np.isfinite(d))
        behind = d[:, (x > 0.15) & (x < 0.1 + M * a0 * 0.04 - 0.05)]
        res[hc] = float(np.mean(np.std(behind, axis=0)))
    assert res[True] < res[False], res


def test_c2_gathers_from_the_two_cells_that_share_the_interface(ref):
    """Reading G11 made observable.  A density ramp along x gives every x-interface the same jump; one cell
    (i0, j0+1) gets a large transverse velocity, which makes eta large on the y-interface (i0, j0+1/2) only.
    With the correction, the x-interface (i0+1/2, j0) — cells i0 and i0+1 share it — gathers that eta, so cell
    (i0+1, j0) responds; the x-interface (i0+3/2, j0) gathers only from cells i0+1 and i0+2, whose eta do not
    depend on the perturbed cell, so cell (i0+2, j0) is untouched to the bit.  With the indices as printed (i-1
    and i+1) it would be the interface (i0+3/2, j0) that sees the large eta, and cell (i0+2, j0) would change."""
    nx, ny, i0, j0, gamma = 24, 12, 10, 5, 1.4
    rho = (1.0 + 0.02 * np.arange(nx))[None, None, :] * np.ones((1, ny, nx))
    vy = np.zeros((1, ny, nx))
    vy_p = vy.copy(); vy_p[0, j0 + 1, i0] = 2.0
    base = wl.conserved(rho, 0.3, vy, 0.0, 1.0, gamma)
    pert = wl.conserved(rho, 0.3, vy_p, 0.0, 1.0, gamma)

    def change(dt, hc):
        out = []
        for u in (base, pert):
            Gd = ref.RefGrid(nx, ny, 1, 4, gamma, (P,) * 6)
            Gd.set_solver(1); Gd.set_hcorrection(hc)
            Gd.set_state(u)
            Gd.step(dt)
            out.append(Gd.get_state()[0, 0])
        d = np.abs(out[1] - out[0])
        return d[j0, i0 + 1], d[j0, i0 + 2]

    dt = 2e-3
    near0, far0 = change(dt, False)
    near1, far1 = change(dt, True)
    _, far2 = change(dt / 4, True)
    # (uncorrected, the perturbed cell reaches (i0+1, j0) through the x-flux at i0+1/2 at O(dt), and (i0+2, j0)
    # only through second-order couplings)
    assert abs(near1 - near0) > 1e-6                            # the shared interface sees the large eta
    assert far1 == 0.0 and far2 == 0.0                          # the next interface does not: no path to that cell


# ---- Eq. C1 pinned quantitatively ---------------------------------------------------------------------
# With PCM (Eq. 25-26) the traced states are the cell averages, so one H-corrected step can be written out by hand
# from the unit-level solver alone (ref.riemann_roe / ref.riemann_roe_eta, pinned above and in test_oracle_roe.py):
# nothing of the oracle's grid code (ctu_step) is used to form the expected values.
def _prim(u, gamma):
    rho = u[0]
    v = u[1:4] / rho
    p = (gamma - 1) * (u[4] - 0.5 * rho * (v ** 2).sum(axis=0))
    return np.concatenate([rho[None], v, p[None]])


def _eta_c1(WL, WR, gamma, d, variant="C1"):
    """eta of one interface from its two input states (primitive, global order), normal direction d."""
    aL, aR = math.sqrt(gamma * WL[4] / WL[0]), math.sqrt(gamma * WR[4] / WR[0])
    if variant == "no_half":
        return abs((WR[1 + d] + aR) - (WL[1 + d] + aL))
    if variant == "u_minus_a":
        return 0.5 * abs((WR[1 + d] - aR) - (WL[1 + d] - aL))
    return 0.5 * abs((WR[1 + d] + aR) - (WL[1 + d] + aL))


def _local(W, d):        # global (rho, vx, vy, vz, p) -> direction-local (rho, vn, vt1, vt2, p), cyclic
    return [W[0], W[1 + d], W[1 + (d + 1) % 3], W[1 + (d + 2) % 3], W[4]]


def _global_flux(f, d):  # local flux (rho, mn, mt1, mt2, E) -> global field order
    out = np.empty(5)
    out[0], out[4] = f[0], f[4]
    out[1 + d], out[1 + (d + 1) % 3], out[1 + (d + 2) % 3] = f[1], f[2], f[3]
    return out


def pcm_roe_hcorr_step_by_hand(ref, u, dt, dx, gamma, variant="C1", eta_states="corrected"):
    """One CTU step, PCM + Roe + H correction, on a 2-D periodic [5][ny][nx] array: steps 1-5 of P:L152-173 with
    C1-C3 written out per interface in Python loops."""
    _, ny, nx = u.shape
    sh = {0: lambda a, s: np.roll(a, -s, axis=2), 1: lambda a, s: np.roll(a, -s, axis=1)}   # a(c + s e_d)
    W = _prim(u, gamma)
    Fs = {}
    for d in (0, 1):                                                   # step 2: F* from the cell averages
        Wp = sh[d](W, 1)
        F = np.empty_like(u)
        for j in range(ny):
            for i in range(nx):
                f, _ = ref.riemann_roe(gamma, _local(W[:, j, i], d), _local(Wp[:, j, i], d))
                F[:, j, i] = _global_flux(f, d)
        Fs[d] = F
    Uh = {d: u + 0.5 * dt / dx * (sh[1 - d](Fs[1 - d], -1) - Fs[1 - d]) for d in (0, 1)}   # step 3, Eq. 23
    Wh = {d: _prim(Uh[d], gamma) for d in (0, 1)}
    src = Wh if eta_states == "corrected" else {0: W, 1: W}
    eta = {}
    for d in (0, 1):                                                   # C1 at interface c + 1/2 along d, stored at c
        Sp = sh[d](src[d], 1)
        eta[d] = np.array([[_eta_c1(src[d][:, j, i], Sp[:, j, i], gamma, d, variant) for i in range(nx)]
                           for j in range(ny)])[None]
    Fh = {}
    for d in (0, 1):                                                   # C2 (reading G11) + C3 + step 4
        e = 1 - d
        own, te = eta[d][0], eta[e][0]
        tem = sh[e](eta[e], -1)[0]
        etaH = np.maximum.reduce([own, te, tem, sh[d](eta[e], 1)[0], sh[d](sh[e](eta[e], -1), 1)[0]])
        Wp = sh[d](Wh[d], 1)
        F = np.empty_like(u)
        for j in range(ny):
            for i in range(nx):
                f, _ = ref.riemann_roe_eta(gamma, _local(Wh[d][:, j, i], d), _local(Wp[:, j, i], d), etaH[j, i])
                F[:, j, i] = _global_flux(f, d)
        Fh[d] = F
    return u + dt / dx * ((sh[0](Fh[0], -1) - Fh[0]) + (sh[1](Fh[1], -1) - Fh[1]))      # step 5, Eq. 24


def test_c1_one_dimensional_two_state_problem_by_hand(ref):
    """1-D, PCM + Roe + H correction, one step: the only interface with a jump has eta = |(u_R+a_R) - (u_L+a_L)|/2
    by hand, its flux must be riemann_roe_eta(W_L, W_R, eta) and the two neighbouring cells change by exactly
    -/+ dt/dx (F - F_uniform).  The states are chosen so that eta exceeds the contact speed |u~| (otherwise C3's
    max() hides it): dropping the 1/2 or taking u - a for u + a changes the flux by far more than the gate."""
    n, gamma, i0 = 16, G, 7
    WL, WR = [1.0, 0.3, 0.0, 0.0, 1.0], [0.5, -0.2, 0.0, 0.0, 0.4]
    rho = np.where(np.arange(n) <= i0, WL[0], WR[0]); vx = np.where(np.arange(n) <= i0, WL[1], WR[1])
    p = np.where(np.arange(n) <= i0, WL[4], WR[4])
    u = wl.conserved(rho, vx, 0.0, 0.0, p, gamma).reshape(5, 1, 1, n)
    Gd = ref.RefGrid(n, 1, 1, 4, gamma, (O,) * 6)
    Gd.set_solver(1); Gd.set_reconstruction(2); Gd.set_hcorrection(True)
    Gd.set_state(u)
    dt, dx = 0.01, 1.0 / n
    Gd.step(dt)
    out = Gd.get_state()[:, 0, 0, :]
    eta = _eta_c1(WL, WR, gamma, 0)
    assert abs(eta - 0.5 * abs((-0.2 + math.sqrt(1.4 * 0.8)) - (0.3 + math.sqrt(1.4)))) < 1e-15
    F, path = ref.riemann_roe_eta(gamma, WL, WR, eta)
    assert path == "roe"
    FL, UL = eq11_and_u(WL); FR, UR = eq11_and_u(WR)
    assert np.allclose(out[:, i0], UL - dt / dx * (F - FL), rtol=0, atol=1e-14)
    assert np.allclose(out[:, i0 + 1], UR + dt / dx * (F - FR), rtol=0, atol=1e-14)
    assert np.array_equal(out[:, :i0], u[:, 0, 0, :i0]) and np.array_equal(out[:, i0 + 2:], u[:, 0, 0, i0 + 2:])
    # the pin discriminates: each plausible mistake in C1 moves the expected cell values far outside the gate
    for variant in ("no_half", "u_minus_a"):
        Fw, _ = ref.riemann_roe_eta(gamma, WL, WR, _eta_c1(WL, WR, gamma, 0, variant))
        assert np.abs((UL - dt / dx * (Fw - FL)) - out[:, i0]).max() > 1e-4, variant
    F0, _ = ref.riemann_roe(gamma, WL, WR)
    assert np.abs((UL - dt / dx * (F0 - FL)) - out[:, i0]).max() > 1e-4


def test_c1_transverse_jump_sets_eta_on_an_interface_with_no_jump_of_its_own(ref):
    """2-D: a shear layer along x (jump in v_y only: u + a equal on both sides, so the x-interface's own eta is 0 and
    the plain Roe flux does not diffuse it, u~ = 0) next to a jump in v_y + a across y.  eta^H of the x-interface is
    then the TRANSVERSE eta of C1, and the shear is diffused at rate eta^H: cell values follow from it by hand."""
    nx, ny, gamma = 8, 6, G
    rho = np.ones((1, ny, nx)); p = np.ones((1, ny, nx)); vx = np.zeros((1, ny, nx)); vy = np.zeros((1, ny, nx))
    vy[0, :, nx // 2:] = 0.4                      # shear across the x-interfaces i = nx/2 - 1/2 and the periodic seam
    p[0, ny // 2:, :] = 1.6                       # pressure (sound-speed) jump across y: eta_y = |a_R - a_L|/2-ish
    u = wl.conserved(rho, vx, vy, 0.0, p, gamma)[:, 0]
    dt, dx = 4e-3, 1.0 / nx
    Gd = ref.RefGrid(nx, ny, 1, 4, gamma, (P,) * 6)
    Gd.set_solver(1); Gd.set_reconstruction(2); Gd.set_hcorrection(True)
    Gd.set_state(u.reshape(5, 1, ny, nx))
    Gd.step(dt)
    out = Gd.get_state()[:, 0]
    want = pcm_roe_hcorr_step_by_hand(ref, u, dt, dx, gamma)
    scale = np.abs(u).max()
    assert np.abs(out - want).max() <= 1e-13 * scale
    G0 = ref.RefGrid(nx, ny, 1, 4, gamma, (P,) * 6)
    G0.set_solver(1); G0.set_reconstruction(2); G0.set_hcorrection(False)
    G0.set_state(u.reshape(5, 1, ny, nx)); G0.step(dt)
    assert np.abs(G0.get_state()[:, 0] - out).max() > 1e-4 * scale          # the correction acts here


def test_c1_random_two_dimensional_states_by_hand_and_the_mistakes_it_excludes(ref):
    """Random piecewise-constant 2-D states, PCM + Roe + H correction, every cell against the hand-written step.
    The same hand-written step with each plausible mistake in C1 — the 1/2 dropped, u - a for u + a, eta from the
    states BEFORE the transverse correction (U* instead of U^{n+1/2}) — misses the oracle by orders of
    magnitude more than the gate, so any of them in cholla_ref.cpp would fail this test."""
    nx, ny, gamma = 7, 6, G
    rng = np.random.default_rng(1281)
    rho = rng.uniform(0.6, 1.6, (1, ny, nx)); p = rng.uniform(0.6, 1.6, (1, ny, nx))
    vx, vy, vz = (rng.normal(0, 0.25, (1, ny, nx)) for _ in range(3))
    u = wl.conserved(rho, vx, vy, vz, p, gamma)[:, 0]
    dt, dx = 0.02, 1.0 / nx                        # CFL ~ 0.25: the transverse correction moves the states visibly
    Gd = ref.RefGrid(nx, ny, 1, 4, gamma, (P,) * 6)
    Gd.set_solver(1); Gd.set_reconstruction(2); Gd.set_hcorrection(True)
    Gd.set_state(u.reshape(5, 1, ny, nx))
    Gd.step(dt)
    out = Gd.get_state()[:, 0]
    scale = np.abs(u).max()
    want = pcm_roe_hcorr_step_by_hand(ref, u, dt, dx, gamma)
    assert np.abs(out - want).max() <= 1e-13 * scale
    for kw in (dict(variant="no_half"), dict(variant="u_minus_a"), dict(eta_states="uncorrected")):
        wrong = pcm_roe_hcorr_step_by_hand(ref, u, dt, dx, gamma, **kw)
        assert np.abs(out - wrong).max() > 1e-7 * scale, kw
