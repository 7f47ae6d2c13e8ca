"""Pins of the oracle's whole CTU step (oracle/cholla_ref.cpp: ghost_fill, compute_dt, ctu_step;
P:L103-175) against what the paper and the physics fix:

* ghost fill == numpy.pad (wrap / edge / symmetric with the normal momentum negated), any mix per face;
* Eq. 22 in closed form on uniform data, and its min over cells/directions;
* uniform states are preserved to the bit under every boundary condition;
* mass, momentum, energy are conserved to round-off under periodic boundaries;
* a 1-D problem embedded in 3-D along x, y or z reproduces the 1-D run to the bit;
* translation invariance under periodic boundaries (pins the edge/corner ghost ordering);
* mirror symmetry to the bit; reflective walls == the mirrored periodic problem;
* second-order L1 convergence on a smooth sound wave, 1-D and oblique 3-D;
* Sod (BASELINE.json config 1): L1 error against the exact solution falls with resolution, the
  contact and the shock sit where the paper says; strong shock; 123;
* a Mach-50 planar shock moves at the Rankine-Hugoniot speed; Sedov-Taylor radius (config 3).
"""
import math

import mpmath as mp
import numpy as np
import pytest

from paper_1410_4194_b200 import workloads as wl
from paper_1410_4194_b200.driver import run

P, R, O = wl.PERIODIC, wl.REFLECTIVE, wl.OUTFLOW


def smooth_state(nx, ny, nz, seed=0, gamma=5.0 / 3.0, amp=0.2):
    rng = np.random.default_rng(seed)
    def f():
        x = (np.arange(nx) + 0.5) / nx; y = (np.arange(ny) + 0.5) / ny; z = (np.arange(nz) + 0.5) / nz
        out = np.zeros((nz, ny, nx))
        for _ in range(3):
            k = rng.integers(-2, 3, 3); ph = rng.uniform(0, 2 * np.pi)
            out += np.sin(2 * np.pi * (k[0] * x[None, None, :] + k[1] * y[None, :, None] + k[2] * z[:, None, None]) + ph)
        return out / 3
    return wl.conserved(1 + amp * f(), amp * f(), amp * f(), amp * f(), 1 + amp * f(), gamma)


# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", [(P, P, P, P, P, P), (O, O, O, O, O, O), (R, R, R, R, R, R), (R, O, P, P, O, R)])
def test_ghost_fill_equals_numpy_pad(ref, bc):
    nx, ny, nz, g = 4, 5, 6, 3
    rng = np.random.default_rng(1)
    u = rng.normal(size=(5, nz, ny, nx))
    G = ref.RefGrid(nx, ny, nz, g, 1.4, bc)
    G.set_state(u)
    got = G.get_padded()
    mode = {P: "wrap", O: "edge", R: "symmetric"}
    want = u.copy()
    for d, axis in ((0, 3), (1, 2), (2, 1)):           # x, then y, then z
        lo, hi = bc[2 * d], bc[2 * d + 1]
        pads = [[(0, 0)] * 4, [(0, 0)] * 4]
        pads[0][axis] = (g, 0); pads[1][axis] = (0, g)
        # pad both sides from the same unpadded array so 'wrap' on one side cannot see the other pad
        a = np.pad(want, pads[0], mode=mode[lo])
        b = np.pad(want, pads[1], mode=mode[hi])
        lo_part = np.take(a, range(g), axis=axis).copy()
        hi_part = np.take(b, range(b.shape[axis] - g, b.shape[axis]), axis=axis).copy()
        if lo == R: lo_part[1 + d] *= -1
        if hi == R: hi_part[1 + d] *= -1
        want = np.concatenate([lo_part, want, hi_part], axis=axis)
    assert np.array_equal(got, want)


def test_inactive_dimensions_have_no_ghosts(ref):
    G = ref.RefGrid(8, 1, 1, 3, 1.4, (O,) * 6)
    assert G.padded_shape == (1, 1, 14)
    G = ref.RefGrid(8, 6, 1, 3, 1.4, (P,) * 6)
    assert G.padded_shape == (1, 12, 14)


def test_init_rejects_bad_arguments(ref):
    for args in ((0, 1, 1, 3, 1.4, (P,) * 6), (8, 1, 1, 2, 1.4, (P,) * 6), (8, 1, 1, 3, 1.0, (P,) * 6),
                 (8, 1, 1, 3, 1.4, (P, O, P, P, P, P)), (8, 2, 1, 3, 1.4, (P,) * 6)):
        with pytest.raises(ValueError):
            ref.RefGrid(*args)


def test_dt_closed_form(ref):
    gamma, nx = 1.4, 16
    rho, vel, p = 1.3, (0.4, -1.1, 0.2), 0.9
    a = math.sqrt(gamma * p / rho)
    for shape, dims in (((nx, 1, 1), (0,)), ((nx, 8, 1), (0, 1)), ((nx, 8, 4), (0, 1, 2))):
        u = wl.conserved(rho, vel[0], vel[1], vel[2], p, gamma).reshape(5, 1, 1, 1) * np.ones((5, shape[2], shape[1], shape[0]))
        G = ref.RefGrid(*shape, 3, gamma, (P,) * 6)
        G.set_state(u)
        want = 0.3 * min((1.0 / nx) / (abs(vel[d]) + a) for d in dims)      # Eq. 22, inactive dims dropped
        assert G.compute_dt(0.3) == pytest.approx(want, rel=1e-14)
    # the minimum is over all cells: one fast cell sets it
    u = wl.conserved(rho, 0.0, 0.0, 0.0, p, gamma).reshape(5, 1, 1, 1) * np.ones((5, 4, 8, nx))
    u[:, 2, 5, 7] = wl.conserved(rho, 0.0, 0.0, -9.0, p, gamma)
    G = ref.RefGrid(nx, 8, 4, 3, gamma, (P,) * 6); G.set_state(u)
    assert G.compute_dt(0.5) == pytest.approx(0.5 * (1.0 / nx) / (9.0 + a), rel=1e-14)
    u[0, 0, 0, 0] = -1.0
    G.set_state(u)
    assert math.isnan(G.compute_dt(0.5))


@pytest.mark.parametrize("bc", [(P,) * 6, (O,) * 6, (R,) * 6, (R, O, P, P, O, R)])
def test_uniform_state_is_preserved_bitwise(ref, bc):
    gamma = 5.0 / 3.0
    u = wl.conserved(0.7, 0.3, -0.45, 0.21, 1.9, gamma).reshape(5, 1, 1, 1) * np.ones((5, 6, 7, 8))
    if R in bc:    # a wall needs zero normal velocity for the state to be uniform across it
        u = wl.conserved(0.7, 0.0, 0.0, 0.0, 1.9, gamma).reshape(5, 1, 1, 1) * np.ones((5, 6, 7, 8))
        if bc[2:4] == (P, P):
            u = wl.conserved(0.7, 0.0, 0.37, 0.0, 1.9, gamma).reshape(5, 1, 1, 1) * np.ones((5, 6, 7, 8))
    G = ref.RefGrid(8, 7, 6, 3, gamma, bc)
    G.set_state(u)
    for _ in range(3):
        G.step(G.compute_dt(0.4))
    assert np.array_equal(G.get_state(), u)


def test_conservation_periodic(ref):
    nx, ny, nz = 12, 10, 8
    u0 = smooth_state(nx, ny, nz, seed=3)
    G = ref.RefGrid(nx, ny, nz, 3, 5.0 / 3.0, (P,) * 6)
    G.set_state(u0)
    for _ in range(4):
        G.step(G.compute_dt(0.4))
    u1 = G.get_state()
    assert not np.array_equal(u0, u1)
    for f in range(5):
        s0, s1 = math.fsum(u0[f].ravel()), math.fsum(u1[f].ravel())
        scale = math.fsum(np.abs(u0[f]).ravel()) + 1.0
        assert abs(s1 - s0) <= 4e-16 * scale * math.sqrt(u0[f].size), (f, s1 - s0)


def test_conservation_2d_and_positivity(ref):
    w = wl.kelvin_helmholtz(32, steps=10)
    G = ref.RefGrid(32, 32, 1, 3, w.gamma, w.bc)
    run(G, w)
    u1 = G.get_state()
    for f in (0, 1, 2, 4):
        assert abs(math.fsum(u1[f].ravel()) - math.fsum(w.u[f].ravel())) <= 1e-13 * (1 + math.fsum(np.abs(w.u[f]).ravel()))
    assert np.all(u1[3] == 0.0) and np.all(u1[0] > 0)


@pytest.mark.parametrize("aniso", [False, True])
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_1d_embedded_in_3d_is_bitwise(ref, axis, aniso):
    """aniso: the two transverse cell widths differ from the sweep's — the result must not notice, which pins
    that the sweep along `axis` uses dx_axis (and only it) in tracing, update and nothing else."""
    n, m = 32, 4
    one = wl.sod(n)
    G1 = ref.RefGrid(n, 1, 1, 3, one.gamma, one.bc)
    dts = []
    run(G1, one, max_steps=12, record_dts=dts)
    u1 = G1.get_state()[:, 0, 0, :]                       # [5][n], momentum along x in slot 1

    shape = [m, m, m]; shape[axis] = n                     # (nx, ny, nz)
    u3 = np.zeros((5, shape[2], shape[1], shape[0]))
    line = one.u[:, 0, 0, :]
    idx = [None, None, None]; idx[2 - axis] = slice(None)
    for f_src, f_dst in ((0, 0), (1, 1 + axis), (4, 4)):
        u3[f_dst] = line[f_src][tuple(idx)]
    bc = tuple(O if d == axis else P for d in range(3) for _ in range(2))
    G3 = ref.RefGrid(*shape, 3, one.gamma, bc)
    # keep the same cell width as the 1-D run (reading S8 ties dx to nx)
    sp = [1.0 / n, 1.0 / n, 1.0 / n]
    if aniso:
        sp = [0.37, 0.011, 2.3]; sp[axis] = 1.0 / n
    G3.set_spacing(*sp)
    G3.set_state(u3)
    if aniso:                                  # Eq. 22 picks each direction's own width
        a = np.sqrt(one.gamma * 1.0 / 1.0)      # fastest signal at t = 0: sound speed of the left state, v = 0
        assert G3.compute_dt(0.4) == pytest.approx(0.4 * min(sp) / a, rel=1e-14)
    for dt in dts:
        G3.step(dt)
    out = G3.get_state()
    for f_src, f_dst in ((0, 0), (1, 1 + axis), (4, 4)):
        want = u1[f_src][tuple(idx)] * np.ones_like(out[0])
        assert np.array_equal(out[f_dst], want), (axis, f_dst)
    for f in (1, 2, 3):
        if f != 1 + axis:
            assert np.all(out[f] == 0.0)


def test_translation_invariance_periodic_bitwise(ref):
    nx, ny, nz = 10, 12, 9
    u0 = smooth_state(nx, ny, nz, seed=5)
    sh = (2, 5, 3)                                         # shift in (z, y, x)
    outs = []
    for u in (u0, np.roll(u0, sh, axis=(1, 2, 3))):
        G = ref.RefGrid(nx, ny, nz, 3, 5.0 / 3.0, (P,) * 6)
        G.set_state(u)
        for _ in range(3):
            G.step(1.5e-2)
        outs.append(G.get_state())
    assert np.array_equal(np.roll(outs[0], sh, axis=(1, 2, 3)), outs[1])


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_mirror_symmetry_bitwise(ref, axis):
    """Mirrored initial data give the mirrored solution to the bit (the paper's implosion and
    explosion tests stay exactly symmetric)."""
    nx, ny, nz = 10, 8, 6
    u0 = smooth_state(nx, ny, nz, seed=8, amp=0.3)
    ax = 3 - axis
    um = np.flip(u0, axis=ax).copy()
    um[1 + axis] *= -1
    outs = []
    for u in (u0, um):
        G = ref.RefGrid(nx, ny, nz, 3, 5.0 / 3.0, (P,) * 6)
        G.set_state(u)
        for _ in range(3):
            G.step(1.2e-2)
        outs.append(G.get_state())
    back = np.flip(outs[1], axis=ax).copy()
    back[1 + axis] *= -1
    assert np.array_equal(outs[0], back)


def test_reflective_walls_equal_the_mirrored_periodic_problem(ref):
    n = 24
    rng = np.random.default_rng(2)
    rho = 1 + 0.3 * rng.uniform(size=n); v = 0.3 * rng.normal(size=n); p = 1 + 0.3 * rng.uniform(size=n)
    half = wl.conserved(rho, v, 0.0, 0.0, p, 1.4).reshape(5, 1, 1, n)
    full = np.concatenate([half, np.flip(half, axis=3) * np.array([1, -1, 1, 1, 1]).reshape(5, 1, 1, 1)], axis=3)
    Gh = ref.RefGrid(n, 1, 1, 3, 1.4, (R, R, P, P, P, P)); Gh.set_state(half)
    Gf = ref.RefGrid(2 * n, 1, 1, 3, 1.4, (P,) * 6); Gf.set_spacing(1.0 / n, 1.0 / n, 1.0 / n); Gf.set_state(full)
    for _ in range(20):
        dt = Gh.compute_dt(0.4)
        assert Gf.compute_dt(0.4) == dt
        Gh.step(dt); Gf.step(dt)
    assert np.array_equal(Gf.get_state()[..., :n], Gh.get_state())


# ------------------------------------------------------------------------------------------------
def l1_wave_error(ref, n, dims):
    shape = (n, n if dims >= 2 else 1, n if dims >= 3 else 1)
    k = (1, 1 if dims >= 2 else 0, 1 if dims >= 3 else 0)
    w = wl.linear_wave(*shape, amp=1e-6, kvec=k)
    G = ref.RefGrid(*shape, 3, w.gamma, w.bc)
    run(G, w)
    return float(np.mean(np.abs(G.get_state() - w.u)))


def test_second_order_convergence_1d(ref):
    """second-order convergence in L1 on the smooth perturbation test."""
    ns = [32, 64, 128, 256]
    errs = [l1_wave_error(ref, n, 1) for n in ns]
    slopes = [math.log(errs[i] / errs[i + 1], 2) for i in range(len(ns) - 1)]
    assert all(e1 < e0 for e0, e1 in zip(errs, errs[1:]))
    assert all(1.8 <= s <= 3.3 for s in slopes), (errs, slopes)
    assert errs[0] < 0.05 * 1e-6                          # error is a small fraction of the amplitude


def test_second_order_convergence_3d_oblique(ref):
    errs = [l1_wave_error(ref, n, 3) for n in (8, 16, 32)]
    slopes = [math.log(errs[i] / errs[i + 1], 2) for i in range(2)]
    assert 1.7 <= slopes[-1] <= 3.3, (errs, slopes)


# ---- exact solution of a left-rarefaction / right-shock Riemann problem, built from the jump
# ---- conditions (independent of the oracle's sampler) -----------------------------------------
def exact_rarefaction_shock(left, right, gamma, guess):
    mp.mp.dps = 30
    rL, uL, pL = [mp.mpf(x) for x in left]; rR, uR, pR = [mp.mpf(x) for x in right]
    g = mp.mpf(gamma)
    ER = pR / (g - 1) + rR * uR ** 2 / 2
    aL = mp.sqrt(g * pL / rL)
    def eqs(p, u, rsl, rsr, S):
        Es = p / (g - 1) + rsr * u ** 2 / 2
        return [rsr * (u - S) - rR * (uR - S), rsr * u * (u - S) + p - (rR * uR * (uR - S) + pR),
                Es * (u - S) + p * u - (ER * (uR - S) + pR * uR), p / rsl ** g - pL / rL ** g,
                u + 2 * mp.sqrt(g * p / rsl) / (g - 1) - (uL + 2 * aL / (g - 1))]
    ps, us, rsl, rsr, S = [float(x) for x in mp.findroot(eqs, guess, tol=1e-25)]
    aL = float(aL); rL, uL, pL = left; rR, uR, pR = right
    head = uL - aL
    tail = us - math.sqrt(gamma * ps / rsl)
    def sample(xi):
        xi = np.asarray(xi, dtype=float)
        # inside the fan: u - a = xi, u + 2a/(g-1) = const, isentropic
        a_f = (2 / (gamma + 1)) * (aL + 0.5 * (gamma - 1) * (uL - xi))
        u_f = xi + a_f
        r_f = rL * (a_f / aL) ** (2 / (gamma - 1))
        p_f = pL * (a_f / aL) ** (2 * gamma / (gamma - 1))
        rho = np.where(xi < head, rL, np.where(xi < tail, r_f, np.where(xi < us, rsl, np.where(xi < S, rsr, rR))))
        u = np.where(xi < head, uL, np.where(xi < tail, u_f, np.where(xi < S, us, uR)))
        p = np.where(xi < head, pL, np.where(xi < tail, p_f, np.where(xi < S, ps, pR)))
        return rho, u, p
    return sample, dict(ps=ps, us=us, S=S, head=head, tail=tail)


def cell_average_exact(sample, n, t, x0=0.5, sub=16):
    xs = (np.arange(n * sub) + 0.5) / (n * sub)
    rho, u, p = sample((xs - x0) / t)
    return [a.reshape(n, sub).mean(axis=1) for a in (rho, u, p)]


def run_tube(ref, w):
    nx = w.shape[0]
    G = ref.RefGrid(nx, 1, 1, 3, w.gamma, w.bc)
    steps, t = run(G, w)
    u = G.get_state()[:, 0, 0, :]
    rho = u[0]; v = u[1] / rho
    p = (w.gamma - 1) * (u[4] - 0.5 * rho * v * v)
    return rho, v, p, steps


def test_sod_l1_error_decreases_and_waves_sit_where_the_paper_says(ref):
    sample, info = exact_rarefaction_shock((1.0, 0.0, 1.0), (0.125, 0.0, 0.1), 1.4, (0.30313, 0.92745, 0.42632, 0.26557, 1.7522))
    errs = []
    for n in (64, 128, 256, 512):
        rho, v, p, steps = run_tube(ref, wl.sod(n))
        er, eu, ep = cell_average_exact(sample, n, 0.2)
        errs.append(np.mean(np.abs(rho - er)) + np.mean(np.abs(v - eu)) + np.mean(np.abs(p - ep)))
        assert np.all(rho > 0) and np.all(p > 0)
        if n == 128:
            x = (np.arange(n) + 0.5) / n
            # shock: where rho falls through the mean of post-shock and ambient density
            mid = 0.5 * (0.26557 + 0.125)
            i_sh = np.max(np.nonzero(rho > mid)[0])
            assert abs(x[i_sh] - (0.5 + 0.2 * info["S"])) <= 1.5 / n      # ~0.85
            assert abs(x[i_sh] - 0.85) < 0.01
            # contact: where rho falls through the mean of the two star densities; ~0.7,
            # spread over a few zones
            midc = 0.5 * (0.42632 + 0.26557)
            i_c = np.max(np.nonzero(rho > midc)[0])
            assert abs(x[i_c] - (0.5 + 0.2 * info["us"])) <= 2.0 / n
            width = np.sum((rho < 0.42632 - 0.05 * 0.16) & (rho > 0.26557 + 0.05 * 0.16) & (np.abs(x - 0.6855) < 0.06))
            assert 1 <= width <= 6
            # plateaus reach the exact star values
            assert abs(rho[int(0.62 * n)] - 0.42632) < 2e-3 and abs(p[int(0.75 * n)] - 0.30313) < 2e-3
            assert 90 <= steps <= 160                                      # reading S13
    assert all(e1 < 0.75 * e0 for e0, e1 in zip(errs, errs[1:])), errs
    assert errs[1] < 0.01


def test_strong_shock_tube(ref):
    """rho 10/1, p 100/1, t = 0.07."""
    sample, info = exact_rarefaction_shock((10.0, 0.0, 100.0), (1.0, 0.0, 1.0), 1.4, (19.9, 3.85, 3.16, 4.65, 4.9))
    n = 100
    rho, v, p, _ = run_tube(ref, wl.riemann_tube(n, (10.0, 0.0, 100.0), (1.0, 0.0, 1.0), 1.4, t_end=0.07))
    er, eu, ep = cell_average_exact(sample, n, 0.07)
    assert np.mean(np.abs(rho - er)) < 0.06 and np.mean(np.abs(p - ep)) < 0.5
    x = (np.arange(n) + 0.5) / n
    i_sh = np.max(np.nonzero(rho > 0.5 * (4.649 + 1.0))[0])
    assert abs(x[i_sh] - (0.5 + 0.07 * info["S"])) <= 1.5 / n
    assert np.all(rho > 0) and np.all(p > 0)


def test_123_problem_near_vacuum(ref):
    """strong double rarefaction.  The paper runs it with PPMP + exact ("not a
    challenge"); its text makes no claim for PPMC.  With the PPMC step as printed the run stays
    positive at CFL 0.1 (at CFL >= 0.2 the central internal energy undershoots and the run fails
    — recorded in DESIGN.md, not a pin)."""
    n = 128
    w = wl.riemann_tube(n, (1.0, -2.0, 0.4), (1.0, 2.0, 0.4), 1.4, t_end=0.15)
    w.cfl = 0.1
    rho, v, p, _ = run_tube(ref, w)
    assert np.all(np.isfinite(rho)) and np.all(rho > 0) and np.all(p > 0)
    assert np.array_equal(rho, rho[::-1]) and np.array_equal(v, -v[::-1])     # mirror symmetric to the bit
    # central density approaches the two-rarefaction star value 0.02185
    assert rho[n // 2] < 0.05 and rho.min() < 0.03


def test_planar_mach50_shock_moves_at_the_rankine_hugoniot_speed(ref):
    """Config 4 without the cloud: the post-shock slab (Eq. 33 region) drives a Mach-50
    shock into (rho 0.1, p 1); the front must advance at 50 a0 = 204.124 and leave the RH plateau."""
    n = 128
    gamma, rho0, p0 = 5.0 / 3.0, 0.1, 1.0
    a0 = math.sqrt(gamma * p0 / rho0); m2 = 2500.0
    r1 = rho0 * (gamma + 1) * m2 / ((gamma - 1) * m2 + 2); p1 = p0 * (2 * gamma * m2 - (gamma - 1)) / (gamma + 1)
    vs = 50 * a0; v1 = vs * (1 - rho0 / r1)
    x0 = 16.0 / n
    t_end = 80.0 / n / vs
    w = wl.riemann_tube(n, (r1, v1, p1), (rho0, 0.0, p0), gamma, t_end=t_end, x0=x0)
    w.cfl = 0.3
    rho, v, p, _ = run_tube(ref, w)
    x = (np.arange(n) + 0.5) / n
    i_sh = np.max(np.nonzero(rho > 0.5 * (r1 + rho0))[0])
    assert abs(x[i_sh] - (x0 + vs * t_end)) <= 1.5 / n
    plate = slice(30, 80)
    # start-up errors of the initial discontinuity leave few-% ripples; the plateau mean is the RH state
    assert np.allclose(rho[plate], r1, rtol=4e-2) and np.allclose(v[plate], v1, rtol=2e-2) and np.allclose(p[plate], p1, rtol=4e-2)
    assert abs(rho[plate].mean() / r1 - 1) < 1e-2 and abs(v[plate].mean() / v1 - 1) < 5e-3 and abs(p[plate].mean() / p1 - 1) < 1e-2


def test_sedov_taylor_radius_octant(ref):
    """Config 3 on the +++ octant (reflective low faces) of a 64^3 box: the shock radius follows
    R = 1.15 (E t^2 / rho)^(1/5) (BASELINE.json config 3).  A captured shock is ~2 cells wide: the
    outer half-rise radius sits ~half a cell ahead of it and the density peak ~half a cell behind,
    so the closed form must lie between them and within one cell of the half-rise radius."""
    n = 32
    w = wl.sedov(n, octant=True)
    dx = w.meta["dx"]
    assert w.meta["hot_cells"] == 160                      # 160 cells within 3.5 dx
    G = ref.RefGrid(n, n, n, 3, w.gamma, w.bc)
    G.set_spacing(dx, dx, dx)
    w.t_end = 0.03
    steps, t = run(G, w)
    u = G.get_state()
    rho = u[0]
    c = (np.arange(n) + 0.5) * dx
    r = np.sqrt(c[None, None, :] ** 2 + c[None, :, None] ** 2 + c[:, None, None] ** 2)
    bins = np.arange(0, 0.5 + dx, dx)
    which = np.digitize(r.ravel(), bins)
    prof = np.array([rho.ravel()[which == b].mean() if np.any(which == b) else np.nan for b in range(1, len(bins))])
    rc = 0.5 * (bins[1:] + bins[:-1])
    ok = np.isfinite(prof) & (rc < 0.5 - 3 * dx)
    prof, rc = prof[ok], rc[ok]
    half = 0.5 * (prof.max() + 1.0)
    i = np.max(np.nonzero(prof > half)[0])
    r_half = rc[i] + (prof[i] - half) / (prof[i] - prof[i + 1]) * dx
    r_peak = rc[np.argmax(prof)]
    want = 1.15 * (1.0 * t * t / 1.0) ** 0.2
    assert abs(r_half - want) <= dx, (r_half, want, steps)
    assert r_peak - 0.5 * dx <= want <= r_half, (r_peak, want, r_half)
    assert prof.max() > 2.0                                # compression toward (g+1)/(g-1) = 4
    # symmetric under exchange of axes to round-off; total energy (8 octants) conserved while the
    # shock is inside the box
    assert np.allclose(rho, rho.transpose(2, 1, 0), rtol=1e-10) and np.allclose(rho, rho.transpose(0, 2, 1), rtol=1e-10)
    e_tot = math.fsum(u[4].ravel()) * dx ** 3 * 8
    assert abs(e_tot - (1.0 + 1e-5 / (w.gamma - 1) * (1 - 160 * dx ** 3))) < 1e-9
