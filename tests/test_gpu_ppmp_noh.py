"""GPU-vs-oracle parity of the last rows of SURVEY.md section 8(f) NEXT-4 (`-m gpu`, through the C ABI):
the PPMP and PLMP reconstructions (ch_set_reconstruction 3 / 4) and the analytic boundary of the Noh strong-shock
test (bc code 4, ch_set_noh / ch_set_time), plus the Noh test itself on the GPU against its analytic solution."""
import math

import numpy as np
import pytest

from paper_1410_4194_b200 import binding, workloads as wl
from paper_1410_4194_b200.driver import run
from tests.parity import ONE_STEP_TOL, RUN_L1_TOL, max_rel_error, rel_l1_error

pytestmark = pytest.mark.gpu

P, R, O, N = wl.PERIODIC, wl.REFLECTIVE, wl.OUTFLOW, wl.NOH
PPMP, PLMP = 3, 4


@pytest.fixture(scope="module")
def ch():
    import paper_1410_4194_b200 as pkg
    pkg.load_library()
    return pkg


CASES = {
    "sod_1d": lambda: wl.sod(128),
    "sod_along_z": lambda: wl.sod(96, axis=2, n_other=5),
    "kh_2d": lambda: wl.kelvin_helmholtz(128),
    "sweep_ragged_3d": lambda: wl.sweep(shape=(70, 45, 37)),
    "sweep_xz_2d": lambda: wl.sweep(shape=(64, 1, 48)),
    "sedov_32": lambda: wl.sedov(32),
    "shock_cloud_48": lambda: wl.shock_cloud(48),
    "rough_3d": lambda: wl.rough_random(38, 21, 13, seed=11, decades=0.3, mach=0.8),
    "rough_1d": lambda: wl.rough_random(600, seed=12, mach=2.0, decades=0.5),
    "smooth_mixed_bc": lambda: wl.smooth_random(41, 29, 23, seed=5, bc=(R, O, P, P, O, R)),
}


def make(ch, ref, w, recon, solver, g=4):
    nx, ny, nz = w.shape
    G = ch.Grid(nx, ny, nz, g, w.gamma, w.bc)
    Rg = ref.RefGrid(nx, ny, nz, g, w.gamma, w.bc)
    for x in (G, Rg):
        x.set_solver(solver)
        x.set_reconstruction(recon)
    return G, Rg


@pytest.mark.parametrize("solver", [0, 1])
@pytest.mark.parametrize("recon", [PPMP, PLMP])
@pytest.mark.parametrize("name", sorted(CASES))
def test_ppmp_plmp_one_step_parity(ch, ref, name, recon, solver):
    w = CASES[name]()
    G, Rg = make(ch, ref, w, recon, solver)
    G.set_state(w.u); Rg.set_state(w.u)
    dt = Rg.compute_dt(w.cfl)
    G.step(dt); Rg.step(dt)
    ur = Rg.get_state()
    if not np.all(np.isfinite(ur)) or np.any(ur[0] <= 0):
        pytest.skip("the oracle's step left the physical regime on this input")
    err = max_rel_error(G.get_state(), ur, w.gamma)
    G.close()
    assert max(err) <= ONE_STEP_TOL, (name, recon, solver, err)


def test_ppmp_steepening_and_flattening_are_exercised(ref):
    """The parity cases above must reach the thresholded branches: on the Sod tube after some steps the contact is
    steepened (PPMP differs from the same run without A35-A41 would need oracle surgery, so instead: the PPMP state
    differs from the PPMC state at the contact AND at the shock by far more than rounding)."""
    w = wl.sod(128)
    a = ref.RefGrid(128, 1, 1, 4, w.gamma, w.bc); a.set_reconstruction(PPMP); run(a, w, max_steps=40)
    b = ref.RefGrid(128, 1, 1, 4, w.gamma, w.bc); b.set_reconstruction(0); run(b, w, max_steps=40)
    assert np.max(np.abs(a.get_state()[0] - b.get_state()[0])) > 1e-3


@pytest.mark.parametrize("recon", [PPMP, PLMP])
def test_ppmp_plmp_runs_match_oracle_and_switch_back(ch, ref, recon):
    for w in (wl.sod(128), wl.sweep(shape=(40, 32, 24))):
        if w.t_end is None:
            w.steps = 12
        G, Rg = make(ch, ref, w, recon, 0)
        dts = []
        run(Rg, w, record_dts=dts)
        run(G, w, dts=dts)
        assert max(rel_l1_error(G.get_state(), Rg.get_state(), w.gamma)) <= RUN_L1_TOL
        run(G, w)                                                  # free-running
        assert max(rel_l1_error(G.get_state(), Rg.get_state(), w.gamma)) <= RUN_L1_TOL
        # back to the default reconstruction: the default kernels again, same bits as a fresh default grid
        G.set_reconstruction(0)
        G.set_state(w.u)
        G.step(dts[0])
        F = ch.Grid(*w.shape, 4, w.gamma, w.bc)
        F.set_state(w.u); F.step(dts[0])
        assert np.array_equal(G.get_state(), F.get_state())
        G.close(); F.close()


def test_reconstruction_refusals(ch):
    G = ch.Grid(16, 16, 1, 3, 1.4, (P,) * 6)
    with pytest.raises(ValueError):
        G.set_reconstruction(PPMP)                                 # 7-cell stencil: nghost >= 4
    G.set_reconstruction(PLMP)
    G.close()
    G = ch.Grid(16, 16, 1, 4, 1.4, (P,) * 6)
    G.set_solver(1); G.set_hcorrection(True)
    with pytest.raises(ValueError):
        G.set_reconstruction(PPMP)
    G.set_hcorrection(False); G.set_reconstruction(PPMP)
    with pytest.raises(ValueError):
        G.set_hcorrection(True)
    with pytest.raises(ValueError):
        G.set_reconstruction(7)
    G.close()


# ---- the analytic (Noh) boundary -----------------------------------------------------------------------
@pytest.mark.parametrize("shape,bc", [((12, 1, 1), (R, N) * 3), ((10, 8, 1), (R, N) * 3), ((7, 6, 5), (R, N) * 3),
                                      ((1, 9, 8), (R, N) * 3), ((9, 7, 6), (O, N, R, N, P, P)), ((8, 8, 8), (N, N, R, O, R, N))])
def test_noh_ghost_fill_is_bit_exact(ch, ref, shape, bc):
    w = wl.noh(shape=shape)
    for g in (3, 4):
        G = ch.Grid(*shape, g, w.gamma, bc)
        Rg = ref.RefGrid(*shape, g, w.gamma, bc)
        for x in (G, Rg):
            x.set_noh(1.3, 2e-6)
            x.set_state(w.u)
        assert np.array_equal(G.get_padded(), Rg.get_padded())     # t = 0
        for x in (G, Rg):
            x.set_time(0.37)
            x.fill_ghosts()
        a, b = G.get_padded(), Rg.get_padded()
        assert np.array_equal(a, b)
        assert G.get_time() == 0.37
        G.close()


def noh_pair(ch, ref, w, hc=True):
    G = ch.Grid(*w.shape, 4, w.gamma, w.bc)
    Rg = ref.RefGrid(*w.shape, 4, w.gamma, w.bc)
    for x in (G, Rg):
        x.set_solver(1)
        x.set_hcorrection(hc)
        x.set_noh(1.0, 1e-6)
    return G, Rg


@pytest.mark.parametrize("dims,n,steps", [(1, 200, 40), (2, 48, 40), (3, 20, 20)])
def test_noh_runs_match_the_oracle(ch, ref, dims, n, steps):
    """The Noh problem as the paper runs it (Roe + H correction, reflecting inner / analytic outer faces): one step
    within the one-step gate, `steps` steps within the run gate (lock-step), and the clocks agree."""
    w = wl.noh(n=n, dims=dims)
    w.t_end, w.steps = None, steps
    G, Rg = noh_pair(ch, ref, w)
    G.set_state(w.u); Rg.set_state(w.u)
    dt = Rg.compute_dt(w.cfl)
    G.step(dt); Rg.step(dt)
    assert max(max_rel_error(G.get_padded(), Rg.get_padded(), w.gamma)) <= ONE_STEP_TOL
    dts = []
    run(Rg, w, record_dts=dts)
    run(G, w, dts=dts)
    assert max(rel_l1_error(G.get_state(), Rg.get_state(), w.gamma)) <= RUN_L1_TOL
    assert abs(G.get_time() - Rg.get_time()) <= 1e-15
    with pytest.raises(RuntimeError):
        G.step_cfl(w.cfl)                                          # analytic faces need the time on the host
    G.close()


def test_noh_3d_on_the_gpu_against_the_analytic_solution(ch):
    """P:L543-565 at 100^3 (the paper: 200^3), PPMC + Roe + H correction, to t = 2: shock at r = t/3 = 0.667,
    rho = 64 behind it, rho = (1 + t/r)^2 ahead of it."""
    n, t_end = 100, 2.0
    w = wl.noh(n=n, dims=3, t_end=t_end)
    G = ch.Grid(n, n, n, 4, w.gamma, w.bc)
    G.set_solver(1); G.set_hcorrection(True); G.set_noh(1.0, 1e-6)
    steps, t = run(G, w)
    u = G.get_state()
    G.close()
    assert abs(t - t_end) < 1e-12 and steps > 300
    c = (np.arange(n) + 0.5) / n
    r = np.sqrt(c[None, None, :] ** 2 + c[None, :, None] ** 2 + c[:, None, None] ** 2)
    rho = u[0]
    assert np.all(np.isfinite(u)) and rho.min() > 0
    post = (r > 0.2) & (r < 0.55)
    assert abs(rho[post].mean() - 64.0) < 2.5, rho[post].mean()
    pre = (r > 0.8) & (r < 1.0)
    assert np.max(np.abs(rho[pre] / (1.0 + t_end / r[pre]) ** 2 - 1.0)) < 0.03
    bins = np.linspace(0.5, 0.85, 36)
    prof = np.array([rho[(r >= a) & (r < b)].mean() for a, b in zip(bins[:-1], bins[1:])])
    rc = 0.5 * (bins[1:] + bins[:-1])
    r_shock = rc[np.max(np.nonzero(prof > 40.0)[0])]
    assert abs(r_shock - t_end / 3.0) < 2.5 / n, r_shock
    # octant symmetry under permutation of the axes, to the level a Mach-1000 shock leaves
    for perm in ((2, 1, 0), (1, 0, 2)):
        d = np.abs(rho - rho.transpose(perm)) / rho
        assert np.median(d) < 1e-4 and d.mean() < 1e-2, (np.median(d), d.mean(), d.max())    # rounding, amplified at the front of a Mach-1000 shock
