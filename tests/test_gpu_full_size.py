"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (`-m gpu`).

At 256^3 every cell is compared (whole_grid_one_step: the oracle re-steps the grid slab by slab).  The oracle
cannot step 384^3 / 512^3 in seconds, so there full-size parity is taken on SAMPLED outputs
the oracle can compute one by one: after one GPU step of the whole grid, sub-boxes of m^3 real cells
(with their 3-deep halo cut from the GPU's pre-step padded store, whose ghost fill is checked
bit-exactly elsewhere) are stepped by the oracle with the same dt and cell widths, and every cell of
every sub-box must agree to <= 1e-12 (north_star's one-step gate; a cell's update depends on nothing
outside its radius-3 neighbourhood).  Sub-boxes sit on domain corners, edges and faces
(so periodic / outflow ghosts take part), across CTA tile seams of every kernel, and at seeded
random interior positions.  Conservation (periodic) holds at any size and is checked on the whole grid.
"""
import math

import numpy as np
import pytest

from paper_1410_4194_b200 import workloads as wl
from paper_1410_4194_b200.driver import run
from tests.parity import ONE_STEP_TOL, RUN_L1_TOL, max_rel_error, max_rel_error_strict, rel_l1_error

pytestmark = pytest.mark.gpu


def subbox_origins(n, m, rng, tiling, extra=6):
    """Origins of m^3 sub-boxes: domain corners / edges / faces, boxes centred on a CTA seam of every kernel (seam
    positions from ch_tiling, i.e. from the tile constants the library is using for THIS grid), random interior."""
    lo, hi, mid = 0, n - m, (n - m) // 2

    def seam(period, which):
        """a box origin such that the box straddles the `which`-th seam of a tiling with this period"""
        if period <= 0:
            return mid
        s = period * max(1, min(which, (n - 1) // period))
        return int(min(max(s - m // 2, lo), hi))

    t = tiling
    # the x pass cuts the flat padded run, so its seams drift through x; the first one falls at x = x_interfaces - g
    pts = [(lo, lo, lo), (hi, hi, hi), (lo, hi, mid), (hi, lo, mid), (mid, mid, lo), (mid, mid, hi),
           (seam(t["x_interfaces_per_cta"], 1), seam(t["march_seg_y"], 1), seam(t["march_seg_z"], 1)),
           (seam(t["march_columns_per_cta"], 1), seam(t["march_seg_y"], 2), seam(t["march_seg_z"], 3)),
           (seam(t["final_tile_x"], 1), seam(t["final_tile_y"], 1), seam(t["final_seg"], 1)),
           (seam(t["final_tile_x"], 10 ** 6), seam(t["final_tile_y"], 10 ** 6), seam(t["final_seg"], 10 ** 6)),
           (seam(t["final_tile_x"], 3), seam(t["final_tile_y"], 7), seam(t["final_seg"], 2))]
    for _ in range(extra):
        pts.append(tuple(int(v) for v in rng.integers(0, n - m + 1, 3)))
    return pts


def sampled_one_step(ref, w, m=12, extra=6, seed=0):
    import paper_1410_4194_b200 as ch
    nx, ny, nz = w.shape
    g = 3
    G = ch.Grid(nx, ny, nz, g, w.gamma, w.bc)
    tiling = G.tiling()
    assert tiling["final_tile_x"] > 0 and tiling["final_seg"] > 0
    G.set_state(w.u)
    dt = G.compute_dt(w.cfl)
    pre = G.get_padded()
    G.step(dt)
    post = G.get_state()
    G.close()
    dx = 1.0 / nx
    worst = 0.0
    rng = np.random.default_rng(seed)
    for (i0, j0, k0) in subbox_origins(nx, m, rng, tiling, extra):
        Rg = ref.RefGrid(m, m, m, g, w.gamma, (wl.OUTFLOW,) * 6)     # its own ghost fill runs after the update only
        Rg.set_spacing(dx, dx, dx)
        Rg.set_padded(pre[:, k0:k0 + m + 2 * g, j0:j0 + m + 2 * g, i0:i0 + m + 2 * g])
        Rg.step(dt)
        ur = Rg.get_state()
        ug = post[:, k0:k0 + m, j0:j0 + m, i0:i0 + m]
        worst = max(worst, max(max_rel_error(ug, ur, w.gamma)))
    return worst, post, dt


def whole_grid_one_step(ref, w, slab=32, pre_steps=0, g=3, setup=None, want_tma=None):
    """One GPU step of the WHOLE grid against the oracle on EVERY cell: the oracle re-steps z-slabs of `slab` planes
    (full x, y extent) cut with their 3-deep halo from the GPU's pre-step padded store (whose ghost fill is
    checked bit-exactly elsewhere), with the same dt and cell widths; a cell's update depends on nothing outside
    its radius-3 neighbourhood, so the slabs together are the oracle's step of the whole grid while
    its ~95 whole-grid work arrays stay at 1/8 of their 256^3 size.  Returns the assembled oracle state."""
    import paper_1410_4194_b200 as ch
    nx, ny, nz = w.shape
    G = ch.Grid(nx, ny, nz, g, w.gamma, w.bc)
    if setup:
        setup(G)
    if want_tma is not None:
        assert G.tiling()["tma"] == want_tma
    G.set_state(w.u)
    for _ in range(pre_steps):
        G.step(G.compute_dt(w.cfl))
    dt = G.compute_dt(w.cfl)
    pre = G.get_padded()
    G.step(dt)
    post = G.get_state()
    G.close()
    dx = 1.0 / nx
    ur = np.empty_like(post)
    for k0 in range(0, nz, slab):
        kn = min(slab, nz - k0)
        Rg = ref.RefGrid(nx, ny, kn, g, w.gamma, (wl.OUTFLOW,) * 6)
        if setup:
            setup(Rg)
        Rg.set_spacing(dx, dx, dx)
        Rg.set_padded(np.ascontiguousarray(pre[:, k0:k0 + kn + 2 * g]))
        Rg.step(dt)
        ur[:, k0:k0 + kn] = Rg.get_state()
        del Rg
    return post, ur, dt


def test_whole_grid_parity_256_sweep(ref):
    """north_star's one-step gate at a size the metric is quoted on, on ALL 256^3 cells x 5 fields of the
    throughput-sweep workload (BASELINE.json config 5), after two steps so the state is not the analytic one.
    Density and energy are gated with no floor in the denominator (strictly positive fields)."""
    w = wl.sweep(256)
    post, ur, _ = whole_grid_one_step(ref, w, pre_steps=2)
    assert post.shape == (5, 256, 256, 256)
    err = max_rel_error(post, ur, w.gamma)
    strict = max_rel_error_strict(post, ur, w.gamma)
    print("whole-grid 256^3 sweep: S11 norm", err, "strict", strict)
    assert max(err) <= ONE_STEP_TOL, err
    assert max(strict) <= ONE_STEP_TOL, strict


# the paper's other method choices on every cell of the 256^3 grid
METHODS_256 = {
    "ppmc_roe": (3, lambda G: G.set_solver(1)),
    "plmc_exact": (3, lambda G: G.set_reconstruction(1)),
    "plmc_roe": (3, lambda G: (G.set_solver(1), G.set_reconstruction(1))),
    "plmp_exact": (3, lambda G: G.set_reconstruction(4)),
    "ppmp_exact": (4, lambda G: G.set_reconstruction(3)),
}


@pytest.mark.parametrize("name", sorted(METHODS_256))
def test_whole_grid_parity_256_other_methods(ref, name):
    """Every cell of the 256^3 throughput-sweep grid after one GPU step with each of the paper's other reconstructions
    and with the Roe + HLLE solver, in the launch configuration bench.py times them in."""
    g, setup = METHODS_256[name]
    w = wl.sweep(256)
    post, ur, _ = whole_grid_one_step(ref, w, pre_steps=1, g=g, setup=setup)
    err = max_rel_error(post, ur, w.gamma)
    strict = max_rel_error_strict(post, ur, w.gamma)
    print(f"whole-grid 256^3 sweep, {name}: S11 norm", err, "strict", strict)
    assert max(err) <= ONE_STEP_TOL, (name, err)
    assert max(strict) <= ONE_STEP_TOL, (name, strict)


@pytest.mark.parametrize("n", [384, 512])
def test_whole_grid_parity_at_the_largest_sizes(ref, n):
    """Every cell of the 384^3 and the 512^3 grid (the size bench.py times; 1.3e8 cells x 5 fields) after one GPU
    step, in the launch configuration the bench uses, against the oracle re-stepping the grid in 32-plane slabs
    (about a minute of the box's host cores at 512^3)."""
    w = wl.sweep(n)
    post, ur, _ = whole_grid_one_step(ref, w, pre_steps=1)
    assert post.shape == (5, n, n, n)
    err = max_rel_error(post, ur, w.gamma)
    strict = max_rel_error_strict(post, ur, w.gamma)
    print(f"whole-grid {n}^3 sweep: S11 norm", err, "strict", strict)
    assert max(err) <= ONE_STEP_TOL, err
    assert max(strict) <= ONE_STEP_TOL, strict


def test_whole_grid_parity_256_shock_cloud(ref):
    """The same on BASELINE.json config 4 (Mach-50 shock + lognormal cloud, outflow faces): every cell of the
    256^3 grid, after five steps (the front has entered fresh cells).  Gate in the S11 norm; the floor-free figure
    for density and energy is printed (cold ambient cells beside the Mach-50 front lose digits to the size of the
    fluxes that pass through them, in the oracle as much as on the GPU)."""
    w = wl.shock_cloud(256)
    post, ur, _ = whole_grid_one_step(ref, w, pre_steps=5)
    err = max_rel_error(post, ur, w.gamma)
    print("whole-grid 256^3 shock-cloud: S11 norm", err, "strict", max_rel_error_strict(post, ur, w.gamma))
    assert max(err) <= ONE_STEP_TOL, err
    assert post[0].min() > 0


def test_whole_grid_parity_256_shock_cloud_h_correction(ref):
    """The H-corrected step (Roe solver + Appendix C, four ghost layers) in its fused form (k_eta + the TMA kernel
    with C2's maxima taken from the staged eta planes) on every cell of the Mach-50 shock-cloud grid: the
    grid-aligned strong shock is what the correction is for."""
    w = wl.shock_cloud(256)

    def hc(G):
        G.set_solver(1); G.set_hcorrection(True)
    post, ur, _ = whole_grid_one_step(ref, w, pre_steps=5, g=4, setup=hc, want_tma=1)
    err = max_rel_error(post, ur, w.gamma)
    print("whole-grid 256^3 shock-cloud, H correction: S11 norm", err, "strict", max_rel_error_strict(post, ur, w.gamma))
    assert max(err) <= ONE_STEP_TOL, err
    assert post[0].min() > 0


@pytest.mark.parametrize("n", [128, 256, 384, 512])
def test_sweep_full_size_sampled_parity_and_conservation(ref, n):
    """Throughput-sweep workload (BASELINE.json config 5) at the sizes the metric is quoted on."""
    w = wl.sweep(n)
    worst, post, _ = sampled_one_step(ref, w)
    assert worst <= ONE_STEP_TOL, worst
    for f in range(5):
        s0, s1 = float(np.sum(w.u[f], dtype=np.longdouble)), float(np.sum(post[f], dtype=np.longdouble))
        scale = float(np.sum(np.abs(w.u[f]), dtype=np.longdouble)) + (w.u[0].size if f in (1, 2, 3) else 0)
        assert abs(s1 - s0) <= 1e-13 * scale, (f, s0, s1)


def test_shock_cloud_256_sampled_parity(ref):
    """BASELINE.json config 4 at full size: one step, sub-boxes on the shock front and in the cloud."""
    w = wl.shock_cloud(256)
    worst, post, _ = sampled_one_step(ref, w, extra=10, seed=4)
    assert worst <= ONE_STEP_TOL, worst
    assert np.all(np.isfinite(post)) and post[0].min() > 0


def test_sedov_128_sampled_parity(ref):
    """BASELINE.json config 3 at full size: one step; the centre sub-box holds the hot cells."""
    w = wl.sedov(128)
    nx = 128
    import paper_1410_4194_b200 as ch
    worst, post, dt = sampled_one_step(ref, w, extra=4, seed=3)
    assert worst <= ONE_STEP_TOL, worst
    # the blast centre itself
    g, m, o = 3, 16, 56
    G = ch.Grid(nx, nx, nx, g, w.gamma, w.bc)
    G.set_state(w.u)
    pre = G.get_padded()
    G.step(dt)
    ug = G.get_state()[:, o:o + m, o:o + m, o:o + m]
    G.close()
    Rg = ref.RefGrid(m, m, m, g, w.gamma, (wl.OUTFLOW,) * 6)
    Rg.set_spacing(1.0 / nx, 1.0 / nx, 1.0 / nx)
    Rg.set_padded(pre[:, o:o + m + 2 * g, o:o + m + 2 * g, o:o + m + 2 * g])
    Rg.step(dt)
    assert max(max_rel_error(ug, Rg.get_state(), w.gamma)) <= ONE_STEP_TOL


def test_kelvin_helmholtz_256_200_steps(ref):
    """BASELINE.json config 2 in full: 256^2, 200 steps at CFL 0.4, lock-step and free-running."""
    import paper_1410_4194_b200 as ch
    w = wl.kelvin_helmholtz(256, steps=200)
    Rg = ref.RefGrid(256, 256, 1, 3, w.gamma, w.bc)
    dts = []
    run(Rg, w, record_dts=dts)
    ur = Rg.get_state()
    G = ch.Grid(256, 256, 1, 3, w.gamma, w.bc)
    run(G, w, dts=dts)
    e_lock = rel_l1_error(G.get_state(), ur, w.gamma)
    run(G, w)
    e_free = rel_l1_error(G.get_state(), ur, w.gamma)
    G.close()
    assert max(e_lock) <= RUN_L1_TOL, e_lock
    assert max(e_free) <= RUN_L1_TOL, e_free


def test_sedov_128_full_run_reaches_the_sedov_taylor_radius():
    """BASELINE.json config 3 in full on the GPU (the oracle cannot run ~2000 steps of 128^3): ambient rho = 1,
    E = 1 in the 160 central cells, run until the closed form R = 1.15 (E t^2 / rho)^(1/5) says 0.4
    (t = 0.071352).  The shell-averaged density's outer half-rise radius must sit within 1.5 cells of it, the
    blast must stay octant-symmetric, and total energy is conserved while the shock is inside the box."""
    import paper_1410_4194_b200 as ch
    n = 128
    w = wl.sedov(n)
    dx = 1.0 / n
    G = ch.Grid(n, n, n, 3, w.gamma, w.bc)
    steps, t = run(G, w)
    u = G.get_state()
    G.close()
    assert abs(t - w.t_end) < 1e-12 and steps > 500
    rho = u[0]
    c = (np.arange(n) + 0.5) * dx - 0.5
    r = np.sqrt(c[None, None, :] ** 2 + c[None, :, None] ** 2 + c[:, None, None] ** 2)
    bins = np.arange(0, 0.5, dx)
    which = np.digitize(r.ravel(), bins)
    prof = np.array([rho.ravel()[which == b].mean() for b in range(1, len(bins))])
    rc = 0.5 * (bins[1:] + bins[:-1])
    half = 0.5 * (prof.max() + 1.0)
    i = np.max(np.nonzero(prof > half)[0])
    r_half = rc[i] + (prof[i] - half) / (prof[i] - prof[i + 1]) * dx
    want = 1.15 * (t * t) ** 0.2
    assert abs(want - 0.4) < 1e-4
    assert abs(r_half - want) <= 1.5 * dx, (r_half, want, steps)
    assert prof.max() > 2.5                                           # compression toward (g+1)/(g-1) = 4
    assert np.allclose(rho, rho[::-1, :, :], rtol=1e-8) and np.allclose(rho, rho.transpose(2, 1, 0), rtol=1e-8)
    e_tot = math.fsum(u[4].ravel()) * dx ** 3
    assert abs(e_tot - (1.0 + 1e-5 / (w.gamma - 1) * (1 - 160 * dx ** 3))) < 1e-8


def test_shock_cloud_256_500_steps_stays_physical():
    """BASELINE.json config 4 in full on the GPU: 500 steps at CFL 0.3.  The Mach-50 shock must have advanced
    at the Rankine-Hugoniot speed (204.124 in code units) through the part of the box it has not yet reached
    the cloud in, density and pressure stay positive everywhere, no non-physical cell is reported."""
    import paper_1410_4194_b200 as ch
    w = wl.shock_cloud(256)
    G = ch.Grid(*w.shape, 3, w.gamma, w.bc)
    steps, t = run(G, w)
    assert steps == 500
    dt_next = G.compute_dt(w.cfl)
    u = G.get_state()
    G.close()
    assert math.isfinite(dt_next) and dt_next > 0
    rho = u[0]
    p = (w.gamma - 1) * (u[4] - 0.5 * (u[1] ** 2 + u[2] ** 2 + u[3] ** 2) / rho)
    assert np.all(np.isfinite(u)) and rho.min() > 0 and p.min() > 0
    # shock position along a line far from the cloud (y = z = 8 cells from the corner): first cell from the +x
    # side whose density exceeds twice the ambient value
    line = rho[8, 8, :]
    front = np.max(np.nonzero(line > 0.2)[0]) + 1
    want = 16 + 204.12414523 * t * 256
    assert abs(front - want) <= 2.5, (front, want, t)


def test_sweep_128_100_steps_match_the_oracle(ref):
    """BASELINE.json config 5 as it is stated — 100 steps at CFL 0.4 — at the size the oracle can run in full
    (128^3, ~90 s of the box's host cores): relative L1 per field <= 1e-8 at the end, lock-step (the oracle's dt fed
    to the GPU) and free-running (its own Eq. 22 every step), and the two clocks agree."""
    import paper_1410_4194_b200 as ch
    w = wl.sweep(128)
    w.steps = 100
    Rg = ref.RefGrid(128, 128, 128, 3, w.gamma, w.bc)
    dts = []
    run(Rg, w, record_dts=dts)
    ur = Rg.get_state()
    G = ch.Grid(128, 128, 128, 3, w.gamma, w.bc)
    run(G, w, dts=dts)
    e_lock = rel_l1_error(G.get_state(), ur, w.gamma)
    gdts = []
    run(G, w, record_dts=gdts)
    e_free = rel_l1_error(G.get_state(), ur, w.gamma)
    G.close()
    print("sweep 128^3 x 100 steps: rel L1 lock-step", e_lock, "free-running", e_free)
    assert len(dts) == 100 and max(e_lock) <= RUN_L1_TOL and max(e_free) <= RUN_L1_TOL
    assert np.allclose(gdts, dts, rtol=1e-9, atol=0)
