"""ch_dt_noalloc (`-m gpu`; collected last on purpose: the suite runs with pytest -x).

The entry point computes Eq. 22 of a padded state with its reduction scratch in a file-scope device
array: no context, no workspace, no allocation.  Its output must equal what the existing path (ch_set_state +
ch_compute_dt on a bound Grid) returns for the same state, on two calls in a row (the second call meets the first
call's contents in the shared scratch), on a state that changes between the calls, after a call that met a
non-physical cell, and it must refuse grids beyond its stated maximum.
"""
import math

import numpy as np
import pytest

from paper_1410_4194_b200 import workloads as wl
from tests.parity import ONE_STEP_TOL

pytestmark = pytest.mark.gpu


def grid_dt(ch, w, nghost, dx, cfl):
    """The existing path: a Grid with bound buffers, ch_compute_dt; returns (dt, padded store as a CUDA tensor)."""
    import torch
    G = ch.Grid(*w.shape, nghost, w.gamma, w.bc)
    G.set_spacing(*dx)
    G.set_state(w.u)
    dt = G.compute_dt(cfl)
    padded = torch.from_numpy(np.ascontiguousarray(G.get_padded())).cuda()
    G.close()
    return dt, padded


@pytest.mark.parametrize("maker,nghost", [(lambda: wl.sweep(shape=(70, 45, 37)), 3),      # ragged last CTA
                                          (lambda: wl.sedov(40), 3),
                                          (lambda: wl.kelvin_helmholtz(64), 4),           # inactive z
                                          (lambda: wl.sod(128), 3)])                      # 1-D, less than one CTA
def test_dt_noalloc_equals_compute_dt_on_two_calls_in_a_row(maker, nghost):
    import torch
    import paper_1410_4194_b200 as ch
    from paper_1410_4194_b200 import binding
    w = maker()
    nx, ny, nz = w.shape
    dx = (1.0 / nx, 1.3 / nx, 0.9 / nx)
    want, padded = grid_dt(ch, w, nghost, dx, w.cfl)
    out = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    mem0 = torch.cuda.memory_allocated()
    got = []
    for _ in range(2):                                   # the second call finds the first one's partials and flag
        binding.dt_noalloc(padded, nx, ny, nz, nghost, w.gamma, *dx, w.cfl, out)
        got.append(float(out.item()))
        out.fill_(-1.0)
    assert torch.cuda.memory_allocated() == mem0         # torch's allocator was not asked for anything
    for g in got:
        assert math.isfinite(g) and g > 0
        assert abs(g - want) <= ONE_STEP_TOL * want, (g, want)
    assert got[0] == got[1]

    # a different state through the same scratch: a hotter state (smaller dt), then the first one again
    w2 = maker()
    w2.u[4] *= 4.0                                        # hotter gas: larger sound speed everywhere
    want2, padded2 = grid_dt(ch, w2, nghost, dx, w.cfl)
    binding.dt_noalloc(padded2, nx, ny, nz, nghost, w.gamma, *dx, w.cfl, out)
    g2 = float(out.item())
    assert abs(g2 - want2) <= ONE_STEP_TOL * want2 and g2 < want
    binding.dt_noalloc(padded, nx, ny, nz, nghost, w.gamma, *dx, w.cfl, out)
    assert abs(float(out.item()) - want) <= ONE_STEP_TOL * want      # stale larger maxima did not survive


def test_dt_noalloc_flags_a_non_physical_cell_and_clears_the_flag_for_the_next_call():
    import torch
    import paper_1410_4194_b200 as ch
    from paper_1410_4194_b200 import binding
    w = wl.sweep(shape=(33, 20, 17))
    nx, ny, nz = w.shape
    dx = (1.0 / nx,) * 3
    want, padded = grid_dt(ch, w, 3, dx, w.cfl)
    bad = padded.clone()
    bad.view(5, nz + 6, ny + 6, nx + 6)[0, 3 + 5, 3 + 4, 3 + 7] = -1.0            # a real cell with rho < 0
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    binding.dt_noalloc(bad, nx, ny, nz, 3, w.gamma, *dx, w.cfl, out)
    assert math.isnan(float(out.item()))
    binding.dt_noalloc(padded, nx, ny, nz, 3, w.gamma, *dx, w.cfl, out)           # the flag must start at zero again
    assert abs(float(out.item()) - want) <= ONE_STEP_TOL * want
    # a ghost cell is not a real cell: garbage there changes nothing
    ghost = padded.clone()
    ghost.view(5, nz + 6, ny + 6, nx + 6)[:, 0, 0, 0] = float("nan")
    binding.dt_noalloc(ghost, nx, ny, nz, 3, w.gamma, *dx, w.cfl, out)
    assert abs(float(out.item()) - want) <= ONE_STEP_TOL * want


def test_dt_noalloc_refuses_sizes_beyond_its_scratch_and_bad_arguments():
    import torch
    from paper_1410_4194_b200 import binding
    assert binding.noalloc_max_cells() == 256 ** 3
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    tiny = torch.zeros(8, dtype=torch.float64, device="cuda")                     # never read: the size check comes first
    with pytest.raises(ValueError, match="16777216"):
        binding.dt_noalloc(tiny, 257, 256, 256, 3, 1.4, 1.0, 1.0, 1.0, 0.4, out)
    with pytest.raises(ValueError):
        binding.dt_noalloc(tiny, 16, 16, 16, 2, 1.4, 1.0, 1.0, 1.0, 0.4, out)     # nghost < 3
    with pytest.raises(ValueError):
        binding.dt_noalloc(tiny, 16, 16, 16, 3, 1.4, 1.0, 1.0, 1.0, 1.5, out)     # cfl > 1
    with pytest.raises(ValueError):
        binding.dt_noalloc(tiny, 16, 16, 16, 3, 1.4, 0.0, 1.0, 1.0, 0.4, out)     # dx = 0
    assert float(out.item()) == 0.0


def test_dt_noalloc_at_its_largest_size():
    """256^3, the stated maximum (65536 partial maxima): against ch_compute_dt on the same state."""
    import torch
    import paper_1410_4194_b200 as ch
    from paper_1410_4194_b200 import binding
    w = wl.sweep(256)
    dx = (1.0 / 256,) * 3
    G = ch.Grid(256, 256, 256, 3, w.gamma, w.bc)
    G.set_state(w.u)
    want = G.compute_dt(w.cfl)
    padded = torch.from_numpy(G.get_padded()).cuda()
    G.close()
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    for _ in range(2):
        binding.dt_noalloc(padded, 256, 256, 256, 3, w.gamma, *dx, w.cfl, out)
        assert abs(float(out.item()) - want) <= ONE_STEP_TOL * want
