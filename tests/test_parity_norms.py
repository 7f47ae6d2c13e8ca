"""The parity norms themselves (tests/parity.py), `-m "not gpu"`: a wrong state must never pass a gate through a
NaN (python's max() skips NaN), and the strict norm has no floor on the strictly positive fields."""
import numpy as np
import pytest

from paper_1410_4194_b200 import workloads as wl
from tests.parity import ONE_STEP_TOL, max_rel_error, max_rel_error_strict, rel_l1_error, within


def state():
    return wl.sweep(shape=(12, 10, 8))


def test_doubled_momenta_fail_every_norm():
    w = state()
    bad = w.u.copy()
    bad[1:4] *= 2.0
    for fn in (max_rel_error, max_rel_error_strict, rel_l1_error):
        err = fn(bad, w.u, w.gamma)
        assert err[0] == 0.0 and err[4] == 0.0
        assert min(err[1:4]) > 1e-3 and not within(err, ONE_STEP_TOL)


def test_non_physical_reference_is_refused():
    w = state()
    ref = w.u.copy()
    ref[0, 3, 4, 5] = -0.175           # what the oracle's Mach-3, +-1-decade 1-D step produces in one cell
    gpu = ref.copy()
    gpu[1:4] *= 2.0
    for fn in (max_rel_error, max_rel_error_strict, rel_l1_error):
        with pytest.raises(AssertionError):
            fn(gpu, ref, w.gamma)


def test_nan_on_either_side_is_refused():
    w = state()
    for side in (0, 1):
        a, b = w.u.copy(), w.u.copy()
        (a if side == 0 else b)[2, 1, 1, 1] = np.nan
        for fn in (max_rel_error, max_rel_error_strict, rel_l1_error):
            with pytest.raises(AssertionError):
                fn(a, b, w.gamma)


def test_within_never_lets_nan_through():
    assert within([0.0, 1e-13], ONE_STEP_TOL)
    assert not within([0.0, float("nan"), 0.0], ONE_STEP_TOL)
    assert not within([2e-12], ONE_STEP_TOL)


def test_strict_norm_has_no_floor_on_density_and_energy():
    """A cold cell (E tiny against the grid RMS) wrong by 1e-5 relative passes the floored norm and fails the
    strict one: the floored gate alone is an absolute gate there."""
    w = state()
    ref = w.u.copy()
    ref[4, 2, 2, 2] = 1.5e-5 + 0.5 * (ref[1, 2, 2, 2] ** 2 + ref[2, 2, 2, 2] ** 2 + ref[3, 2, 2, 2] ** 2) / ref[0, 2, 2, 2]
    ref[4] *= 1.0
    big = ref.copy()
    big[4, 0, 0, 0] = 1e4                        # a hot cell sets the RMS
    gpu = big.copy()
    gpu[4, 2, 2, 2] *= 1.0 + 1e-5
    assert max_rel_error(gpu, big, w.gamma)[4] < 1e-9
    assert max_rel_error_strict(gpu, big, w.gamma)[4] > 5e-6
