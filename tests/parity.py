"""Error norms used by the GPU-vs-oracle parity tests (numpy only; none of the method's arithmetic
beyond the definitions of the natural field scales, reading S11).

per-cell relative error of field f:  |gpu - ref| / max(|ref|, s_f)  where s_f is the grid RMS of the
field's natural scale: rho for density, rho(|V| + a) for the momenta, E for the energy.  north_star
gates: one step max <= 1e-12; end of run relative L1 (sum|gpu-ref| / sum|ref|, momenta against
sum rho(|V|+a)) <= 1e-8 per field.

The momenta cross zero, so their denominator is floored at the grid RMS of rho(|V| + a).  Density and
energy are strictly positive: `max_rel_error_strict` gates them with NO floor (|gpu - ref| / |ref|).

A norm is only meaningful on a physical reference state: both functions raise AssertionError if
either state holds a non-finite value or the reference holds rho <= 0 (python's max() silently skips
NaN, so a NaN scale must never reach a comparison).  Cases whose oracle step leaves the physical
regime are tested on what both sides REPORT (CH_ENONPHYS), not with these norms.
"""
import numpy as np

ONE_STEP_TOL = 1e-12
RUN_L1_TOL = 1e-8


def check_physical(u_gpu, u_ref):
    assert np.all(np.isfinite(u_ref)), "oracle state holds non-finite values: no norm is defined on it"
    assert np.all(np.isfinite(u_gpu)), "GPU state holds non-finite values"
    assert np.all(u_ref[0] > 0.0), "oracle state holds rho <= 0: the case has left the physical regime"


def within(err, tol):
    """True iff every entry is a number and <= tol (never lets a NaN through)."""
    return all((e == e) and e <= tol for e in err)


def field_scales(u, gamma):
    rho = u[0]
    v2 = (u[1] ** 2 + u[2] ** 2 + u[3] ** 2) / rho ** 2
    p = np.maximum((gamma - 1.0) * (u[4] - 0.5 * rho * v2), 1e-20)
    mom = rho * (np.sqrt(v2) + np.sqrt(gamma * p / rho))
    return [rho, mom, mom, mom, u[4]]


def max_rel_error(u_gpu, u_ref, gamma):
    """Max over cells of the S11 per-cell relative error, per field -> list of 5 floats."""
    check_physical(u_gpu, u_ref)
    out = []
    for f, nat in enumerate(field_scales(u_ref, gamma)):
        s = float(np.sqrt(np.mean(nat.astype(np.float64) ** 2)))
        assert np.isfinite(s) and s > 0.0, (f, s)
        denom = np.maximum(np.abs(u_ref[f]), s)
        out.append(float(np.max(np.abs(u_gpu[f] - u_ref[f]) / denom)))
    assert not any(np.isnan(out)), out
    return out


def max_rel_error_strict(u_gpu, u_ref, gamma):
    """As max_rel_error, but density and energy (strictly positive fields) are gated per cell against
    |ref| alone, with no RMS floor; the momenta keep the floor because they cross zero."""
    check_physical(u_gpu, u_ref)
    out = max_rel_error(u_gpu, u_ref, gamma)
    for f in (0, 4):
        assert np.all(u_ref[f] > 0.0), f
        out[f] = float(np.max(np.abs(u_gpu[f] - u_ref[f]) / np.abs(u_ref[f])))
    return out


def rel_l1_error(u_gpu, u_ref, gamma):
    check_physical(u_gpu, u_ref)
    out = []
    for f, nat in enumerate(field_scales(u_ref, gamma)):
        out.append(float(np.sum(np.abs(u_gpu[f] - u_ref[f])) / np.sum(np.abs(nat))))
    assert not any(np.isnan(out)), out
    return out
