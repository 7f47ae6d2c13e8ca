"""Error norms used by the GPU-vs-oracle parity tests (numpy only; none of the method's arithmetic
beyond the definitions of the natural field scales, reading S11).

per-cell relative error of field f:  |gpu - ref| / max(|ref|, s_f)  where s_f is the grid RMS of the
field's natural scale: rho for density, rho(|V| + a) for the momenta, E for the energy.  north_star
gates: one step max <= 1e-12; end of run relative L1 (sum|gpu-ref| / sum|ref|, momenta against
sum rho(|V|+a)) <= 1e-8 per field.
"""
import numpy as np

ONE_STEP_TOL = 1e-12
RUN_L1_TOL = 1e-8


def field_scales(u, gamma):
    rho = u[0]
    v2 = (u[1] ** 2 + u[2] ** 2 + u[3] ** 2) / rho ** 2
    p = np.maximum((gamma - 1.0) * (u[4] - 0.5 * rho * v2), 1e-20)
    mom = rho * (np.sqrt(v2) + np.sqrt(gamma * p / rho))
    return [rho, mom, mom, mom, u[4]]


def max_rel_error(u_gpu, u_ref, gamma):
    """Max over cells of the S11 per-cell relative error, per field -> list of 5 floats."""
    out = []
    for f, nat in enumerate(field_scales(u_ref, gamma)):
        s = float(np.sqrt(np.mean(nat.astype(np.float64) ** 2)))
        denom = np.maximum(np.abs(u_ref[f]), s)
        out.append(float(np.max(np.abs(u_gpu[f] - u_ref[f]) / denom)))
    return out


def rel_l1_error(u_gpu, u_ref, gamma):
    out = []
    for f, nat in enumerate(field_scales(u_ref, gamma)):
        out.append(float(np.sum(np.abs(u_gpu[f] - u_ref[f])) / np.sum(np.abs(nat))))
    return out
