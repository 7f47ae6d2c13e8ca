"""Seeded synthetic inputs (initial conditions) for the workloads BASELINE.json names.

This module serves BOTH the CUDA path and the oracle and therefore holds none of the method's
arithmetic: it only writes initial data (primitive fields -> the conserved vector of Eq. 9,
P:L65, with E from Eq. 6-8) as numpy arrays `u[5][nz][ny][nx]`, field order
rho, rho*u, rho*v, rho*w, E, x fastest.  numpy only; imports neither the CUDA binding nor oracle/.

Box: x in [0,1], cubic cells of width 1/nx, cell centres (i+1/2)/nx (reading S8).
Every generator returns a `Workload` (state + boundary codes + gamma + CFL + run length).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

PERIODIC, REFLECTIVE, OUTFLOW, NOH = 1, 2, 3, 4      # 4: the analytic inflow boundary of the Noh test


@dataclass
class Workload:
    name: str
    u: np.ndarray                 # [5][nz][ny][nx] conserved
    gamma: float
    bc: tuple                     # (x-, x+, y-, y+, z-, z+)
    cfl: float
    steps: int | None = None      # fixed step count, or
    t_end: float | None = None    # run to this time (last dt clipped)
    meta: dict = field(default_factory=dict)

    @property
    def shape(self):              # (nx, ny, nz)
        return self.u.shape[3], self.u.shape[2], self.u.shape[1]


def conserved(rho, vx, vy, vz, p, gamma) -> np.ndarray:
    """Primitive fields -> conserved vector (Eq. 6-9)."""
    rho, vx, vy, vz, p = np.broadcast_arrays(*(np.asarray(a, dtype=np.float64) for a in (rho, vx, vy, vz, p)))
    u = np.empty((5,) + rho.shape, dtype=np.float64)
    u[0] = rho
    u[1] = rho * vx
    u[2] = rho * vy
    u[3] = rho * vz
    u[4] = p / (gamma - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz)
    return u


def centres(nx, ny, nz):
    """Cell-centre coordinates as broadcastable [nz,1,1],[1,ny,1],[1,1,nx] arrays (x,y,z order returned)."""
    d = 1.0 / nx
    x = ((np.arange(nx) + 0.5) * d).reshape(1, 1, nx)
    y = ((np.arange(ny) + 0.5) * d).reshape(1, ny, 1)
    z = ((np.arange(nz) + 0.5) * d).reshape(nz, 1, 1)
    return x, y, z


# ---- config 1: Sod shock tube (stands for P:L447-451; BASELINE.json ICs, reading S12) --------
def sod(nx=128, axis=0, n_other=1) -> Workload:
    gamma = 1.4
    shape = [n_other, n_other, n_other]
    shape[2 - axis] = nx
    s = ((np.arange(nx) + 0.5) / nx)
    view = [1, 1, 1]
    view[2 - axis] = nx
    s = s.reshape(view)
    left = np.broadcast_to(s < 0.5, shape)
    rho = np.where(left, 1.0, 0.125)
    p = np.where(left, 1.0, 0.1)
    zero = np.zeros(shape)
    bc = (OUTFLOW,) * 6 if n_other == 1 else tuple(OUTFLOW if d == axis else PERIODIC for d in range(3) for _ in range(2))
    return Workload("sod", conserved(rho, zero, zero, zero, p, gamma), gamma, bc, 0.4, t_end=0.2)


# ---- Noh's strong shock (section 4.3.1; the consumer of the custom boundary and the H correction) ----
def noh(n=64, dims=3, t_end=2.0, shape=None, rho0=1.0, p0=1e-6, cfl=0.4) -> Workload:
    """Octant [0,1]^dims: rho = rho0, p = p0, unit velocity toward the origin; reflecting inner faces, analytic
    (NOH) outer faces; gamma = 5/3.  `shape` overrides (n, dims) with an explicit (nx, ny, nz); dimensions of
    size 1 are inactive."""
    gamma = 5.0 / 3.0
    if shape is None:
        shape = tuple(n if d < dims else 1 for d in range(3))
    nx, ny, nz = shape
    x, y, z = centres(nx, ny, nz)
    x = x if nx > 1 else np.zeros((1, 1, 1))
    y = y if ny > 1 else np.zeros((1, 1, 1))
    z = z if nz > 1 else np.zeros((1, 1, 1))
    X, Y, Z = np.broadcast_arrays(x, y, z)
    X, Y, Z = (np.broadcast_to(a, (nz, ny, nx)) for a in (X, Y, Z))
    r = np.sqrt(X * X + Y * Y + Z * Z)
    rho = np.full((nz, ny, nx), rho0)
    u = conserved(rho, -X / r, -Y / r, -Z / r, np.full((nz, ny, nx), p0), gamma)
    bc = (REFLECTIVE, NOH) * 3
    return Workload("noh", u, gamma, bc, cfl, t_end=t_end, meta={"rho0": rho0, "p0": p0})


# ---- config 2: Kelvin-Helmholtz (stands for P:L535-541) --------------------------------------
def kelvin_helmholtz(n=256, seed=1410, steps=200) -> Workload:
    gamma = 1.4
    x, y, z = centres(n, n, 1)
    inner = np.broadcast_to(np.abs(y - 0.5) < 0.25, (1, n, n))
    rho = np.where(inner, 2.0, 1.0)
    vx = np.where(inner, 0.5, -0.5)
    rng = np.random.default_rng(seed)
    vy = rng.uniform(-0.01, 0.01, size=(1, n, n))      # array order [j][i]
    u = conserved(rho, vx, vy, 0.0, 2.5, gamma)
    return Workload("kelvin_helmholtz", u, gamma, (PERIODIC,) * 6, 0.4, steps=steps)


# ---- config 3: Sedov-Taylor blast (not in the paper; BASELINE.json config 3) -----------------
def sedov(n=128, octant=False, r_cells=3.5) -> Workload:
    """Full box [0,1]^3 with outflow faces, or (octant=True) the +++ octant of a 2n box with
    reflective low faces — same cell width 1/(2n)·... see meta['dx']."""
    gamma = 5.0 / 3.0
    if octant:
        # octant of a box with N=2n cells per side: centre at the low corner, dx = 1/(2n)
        dx = 1.0 / (2 * n)
        c = (np.arange(n) + 0.5) * dx
        X, Y, Z = c.reshape(1, 1, n), c.reshape(1, n, 1), c.reshape(n, 1, 1)
        r = np.sqrt(X * X + Y * Y + Z * Z)
        bc = (REFLECTIVE, OUTFLOW) * 3
    else:
        dx = 1.0 / n
        X, Y, Z = centres(n, n, n)
        r = np.sqrt((X - 0.5) ** 2 + (Y - 0.5) ** 2 + (Z - 0.5) ** 2)
        bc = (OUTFLOW,) * 6
    hot = r < r_cells * dx
    ncell = int(hot.sum()) * (8 if octant else 1)
    e = 1.0 / (ncell * dx ** 3)                       # total energy E=1 as uniform internal energy
    p = np.where(hot, (gamma - 1.0) * e, 1e-5)
    u = conserved(1.0, 0.0, 0.0, 0.0, p, gamma)
    return Workload("sedov", u, gamma, bc, 0.4, t_end=0.071352,
                    meta=dict(dx=dx, hot_cells=ncell, octant=octant))


# ---- config 4: shock / turbulent cloud (synthetic stand-in for P:L567-610) -------------------
def gaussian_random_field(n, seed, slope=-11.0 / 3.0):
    """Gaussian random field on n^3 with P(k) ∝ k^slope: white noise -> FFT -> |k|^(slope/2) -> inverse."""
    rng = np.random.default_rng(seed)
    white = rng.standard_normal((n, n, n))
    wk = np.fft.rfftn(white)
    k1 = np.fft.fftfreq(n) * n
    kr = np.fft.rfftfreq(n) * n
    kk = np.sqrt(k1.reshape(n, 1, 1) ** 2 + k1.reshape(1, n, 1) ** 2 + kr.reshape(1, 1, -1) ** 2)
    amp = np.zeros_like(kk)
    nz = kk > 0
    amp[nz] = kk[nz] ** (slope / 2.0)
    return np.fft.irfftn(wk * amp, s=(n, n, n))


def shock_cloud(n=256, seed=4194, steps=500, mach=50.0, sigma=1.0) -> Workload:
    gamma = 5.0 / 3.0
    rho0, p0 = 0.1, 1.0
    s = n / 256.0
    dx = 1.0 / n
    X, Y, Z = centres(n, n, n)
    cx, cy, cz = 80.0 * s * dx, 128.0 * s * dx, 128.0 * s * dx
    cloud = np.sqrt((X - cx) ** 2 + (Y - cy) ** 2 + (Z - cz) ** 2) < 32.0 * s * dx
    g = gaussian_random_field(n, seed)
    gc = g[cloud]
    g = (g - gc.mean()) / gc.std()
    rho_c = np.exp(sigma * g - 0.5 * sigma * sigma)
    for _ in range(3):                                   # rescale to mean 10x ambient, floor at ambient
        rho_c = rho_c * (10.0 * rho0 / rho_c[cloud].mean())
        rho_c = np.maximum(rho_c, rho0)
    rho = np.where(cloud, rho_c, rho0)
    # Rankine-Hugoniot post-shock state for a Mach `mach` shock moving in +x into (rho0, p0, 0)
    a0 = np.sqrt(gamma * p0 / rho0)
    m2 = mach * mach
    r1 = rho0 * (gamma + 1.0) * m2 / ((gamma - 1.0) * m2 + 2.0)
    p1 = p0 * (2.0 * gamma * m2 - (gamma - 1.0)) / (gamma + 1.0)
    vs = mach * a0
    v1 = vs * (1.0 - rho0 / r1)
    post = np.broadcast_to(X < 16.0 * s * dx, (n, n, n))
    rho = np.where(post, r1, rho)
    vx = np.where(post, v1, 0.0)
    p = np.where(post, p1, p0)
    u = conserved(rho, vx, 0.0, 0.0, p, gamma)
    return Workload("shock_cloud", u, gamma, (OUTFLOW,) * 6, 0.3, steps=steps,
                    meta=dict(post=(r1, v1, p1), shock_speed=vs))


# ---- config 5: throughput sweep (stands for the 3-D sound-wave workload) -------------
def _sinusoid_sum(nx, ny, nz, seed):
    rng = np.random.default_rng(seed)
    cand = np.array([(a, b, c) for a in range(-8, 9) for b in range(-8, 9) for c in range(-8, 9)
                     if 1 <= a * a + b * b + c * c <= 64])
    ks = cand[rng.integers(0, len(cand), size=8)]
    ph = rng.uniform(0.0, 2.0 * np.pi, size=8)
    # unit box in every direction for this workload: coordinates (i+1/2)/n_d so the field is periodic.
    # sin(tx + ty + tz + ph) = sin(tx+ty+ph) cos(tz) + cos(tx+ty+ph) sin(tz): the sum over the 8 modes
    # is one [nz,16] x [16,ny*nx] product (keeps 512^3 generation to seconds).
    x = ((np.arange(nx) + 0.5) / nx).reshape(1, 1, nx)
    y = ((np.arange(ny) + 0.5) / ny).reshape(1, ny, 1)
    z = ((np.arange(nz) + 0.5) / nz).reshape(nz, 1)
    kx, ky, kz = (ks[:, d].astype(np.float64).reshape(8, 1, 1) for d in range(3))
    txy = 2.0 * np.pi * (kx * x + ky * y) + ph.reshape(8, 1, 1)           # [8,ny,nx]
    tz = 2.0 * np.pi * z * kz.reshape(1, 8)                                  # [nz,8]
    A = np.concatenate([np.cos(tz), np.sin(tz)], axis=1)                    # [nz,16]
    B = np.concatenate([np.sin(txy), np.cos(txy)], axis=0).reshape(16, ny * nx)
    return (A @ B).reshape(nz, ny, nx) / 8.0


def sweep(n=256, steps=100, shape=None) -> Workload:
    gamma = 5.0 / 3.0
    nx, ny, nz = shape if shape is not None else (n, n, n)
    rho = 1.0 + 0.1 * _sinusoid_sum(nx, ny, nz, 41940)
    vx = 0.1 * _sinusoid_sum(nx, ny, nz, 41941)
    vy = 0.1 * _sinusoid_sum(nx, ny, nz, 41942)
    vz = 0.1 * _sinusoid_sum(nx, ny, nz, 41943)
    u = conserved(rho, vx, vy, vz, 1.0, gamma)
    return Workload("sweep", u, gamma, (PERIODIC,) * 6, 0.4, steps=steps)


# ---- extra inputs used by the pins -------------------------------------------------------------
def linear_wave(nx, ny=1, nz=1, amp=1e-6, kvec=(1, 0, 0)) -> Workload:
    """Right-going sound wave on rho0=1, p0=1/gamma (a0=1), gamma=5/3 (P:L445 names the test only)."""
    gamma = 5.0 / 3.0
    x = ((np.arange(nx) + 0.5) / nx).reshape(1, 1, nx)
    y = ((np.arange(ny) + 0.5) / nx).reshape(1, ny, 1)
    z = ((np.arange(nz) + 0.5) / nx).reshape(nz, 1, 1)
    k = np.asarray(kvec, dtype=np.float64)
    khat = k / np.linalg.norm(k)
    phase = 2.0 * np.pi * (k[0] * x + k[1] * y + k[2] * z)
    s = amp * np.sin(phase) * np.ones((nz, ny, nx))
    u = conserved(1.0 + s, khat[0] * s, khat[1] * s, khat[2] * s, 1.0 / gamma + s, gamma)
    return Workload("linear_wave", u, gamma, (PERIODIC,) * 6, 0.4, t_end=1.0 / np.linalg.norm(k),
                    meta=dict(amp=amp))


def riemann_tube(nx, left, right, gamma=1.4, t_end=0.2, x0=0.5) -> Workload:
    """1-D Riemann problem (rho,u,p) left/right of x0, outflow ends."""
    s = ((np.arange(nx) + 0.5) / nx).reshape(1, 1, nx)
    L = s < x0
    rho = np.where(L, left[0], right[0])
    vx = np.where(L, left[1], right[1])
    p = np.where(L, left[2], right[2])
    return Workload("riemann_tube", conserved(rho, vx, 0.0, 0.0, p, gamma), gamma, (OUTFLOW,) * 6, 0.4, t_end=t_end)


def smooth_random(nx, ny=1, nz=1, seed=0, gamma=5.0 / 3.0, amp=0.2, bc=(PERIODIC,) * 6, steps=1, cfl=0.4) -> Workload:
    """Seeded smooth state of O(1) density/pressure with `amp`-sized variations in every primitive
    field (three random low-|k| sinusoids each): the generic parity-test input, any grid shape."""
    rng = np.random.default_rng(seed)
    x = ((np.arange(nx) + 0.5) / nx).reshape(1, 1, nx)
    y = ((np.arange(ny) + 0.5) / ny).reshape(1, ny, 1)
    z = ((np.arange(nz) + 0.5) / nz).reshape(nz, 1, 1)

    def f():
        out = np.zeros((nz, ny, nx))
        for _ in range(3):
            k = rng.integers(-2, 3, 3)
            ph = rng.uniform(0.0, 2.0 * np.pi)
            out += np.sin(2.0 * np.pi * (k[0] * x + k[1] * y + k[2] * z) + ph)
        return out / 3.0

    u = conserved(1.0 + amp * f(), amp * f(), amp * f(), amp * f(), 1.0 + amp * f(), gamma)
    return Workload("smooth_random", u, gamma, tuple(bc), cfl, steps=steps)


def rough_random(nx, ny=1, nz=1, seed=0, gamma=1.4, mach=2.0, bc=(OUTFLOW,) * 6, steps=1, cfl=0.3,
                 decades=1.0) -> Workload:
    """Seeded cell-wise random state (log-uniform density and pressure over 2*`decades` decades,
    velocities up to `mach` sound speeds): every interface is a strong Riemann problem, so every
    sampling branch, limiter branch and many Newton iteration counts are exercised in one step.
    In 2-D/3-D use decades <= 0.5: with cell-to-cell density ratios of 100 the Eq. 23 transverse
    correction drives face densities negative (the method has no fallback for that) and the
    step is undefined for oracle and GPU alike."""
    rng = np.random.default_rng(seed)
    shp = (nz, ny, nx)
    rho = 10.0 ** rng.uniform(-decades, decades, shp)
    p = 10.0 ** rng.uniform(-decades, decades, shp)
    a = np.sqrt(gamma * p / rho)
    v = [mach * a * rng.uniform(-1.0, 1.0, shp) for _ in range(3)]
    u = conserved(rho, v[0], v[1], v[2], p, gamma)
    return Workload("rough_random", u, gamma, tuple(bc), cfl, steps=steps)
