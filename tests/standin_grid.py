"""A stand-in "grid" for the host-logic tests of paper_1410_4194_b200/decomp.py (`-m "not gpu"`): the call surface
the block drivers use (set_state, halo_cells / halo_pack / halo_unpack, fill_dim, compute_dt, step, get_state) on a
numpy padded array.  Index work only plus a toy update that reads every ghost cell within its radius, corners
included, so that a wrong message, a wrong order of directions or a missing corner changes the result.  It holds none
of the hydro method and exists so that the exchange schedule can run under gloo on CPU."""
import numpy as np
import torch

PERIODIC, REFLECTIVE, OUTFLOW, NOH, EXCHANGE = 1, 2, 3, 4, 5


class StandInGrid:
    def __init__(self, nx, ny, nz, nghost, gamma, bc, device="cpu"):
        self.n = (nx, ny, nz)
        self.g = tuple(nghost if n > 1 else 0 for n in self.n)
        self.bc = tuple(bc)
        self.device = "cpu"
        self.pd = tuple(n + 2 * g for n, g in zip(self.n, self.g))
        self.u = np.zeros((5, self.pd[2], self.pd[1], self.pd[0]))
        self.origin = (0, 0, 0)

    def set_origin(self, i0, j0, k0):
        self.origin = (i0, j0, k0)

    def _real(self):
        gx, gy, gz = self.g
        nx, ny, nz = self.n
        return (slice(None), slice(gz, gz + nz), slice(gy, gy + ny), slice(gx, gx + nx))

    def set_state(self, u):
        self.u[self._real()] = u

    def get_state(self):
        return self.u[self._real()].copy()

    def set_spacing(self, *a):
        pass

    def _slab(self, d, lo, hi):
        """index of layers [lo, hi) (real-cell coordinates) along d; directions before d padded, after d real"""
        idx = [slice(None)] * 4
        for e in range(3):
            ax = 3 - e
            if e == d:
                idx[ax] = slice(lo + self.g[e], hi + self.g[e])
            elif e < d:
                idx[ax] = slice(0, self.pd[e])
            else:
                idx[ax] = slice(self.g[e], self.g[e] + self.n[e])
        return tuple(idx)

    def halo_cells(self, d):
        v = self.u[self._slab(d, 0, self.g[d])]
        return v[0].size

    def halo_pack(self, face, buf):
        d, side = face // 2, face & 1
        g, n = self.g[d], self.n[d]
        v = self.u[self._slab(d, 0, g)] if side == 0 else self.u[self._slab(d, n - g, n)]
        buf.copy_(torch.from_numpy(np.ascontiguousarray(v).ravel()))

    def halo_unpack(self, face, buf):
        d, side = face // 2, face & 1
        g, n = self.g[d], self.n[d]
        sl = self._slab(d, -g, 0) if side == 0 else self._slab(d, n, n + g)
        self.u[sl] = buf.numpy().reshape(self.u[sl].shape)

    def fill_dim(self, d):
        g, n = self.g[d], self.n[d]
        if g == 0:
            return
        for side in (0, 1):
            bc = self.bc[2 * d + side]
            if bc == EXCHANGE:
                continue
            for l in range(1, g + 1):
                gi = -l if side == 0 else n - 1 + l
                if bc == PERIODIC:
                    si = n - l if side == 0 else l - 1
                elif bc == REFLECTIVE:
                    si = l - 1 if side == 0 else n - l
                else:
                    si = 0 if side == 0 else n - 1
                v = self.u[self._slab(d, si, si + 1)].copy()
                if bc == REFLECTIVE:
                    v[1 + d] = -v[1 + d]
                self.u[self._slab(d, gi, gi + 1)] = v

    def compute_dt(self, cfl):
        return cfl / (1.0 + float(np.max(np.abs(self.u[self._real()]))))

    def step(self, dt):
        """u += dt * (box average over the 3^3 neighbourhood, with weights that tell the 26 neighbours apart - u)"""
        gx, gy, gz = self.g
        nx, ny, nz = self.n
        acc = np.zeros_like(self.u[self._real()])
        wsum = 0.0
        for dk in (-1, 0, 1) if gz else (0,):
            for dj in (-1, 0, 1) if gy else (0,):
                for di in (-1, 0, 1) if gx else (0,):
                    wgt = 1.0 + 0.25 * di + 0.125 * dj + 0.0625 * dk + 0.03125 * di * dj * (dk + 2)
                    acc += wgt * self.u[:, gz + dk:gz + dk + nz, gy + dj:gy + dj + ny, gx + di:gx + di + nx]
                    wsum += wgt
        new = self.u[self._real()] + dt * (acc / wsum - self.u[self._real()])
        self.u[self._real()] = new

    def sync(self):
        pass
