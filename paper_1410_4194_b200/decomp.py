"""Block decomposition of the domain (section 3.7 of the paper): host logic only.

A domain of nx x ny x nz cells is cut into bx x by x bz blocks; every block is a grid of its own (a `Grid` of
binding.py on a GPU) whose interior faces carry the code EXCHANGE.  After `set_state` and after every step the ghost
cells are filled direction by direction, x then y then z, each direction over the padded extent of the directions
before it, so edge and corner ghosts ride along and a block sends at most six messages; the time step
is the minimum over the blocks.  No arithmetic of the method lives here: packing, unpacking and the local
fills are kernels of the library (ch_halo_pack / ch_halo_unpack / ch_fill_dim), this module only decides who talks
to whom and in which order.

Two drivers share the `Topology`:
* `BlockGrid`      every block in THIS process (one GPU or several): transfers are device copies.  This is how the
                   decomposition is verified on a single GPU: its result equals the undivided grid's bit for bit.
* `RankBlockGrid`  one block per rank of torch.distributed (NCCL across GPUs, gloo in the CPU tests): transfers are
                   point-to-point send / recv of the packed slabs, the time step an all-reduce(MIN).
Both take a `grid_factory(nx, ny, nz, nghost, gamma, bc, device)` so that the tests can drive the same host logic
with a stand-in grid.
"""
from __future__ import annotations

import numpy as np

PERIODIC, REFLECTIVE, OUTFLOW, NOH, EXCHANGE = 1, 2, 3, 4, 5


def split(n: int, parts: int):
    """Contiguous near-equal ranges: [(start, stop)] * parts."""
    base, extra = divmod(n, parts)
    out, s = [], 0
    for p in range(parts):
        e = s + base + (1 if p < extra else 0)
        out.append((s, e))
        s = e
    return out


class Topology:
    def __init__(self, shape, blocks, bc):
        self.shape = tuple(int(v) for v in shape)          # (nx, ny, nz)
        self.blocks = tuple(int(v) for v in blocks)        # (bx, by, bz)
        self.bc = tuple(int(v) for v in bc)                # global faces x-, x+, y-, y+, z-, z+
        for n, b in zip(self.shape, self.blocks):
            if b < 1 or b > n:
                raise ValueError("more blocks than cells along a direction")
        self.ranges = [split(n, b) for n, b in zip(self.shape, self.blocks)]
        self.nblocks = self.blocks[0] * self.blocks[1] * self.blocks[2]

    def coords(self, bid):
        bx, by, _ = self.blocks
        return (bid % bx, (bid // bx) % by, bid // (bx * by))

    def bid(self, c):
        bx, by, _ = self.blocks
        return c[0] + bx * (c[1] + by * c[2])

    def extent(self, bid):
        c = self.coords(bid)
        return [self.ranges[d][c[d]] for d in range(3)]

    def block_shape(self, bid):
        return tuple(e - s for s, e in self.extent(bid))

    def origin(self, bid):
        return tuple(s for s, _ in self.extent(bid))

    def neighbour(self, bid, face):
        """Block behind `face` of block `bid`, or None at a domain face with a local rule."""
        d, side = face // 2, face & 1
        c = list(self.coords(bid))
        c[d] += 1 if side else -1
        if 0 <= c[d] < self.blocks[d]:
            return self.bid(c)
        if self.bc[2 * d] == PERIODIC and self.blocks[d] > 1:
            c[d] %= self.blocks[d]
            return self.bid(c)
        return None

    def block_bc(self, bid):
        return tuple(EXCHANGE if self.neighbour(bid, f) is not None else self.bc[f] for f in range(6))

    def transfers(self, d):
        """Messages of direction d: [(src block, src face, dst block, dst face)]; the real layers next to `src face`
        become the ghost layers behind `dst face`."""
        out = []
        for b in range(self.nblocks):
            for side in (0, 1):
                f = 2 * d + side
                nb = self.neighbour(b, f)
                if nb is not None:
                    out.append((nb, f ^ 1, b, f))
        return out


class BlockGrid:
    """All blocks in this process.  `devices`: one device for all blocks, or one per block."""

    def __init__(self, shape, blocks, nghost, gamma, bc, grid_factory, devices="cuda:0"):
        self.topo = Topology(shape, blocks, bc)
        t = self.topo
        if isinstance(devices, (str,)) or not hasattr(devices, "__len__"):
            devices = [devices] * t.nblocks
        self.devices = list(devices)
        self.grids = []
        for b in range(t.nblocks):
            G = grid_factory(*t.block_shape(b), nghost, gamma, t.block_bc(b), self.devices[b])
            if hasattr(G, "set_origin"):
                G.set_origin(*t.origin(b))
            self.grids.append(G)
        self.messages = 0

    def _alloc(self, G, d):
        import torch
        return torch.empty(5 * G.halo_cells(d), dtype=torch.float64, device=getattr(G, "device", "cpu"))

    def exchange(self):
        """Ghost fill of the whole decomposed domain: x, then y, then z."""
        for d in range(3):
            if self.topo.shape[d] == 1:
                continue
            for src, sf, dst, df in self.topo.transfers(d):
                S, D = self.grids[src], self.grids[dst]
                buf = self._alloc(S, d)
                S.halo_pack(sf, buf)
                if getattr(S, "device", None) != getattr(D, "device", None):
                    if hasattr(S, "sync"):
                        S.sync()
                    buf = buf.to(D.device)
                D.halo_unpack(df, buf)
                self.messages += 1
            for G in self.grids:
                G.fill_dim(d)

    def set_state(self, u):
        for b, G in enumerate(self.grids):
            (x0, x1), (y0, y1), (z0, z1) = self.topo.extent(b)
            G.set_state(np.ascontiguousarray(u[:, z0:z1, y0:y1, x0:x1]))
        self.exchange()

    def get_state(self):
        nx, ny, nz = self.topo.shape
        out = np.empty((5, nz, ny, nx))
        for b, G in enumerate(self.grids):
            (x0, x1), (y0, y1), (z0, z1) = self.topo.extent(b)
            out[:, z0:z1, y0:y1, x0:x1] = G.get_state()
        return out

    def set_spacing(self, dx, dy, dz):
        for G in self.grids:
            G.set_spacing(dx, dy, dz)

    def compute_dt(self, cfl) -> float:
        dts = [G.compute_dt(cfl) for G in self.grids]
        if any(not d == d for d in dts):
            return float("nan")                                     # a non-physical cell in any block
        return min(dts)

    def step(self, dt):
        if not dt == dt:
            raise FloatingPointError("non-physical state in a block")
        for G in self.grids:
            G.step(dt)
        self.exchange()

    def close(self):
        for G in self.grids:
            if hasattr(G, "close"):
                G.close()


class RankBlockGrid:
    """One block per rank of torch.distributed.  `dist` is the initialised torch.distributed module."""

    def __init__(self, shape, blocks, nghost, gamma, bc, grid_factory, dist, device="cpu"):
        self.topo = Topology(shape, blocks, bc)
        self.dist = dist
        self.rank = dist.get_rank()
        if dist.get_world_size() != self.topo.nblocks:
            raise ValueError("world size must equal the number of blocks")
        t = self.topo
        self.device = device
        # gloo moves host tensors only: slabs are staged through the host there; NCCL sends device tensors as they are
        self.wire = "cpu" if dist.get_backend() == "gloo" else device
        self.G = grid_factory(*t.block_shape(self.rank), nghost, gamma, t.block_bc(self.rank), device)
        if hasattr(self.G, "set_origin"):
            self.G.set_origin(*t.origin(self.rank))
        self.messages = 0

    def exchange(self):
        import torch
        dist, G = self.dist, self.G
        for d in range(3):
            if self.topo.shape[d] == 1:
                continue
            mine = [m for m in self.topo.transfers(d) if m[0] == self.rank or m[2] == self.rank]
            sends, recvs, ops = [], [], []
            for src, sf, dst, df in mine:
                # tag = destination face: two blocks can exchange two slabs of one direction (periodic, two blocks)
                if src == self.rank:
                    buf = torch.empty(5 * G.halo_cells(d), dtype=torch.float64, device=self.device)
                    G.halo_pack(sf, buf)
                    sends.append([dst, df, buf])
                if dst == self.rank:
                    buf = torch.empty(5 * G.halo_cells(d), dtype=torch.float64, device=self.wire)
                    recvs.append([src, df, buf])
            if hasattr(G, "sync"):
                G.sync()                                            # packed slabs complete before they are sent
            if self.wire != self.device:
                for s_ in sends:
                    s_[2] = s_[2].to(self.wire)
            local = []
            for dst, df, buf in sends:
                if dst == self.rank:
                    local.append((df, buf))
                else:
                    ops.append(dist.P2POp(dist.isend, buf, dst, tag=df))
            for src, df, buf in recvs:
                if src != self.rank:
                    ops.append(dist.P2POp(dist.irecv, buf, src, tag=df))
            if ops:
                for w in dist.batch_isend_irecv(ops):
                    w.wait()
            for src, df, buf in recvs:
                if src == self.rank:
                    buf = next(b for f, b in local if f == df)
                if str(buf.device) != str(torch.device(self.device)):
                    buf = buf.to(self.device)
                G.halo_unpack(df, buf)
                self.messages += 1
            if hasattr(G, "sync") and self.wire != self.device:
                G.sync()                                            # staged copies stay alive until they are unpacked
            G.fill_dim(d)

    def set_state(self, u_global):
        (x0, x1), (y0, y1), (z0, z1) = self.topo.extent(self.rank)
        self.G.set_state(np.ascontiguousarray(u_global[:, z0:z1, y0:y1, x0:x1]))
        self.exchange()

    def compute_dt(self, cfl) -> float:
        import torch
        t = torch.tensor([self.G.compute_dt(cfl)], dtype=torch.float64, device=self.wire)
        nan = torch.isnan(t).to(torch.float64)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MIN)
        self.dist.all_reduce(nan, op=self.dist.ReduceOp.MAX)        # a NaN on any rank must reach every rank
        return float("nan") if float(nan.item()) > 0 else float(t.item())

    def step(self, dt):
        self.G.step(dt)
        self.exchange()

    def get_local_state(self):
        return self.G.get_state()
