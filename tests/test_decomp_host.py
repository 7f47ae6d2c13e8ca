"""Host logic of the block decomposition (paper_1410_4194_b200/decomp.py), `-m "not gpu"`: the topology,
the x -> y -> z message schedule that carries edges and corners with at most six messages per block,
the minimum of the blocks' time steps, in one process and over gloo with one block per rank.  The grids are
stand-ins (tests/standin_grid.py): index work and a toy update that reads every ghost within its radius."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

from paper_1410_4194_b200 import decomp
from tests.standin_grid import StandInGrid

P, R, O = decomp.PERIODIC, decomp.REFLECTIVE, decomp.OUTFLOW


def field(shape, seed=0):
    nx, ny, nz = shape
    return np.random.default_rng(seed).normal(size=(5, nz, ny, nx))


def single(shape, bc, u, steps, g=3):
    G = StandInGrid(*shape, g, 1.4, bc)
    G.set_state(u)
    for d in range(3):
        G.fill_dim(d)
    dts = []
    for _ in range(steps):
        dt = G.compute_dt(0.4)
        dts.append(dt)
        G.step(dt)
        for d in range(3):
            G.fill_dim(d)
    return G.get_state(), dts


def test_topology_and_schedule():
    t = decomp.Topology((10, 7, 5), (3, 2, 1), (P, P, R, O, O, O))
    assert [t.block_shape(b) for b in range(6)] == [(4, 4, 5), (3, 4, 5), (3, 4, 5), (4, 3, 5), (3, 3, 5), (3, 3, 5)]
    assert t.origin(4) == (4, 4, 0)
    assert t.block_bc(0) == (5, 5, R, 5, O, O) and t.block_bc(5) == (5, 5, 5, O, O, O)
    assert t.neighbour(0, 0) == 2 and t.neighbour(2, 1) == 0 and t.neighbour(0, 2) is None and t.neighbour(0, 4) is None
    # every block: at most six messages per exchange, one per EXCHANGE face
    per_block = {b: 0 for b in range(6)}
    for d in range(3):
        for src, sf, dst, df in t.transfers(d):
            assert sf == df ^ 1 and t.neighbour(dst, df) == src
            per_block[dst] += 1
    assert all(v == sum(c == 5 for c in t.block_bc(b)) <= 6 for b, v in per_block.items())
    with pytest.raises(ValueError):
        decomp.Topology((4, 4, 4), (5, 1, 1), (P,) * 6)


@pytest.mark.parametrize("shape,blocks,bc", [((12, 10, 8), (2, 2, 2), (P,) * 6), ((13, 9, 7), (3, 1, 2), (R, O, P, P, O, R)),
                                             ((16, 11, 1), (2, 3, 1), (P, P, O, R, P, P)), ((9, 1, 1), (3, 1, 1), (O, R, P, P, P, P))])
def test_blocks_in_one_process_equal_the_undivided_grid_bitwise(shape, blocks, bc):
    u = field(shape)
    want, dts = single(shape, bc, u, 4)
    B = decomp.BlockGrid(shape, blocks, 3, 1.4, bc, StandInGrid, devices="cpu")
    B.set_state(u)
    got_dts = []
    for _ in range(4):
        dt = B.compute_dt(0.4)
        got_dts.append(dt)
        B.step(dt)
    assert got_dts == dts                                    # the minimum over the blocks is the global time step
    assert np.array_equal(B.get_state(), want)               # corners included: the toy update reads all 26 neighbours
    # padded stores agree with the undivided grid's ghosts too (block 0, its low corner)
    n_faces = sum(sum(c == 5 for c in B.topo.block_bc(b)) for b in range(B.topo.nblocks))
    assert B.messages == 5 * n_faces                          # set_state + 4 steps, one message per EXCHANGE face each


def test_wrong_order_of_directions_is_caught():
    """z before x leaves stale corners: the check above is sensitive to the schedule."""
    shape, blocks, bc = (12, 10, 8), (2, 2, 2), (P,) * 6
    u = field(shape)
    want, _ = single(shape, bc, u, 2)

    class Reversed(decomp.BlockGrid):
        def exchange(self):
            for d in (2, 1, 0):
                for src, sf, dst, df in self.topo.transfers(d):
                    buf = self._alloc(self.grids[src], d)
                    self.grids[src].halo_pack(sf, buf)
                    self.grids[dst].halo_unpack(df, buf)
                for G in self.grids:
                    G.fill_dim(d)
    B = Reversed(shape, blocks, 3, 1.4, bc, StandInGrid, devices="cpu")
    B.set_state(u)
    for _ in range(2):
        B.step(B.compute_dt(0.4))
    assert not np.array_equal(B.get_state(), want)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank, world, port, shape, blocks, bc, steps, out):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    u = field(shape)
    G = decomp.RankBlockGrid(shape, blocks, 3, 1.4, bc, StandInGrid, dist, device="cpu")
    G.set_state(u)
    dts = []
    for _ in range(steps):
        dt = G.compute_dt(0.4)
        dts.append(dt)
        G.step(dt)
    np.save(os.path.join(out, f"r{rank}.npy"), G.get_local_state())
    np.save(os.path.join(out, f"dt{rank}.npy"), np.array(dts))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("shape,blocks,bc", [((12, 10, 8), (2, 1, 1), (P,) * 6), ((9, 14, 6), (1, 2, 1), (R, O, O, R, P, P))])
def test_one_block_per_rank_over_gloo(tmp_path, shape, blocks, bc):
    """world_size 2, gloo: point-to-point slabs (periodic with two blocks: both faces of a rank talk to the other
    rank) and the all-reduce(MIN) of dt.  Result = the undivided grid, bitwise."""
    steps = 3
    want, dts = single(shape, bc, field(shape), steps)
    mp.spawn(_rank_main, args=(2, _free_port(), shape, blocks, bc, steps, str(tmp_path)), nprocs=2, join=True)
    topo = decomp.Topology(shape, blocks, bc)
    for r in range(2):
        (x0, x1), (y0, y1), (z0, z1) = topo.extent(r)
        assert np.array_equal(np.load(tmp_path / f"r{r}.npy"), want[:, z0:z1, y0:y1, x0:x1])
        assert np.load(tmp_path / f"dt{r}.npy").tolist() == dts
