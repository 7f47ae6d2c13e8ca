"""Block decomposition on the GPU (`-m gpu`), verified on ONE device: the
blocks of a decomposed domain are separate contexts of the library on the same GPU, their ghost layers travel through
ch_halo_pack / ch_halo_unpack in the paper's x -> y -> z order and every block steps with the minimum of the blocks'
Eq. 22 time steps.  Because a cell's arithmetic does not depend on where it sits in a grid (every function
shared between warm-up and loop code spells out its multiply-adds), the decomposed run must equal the undivided run
BIT FOR BIT, for every kernel form that a block's shape selects (TMA-fed or plain, fused or unfused)."""
import numpy as np
import pytest

from paper_1410_4194_b200 import decomp, workloads as wl

pytestmark = pytest.mark.gpu
P, R, O, N = wl.PERIODIC, wl.REFLECTIVE, wl.OUTFLOW, wl.NOH


@pytest.fixture(scope="module")
def ch():
    import paper_1410_4194_b200 as pkg
    pkg.load_library()
    return pkg


def factory(ch, setup=None):
    def make(nx, ny, nz, g, gamma, bc, device):
        G = ch.Grid(nx, ny, nz, g, gamma, bc, device=device)
        if setup:
            setup(G)
        return G
    return make


def compare(ch, w, blocks, steps, g=3, setup=None, dx=None):
    nx, ny, nz = w.shape
    S = ch.Grid(nx, ny, nz, g, w.gamma, w.bc)
    if setup:
        setup(S)
    B = decomp.BlockGrid(w.shape, blocks, g, w.gamma, w.bc, factory(ch, setup), devices="cuda:0")
    d = 1.0 / nx
    B.set_spacing(d, d, d)                     # a block's default width is 1 / its own nx (reading S8)
    S.set_state(w.u)
    B.set_state(w.u)
    for n in range(steps):
        dt_s, dt_b = S.compute_dt(w.cfl), B.compute_dt(w.cfl)
        assert dt_s == dt_b, (n, dt_s, dt_b)   # the minimum over the blocks IS the global Eq. 22 value (max is exact)
        S.step(dt_s)
        B.step(dt_b)
    a, b = S.get_state(), B.get_state()
    # ghosts of block 0 against the undivided grid's padded store
    G0 = B.grids[0]
    p0, ps = G0.get_padded(), S.get_padded()
    (x0, x1), (y0, y1), (z0, z1) = B.topo.extent(0)
    gx, gy, gz = (g if n > 1 else 0 for n in (nx, ny, nz))
    sub = ps[:, z0:z1 + 2 * gz, y0:y1 + 2 * gy, x0:x1 + 2 * gx]
    S.close(); B.close()
    assert np.all(np.isfinite(a))
    assert np.array_equal(a, b)
    assert np.array_equal(p0, sub)             # edges and corners included
    return B


@pytest.mark.parametrize("blocks", [(2, 2, 1), (1, 2, 3), (3, 1, 2), (2, 2, 2)])
def test_periodic_sweep_blocks_equal_the_undivided_grid_bitwise(ch, blocks):
    compare(ch, wl.sweep(shape=(48, 40, 36)), blocks, 3)


def test_mixed_faces_and_ragged_blocks(ch):
    compare(ch, wl.smooth_random(41, 29, 23, seed=5, bc=(R, O, P, P, O, R)), (3, 2, 2), 3)
    compare(ch, wl.rough_random(45, 31, 26, seed=11, decades=0.5), (2, 3, 2), 2)


def test_two_dimensional_and_one_dimensional_domains(ch):
    compare(ch, wl.kelvin_helmholtz(64), (2, 2, 1), 5)
    compare(ch, wl.sod(128), (4, 1, 1), 10)


def test_other_methods_decompose_too(ch):
    def roe_plmc(G):
        G.set_solver(1); G.set_reconstruction(1)
    compare(ch, wl.sweep(shape=(40, 36, 24)), (2, 2, 1), 2, setup=roe_plmc)

    def ppmp(G):
        G.set_reconstruction(3)
    compare(ch, wl.sweep(shape=(40, 36, 24)), (2, 1, 2), 2, g=4, setup=ppmp)

    def hcorr(G):
        G.set_solver(1); G.set_hcorrection(True)
    compare(ch, wl.sweep(shape=(40, 36, 24)), (2, 2, 1), 2, g=4, setup=hcorr)


def test_noh_octant_in_blocks(ch):
    """Analytic faces need global coordinates (ch_set_origin) and the global clock."""
    def setup(G):
        G.set_solver(1); G.set_hcorrection(True); G.set_noh(1.0, 1e-6)
    w = wl.noh(n=36, dims=3)
    compare(ch, w, (2, 2, 1), 6, g=4, setup=setup)
    w = wl.noh(n=64, dims=2)
    compare(ch, w, (2, 2, 1), 10, g=4, setup=setup)


def test_messages_per_block_and_refusals(ch):
    w = wl.sweep(shape=(24, 24, 24))
    B = decomp.BlockGrid(w.shape, (2, 2, 2), 3, w.gamma, w.bc, factory(ch), devices="cuda:0")
    B.set_state(w.u)
    assert B.messages == 8 * 6                                    # six messages per block
    with pytest.raises(RuntimeError):
        B.grids[0].step_cfl(0.4)                                  # a block needs the global minimum of dt
    B.close()


def _gpu_rank(rank, world, port, shape, blocks, steps, out):
    import os
    import torch
    import torch.distributed as dist
    import paper_1410_4194_b200 as pkg
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    w = wl.sweep(shape=shape)
    G = decomp.RankBlockGrid(shape, blocks, 3, w.gamma, w.bc,
                             lambda nx, ny, nz, g, gamma, bc, dev: pkg.Grid(nx, ny, nz, g, gamma, bc, device=dev), dist, device="cuda:0")
    G.G.set_spacing(*(1.0 / shape[0],) * 3)
    G.set_state(w.u)
    dts = []
    for _ in range(steps):
        dt = G.compute_dt(w.cfl)
        dts.append(dt)
        G.step(dt)
    np.save(os.path.join(out, f"r{rank}.npy"), G.get_local_state())
    np.save(os.path.join(out, f"dt{rank}.npy"), np.array(dts))
    dist.barrier()
    dist.destroy_process_group()


def test_one_block_per_rank_with_the_real_library(ch, tmp_path):
    """RankBlockGrid (one block per torch.distributed rank: point-to-point slabs, all-reduce(MIN) of dt) driving the
    CUDA library: two host processes, both on this one GPU, gloo between them (slabs staged through the host; the
    ranks' kernels never wait on one another — each process blocks on the host in send / recv).  Periodic with two
    blocks: both faces of a rank talk to the other rank.  Result = the undivided grid, bit for bit."""
    import socket
    import torch.multiprocessing as mp
    shape, blocks, steps = (32, 24, 20), (2, 1, 1), 3
    w = wl.sweep(shape=shape)
    S = ch.Grid(*shape, 3, w.gamma, w.bc)
    S.set_state(w.u)
    dts = []
    for _ in range(steps):
        dt = S.compute_dt(w.cfl)
        dts.append(dt)
        S.step(dt)
    want = S.get_state()
    S.close()
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_gpu_rank, args=(2, port, shape, blocks, steps, str(tmp_path)), nprocs=2, join=True)
    topo = decomp.Topology(shape, blocks, w.bc)
    for r in range(2):
        (x0, x1), (y0, y1), (z0, z1) = topo.extent(r)
        assert np.array_equal(np.load(tmp_path / f"r{r}.npy"), want[:, z0:z1, y0:y1, x0:x1])
        assert np.load(tmp_path / f"dt{r}.npy").tolist() == dts
