"""f4: slab-decomposed 3D transform.  Host logic on CPU (gloo, world size 2: slab arithmetic, handle
exchange in rank order); on the GPU the decomposition against the oracle's undecomposed transform with R slabs on one
device processed one after the other (paper_2606_13283_b200/slab.py VirtualSlabs)."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_slab_plan_tiles_both_axes():
    from paper_2606_13283_b200.slab import SlabPlan, slab_ranges
    assert slab_ranges(12, 3) == [(0, 4), (4, 8), (8, 12)]
    with pytest.raises(ValueError):
        slab_ranges(10, 4)
    grid = (24, 16, 36)
    for world in (1, 2, 4):
        plans = [SlabPlan(grid, world, r) for r in range(world)]
        assert sum(p.nzl for p in plans) == 36 and sum(p.nyl for p in plans) == 16
        assert all(p.slab_elems == 24 * 16 * 36 // world for p in plans)
        for p in plans:
            assert p.z_slab_shape == (36 // world, 16, 24) and p.y_slab_shape == (36, 16 // world, 24)
            assert all(plans[0].owner_after_forward(iy) == p.rank for iy in range(p.y_lo, p.y_hi))
            assert all(plans[0].owner_after_inverse(iz) == p.rank for iz in range(p.z_lo, p.z_hi))
    with pytest.raises(ValueError):
        SlabPlan(grid, 2, 2)


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from paper_2606_13283_b200.slab import SlabPlan, exchange_handles
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        handles = exchange_handles(bytes([rank]) * 64)
        plan = SlabPlan((8, 12, 16), world, rank)
        q.put((rank, [h[0] for h in handles], [len(h) for h in handles], (plan.z_lo, plan.z_hi, plan.y_lo, plan.y_hi)))
    finally:
        dist.destroy_process_group()


def test_handle_exchange_world_size_2_gloo():
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, firsts, lens, rng in got:
        assert firsts == [0, 1] and lens == [64, 64]          # every rank sees every handle, in rank order
        assert rng == ((0, 8, 0, 6) if rank == 0 else (8, 16, 6, 12))


@pytest.mark.gpu
@pytest.mark.parametrize("grid,world", [((8, 12, 16), 1), ((24, 16, 36), 2), ((24, 16, 36), 4), ((9, 6, 12), 3), ((64, 32, 16), 8)])
def test_slab_transform_matches_the_undecomposed_one(orc, grid, world):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU test run without a CUDA device")
    import arche_inputs as ai
    from paper_2606_13283_b200 import Arche, ArcheError
    from paper_2606_13283_b200.slab import VirtualSlabs
    nx, ny, nz = grid
    cfg = ai.make_small(n_ions=2, grid=grid, cell=[6.0, 5.0, 7.0], seed=61)
    g = Arche(cfg)
    rng = np.random.default_rng(7)
    f = rng.normal(size=(nz, ny, nx)) + 1j * rng.normal(size=(nz, ny, nx))
    vs = VirtualSlabs(g, world)
    vs.load(f)
    vs.forward()
    ref = orc.fft3d(f, -1)
    got = vs.spectrum().cpu().numpy()
    assert np.abs(got - ref).max() < 1e-12 * np.abs(ref).max()
    assert np.abs(got - g.fft3d(torch.as_tensor(f), -1).cpu().numpy()).max() < 1e-12 * np.abs(ref).max()
    vs.inverse()                                   # and back: N f
    back = vs.field().cpu().numpy()
    assert np.abs(back - f * (nx * ny * nz)).max() < 1e-12 * np.abs(f).max() * nx * ny * nz
    if world > 1 and (ny % (world + 1) or nz % (world + 1)):
        with pytest.raises(ArcheError):            # axis lengths that do not split
            g.fft3d_slab_finish(vs.y[0].data_ptr(), world + 1, -1)


@pytest.mark.gpu
def test_ipc_export_round_trip_within_a_process(orc):
    """arche_slab_alloc / arche_ipc_export: a handle is produced for a slab buffer (opening it needs a second process,
    which one GPU box cannot give to a parity test); the buffer is usable as a transform operand."""
    import ctypes as C
    import torch
    import arche_inputs as ai
    from paper_2606_13283_b200 import Arche
    cfg = ai.make_small(n_ions=2, grid=(8, 12, 16), cell=[6.0, 5.0, 7.0], seed=61)
    g = Arche(cfg)
    p = C.c_void_p()
    assert g.lib.arche_slab_alloc(16 * 8 * 12 * 16, C.byref(p)) == 0 and p.value
    h = C.create_string_buffer(64)
    assert g.lib.arche_ipc_export(p.value, h) == 0 and any(h.raw)
    assert g.lib.arche_slab_free(p.value) == 0


@pytest.mark.gpu
def test_slabfft_object_in_a_world_of_one(orc):
    """paper_2606_13283_b200.slab.SlabFFT, the one-process-per-GPU object, in a process group of size 1 (gloo): buffer
    allocation and IPC export, the handle exchange, the views over library-owned memory, barriers, both directions.
    (Opening a peer's handle needs a second GPU process; the decomposition itself is covered by VirtualSlabs above.)"""
    import torch
    import torch.distributed as dist
    import arche_inputs as ai
    from paper_2606_13283_b200 import Arche
    from paper_2606_13283_b200.slab import SlabFFT
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=0, world_size=1)
    try:
        grid = (24, 16, 36)
        cfg = ai.make_small(n_ions=2, grid=grid, cell=[6.0, 5.0, 7.0], seed=61)
        g = Arche(cfg)
        fft = SlabFFT(g)
        assert fft.plan.z_slab_shape == (36, 16, 24) and fft.peer_y == [fft.buf.y] and fft.peer_z == [fft.buf.z]
        rng = np.random.default_rng(9)
        f = rng.normal(size=(36, 16, 24)) + 1j * rng.normal(size=(36, 16, 24))
        fft.z_slab().copy_(torch.as_tensor(f))
        fft.forward()
        ref = orc.fft3d(f, -1)
        assert np.abs(fft.y_slab().cpu().numpy() - ref).max() < 1e-12 * np.abs(ref).max()
        fft.z_slab().zero_()
        fft.inverse()
        assert np.abs(fft.z_slab().cpu().numpy() - f * f.size).max() < 1e-12 * np.abs(f).max() * f.size
        fft.close()
    finally:
        dist.destroy_process_group()
