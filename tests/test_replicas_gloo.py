"""N > 1 path of bench.py on CPU: the hot path does not shard without an FFT transpose, so
`bench.py --gpus N` runs N independent replicas and reduces the timings with MAX over ranks.  These world_size-2 gloo
tests cover that host logic: rank-dependent replica inputs, the MAX reduction and the aggregate throughput formula."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import arche_inputs as ai
    import bench
    cfg = ai.make_config("c1")
    rep = bench.replica_config(cfg, rank, world)
    t_local = [1.0 + rank, 5.0 - rank]                 # rank 1 is slower on the first, faster on the second timing
    t_max = bench.max_over_ranks(t_local)
    dist.barrier()
    d = rep["pos"] - cfg["pos"]
    d -= cfg["cell"] * np.rint(d / cfg["cell"])          # minimum image: replicas are wrapped back into the cell
    q.put((rank, rep["pos"].copy(), t_max, float(np.abs(d).max())))
    dist.destroy_process_group()


def test_two_rank_replicas_and_max_reduction():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, pos0, tmax0, d0), (r1, pos1, tmax1, d1) = out
    assert tmax0 == tmax1 == [2.0, 5.0]                # MAX over ranks, identical on every rank
    assert not np.allclose(pos0, pos1)                 # independent replicas
    assert 0.0 < d0 < 1.0 and 0.0 < d1 < 1.0           # thermal displacement, still the same workload
    # whole-job throughput as bench.py forms it: all ranks' steps over the slowest rank's time
    steps = 7
    assert abs(2 * steps / tmax0[0] - 7.0) < 1e-12


def test_single_rank_is_identity():
    import arche_inputs as ai
    import bench
    cfg = ai.make_config("c1")
    assert bench.replica_config(cfg, 0, 1) is cfg
    assert bench.max_over_ranks([3.0, 4.0]) == [3.0, 4.0]
