"""Host logic of bench.py's N > 1 path (replicas) on CPU: two gloo ranks."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _rank_main(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import lp_inputs as I
    w = bench.rank_workload(I.workload(1), rank)
    x, y, z, pid = I.make_particles(w)
    ms = 10.0 + 5.0 * rank                               # rank 1 is the slow one
    ms_max = bench.reduce_max(ms, dist, torch.device("cpu"))
    rate = bench.aggregate_rate(world, w.np, 4, ms_max * 1e-3)
    torch.save({"seed": w.seed, "x0": float(x[0]), "np": w.np, "ms_max": ms_max, "rate": rate},
               os.path.join(out, "r%d.pt" % rank))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_replicas(tmp_path):
    world, port = 2, 29500 + os.getpid() % 2000
    mp.spawn(_rank_main, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    r = [torch.load(os.path.join(str(tmp_path), "r%d.pt" % k)) for k in range(world)]
    assert r[0]["seed"] != r[1]["seed"] and r[0]["x0"] != r[1]["x0"]       # own particle set per rank
    assert r[0]["ms_max"] == r[1]["ms_max"] == 15.0                          # max over ranks
    expect = world * r[0]["np"] * 4 / 15.0e-3
    assert np.isclose(r[0]["rate"], expect) and np.isclose(r[1]["rate"], expect)


def test_single_rank_is_identity():
    import bench
    import lp_inputs as I
    w = I.workload(1)
    assert bench.rank_workload(w, 0) is w
    assert bench.reduce_max(3.5, None, None) == 3.5
    assert bench.aggregate_rate(1, 1000, 10, 0.5) == 20000.0
