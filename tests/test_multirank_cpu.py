"""World-size-2 gloo test (CPU) of the only multi-rank logic the path has.  The update path does
not shard (north_star: no sharding, no collectives): bench.py --gpus N runs N independent replica
sets and aggregates work = SUM over ranks, time = MAX over ranks."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    import synth
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, ups, bts = bench.reduce_over_ranks(dist, 10.0 + 5.0 * rank, 1000.0 * (rank + 1), 12000.0 * (rank + 1),
                                           torch.device("cpu"))
    # ranks draw different replica sets: data seeds differ per rank, schedules are per-ctx
    w = synth.workload("mlp3_k4")
    a = torch.empty(w.K, 64)
    synth.fill_grad_(w, 0, 0, a, data_seed=w.seed + 1000 * rank)
    gathered = [torch.empty_like(a) for _ in range(world)]
    dist.all_gather(gathered, a)
    out[rank] = (ms, ups, bts, bool(torch.equal(gathered[0], gathered[1])))
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_only_aggregation_world2():
    world, port = 2, 29500 + os.getpid() % 2000
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        for rank in range(world):
            ms, ups, bts, same = out[rank]
            assert ms == 15.0 and ups == 3000.0 and bts == 36000.0     # MAX time, SUM work
            assert not same                                            # independent replica sets


def test_single_process_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks(None, 3.0, 5, 7, torch.device("cpu")) == (3.0, 5.0, 7.0)
