"""bench.py --gpus N runs N independent replicas (the path does not shard: DESIGN.md section 7).  The only
multi-rank logic is the aggregation of the per-rank timings and work: covered here with two gloo ranks on CPU."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _rank_main(rank: int, world: int, port: int, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r took (1 + r) s for 100 (1 + r) pairs device-resident, (2 + r) s for 10 (1 + r) pairs end to end
    got = bench.aggregate_replicas(torch, dist, "cpu", 1.0 + rank, 2.0 + rank, 100.0 * (1 + rank), 10.0 * (1 + rank))
    out.put((rank, got))
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_time_is_max_and_work_is_sum():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank in (0, 1):
        sec, sec_e2e, pairs, pairs_e2e = res[rank]
        assert (sec, sec_e2e, pairs, pairs_e2e) == (2.0, 3.0, 300.0, 30.0)
    # the job's throughput is whole-job work over the slowest rank's time
    assert res[0][2] / res[0][0] == 150.0


def test_single_process_passes_through():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate_replicas(torch, None, "cpu", 1.5, 2.5, 7.0, 3.0) == (1.5, 2.5, 7.0, 3.0)
