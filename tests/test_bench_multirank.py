"""The N>1 host logic of bench.py on CPU: two ranks over gloo (the data path has no collective: ranks optimise
independent plans; only the timing is reduced -- max over ranks -- and the whole-job rate is formed on rank 0)."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    import bench
    ws, rk, lr = bench._dist_init()
    assert (ws, rk, lr) == (world, rank, rank)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r "measured" (10 + r) ms for K = 50 steps and (0.5 + r) s end to end
    ms, e2e_s = bench.max_over_ranks([10.0 + rank, 0.5 + rank], dist, "cpu")
    dist.barrier()
    q.put((rank, ms, e2e_s, bench.whole_job_rate(50, ws, ms * 1e-3)))
    dist.destroy_process_group()


def test_two_ranks_max_time_and_whole_job_rate():
    world, port = 2, 29541
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, e2e_s, rate in res:
        assert ms == 11.0 and e2e_s == 1.5                     # the slowest rank's times, on every rank
        assert abs(rate - 2 * 50 / 11.0e-3) < 1e-6             # all ranks' iterations / max time


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([3.0, 4.0], None, "cpu") == [3.0, 4.0]
    assert bench.whole_job_rate(50, 1, 0.025) == 2000.0
