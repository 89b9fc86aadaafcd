"""One plan on several GPUs: the partition of the labelled voxels, the aggregation of the ranks' partial
sums, and the sharded iteration.

CPU (`-m "not gpu"`): fredopt_shard_range is pure host code; a world-size-2 gloo run sums the partial transposed products,
proximity and cost of two half-plans (computed by the fp64 oracle over each rank's voxel range) and compares with the whole plan.
GPU (`-m gpu`): the ranks of a sharded plan are emulated on ONE device by threads whose reduction callback exchanges the partial
sums on the host side (stream synchronisation + a thread barrier: no kernel ever waits for another kernel); the sharded
trajectory must match the unsharded plan to rounding and the oracle within the parity bar.
"""
import os
import sys
import threading

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2509_20012_b200 import plangen as pg

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


# ------------------------------------------------------------------------------------------ partition (CPU)
@pytest.mark.parametrize("world", [1, 2, 3, 8])
def test_shard_ranges_cover_every_voxel_once_and_balance_the_labelled_non_zeros(plan0, world):
    from paper_2509_20012_b200 import fredopt
    rp, _, _, _, lab = plan0.to_numpy()
    cuts = [fredopt.shard_range(rp, lab, r, world) for r in range(world)]
    assert cuts[0][0] == 0 and cuts[-1][1] == plan0.n_rows
    for r in range(world - 1):
        assert cuts[r][1] == cuts[r + 1][0]                       # contiguous, disjoint
    w = np.where(lab != 0, np.diff(rp) + 1, 0)
    tot = w.sum()
    for b, e in cuts:
        assert abs(w[b:e].sum() - tot / world) <= w.max() + 1     # balanced to within one row
    with pytest.raises(fredopt.FredoptError):
        fredopt.shard_range(rp, lab, world, world)


def _gloo_worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    from oracle import oracle as om
    from paper_2509_20012_b200 import fredopt
    dist.init_process_group("gloo", rank=rank, world_size=world)
    plan = pg.build_plan(pg.config_spec(0))
    rp, ci, vd, vl, lab = plan.to_numpy()
    b, e = fredopt.shard_range(rp, lab, rank, world)
    mine = np.zeros(plan.n_rows, bool); mine[b:e] = True
    whole = om.from_plan(plan)
    # this rank's half-plan: the labels outside its voxel range are cleared (what a sharded fredopt_create keeps)
    half = om.Oracle.create(plan.n_rows, plan.n_cols, (rp, ci, vd), (rp, ci, vl), np.where(mine, lab, 0).astype(np.int32), plan.bounds)
    x = plan.x0.astype(np.float64) * (1 + 0.2 * (pg.uniform01_array(3, plan.n_cols) - 0.5))
    u = pg.uniform01_array(11, plan.n_rows) - 0.4
    v = pg.uniform01_array(12, plan.n_rows) - 0.6
    part, _ = half.transpose(u, v, active_only=True)             # partial S-vector of the labelled rows of this range
    t = torch.from_numpy(part.copy()); dist.all_reduce(t)
    full, full_abs = whole.transpose(u, v, active_only=True)
    err_t = float(np.max(np.abs(t.numpy() - full) / np.maximum(full_abs, 1e-300)))
    # set counts add up; with the whole plan's W the partial proximities and costs add up too
    cnt = torch.tensor([float(half.stats()["n_sets"]), float(half.stats()["n_zero_norm_sets"])], dtype=torch.float64); dist.all_reduce(cnt)
    Wl = torch.tensor([half.stats()["W"]], dtype=torch.float64); dist.all_reduce(Wl)
    scale = half.stats()["W"] / float(Wl[0]) if half.stats()["W"] > 0 else 0.0      # w^ of the whole plan = w / W_whole
    pr = torch.tensor([half.proximity(x)[0] * scale, float(half.proximity(x)[1]), half.cost(x) * scale], dtype=torch.float64)
    dist.all_reduce(pr)
    pw, nw = whole.proximity(x)
    q.put((rank, b, e, err_t, int(cnt[0]) == whole.stats()["n_sets"], int(cnt[1]) == whole.stats()["n_zero_norm_sets"],
           abs(float(Wl[0]) - whole.stats()["W"]) <= 1e-15 * whole.stats()["W"], abs(float(pr[0]) - pw) <= 1e-14 * pw, int(pr[1]) == nw,
           abs(float(pr[2]) - whole.cost(x)) <= 1e-14 * whole.cost(x)))
    dist.destroy_process_group()


def test_two_half_plans_sum_to_the_whole_plan_over_gloo():
    world, port = 2, 29553
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_gloo_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=300) for _ in range(world))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] == 0 and res[0][2] == res[1][1] and res[1][2] == 32 ** 3          # the two ranges tile the grid
    for r in res:
        assert r[3] <= 1e-15, f"partial transposed products do not add up: {r[3]:.2e}"
        assert all(r[4:]), r


# ------------------------------------------------------------------------------------------ sharded iteration (one GPU, emulated ranks)
class _EmulatedComm:
    """All-reduce among threads of one process: host-side exchange, identical summation order on every rank."""

    def __init__(self, world, fredopt):
        self.world, self.f = world, fredopt
        self.barrier = threading.Barrier(world)
        self.views = [None] * world
        self.calls = [0] * world

    def fn(self, rank):
        def reduce(ptr, n, stream):
            torch.cuda.synchronize()
            self.views[rank] = torch.as_tensor(self.f.DeviceDoubles(ptr, n), device="cuda")
            self.calls[rank] += 1
            self.barrier.wait()
            tot = self.views[0].clone()
            for r in range(1, self.world):
                tot += self.views[r]
            torch.cuda.synchronize()
            self.barrier.wait()
            self.views[rank].copy_(tot)
            torch.cuda.synchronize()
            self.barrier.wait()
        return reduce


def _run_sharded(fredopt, world, make_plan, run):
    comm = _EmulatedComm(world, fredopt)
    out, err = [None] * world, []

    def work(rank):
        try:
            torch.cuda.set_device(0)
            gp = make_plan(rank, world)
            gp.set_reduce(comm.fn(rank))
            out[rank] = run(gp)
        except BaseException as e:          # noqa: BLE001  (reported below; a dead thread would otherwise hang the barrier)
            err.append(e)
            comm.barrier.abort()
    ts = [threading.Thread(target=work, args=(r,)) for r in range(world)]
    for t in ts:
        t.start()
    for t in ts:
        t.join(timeout=600)
    assert not err, err
    return out, comm


@pytest.mark.gpu
@pytest.mark.parametrize("world", [2, 3])
@pytest.mark.parametrize("beta0", [0.0, 1.0])
def test_sharded_plan_matches_the_whole_plan_and_the_oracle(plan0, world, beta0):
    from oracle import oracle as om
    from paper_2509_20012_b200 import fredopt
    sp = plan0.spec

    def run(gp):
        gp.set_option(fredopt.OPT_REDUCTIONS, 2)
        gp.set_weights(plan0.x0)
        gp.iterate(20, sp.lam, beta0, sp.a)
        x = gp.get_weights_f64(np.empty(plan0.n_cols, np.float64))
        return x, gp.stats(), gp.proximity(None)

    res, comm = _run_sharded(fredopt, world, lambda r, w: fredopt.from_plan(plan0, shard_rank=r, shard_world=w), run)
    for r in range(1, world):                                     # the replicated weights stay identical bit for bit
        assert np.array_equal(res[r][0], res[0][0]) and res[r][2] == res[0][2]
    assert sum(s["n_active_rows"] for _, s, _ in res) == int((plan0.labels != 0).sum())
    whole = fredopt.from_plan(plan0); whole.set_option(fredopt.OPT_REDUCTIONS, 2)
    whole.set_weights(plan0.x0); whole.iterate(20, sp.lam, beta0, sp.a)
    xw = whole.get_weights_f64(np.empty(plan0.n_cols, np.float64))
    assert np.linalg.norm(res[0][0] - xw) <= 1e-12 * np.linalg.norm(xw)
    sw = whole.stats()
    assert all(res[0][1][k] == sw[k] for k in ("k", "s", "trials", "n_sets", "n_zero_norm_sets", "n_violated"))
    assert abs(res[0][1]["prox"] - sw["prox"]) <= 1e-10 * abs(sw["prox"])
    orc = om.from_plan(plan0); orc.set_option(om.OPT_REDUCTIONS, 2)
    orc.set_x(plan0.x0); orc.iterate(20, sp.lam, beta0, sp.a)
    xo = orc.get_x()
    assert np.linalg.norm(res[0][0] - xo) <= 1e-4 * np.linalg.norm(xo)
    po, no = orc.proximity(None)
    assert res[0][2][1] == no and abs(res[0][2][0] - po) <= 1e-6 * po
    # three reductions per superiorized reduction step... : set counts + per iteration (2 + 1 per reduction) + proximity
    per_it = (2 * 2 + 1) if beta0 else 1
    assert comm.calls[0] == 1 + 20 * per_it + 1


@pytest.mark.gpu
def test_sharded_plan_refuses_what_it_cannot_do(plan0):
    from paper_2509_20012_b200 import fredopt
    gp = fredopt.from_plan(plan0, shard_rank=0, shard_world=2)
    gp.set_weights(plan0.x0)
    with pytest.raises(fredopt.FredoptError) as e:                # no reduction set
        gp.iterate(1, 1.0, 1.0, 0.99)
    assert e.value.code == fredopt.INVALID_ARG
    with pytest.raises(fredopt.FredoptError) as e:
        gp.percentile_value(0, 1, 0.3)
    assert e.value.code == fredopt.UNSUPPORTED
    for bad in (dict(shard_rank=2, shard_world=2), dict(shard_rank=-1, shard_world=2), dict(shard_rank=1, shard_world=0)):
        with pytest.raises(fredopt.FredoptError):
            fredopt.from_plan(plan0, **bad)
    # the all-voxel calls still cover every voxel
    d = np.empty(plan0.n_rows, np.float32); d2 = np.empty(plan0.n_rows, np.float32)
    gp.dose_let(plan0.x0, d, None)
    fredopt.from_plan(plan0).dose_let(plan0.x0, d2, None)
    assert np.array_equal(d, d2)
