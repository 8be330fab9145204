"""Multi-GPU host logic on CPU: id split + 16-byte min exchange over gloo, world_size 2
(SURVEY §8(e)); the evaluator here is the oracle, the exchange code is the product's."""
import os, socket
import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp
from paper_1909_10286_b200 import sharding, workloads as wl


def test_split_range_partitions_exactly():
    for budget in (0, 1, 7, 1 << 16, (1 << 32) + 5):
        for world in (1, 2, 3, 8):
            parts = [sharding.split_range(budget, world, r, first_id=11) for r in range(world)]
            assert parts[0][0] == 11 and sum(n for _, n in parts) == budget
            for (f0, n0), (f1, _) in zip(parts, parts[1:]):
                assert f1 == f0 + n0
            assert max(n for _, n in parts) - min(n for _, n in parts) <= 1


def test_combine_orders_by_cost_then_id():
    inf = float("inf")
    assert sharding.combine([(3.0, 9), (2.0, 50), (2.0, 7), None]) == (2.0, 7)
    assert sharding.combine([(inf, 4), (inf, 2)]) == (inf, 2)
    assert sharding.combine([None, (inf, 1 << 63)]) == (inf, 1 << 63)
    with pytest.raises(ValueError):
        sharding.combine([None, None])


def _worker(rank, world, port, budget, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import lgo
    inst = wl.make("toy"); o = lgo.Oracle(inst)
    res = sharding.search_sharded(lambda seed, n, first: o.search(seed, n, first_id=first), 0, budget, rank, world)
    res1 = sharding.search_sharded(lambda seed, n, first: o.search(seed, n, first_id=first), 0, 1, rank, world, first_id=5)
    q.put((rank, res, res1))
    dist.barrier(); dist.destroy_process_group()


def test_two_rank_search_equals_single_rank():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    budget = 6001
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, budget, q)) for r in range(2)]
    [p.start() for p in ps]
    got = [q.get(timeout=120) for _ in ps]
    [p.join(60) for p in ps]
    from oracle import lgo
    inst = wl.make("toy"); o = lgo.Oracle(inst)
    want = o.search(0, budget); want1 = o.search(0, 1, first_id=5)
    for _, res, res1 in got:
        assert res == want and res1 == want1     # budget 1: rank 1 has no ids and passes None


def _ls_worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import lgo
    inst = wl.make("small"); o = lgo.Oracle(inst)
    p0 = o.init_plan()
    fn = lambda plan, seed, n_iters, n_workers, thresh: o.local_search(plan, seed, n_iters, n_workers, thresh)
    x, c, eps = sharding.local_search_eps_grid(fn, p0, 3, 25, 64, [0.0, 0.25, 0.5, 0.75, 1.0], rank, world)
    q.put((rank, {k: np.asarray(v).tolist() for k, v in x.items()}, c, eps))
    dist.barrier(); dist.destroy_process_group()


def test_eps_grid_shares_cover_the_grid():
    for n in (1, 5, 8):
        for world in (1, 2, 3, 8):
            got = sorted(k for r in range(world) for k in sharding.eps_grid_shares(n, world, r))
            assert got == list(range(n))


def test_two_rank_eps_grid_equals_single_rank():
    """the loop is run for eps in {0, 0.25, ..., 1} and the best is returned; ranks split the grid."""
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_ls_worker, args=(r, 2, port, q)) for r in range(2)]
    [p.start() for p in ps]
    got = [q.get(timeout=180) for _ in ps]
    [p.join(60) for p in ps]
    from oracle import lgo
    inst = wl.make("small"); o = lgo.Oracle(inst)
    p0 = o.init_plan()
    fn = lambda plan, seed, n_iters, n_workers, thresh: o.local_search(plan, seed, n_iters, n_workers, thresh)
    wx, wc, weps = sharding.local_search_eps_grid(fn, p0, 3, 25, 64, [0.0, 0.25, 0.5, 0.75, 1.0], 0, 1)
    runs = [o.local_search(p0, 3, 25, 64, min(int(e * 2**32), 0xFFFFFFFF))[1] for e in (0.0, 0.25, 0.5, 0.75, 1.0)]
    assert wc == min(runs)
    for _, x, c, eps in got:
        assert c == wc and eps == weps
        for k in wx:
            assert x[k] == np.asarray(wx[k]).tolist()
