"""World-size-2 (and 3) gloo test of the timeslice sharding: the gather of per-rank
correlator rows reproduces the full C[p][t] on every rank, also for T not divisible by the world size and T < world."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2411_08962_b200.sharding import gather_correlator, timeslices_of_rank


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _full(n_mom, T):
    t = torch.arange(T, dtype=torch.float64)
    p = torch.arange(n_mom, dtype=torch.float64)[:, None]
    return torch.complex(1000.0 * p + t, -0.5 * t - p)


def _worker(rank, world, port, T, n_mom, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = timeslices_of_rank(T, rank, world)
        full = _full(n_mom, T)
        got = gather_correlator(full[:, mine].contiguous(), T)
        q.put((rank, bool(torch.equal(got, full))))
    finally:
        dist.destroy_process_group()


def _sharded_worker(rank, world, port, T, n_mom, q):
    """contract_sharded end to end with the device call replaced by a stand-in that returns, for the rank's local
    timeslices, rows that encode WHICH global timeslice they belong to: checks the split, the order of the local rows and
    the gather as bench.py --gpus N uses them (the real device call needs a GPU and is covered by the gpu tests)."""
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_2411_08962_b200 import binding, sharding
        mine = timeslices_of_rank(T, rank, world)
        full = _full(n_mom, T)
        U_local = torch.tensor(mine, dtype=torch.float64).reshape(-1, 1, 1, 1)      # "propagators": the timeslice index itself

        def fake_contract(U, D, terms, momenta, L, T_local, **kw):
            assert T_local == U.shape[0] == len(mine) and kw == {"workspace": None}
            ts = U.reshape(-1).to(torch.long)
            return full[:, ts].contiguous()
        binding.contract, saved = fake_contract, binding.contract
        try:
            got = sharding.contract_sharded(U_local, U_local, None, [(0, 0, 0)] * n_mom, 1, T, workspace=None)
        finally:
            binding.contract = saved
        q.put((rank, bool(torch.equal(got, full))))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,T", [(2, 8), (3, 7), (2, 1)])
def test_contract_sharded_plumbing_gloo(world, T):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_sharded_worker, args=(r, world, port, T, 2, q)) for r in range(world)]
    for p in procs:
        p.start()
    results = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert sorted(results) == [(r, True) for r in range(world)]


def test_timeslices_of_rank_partition():
    for T in (0, 1, 5, 8, 64):
        for world in (1, 2, 3, 8):
            parts = [timeslices_of_rank(T, r, world) for r in range(world)]
            assert sorted(t for p in parts for t in p) == list(range(T))
            assert all(p == sorted(p) for p in parts)
    with pytest.raises(ValueError):
        timeslices_of_rank(4, 2, 2)


@pytest.mark.parametrize("world,T", [(2, 8), (2, 5), (3, 2)])
def test_gather_correlator_gloo(world, T):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, T, 2, q)) for r in range(world)]
    for p in procs:
        p.start()
    results = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert sorted(results) == [(r, True) for r in range(world)]


def test_gather_correlator_single_process():
    full = _full(3, 7)
    assert torch.equal(gather_correlator(full, 7), full)
