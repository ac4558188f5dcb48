"""N > 1 plumbing (replicas only) on CPU: two gloo ranks.  No GPU, no kernels: this covers the
sharding of independent registrations over ranks and the max-over-ranks / whole-job reductions bench.py uses."""
import importlib.util
import os
import socket
import sys

import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _replicas():
    # loaded by path: importing the package itself needs the built CUDA library
    spec = importlib.util.spec_from_file_location("_disc_replicas", os.path.join(ROOT, "paper_1204_6295_b200", "replicas.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    rep = _replicas()
    mine = rep.shard_cases(7, rank, world)
    ms = 10.0 + 5.0 * rank                      # rank 1 is the slow one
    units = 100.0 * len(mine)
    value, ms_max = rep.whole_job_throughput(units, ms, dist)
    q.put((rank, mine, rep.max_over_ranks(ms, dist), value, ms_max))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_shard_and_reduce():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, c0, m0, v0, t0), (r1, c1, m1, v1, t1) = out
    assert sorted(c0 + c1) == list(range(7)) and not set(c0) & set(c1)       # disjoint and covering
    assert m0 == m1 == 15.0 and t0 == t1 == 15.0                             # max over ranks, same on every rank
    assert v0 == v1 == pytest.approx(700.0 / 15e-3)                          # all units / slowest rank


def test_single_process_is_identity():
    rep = _replicas()
    assert rep.shard_cases(5, 0, 1) == [0, 1, 2, 3, 4]
    assert rep.max_over_ranks(3.5) == 3.5
    v, ms = rep.whole_job_throughput(10.0, 2.0)
    assert v == pytest.approx(5000.0) and ms == 2.0
    with pytest.raises(ValueError):
        rep.shard_cases(3, 2, 2)
