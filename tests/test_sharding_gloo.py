"""The N > 1 path on CPU: world_size-2 gloo processes run the host-side sharding logic (-m "not gpu")."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1303_5057_b200 import sharding
from paper_1303_5057_b200.workloads import shard_range


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_total, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        rng = np.random.default_rng(7)
        full = torch.from_numpy(rng.integers(0, 4, size=n_total, dtype=np.uint8))      # a status array, same on all ranks
        lo, hi = shard_range(n_total, rank, world)
        got = sharding.gather_bytes(full[lo:hi].clone(), n_total)
        ok = torch.equal(got, full)
        hist = {f"s{s}": int((full[lo:hi] == s).sum()) for s in range(4)}
        tot = sharding.sum_counters(hist, "cpu")
        ok &= all(tot[f"s{s}"] == int((full == s).sum()) for s in range(4))
        ok &= sharding.max_time_ms(10.0 + rank, "cpu") == 10.0 + world - 1
        try:
            sharding.gather_bytes(full[lo:hi + 1].clone() if hi < n_total else full[lo:hi - 1].clone(), n_total)
            ok = False
        except ValueError:
            pass
        q.put((rank, bool(ok)))
    finally:
        dist.destroy_process_group()


def test_status_gather_and_counter_reduction_world_size_2():
    ctx = mp.get_context("spawn")
    for n_total in (1001, 4096):                       # uneven and even split
        q = ctx.Queue()
        port = _free_port()
        procs = [ctx.Process(target=_worker, args=(r, 2, port, n_total, q)) for r in range(2)]
        for p in procs:
            p.start()
        res = sorted(q.get(timeout=120) for _ in procs)
        for p in procs:
            p.join(timeout=60)
            assert p.exitcode == 0
        assert res == [(0, True), (1, True)]


def test_shard_ranges_tile_the_batch():
    for n in (0, 1, 7, 1000, 2 ** 30):
        for world in (1, 2, 3, 8):
            edges = [shard_range(n, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n
            assert all(edges[r][1] == edges[r + 1][0] for r in range(world - 1))
            sizes = [b - a for a, b in edges]
            assert max(sizes) - min(sizes) <= 1
