"""N > 1 path on the CPU: world_size-2 gloo run of the DM-row sharding plumbing.

The one exchange step of a sharded run is the all-gather of the 80-byte spd_stats_t structs followed by an eq. 2 fold in
rank order.  Without a GPU the fold itself cannot run (it is a CUDA kernel, covered by
test_parity_gpu.py::test_stats_merge_equals_whole); here each rank fills its struct from the ORACLE's Chan triple of
its own rows, the structs go through paper_1611_09704_b200.shard.gather_stats over gloo, and the gathered triples,
folded in rank order with the oracle's eq. 2, must reproduce the whole-array statistics.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import gen
from oracle import spd_oracle as O
from paper_1611_09704_b200 import binding as B
from paper_1611_09704_b200 import shard as S


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_dm, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = gen.custom_config(n_dm, 4096, cid=77, mu=3.0, sigma=2.0)
        lo, hi = S.row_partition(n_dm, world, rank)
        a = np.zeros(1, dtype=B.STATS_DTYPE)
        if hi > lo:
            x = gen.make_rows(cfg, list(range(lo, hi)))
            o = O.stats(x)
            a["n"], a["T"], a["S"], a["mean"], a["sigma"] = o.n, o.T, o.S, o.mean, o.sigma
        local = torch.from_numpy(a.view(np.uint8).copy())
        parts = S.gather_stats(local).numpy().view(B.STATS_DTYPE)
        q.put((rank, lo, hi, parts.tobytes()))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_dm", [7, 1])
def test_row_sharded_stats_exchange_world2(n_dm):
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_dm, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # every rank holds the same gathered structs, in rank order
    assert res[0][3] == res[1][3]
    parts = np.frombuffer(res[0][3], dtype=B.STATS_DTYPE)
    assert [r[1] for r in res] == [0, res[0][2]] and res[1][2] == n_dm          # contiguous cover of the rows
    assert int(parts["n"].sum()) == n_dm * 4096
    # eq. 2 fold in rank order == statistics of the whole array
    cfg = gen.custom_config(n_dm, 4096, cid=77, mu=3.0, sigma=2.0)
    whole = O.stats(gen.make_rows(cfg, list(range(n_dm))))
    acc = np.array([0.0, 0.0, 0.0])
    for p in parts:
        acc = O.merge(acc, np.array([float(p["n"]), float(p["T"]), float(p["S"])]))
    n, T, Ssum = acc
    assert n == whole.n
    assert abs(T / n - whole.mean) <= 1e-12 * max(abs(whole.mean), whole.sigma)
    assert abs(np.sqrt(Ssum / n) - whole.sigma) <= 1e-12 * whole.sigma


def test_row_partition_covers_rows_exactly_once():
    for n_dm in (0, 1, 5, 6000, 4097):
        for world in (1, 2, 3, 8):
            blocks = [S.row_partition(n_dm, world, r) for r in range(world)]
            assert blocks[0][0] == 0 and blocks[-1][1] == n_dm
            assert all(blocks[i][1] == blocks[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in blocks]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        S.row_partition(4, 2, 2)
