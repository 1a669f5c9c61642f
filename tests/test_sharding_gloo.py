"""Multi-GPU HOST LOGIC only, on CPU: templates shard across ranks with no
data-path collective; the only exchange is the max-over-ranks of the timing.  world_size 2, gloo.  No device call is
made here (the oracle stands in for it so that the partition and the gather can be checked without a GPU); the device
path of the same split -- two ranks filtering their shards through spiir_filter, gathered rows against the oracle and
bitwise against the single-bank run -- is tests/test_sharding_gpu.py (-m gpu)."""
import os
import socket

import numpy as np
import pytest

import spiir_inputs


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_shard_templates_balances_and_partitions():
    import paper_1602_05573_b200 as pkg
    inp = spiir_inputs.make_config(4, n_templates=500, n_samples=16)
    kt = np.diff(inp.offsets)
    for world in (1, 2, 3, 8):
        parts = pkg.shard_templates(inp.offsets, world)
        assert len(parts) == world
        allt = np.concatenate(parts)
        assert np.array_equal(np.sort(allt), np.arange(500))               # a partition
        loads = np.array([kt[p].sum() for p in parts])
        assert loads.max() - loads.min() <= kt.max()                       # LPT bound
        assert all(np.array_equal(p, np.sort(p)) for p in parts)
    assert [p.tolist() for p in pkg.shard_templates(np.array([0, 5, 5 + 9, 5 + 9 + 9]), 2)] == [[0, 1], [2]]
    with pytest.raises(ValueError):
        pkg.shard_templates(inp.offsets, 0)


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    os.environ.setdefault("GLOO_SOCKET_IFNAME", "lo")      # the container hostname may not resolve
    import torch
    import torch.distributed as dist
    import oracle
    import paper_1602_05573_b200 as pkg
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        inp = spiir_inputs.make_random_bank(123, [64, 300, 17, 128, 90, 256, 33], 600, d_max=200)
        mine = pkg.shard_templates(inp.offsets, world)[rank]
        sub = inp.select_templates(mine)
        # every rank filters the same strain with its own slice (here with the CPU oracle standing in for the
        # device call: this test covers the sharding and the gather of results, not the kernels)
        part = oracle.run_inputs(sub)
        # what bench.py exchanges: the step time, max over ranks
        t = torch.tensor([1.0 + rank], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        # a consumer that wants all rows in one place gathers them; rows land at their template index
        gathered = [None] * world
        dist.all_gather_object(gathered, (mine, part))
        full = np.empty((inp.n_templates, inp.n_samples), np.complex128)
        for idx, rows in gathered:
            full[idx] = rows
        ok = np.array_equal(full, oracle.run_inputs(inp)) and float(t.item()) == float(world)
        q.put((rank, bool(ok), int(sub.n_filters)))
    finally:
        dist.destroy_process_group()


def test_two_ranks_shard_a_bank_and_reassemble_it():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [True, True]
    assert sum(r[2] for r in res) == 64 + 300 + 17 + 128 + 90 + 256 + 33
    assert abs(res[0][2] - res[1][2]) <= 300
