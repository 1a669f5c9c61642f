"""Device path of the multi-GPU split ("a fairly small number of desktop
GPUs", L307 independence of the filters): ONE bank is split over two ranks by `shard_templates`, every rank filters
the same strain with its own shard through spiir_filter (C ABI), the rows are gathered on rank 0 and must equal
 - the oracle within the north_star tolerance, and
 - the single-bank GPU run BITWISE (a template's layout and summation tree do not depend on its position in the bank
   or on its neighbours, so splitting the bank cannot change a single bit).
The test box has one GPU: the two ranks are two processes on cuda:0 (independent kernels; nobody waits on a peer), the
exchange goes over gloo.  No data-path collective exists in this split; the gather only serves the comparison."""
import os
import socket

import numpy as np
import pytest

import spiir_inputs

pytestmark = pytest.mark.gpu
TOL = 1e-4


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _bank():
    return spiir_inputs.make_config(4, n_templates=300, n_samples=2048)


def _filter(pkg, torch, inp, path, chunk, F):
    opt = pkg.SpiirOptions(path=path, filters_per_thread=F, window_copies=2)
    x = torch.from_numpy(inp.x).cuda()
    snr = torch.full((inp.n_templates, inp.n_samples), float("nan"), dtype=torch.complex64, device="cuda")
    with pkg.SpiirBank(inp.offsets, inp.a1, inp.b0, inp.delays, 0, opt) as bank:
        for c0 in range(0, inp.n_samples, chunk):
            pkg.spiir_filter(bank.handle, x[c0:c0 + chunk], snr[:, c0:c0 + chunk])
        torch.cuda.synchronize()
    return snr.cpu().numpy()


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    os.environ.setdefault("GLOO_SOCKET_IFNAME", "lo")
    import torch
    import torch.distributed as dist
    import paper_1602_05573_b200 as pkg
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        torch.cuda.set_device(0)
        pkg.load_library()
        inp = _bank()
        parts = pkg.shard_templates(inp.offsets, world)
        out = {}
        for name, path, chunk, F in (("throughput", 1, 512, 8), ("stream", 3, 16, 4)):
            part = _filter(pkg, torch, inp.select_templates(parts[rank]), path, chunk, F)
            gathered = [None] * world
            dist.all_gather_object(gathered, (parts[rank], part))
            if rank == 0:
                full = np.full((inp.n_templates, inp.n_samples), np.nan, np.complex64)
                for idx, rows in gathered:
                    full[idx] = rows
                out[name] = full
        if rank == 0:
            import oracle
            ref = oracle.run_inputs(inp)
            res = {}
            for name, path, chunk, F in (("throughput", 1, 512, 8), ("stream", 3, 16, 4)):
                single = _filter(pkg, torch, inp, path, chunk, F)
                err = (np.abs(out[name].astype(np.complex128) - ref).max(axis=1) / np.abs(ref).max(axis=1)).max()
                res[name] = (float(err), bool(np.array_equal(out[name].view(np.float32), single.view(np.float32))))
            kt = np.diff(inp.offsets)
            q.put((res, [int(kt[p].sum()) for p in parts]))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_ranks_filter_one_sharded_bank_on_the_device():
    import torch
    import torch.multiprocessing as mp
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    import paper_1602_05573_b200 as pkg
    if not pkg.library_path().exists():
        import __graft_entry__ as entry
        entry.build()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res, loads = q.get(timeout=600)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    for name, (err, bitwise) in res.items():
        assert err <= TOL, (name, err)
        assert bitwise, f"{name}: sharded rows differ from the single-bank GPU run"
    assert abs(loads[0] - loads[1]) <= 2048          # LPT balance: within one template of each other
