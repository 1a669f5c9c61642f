"""spiir_filter_static: the entry point that allocates nothing (include/spiir.h) against the existing spiir_filter path.

Collected last on purpose (the file name sorts behind every other test file): the run uses pytest -x.
The partial sums of the tiny-chunk streaming kernels go to a 4 MiB file-scope device array instead of a cudaMalloc'ed buffer;
the kernels are the same, so the two paths must agree bitwise -- and, like every GPU path here, with the oracle within
max|gpu - ref| <= 1e-4 max|ref| per template.  Two calls in a row (and more) share the array and must not disturb each other.
"""
import numpy as np
import pytest

import spiir_inputs

pytestmark = pytest.mark.gpu

TOL = 1e-4


@pytest.fixture(scope="module")
def env():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    import oracle
    import paper_1602_05573_b200 as pkg
    if not pkg.library_path().exists():
        import __graft_entry__ as entry
        entry.build()
    pkg.load_library()
    return pkg, oracle, torch


def run(pkg, torch, inp, chunks, static):
    x = torch.from_numpy(inp.x).cuda()
    snr = torch.full((inp.n_templates, inp.n_samples), float("nan"), dtype=torch.complex64, device="cuda")
    fn = pkg.spiir_filter_static if static else pkg.spiir_filter
    with pkg.SpiirBank(inp.offsets, inp.a1, inp.b0, inp.delays, 0, pkg.SpiirOptions(path=pkg.PATH_STREAM)) as bank:
        pos = 0
        for c in chunks:
            fn(bank.handle, x[pos:pos + c], snr[:, pos:pos + c])
            pos += c
        torch.cuda.synchronize()
    return snr


def test_static_entry_matches_spiir_filter_on_consecutive_calls(env):
    pkg, oracle, torch = env
    inp = spiir_inputs.make_random_bank(91, [700, 64, 2048, 130, 1, 300, 1500, 90], 2 * 16 + 64 + 7 + 40 * 16, d_max=900)
    chunks = [16, 16, 64, 7] + [16] * 40            # two calls in a row first, then other sizes: the array is shared
    ref = oracle.run_inputs(inp)
    want = run(pkg, torch, inp, chunks, static=False)
    got = run(pkg, torch, inp, chunks, static=True)
    assert torch.isfinite(torch.view_as_real(got)).all()
    # after the first two calls already
    assert torch.equal(torch.view_as_real(got[:, :32]), torch.view_as_real(want[:, :32]))
    assert torch.equal(torch.view_as_real(got), torch.view_as_real(want))          # same kernels, same order: bitwise
    g = got.cpu().numpy().astype(np.complex128)
    err = np.abs(g - ref).max(axis=1) / np.abs(ref).max(axis=1)
    assert err.max() <= TOL, f"max relative error {err.max():.3e} at template {int(err.argmax())}"
    # a second bank through the same array right afterwards, and mixed with spiir_filter on one bank
    inp2 = spiir_inputs.make_random_bank(92, [256] * 12, 64 + 16, d_max=300)
    a = run(pkg, torch, inp2, [64, 16], static=True)
    b = run(pkg, torch, inp2, [64, 16], static=False)
    assert torch.equal(torch.view_as_real(a), torch.view_as_real(b))
    x = torch.from_numpy(inp2.x).cuda()
    c = torch.empty_like(a)
    with pkg.SpiirBank(inp2.offsets, inp2.a1, inp2.b0, inp2.delays, 0, pkg.SpiirOptions(path=pkg.PATH_STREAM)) as bank:
        pkg.spiir_filter(bank.handle, x[:64], c[:, :64])
        pkg.spiir_filter_static(bank.handle, x[64:], c[:, 64:])
        torch.cuda.synchronize()
    assert torch.equal(torch.view_as_real(c), torch.view_as_real(b))


def test_static_entry_rejects_what_it_cannot_serve_without_allocating(env):
    pkg, _, torch = env
    inp = spiir_inputs.make_random_bank(93, [128] * 4, 256, d_max=100)
    x = torch.from_numpy(inp.x).cuda()
    snr = torch.empty((inp.n_templates, inp.n_samples), dtype=torch.complex64, device="cuda")
    with pkg.SpiirBank(inp.offsets, inp.a1, inp.b0, inp.delays, 0, pkg.SpiirOptions(path=pkg.PATH_STREAM)) as bank:
        with pytest.raises(pkg.SpiirError) as ei:                   # more samples than the streaming kernels take per call
            pkg.spiir_filter_static(bank.handle, x[:65], snr[:, :65])
        assert ei.value.code == -1 and "64" in str(ei.value)
        pkg.spiir_filter_static(bank.handle, x[:64], snr[:, :64])   # the bank is still usable
    with pkg.SpiirBank(inp.offsets, inp.a1, inp.b0, inp.delays, 0, pkg.SpiirOptions()) as bank:
        with pytest.raises(pkg.SpiirError) as ei:                   # not a streaming bank
            pkg.spiir_filter_static(bank.handle, x[:16], snr[:, :16])
        assert ei.value.code == -1 and "SPIIR_PATH_STREAM" in str(ei.value)
    # more warp tiles than the static array holds: 8193 templates of one tile each
    big = spiir_inputs.make_random_bank(94, [8] * 8193, 16, d_max=50)
    xb = torch.from_numpy(big.x).cuda()
    sb = torch.empty((big.n_templates, 16), dtype=torch.complex64, device="cuda")
    with pkg.SpiirBank(big.offsets, big.a1, big.b0, big.delays, 0, pkg.SpiirOptions(path=pkg.PATH_STREAM)) as bank:
        with pytest.raises(pkg.SpiirError) as ei:
            pkg.spiir_filter_static(bank.handle, xb, sb)
        assert ei.value.code == -1 and "8192" in str(ei.value)
        pkg.spiir_filter(bank.handle, xb, sb)                       # the allocating path serves it
        torch.cuda.synchronize()
