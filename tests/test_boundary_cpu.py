"""CPU-side checks of the C-ABI boundary: the library loads, exports every symbol include/spiir.h declares,
validates arguments, and fails loudly (never falls back) when no CUDA device is present."""
import ctypes
import re
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def pkg():
    import __graft_entry__ as entry
    entry.build()
    import paper_1602_05573_b200 as p
    return p


def test_header_symbols_are_exported(pkg):
    header = (ROOT / "include" / "spiir.h").read_text()
    declared = set(re.findall(r"\b(spiir_[a-z_0-9]+)\s*\(", header))
    declared -= {"spiir_options"}
    assert {"spiir_bank_create", "spiir_filter", "spiir_bank_destroy"} <= declared
    lib = pkg.load_library()
    for name in sorted(declared):
        assert hasattr(lib, name), f"{name} declared in include/spiir.h but not exported"
    assert declared == set(pkg.binding.EXPORTS)
    assert pkg.spiir_version() >= 100


def test_no_torch_types_in_the_abi():
    header = (ROOT / "include" / "spiir.h").read_text()
    assert "torch" not in header.lower() and "at::" not in header and 'extern "C"' in header


def test_argument_validation_happens_before_any_device_work(pkg):
    off = np.array([0, 2], np.int64)
    a1 = np.array([0.5, 0.5j], np.complex64)
    b0 = np.ones(2, np.complex64)
    d = np.zeros(2, np.int32)
    cases = [
        (np.array([0, 0], np.int64), a1[:0], b0[:0], d[:0], "no filters"),
        (off, np.array([1.0, 0.5j], np.complex64), b0, d, "|a1| >= 1"),
        (off, np.array([np.nan, 0.5j], np.complex64), b0, d, "non-finite"),
        (off, a1, b0, np.array([0, -1], np.int32), "negative delay"),
    ]
    for o, a, b, dd, what in cases:
        with pytest.raises(pkg.SpiirError) as ei:
            pkg.spiir_bank_create(o, a, b, dd)
        assert ei.value.code == -1 and what in str(ei.value), what
    with pytest.raises(pkg.SpiirError) as ei:
        pkg.spiir_bank_create(off, a1, b0, d, options=pkg.SpiirOptions(filters_per_thread=3))
    assert ei.value.code == -1
    lib = pkg.load_library()
    assert lib.spiir_bank_num_templates(None) == -1 and lib.spiir_bank_destroy(None) == 0
    assert lib.spiir_filter(None, None, 0, None, 0, None) == -1


def test_every_invalid_blocking_pair_is_rejected_at_create(pkg):
    # spiir.h lists the valid (filters_per_thread, warps_per_cta) pairs as a create-time contract: every other pair must
    # come back SPIIR_EINVAL from spiir_bank_create itself (before any device work), not from the first spiir_filter
    off = np.array([0, 300], np.int64)
    rng = np.random.default_rng(3)
    a1 = (0.9 * np.exp(1j * rng.uniform(0, 1, 300))).astype(np.complex64)
    b0 = np.ones(300, np.complex64)
    d = rng.integers(0, 50, 300).astype(np.int32)
    valid = {(16, 8), (8, 8), (8, 16), (4, 8), (4, 16), (4, 32), (2, 32), (1, 32)}
    import torch
    for F in (1, 2, 4, 8, 16):
        for W in (8, 16, 32):
            opt = pkg.SpiirOptions(filters_per_thread=F, warps_per_cta=W)
            if (F, W) in valid:
                if torch.cuda.is_available():
                    pkg.spiir_bank_destroy(pkg.spiir_bank_create(off, a1, b0, d, options=opt))
                else:
                    with pytest.raises(pkg.SpiirError) as ei:
                        pkg.spiir_bank_create(off, a1, b0, d, options=opt)
                    assert ei.value.code == -3                     # got past the validation, stopped at "no device"
            else:
                with pytest.raises(pkg.SpiirError) as ei:
                    pkg.spiir_bank_create(off, a1, b0, d, options=opt)
                assert ei.value.code == -1 and "unsupported blocking" in str(ei.value), (F, W)
    # the streaming path comes with 8 warps: filters_per_thread 1 and 2 have no kernel there
    for F in (1, 2):
        with pytest.raises(pkg.SpiirError) as ei:
            pkg.spiir_bank_create(off, a1, b0, d, options=pkg.SpiirOptions(path=pkg.PATH_STREAM, filters_per_thread=F))
        assert ei.value.code == -1
    # scan_launches is 0, 1 or 3
    opt = pkg.SpiirOptions()
    opt.scan_launches = 7
    with pytest.raises(pkg.SpiirError) as ei:
        pkg.spiir_bank_create(off, a1, b0, d, options=opt)
    assert ei.value.code == -1 and "scan_launches" in str(ei.value)


def test_fails_loudly_without_a_gpu(pkg):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(pkg.SpiirError) as ei:
        pkg.spiir_bank_create(np.array([0, 1], np.int64), np.array([0.5], np.complex64),
                              np.ones(1, np.complex64), np.zeros(1, np.int32))
    assert ei.value.code == -3 and "no CPU fallback" in str(ei.value)


def test_product_never_imports_the_oracle():
    for path in list((ROOT / "paper_1602_05573_b200").rglob("*.py")) + list((ROOT / "paper_1602_05573_b200").rglob("*.cu*")) \
            + list((ROOT / "paper_1602_05573_b200").rglob("*.hpp")):
        text = path.read_text()
        assert "oracle" not in text, f"{path} mentions the oracle"
    for path in (ROOT / "oracle").rglob("*"):
        if path.is_file() and path.suffix in (".py", ".c", ".h"):
            assert "paper_1602_05573_b200" not in path.read_text().replace("paper_1602_05573_b200/ (the CUDA path)", "") \
                .replace("(``paper_1602_05573_b200``)", ""), f"{path} references the CUDA package"
