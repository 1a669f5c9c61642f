"""CPU oracle for the SPIIR template-bank filter -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with the CUDA path
(``paper_1602_05573_b200``) and neither imports the other.

The arithmetic lives in ``spiir_oracle.c`` (plain C, IEEE double, loop order template -> sample ->
filter; see that file's header for the passages it follows: BASELINE.json:north_star formula,
PAPER.md:L303, L323-L329, L339).  This file only compiles it with gcc and marshals numpy arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "spiir_oracle.c"
_LIB = _HERE / "_build" / "libspiir_oracle.so"
# Baseline x86-64 ISA on purpose (the built .so travels to another machine); contraction off so the
# result is the plain IEEE-double evaluation of the written expression on any host.
_CFLAGS = ["-O3", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-Wall"]

_lib = None


def build(force: bool = False) -> Path:
    """Compile the oracle (building the checker is not using it)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        _LIB.parent.mkdir(exist_ok=True)
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        subprocess.run(["gcc", *_CFLAGS, "-o", str(tmp), str(_SRC)], check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(str(build()))
        c_i64p = ctypes.POINTER(ctypes.c_int64)
        c_i32p = ctypes.POINTER(ctypes.c_int32)
        c_f32p = ctypes.POINTER(ctypes.c_float)
        c_f64p = ctypes.POINTER(ctypes.c_double)
        lib.spiir_oracle_run.restype = ctypes.c_int
        lib.spiir_oracle_run.argtypes = [ctypes.c_int32, c_i64p, c_f32p, c_f32p, c_i32p, c_f32p,
                                         ctypes.c_int64, c_f64p, ctypes.c_int64, ctypes.c_int32]
        lib.spiir_oracle_stream_create.restype = ctypes.c_void_p
        lib.spiir_oracle_stream_create.argtypes = [ctypes.c_int32, c_i64p, c_f32p, c_f32p, c_i32p]
        lib.spiir_oracle_stream_filter.restype = ctypes.c_int
        lib.spiir_oracle_stream_filter.argtypes = [ctypes.c_void_p, c_f32p, ctypes.c_int64, c_f64p,
                                                   ctypes.c_int64, ctypes.c_int32]
        lib.spiir_oracle_stream_destroy.restype = None
        lib.spiir_oracle_stream_destroy.argtypes = [ctypes.c_void_p]
        lib.spiir_oracle_filter_outputs.restype = ctypes.c_int
        lib.spiir_oracle_filter_outputs.argtypes = [ctypes.c_int64, c_f32p, c_f32p, c_i32p, c_f32p,
                                                    ctypes.c_int64, c_f64p]
        lib.spiir_oracle_max_threads.restype = ctypes.c_int32
        _lib = lib
    return _lib


def _p(arr, ctype):
    return arr.ctypes.data_as(ctypes.POINTER(ctype))


def _bank_arrays(offsets, a1, b0, delays):
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    a1 = np.ascontiguousarray(a1, dtype=np.complex64)
    b0 = np.ascontiguousarray(b0, dtype=np.complex64)
    delays = np.ascontiguousarray(delays, dtype=np.int32)
    K = int(offsets[-1])
    if not (a1.shape == b0.shape == delays.shape == (K,)):
        raise ValueError("bank arrays must all have offsets[-1] entries")
    return offsets, a1, b0, delays


def max_threads() -> int:
    return int(_load().spiir_oracle_max_threads())


def run(offsets, a1, b0, delays, x, n_threads: int = 0) -> np.ndarray:
    """One-shot oracle: complex128 SNR[T][N] for the whole strain series ``x`` (float32)."""
    lib = _load()
    offsets, a1, b0, delays = _bank_arrays(offsets, a1, b0, delays)
    x = np.ascontiguousarray(x, dtype=np.float32)
    T, N = offsets.size - 1, x.size
    snr = np.empty((T, N), dtype=np.complex128)
    rc = lib.spiir_oracle_run(T, _p(offsets, ctypes.c_int64), _p(a1.view(np.float32), ctypes.c_float),
                              _p(b0.view(np.float32), ctypes.c_float), _p(delays, ctypes.c_int32),
                              _p(x, ctypes.c_float), N, _p(snr.view(np.float64), ctypes.c_double),
                              N, n_threads)
    if rc != 0:
        raise RuntimeError(f"spiir_oracle_run failed ({rc})")
    return snr


def run_inputs(inp, n_threads: int = 0) -> np.ndarray:
    return run(inp.offsets, inp.a1, inp.b0, inp.delays, inp.x, n_threads)


def filter_outputs(a1, b0, delays, x) -> np.ndarray:
    """Per-filter outputs y_k[n] (complex128 [K][N]) of one template, not summed."""
    lib = _load()
    a1 = np.ascontiguousarray(a1, dtype=np.complex64)
    b0 = np.ascontiguousarray(b0, dtype=np.complex64)
    delays = np.ascontiguousarray(delays, dtype=np.int32)
    x = np.ascontiguousarray(x, dtype=np.float32)
    K, N = a1.size, x.size
    y = np.empty((K, N), dtype=np.complex128)
    rc = lib.spiir_oracle_filter_outputs(K, _p(a1.view(np.float32), ctypes.c_float),
                                         _p(b0.view(np.float32), ctypes.c_float),
                                         _p(delays, ctypes.c_int32), _p(x, ctypes.c_float), N,
                                         _p(y.view(np.float64), ctypes.c_double))
    if rc != 0:
        raise RuntimeError(f"spiir_oracle_filter_outputs failed ({rc})")
    return y


def peaks(snr: np.ndarray, j0: int = 0, n: int | None = None):
    """power[t] = max_j |snr[t, j0 + j]|^2 over j in [0, n), index[t] = first such j.  snr complex128 [T][N]."""
    lib = _load()
    snr = np.ascontiguousarray(snr, dtype=np.complex128)
    T, N = snr.shape
    n = N - j0 if n is None else n
    if n < 1 or j0 < 0 or j0 + n > N:
        raise ValueError("need 0 <= j0 and 1 <= n <= N - j0")
    power = np.empty(T, dtype=np.float64)
    index = np.empty(T, dtype=np.int64)
    lib.spiir_oracle_peaks.restype = ctypes.c_int
    rc = lib.spiir_oracle_peaks(ctypes.c_int32(T), _p(snr.view(np.float64), ctypes.c_double), ctypes.c_int64(N),
                                ctypes.c_int64(j0), ctypes.c_int64(n), _p(power, ctypes.c_double),
                                _p(index, ctypes.c_int64))
    if rc != 0:
        raise RuntimeError(f"spiir_oracle_peaks failed ({rc})")
    return power, index


class Stream:
    """Streaming oracle: state and the whole input past are carried across ``filter`` calls."""

    def __init__(self, offsets, a1, b0, delays):
        self._lib = _load()
        self._arrs = _bank_arrays(offsets, a1, b0, delays)
        offsets, a1, b0, delays = self._arrs
        self.n_templates = offsets.size - 1
        self._h = self._lib.spiir_oracle_stream_create(
            self.n_templates, _p(offsets, ctypes.c_int64), _p(a1.view(np.float32), ctypes.c_float),
            _p(b0.view(np.float32), ctypes.c_float), _p(delays, ctypes.c_int32))
        if not self._h:
            raise MemoryError("spiir_oracle_stream_create failed")

    def filter(self, x, n_threads: int = 0) -> np.ndarray:
        x = np.ascontiguousarray(x, dtype=np.float32)
        n = x.size
        snr = np.empty((self.n_templates, n), dtype=np.complex128)
        rc = self._lib.spiir_oracle_stream_filter(self._h, _p(x, ctypes.c_float), n,
                                                  _p(snr.view(np.float64), ctypes.c_double), n, n_threads)
        if rc != 0:
            raise RuntimeError(f"spiir_oracle_stream_filter failed ({rc})")
        return snr

    def close(self):
        if self._h:
            self._lib.spiir_oracle_stream_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
