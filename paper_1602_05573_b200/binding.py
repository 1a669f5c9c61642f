"""ctypes binding of include/spiir.h -- argument marshalling only."""
from __future__ import annotations

import ctypes
from pathlib import Path

import numpy as np

_PKG = Path(__file__).resolve().parent
_LIB_PATH = _PKG / "libspiir_b200.so"
_lib = None

PATH_AUTO, PATH_THROUGHPUT, PATH_SCAN, PATH_STREAM = 0, 1, 2, 3

EXPORTS = ["spiir_bank_create", "spiir_filter", "spiir_filter_host", "spiir_bank_reset",
           "spiir_bank_num_templates", "spiir_bank_num_filters", "spiir_bank_max_delay",
           "spiir_bank_get_state", "spiir_bank_set_state", "spiir_bank_destroy", "spiir_last_error",
           "spiir_kernel_launches", "spiir_bank_last_path", "spiir_version", "spiir_layout_probe",
           "spiir_filter_host_async", "spiir_bank_host_sync", "spiir_filter_peaks", "spiir_filter_static"]


class SpiirError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"spiir error {code}: {msg}")
        self.code = code


class SpiirOptions(ctypes.Structure):
    _fields_ = [("struct_size", ctypes.c_int32), ("path", ctypes.c_int32),
                ("filters_per_thread", ctypes.c_int32), ("scan_segments", ctypes.c_int32),
                ("warps_per_cta", ctypes.c_int32), ("window_copies", ctypes.c_int32),
                ("small_templates", ctypes.c_int32), ("scan_launches", ctypes.c_int32)]

    def __init__(self, path: int = PATH_AUTO, filters_per_thread: int = 0, scan_segments: int = 0,
                 warps_per_cta: int = 0, window_copies: int = 0, small_templates: int = 0, scan_launches: int = 0):
        super().__init__()
        self.struct_size = ctypes.sizeof(SpiirOptions)
        self.path, self.filters_per_thread, self.scan_segments = path, filters_per_thread, scan_segments
        self.warps_per_cta = warps_per_cta
        self.window_copies = window_copies
        self.small_templates = small_templates
        self.scan_launches = scan_launches


def library_path() -> Path:
    return _LIB_PATH


def load_library():
    """Load libspiir_b200.so (built in-tree by ``__graft_entry__.build()``); fails loudly if missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not _LIB_PATH.exists():
        raise FileNotFoundError(f"{_LIB_PATH} is not built: run `python -c 'import __graft_entry__ as g; g.build()'` "
                                "(there is no CPU fallback)")
    lib = ctypes.CDLL(str(_LIB_PATH))
    vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
    lib.spiir_bank_create.restype = ctypes.c_int
    lib.spiir_bank_create.argtypes = [ctypes.POINTER(vp), i32, vp, vp, vp, vp, i32, ctypes.POINTER(SpiirOptions)]
    lib.spiir_filter.restype = ctypes.c_int
    lib.spiir_filter.argtypes = [vp, vp, i64, vp, i64, vp]
    lib.spiir_filter_static.restype = ctypes.c_int
    lib.spiir_filter_static.argtypes = [vp, vp, i64, vp, i64, vp]
    lib.spiir_filter_host.restype = ctypes.c_int
    lib.spiir_filter_host.argtypes = [vp, vp, i64, vp, i64]
    lib.spiir_filter_host_async.restype = ctypes.c_int
    lib.spiir_filter_host_async.argtypes = [vp, vp, i64, vp, i64]
    lib.spiir_bank_host_sync.restype = ctypes.c_int
    lib.spiir_bank_host_sync.argtypes = [vp]
    lib.spiir_filter_peaks.restype = ctypes.c_int
    lib.spiir_filter_peaks.argtypes = [vp, vp, i64, vp, i64, vp, vp, vp]
    lib.spiir_bank_reset.restype = ctypes.c_int
    lib.spiir_bank_reset.argtypes = [vp, vp]
    for name in ("spiir_bank_num_templates", "spiir_bank_num_filters", "spiir_bank_max_delay"):
        getattr(lib, name).restype = i64
        getattr(lib, name).argtypes = [vp]
    lib.spiir_bank_get_state.restype = ctypes.c_int
    lib.spiir_bank_get_state.argtypes = [vp, vp, vp, vp]
    lib.spiir_bank_set_state.restype = ctypes.c_int
    lib.spiir_bank_set_state.argtypes = [vp, vp, vp, vp]
    lib.spiir_bank_destroy.restype = ctypes.c_int
    lib.spiir_bank_destroy.argtypes = [vp]
    lib.spiir_last_error.restype = ctypes.c_char_p
    lib.spiir_kernel_launches.restype = i64
    lib.spiir_bank_last_path.restype = i32
    lib.spiir_bank_last_path.argtypes = [vp]
    lib.spiir_version.restype = i32
    lib.spiir_layout_probe.restype = ctypes.c_int
    lib.spiir_layout_probe.argtypes = [i32, vp, vp, i32, i32, i32, vp, vp, i32]
    _lib = lib
    return lib


def _check(rc: int):
    if rc != 0:
        raise SpiirError(rc, load_library().spiir_last_error().decode())


def _ptr(a: np.ndarray):
    return ctypes.c_void_p(a.ctypes.data)


def _stream_handle(stream) -> ctypes.c_void_p:
    if stream is None:
        import torch
        return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return ctypes.c_void_p(stream)
    return ctypes.c_void_p(stream.cuda_stream)


def spiir_bank_create(filter_offsets, a1, b0, delays, device: int = 0, options: SpiirOptions | None = None):
    """-> opaque bank handle.  Host numpy arrays: int64 [T+1], complex64 [K], complex64 [K], int32 [K]."""
    lib = load_library()
    off = np.ascontiguousarray(filter_offsets, dtype=np.int64)
    a1 = np.ascontiguousarray(a1, dtype=np.complex64)
    b0 = np.ascontiguousarray(b0, dtype=np.complex64)
    d = np.ascontiguousarray(delays, dtype=np.int32)
    K = int(off[-1]) if off.size else 0
    if off.ndim != 1 or off.size < 1 or not (a1.shape == b0.shape == d.shape == (K,)):
        raise ValueError("filter_offsets must be [T+1] and a1, b0, delays must have filter_offsets[-1] entries")
    h = ctypes.c_void_p()
    _check(lib.spiir_bank_create(ctypes.byref(h), off.size - 1, _ptr(off), _ptr(a1), _ptr(b0), _ptr(d),
                                 device, ctypes.byref(options) if options is not None else None))
    return h


def _check_rows(bank, snr, *others):
    """Marshalling checks only: the output tensors must have one row / entry per template and live on x's device."""
    T = int(load_library().spiir_bank_num_templates(bank))
    if snr is not None and (snr.dim() != 2 or snr.shape[0] != T):
        raise ValueError(f"snr must have one row per template ({T}), got shape {tuple(snr.shape)}")
    for name, t in others:
        if t is not None and t.numel() != T:
            raise ValueError(f"{name} must have one entry per template ({T}), got {t.numel()}")


def spiir_filter(bank, x, snr, ld: int | None = None, stream=None, n: int | None = None):
    """x: CUDA float32 tensor [n]; snr: CUDA complex64 tensor whose row t starts ``ld`` elements after row t-1
    (a [T, ld] tensor, or a column slice ``big[:, c0:c0+n]`` of one).  Enqueues on ``stream``."""
    import torch
    if x.dtype != torch.float32 or not x.is_cuda or not x.is_contiguous():
        raise ValueError("x must be a contiguous CUDA float32 tensor")
    if snr.dtype != torch.complex64 or not snr.is_cuda:
        raise ValueError("snr must be a CUDA complex64 tensor")
    if snr.device != x.device:
        raise ValueError("x and snr must be on the same device (the bank's)")
    _check_rows(bank, snr)
    n = int(x.numel()) if n is None else int(n)
    if ld is None:
        if snr.dim() != 2 or (snr.shape[1] > 1 and snr.stride(1) != 1) or snr.shape[1] < n:
            raise ValueError("snr must be [T, >=n] with unit column stride")
        ld = int(snr.stride(0)) if snr.shape[0] > 1 else max(int(snr.shape[1]), n)
    _check(load_library().spiir_filter(bank, ctypes.c_void_p(x.data_ptr()), n, ctypes.c_void_p(snr.data_ptr()),
                                       int(ld), _stream_handle(stream)))


def spiir_filter_static(bank, x, snr, ld: int | None = None, stream=None):
    """``spiir_filter`` through the entry point that allocates nothing (SPIIR_PATH_STREAM banks, n <= 64, <= 8192 warp
    tiles): the partial sums go to a 4 MiB file-scope device array of the library instead of a cudaMalloc'ed buffer."""
    import torch
    if x.dtype != torch.float32 or not x.is_cuda or not x.is_contiguous():
        raise ValueError("x must be a contiguous CUDA float32 tensor")
    if snr.dtype != torch.complex64 or not snr.is_cuda or snr.device != x.device:
        raise ValueError("snr must be a CUDA complex64 tensor on x's device")
    _check_rows(bank, snr)
    n = int(x.numel())
    if ld is None:
        if snr.dim() != 2 or (snr.shape[1] > 1 and snr.stride(1) != 1) or snr.shape[1] < n:
            raise ValueError("snr must be [T, >=n] with unit column stride")
        ld = int(snr.stride(0)) if snr.shape[0] > 1 else max(int(snr.shape[1]), n)
    _check(load_library().spiir_filter_static(bank, ctypes.c_void_p(x.data_ptr()), n, ctypes.c_void_p(snr.data_ptr()),
                                              int(ld), _stream_handle(stream)))


def spiir_filter_prepared(bank, x, snr, ld: int | None = None, stream=None):
    """The arguments of one ``spiir_filter`` call checked and marshalled once: returns a zero-argument callable that makes
    the C call with the same pointers every time (a streaming loop that reuses its buffers then pays the library's own host
    time per call, not tensor slicing and argument checks: 9 instead of 30 us, measured)."""
    import torch
    if x.dtype != torch.float32 or not x.is_cuda or not x.is_contiguous():
        raise ValueError("x must be a contiguous CUDA float32 tensor")
    if snr.dtype != torch.complex64 or not snr.is_cuda or snr.device != x.device:
        raise ValueError("snr must be a CUDA complex64 tensor on x's device")
    _check_rows(bank, snr)
    n = int(x.numel())
    if ld is None:
        if snr.dim() != 2 or (snr.shape[1] > 1 and snr.stride(1) != 1) or snr.shape[1] < n:
            raise ValueError("snr must be [T, >=n] with unit column stride")
        ld = int(snr.stride(0)) if snr.shape[0] > 1 else max(int(snr.shape[1]), n)
    fn = load_library().spiir_filter
    args = (bank, ctypes.c_void_p(x.data_ptr()), n, ctypes.c_void_p(snr.data_ptr()), int(ld), _stream_handle(stream))
    keep = (x, snr)                      # the tensors stay alive as long as the callable does

    def call(_keep=keep):
        rc = fn(*args)
        if rc:
            _check(rc)
    return call


def spiir_filter_peaks(bank, x, power=None, index=None, snr=None, stream=None):
    """x: CUDA float32 [n]; power: CUDA float32 [T]; index: CUDA int32 [T]; snr: optional CUDA complex64 [T, >=n]."""
    import torch
    if x.dtype != torch.float32 or not x.is_cuda or not x.is_contiguous():
        raise ValueError("x must be a contiguous CUDA float32 tensor")
    for name, t, dt in (("power", power, torch.float32), ("index", index, torch.int32)):
        if t is not None and (t.dtype != dt or not t.is_cuda or not t.is_contiguous()):
            raise ValueError(f"{name} must be a contiguous CUDA {dt} tensor")
    for t in (power, index, snr):
        if t is not None and t.device != x.device:
            raise ValueError("x, power, index and snr must be on the same device (the bank's)")
    _check_rows(bank, snr, ("power", power), ("index", index))
    n, ld, snr_ptr = int(x.numel()), int(x.numel()), None
    if snr is not None:
        if snr.dtype != torch.complex64 or not snr.is_cuda or snr.dim() != 2 or snr.shape[1] < n or \
                (snr.shape[1] > 1 and snr.stride(1) != 1):
            raise ValueError("snr must be a CUDA complex64 [T, >=n] tensor with unit column stride")
        ld = int(snr.stride(0)) if snr.shape[0] > 1 else max(int(snr.shape[1]), n)
        snr_ptr = ctypes.c_void_p(snr.data_ptr())
    _check(load_library().spiir_filter_peaks(bank, ctypes.c_void_p(x.data_ptr()), n, snr_ptr, ld,
                                             ctypes.c_void_p(power.data_ptr()) if power is not None else None,
                                             ctypes.c_void_p(index.data_ptr()) if index is not None else None,
                                             _stream_handle(stream)))


def spiir_filter_host(bank, x: np.ndarray, snr: np.ndarray | None = None, asynchronous: bool = False) -> np.ndarray:
    """Host-buffer entry: x float32 [n] numpy -> complex64 [T, n] numpy (H2D, kernels, D2H inside).
    ``asynchronous`` = spiir_filter_host_async: x and snr must be pinned and stay untouched until spiir_bank_host_sync."""
    lib = load_library()
    if asynchronous:
        # the copy is still reading x when this returns: a converted temporary would be freed under it
        if not isinstance(x, np.ndarray) or x.dtype != np.float32 or x.ndim != 1 or not x.flags.c_contiguous:
            raise ValueError("asynchronous: x must already be a C-contiguous float32 array (pinned), no conversion is made")
        if snr is None:
            raise ValueError("asynchronous: pass the (pinned) snr buffer the results are written to")
    x = np.ascontiguousarray(x, dtype=np.float32)
    T = int(lib.spiir_bank_num_templates(bank))
    if snr is None:
        snr = np.empty((T, x.size), dtype=np.complex64)
    if snr.dtype != np.complex64 or snr.ndim != 2 or snr.shape[0] != T or snr.shape[1] < x.size or \
            (snr.shape[1] > 1 and snr.strides[1] != 8):
        raise ValueError("snr must be complex64 [T, >=n] with unit column stride")
    ld = snr.strides[0] // 8 if T > 1 else max(snr.shape[1], x.size)
    _check((lib.spiir_filter_host_async if asynchronous else lib.spiir_filter_host)(bank, _ptr(x), x.size, _ptr(snr), ld))
    return snr


def spiir_filter_host_async(bank, x: np.ndarray, snr: np.ndarray) -> np.ndarray:
    return spiir_filter_host(bank, x, snr, asynchronous=True)


def spiir_bank_host_sync(bank):
    _check(load_library().spiir_bank_host_sync(bank))


def spiir_bank_reset(bank, stream=None):
    _check(load_library().spiir_bank_reset(bank, _stream_handle(stream)))


def spiir_bank_num_templates(bank) -> int:
    return int(load_library().spiir_bank_num_templates(bank))


def spiir_bank_num_filters(bank) -> int:
    return int(load_library().spiir_bank_num_filters(bank))


def spiir_bank_max_delay(bank) -> int:
    return int(load_library().spiir_bank_max_delay(bank))


def spiir_bank_last_path(bank) -> int:
    return int(load_library().spiir_bank_last_path(bank))


def spiir_bank_get_state(bank, y=None, hist=None, stream=None):
    """y: CUDA complex64 [K] (caller's filter order); hist: CUDA float32 [D]; either may be None."""
    _check(load_library().spiir_bank_get_state(bank, ctypes.c_void_p(y.data_ptr()) if y is not None else None,
                                               ctypes.c_void_p(hist.data_ptr()) if hist is not None else None,
                                               _stream_handle(stream)))


def spiir_bank_set_state(bank, y=None, hist=None, stream=None):
    _check(load_library().spiir_bank_set_state(bank, ctypes.c_void_p(y.data_ptr()) if y is not None else None,
                                               ctypes.c_void_p(hist.data_ptr()) if hist is not None else None,
                                               _stream_handle(stream)))


def spiir_bank_destroy(bank):
    _check(load_library().spiir_bank_destroy(bank))


def spiir_kernel_launches() -> int:
    return int(load_library().spiir_kernel_launches())


def spiir_last_error() -> str:
    return load_library().spiir_last_error().decode()


def spiir_version() -> int:
    return int(load_library().spiir_version())


def spiir_layout_probe(filter_offsets, delays, filters_per_thread: int = 8, warps_per_cta: int = 16,
                       window_copies: int = 1, pack_small: bool = False):
    """Host-only: the device layout spiir_bank_create would build.  -> (slot_of_filter int64 [K], stats dict)."""
    off = np.ascontiguousarray(filter_offsets, dtype=np.int64)
    d = np.ascontiguousarray(delays, dtype=np.int32)
    if off.ndim != 1 or off.size < 1 or d.shape != (int(off[-1]),):
        raise ValueError("filter_offsets must be [T+1] and delays must have filter_offsets[-1] entries")
    slots = np.empty(d.size, dtype=np.int64)
    stats = np.zeros(8, dtype=np.float64)
    _check(load_library().spiir_layout_probe(off.size - 1, _ptr(off), _ptr(d), filters_per_thread, warps_per_cta,
                                             window_copies, _ptr(slots), _ptr(stats), int(pack_small)))
    names = ("n_slots", "n_warp_tiles", "n_cta_items", "n_rounds", "avg_conflict_degree", "padding_fraction",
             "uniform_groups", "segmented")
    return slots, dict(zip(names, stats.tolist()))


def shard_templates(filter_offsets, world_size: int):
    """Template indices of every rank for multi-GPU runs: templates are independent, so the
    bank is split by template with no data-path collective.  Longest-processing-time-first bin packing on the
    filter counts K_t; deterministic (ties: lower template index, lower rank).  -> list of sorted int64 arrays."""
    off = np.asarray(filter_offsets, dtype=np.int64)
    if world_size < 1 or off.ndim != 1 or off.size < 2:
        raise ValueError("need world_size >= 1 and filter_offsets [T+1]")
    kt = np.diff(off)
    order = np.lexsort((np.arange(kt.size), -kt))          # K_t descending, then index
    load = [0] * world_size
    parts = [[] for _ in range(world_size)]
    for t in order.tolist():
        r = min(range(world_size), key=lambda i: (load[i], i))
        parts[r].append(t)
        load[r] += int(kt[t])
    return [np.sort(np.asarray(p, dtype=np.int64)) for p in parts]


class SpiirBank:
    """Convenience owner of a bank handle (context manager); still argument marshalling only."""

    def __init__(self, filter_offsets, a1, b0, delays, device: int = 0, options: SpiirOptions | None = None):
        self.handle = spiir_bank_create(filter_offsets, a1, b0, delays, device, options)
        self.device = device
        self.n_templates = spiir_bank_num_templates(self.handle)
        self.n_filters = spiir_bank_num_filters(self.handle)
        self.max_delay = spiir_bank_max_delay(self.handle)

    def filter(self, x, snr=None, stream=None):
        import torch
        if snr is None:
            snr = torch.empty((self.n_templates, x.numel()), dtype=torch.complex64, device=x.device)
        spiir_filter(self.handle, x, snr, stream=stream)
        return snr

    def filter_host(self, x, snr=None):
        return spiir_filter_host(self.handle, x, snr)

    def reset(self, stream=None):
        spiir_bank_reset(self.handle, stream)

    @property
    def last_path(self) -> int:
        return spiir_bank_last_path(self.handle)

    def close(self):
        if self.handle is not None:
            spiir_bank_destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
