"""B200-native SPIIR template-bank filter (arxiv 1602.05573 section 3).

Thin Python binding over the C-ABI library ``libspiir_b200.so`` (``include/spiir.h``): the functions
here have the same names as the C entry points and only marshal arguments; every step of the hot path
runs in the library's CUDA kernels.  There is no CPU fallback: without the built library or without a
CUDA device the calls raise.
"""
from .binding import (SpiirError, SpiirOptions, SpiirBank, spiir_bank_create, spiir_filter, spiir_filter_prepared, spiir_filter_static,  # noqa: F401
                      spiir_filter_peaks, spiir_filter_host, spiir_filter_host_async, spiir_bank_host_sync, spiir_bank_reset, spiir_bank_destroy, spiir_bank_num_templates,
                      spiir_bank_num_filters, spiir_bank_max_delay, spiir_bank_get_state,
                      spiir_bank_set_state, spiir_kernel_launches, spiir_last_error, spiir_version,
                      spiir_bank_last_path, spiir_layout_probe, shard_templates, load_library, library_path,
                      PATH_AUTO, PATH_THROUGHPUT, PATH_SCAN, PATH_STREAM)
