"""paper_1603_08357_b200 -- B200-native bond-list connected-component labeling (Komura, arXiv 1603.08357).

The product is the C-ABI CUDA library `libccl.so` (include/ccl.h).  This package is its thin Python binding: argument
marshalling only; PyTorch is used for device memory and streams.  There is no CPU fallback: importing `binding`
fails loudly if the library cannot be built or loaded.
"""
from .binding import (CclError, Stats, cluster_stats, cluster_stats_static, gen_cayley3, gen_honeycomb, gen_occupancy, gen_regular, gen_triangular, gen_wrap_vectors, wrap,  # noqa: F401
                      label, label_batch, label_nn, label_bits, label_bits_host, label_sweep_host, relabel_sequential, last_error, launch_count, lib, set_option, set_profile_events, set_tuning, scratch_bytes, trim_scratch,
                      validate_bonds, version)
