"""paper_1711_06203_b200 -- B200-native per-zone nuclear burn (arXiv 1711.06203, section 4).

Thin Python binding over the C ABI of include/burnzones.h (libburn.so, hand-written fp64 CUDA
for sm_100a).  PyTorch is used for device memory and streams only.  There is no CPU fallback:
without the built library or without a CUDA device every compute call raises.
"""
from .binding import (  # noqa: F401
    BurnError, Net, net_create, burn_zones, burn_zones_src, strang_step, burn_zones_host, net_destroy, get_counters,
    fp64_peak_probe, library_path, COUNTER_NAMES, EXPORTED_SYMBOLS, burn_zones_static, STATIC_SCRATCH_BYTES,
)
from .sharding import shard_range, shard_workload  # noqa: F401
