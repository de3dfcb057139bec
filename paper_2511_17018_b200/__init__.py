"""paper_2511_17018_b200 -- B200-native (sm_100a) TPC clusterizer.

The product is ``libtpcclus.so`` (C ABI in ``include/tpcclus.h``, CUDA in ``csrc/``); this
package is its thin ctypes binding.  PyTorch appears only as the owner of device memory and
streams.  There is no CPU fallback: importing works without a GPU (so the build can be
checked), every compute call needs one.
"""
from .binding import (  # noqa: F401
    CLUSTER16_DTYPE, CLUSTER_DTYPE, COG_GATED, COG_SHARED, DIGIT_DTYPE, FLAG_EDGE_PAD, FLAG_EDGE_TIME, FLAG_SATURATED, MODE_DETERMINISTIC, MODE_FAST,
    RTC, STATUS_BAD_DIGITS, STATUS_INTERNAL, STATUS_NO_PACKED, STATUS_OVERFLOW, Clusterizer, TpcclusError, lib, tpcclus_params, tpcclus_out,
    tpcclus_set_rtc_cache_dir, tpcclus_pack_noalloc, NOALLOC_MAX_ROWS,
)
