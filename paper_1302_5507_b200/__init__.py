"""B200-native batched semi-global affine-gap alignment (SOAP3-dp gapped-alignment stage).

The product is the C-ABI library ``libsdp.so`` (``include/sdp.h``) built from ``csrc/``; this
package is its thin Python binding plus the seeded input generators. There is no CPU fallback:
every entry point raises if the CUDA library is missing.
"""
__all__ = ["workloads", "shard"]

from . import shard, workloads  # noqa: E402,F401
from .binding import (  # noqa: E402,F401
    Context,
    DeviceBatch,
    HostResult,
    SDP_NO_PAIR,
    SdpError,
    best_per_read_static,
    load_library,
    sdp_measure_dpx_rate,
    sdp_version,
)

__all__ += ["Context", "DeviceBatch", "HostResult", "SdpError", "best_per_read_static", "load_library", "sdp_measure_dpx_rate",
            "sdp_version"]
