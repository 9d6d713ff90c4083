"""B200-native (sm_100a) hot path of arXiv 2201.06914: FD wave propagation with the randomized-trace
imaging condition fused into the time loop.  Thin Python binding over the C ABI in include/rtm.h.

There is no CPU fallback: importing the binding fails loudly if the CUDA library is missing."""
from .binding import (RTMError, Rtm, RtmConfig, coeffs_host, coeffs_host3, lib_path, load_library, offset_gather_static, probes_dtt_host, probes_qr_host,
                      workspace_bytes)  # noqa: F401
