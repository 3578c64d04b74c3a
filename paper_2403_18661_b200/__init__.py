"""B200-native (sm_100a) Aframe streaming detection statistic (arXiv 2403.18661).

The product is the C-ABI library declared in include/aframe.h (built from csrc/ into
libaframe_b200.so); this package is its thin ctypes binding.  No CPU fallback exists.
"""
from .binding import (  # noqa: F401
    AframeError, Context, Stream, Weights, aframe_config, default_config, describe_shared_plan, describe_stream_plan, load_library, LIB_PATH, EXPORTS,
    OK, EINVAL, ESHAPE, ENOMEM, ECUDA, ESTATE, EUNSUPPORTED, FP32, BF16, F16,
)
