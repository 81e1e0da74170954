"""B200-native finite-volume step of the 2-D Shallow-Water Equations (arXiv 2010.14416).

`binding` wraps the C ABI of libswe_b200 (include/swe.h); `workloads` holds the seeded
synthetic inputs.  The CUDA library is the only compute path.
"""
from .binding import (LOOP_AUTO, LOOP_GRAPH, LOOP_LAUNCH, LOOP_PERSISTENT, ORDER_HILBERT,  # noqa: F401
                      ORDER_IDENTITY, ORDER_RCM, SweError, SweMesh, load_library)
