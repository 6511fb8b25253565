"""B200-native geometric-network simulation step (arxiv 0908.3934 hot path) behind a C ABI.

`include/gn.h` declares the boundary; `csrc/` holds the CUDA kernels and host logic compiled into
`libgn.so`; `binding` is the thin Python layer with the same names.
"""
from .binding import (  # noqa: F401
    GN_ACC, GN_BIAS, GN_CA, GN_DELIVER_AUTO, GN_DELIVER_QUEUE, GN_DELIVER_RESIDENT, GN_DELIVER_RING, GN_DELIVER_RING_STEPWISE, GN_DRIVER, GN_DRIVER_FUSED, GN_DRIVER_PERSISTENT,
    GN_DRIVER_PLASTIC, GN_DRIVER_QUEUE, GN_DRIVER_RESIDENT, GN_DRIVER_RING, GN_COUNTERS, GN_DELAYS, GN_E_BAD_GRAPH, GN_E_CUDA, GN_E_INVALID_ARG, GN_E_OVERFLOW_RISK,
    GN_E_RANGE_EVICTED, GN_E_WORKSPACE_TOO_SMALL, GN_FAULTS, GN_H, GN_M, GN_MODEL_HODGKIN_HUXLEY, GN_MODEL_IZHIKEVICH, GN_OK, GN_P, GN_R, GN_REFR, GN_RING, GN_STEP, GN_V, GN_W,
    GN_STATIC_MAX_VERTICES, GN_WEIGHTS, GN_WEIGHTS_FX, EXPORTS, GnError, GnNet, create_from_inputs, gn_class_params, gn_config, gn_create,
    gn_check_headroom_static, gn_debug_ceilings, gn_debug_stream_ceilings, gn_debug_words, gn_destroy, gn_observe, gn_profile, gn_profile_read, gn_query_workspace, gn_read_raster, gn_read_state, gn_step,
    gn_write_state, lib, make_config)
from .build import build  # noqa: F401
