"""B200-native grouped MoE-layer forward pass (BrownoutMoE full-brownout hot path).

The product is the C-ABI library declared in include/bm.h (hand-written sm_100a CUDA kernels under
csrc/); this package is its thin Python binding.  Importing the package does not load CUDA; the first
call loads (and if needed builds) libbm.so.
"""
from .binding import (  # noqa: F401
    BM_DEV_BAD_GROUP_MAP, BM_DEV_BAD_ROUTING, BM_DEV_NONFINITE_LOGIT, BM_PATH_AUTO, BM_PATH_DECODE,
    BM_PATH_PREFILL, BM_PATH_SIMT, BM_PATH_GEMV, BM_DECODE_MAX_T, BmError, Routing, alloc_workspace, bm_device_status, bm_moe_forward,
    bm_moe_layer_host, bm_moe_layer, bm_route, bm_route_partial, bm_unite_weights, bm_expert_histogram, bm_expert_outputs,
    bm_cosine_gram, bm_group_mse, bm_moe_forward_f32, bm_round_bf16, launch_count, lib, profile_enable, profile_read, profile_read_kinds, status_string,
    workspace_bytes, KERNELS, Salc, bm_salc_cold_mask, set_option, get_option, options, bm_forward_info, bm_host_chunks, BM_MAX_S,
    bm_route_static, bm_route_static_status, BM_ERR_LIMIT, BM_STATIC_ROUTE_BYTES, BM_STATIC_ROUTE_MAX_T,
)
from .tp import shard_f, tp_moe_forward  # noqa: F401,E402
from . import tp  # noqa: F401,E402
