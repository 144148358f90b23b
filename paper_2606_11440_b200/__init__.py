"""paper_2606_11440_b200 — B200-native (sm_100a) rollout + returns of the INFRAMIND hierarchical CMDP.

The product is libinframind.so (C ABI in include/inframind.h, CUDA sources in csrc/); this package only
builds it (build.py) and marshals arguments to it (binding.py).  No CPU fallback exists.
"""
from .binding import (  # noqa: F401
    InfraMind, IMError, load_library, marshal_spec, EXPORTS, gae_static, IM_GAE_STATIC_MAX_ENVS,
    IM_FLAG_LOG_DECISIONS, IM_FLAG_LOG_LOGITS,
    IM_TEL_SNAPSHOT, IM_TEL_COUNTERS, IM_TEL_REW, IM_TEL_COST, IM_TEL_VAL, IM_TEL_DONE, IM_TEL_MISS, IM_TEL_ADV,
    IM_TEL_RET, IM_TEL_SCALARS, IM_TEL_DECISIONS_EXEC, IM_TEL_DECISIONS_PLAN, IM_TEL_QUERIES, IM_TEL_UNORM,
    IM_TEL_STATE, IM_TEL_QUEUE_ORDER, IM_TEL_TABLES, IM_TEL_LOGITS_EXEC, IM_TEL_LOGITS_PLAN, IM_TEL_SUMS,
)
