"""B200-native Line Segment Tracking object-building chain (arxiv 2407.18231) -- Python binding.

The product is the C-ABI CUDA library ``liblst_b200.so`` (include/lst.h, csrc/); this package only
marshals arguments.  It never imports ``oracle`` and has no CPU fallback.
"""
from .binding import (ABI_SYMBOLS, LST_ERR_ARG, LST_ERR_CAPACITY, LST_ERR_CUDA, LST_ERR_GEOMETRY, LST_ERR_LIMIT, LST_OK,  # noqa: F401
                      LST_SCAN_STATIC_MAX_N,
                      LstError, library_path, lst_caps, lst_default_caps, lst_default_params, lst_free,
                      lst_load_geometry, lst_params, lst_workspace_bytes)
from .api import (event_out_to_dict, lst_ctx_create, lst_ctx_fetch_event, lst_ctx_fetch_tc,  # noqa: F401
                  lst_ctx_kernel_times, lst_ctx_launch_count, lst_ctx_run, lst_ctx_set_blocks_per_sm, lst_ctx_set_graph, lst_ctx_set_timing, lst_ctx_sync,
                  lst_run_event, make_hits, make_pls, lst_ctx_stat, LST_STAT_PT_QUEUE, LST_STAT_WORKSPACE_MB,
                  lst_scan_counts, lst_scan_counts_static, lst_ctx_audit, AUDIT_STAGES)
