"""B200-native SAP attention hot path (arxiv/paper_2606_30460): Python binding of the C-ABI library."""
from .api import (Stitched, sap_attn_fwd_items, sap_attn_bwd_items, sap_axpy, sap_attn_fwd_chunks, sap_attn_bwd_begin, sap_attn_bwd_chunks, sap_attn_bwd_end, Plan, SapError, sap_plan, sap_attn_fwd, sap_attn_fwd_partial, sap_lse_merge, sap_attn_bwd, sap_attn_bwd_static,
                  sap_workspace_bytes, sap_launch_count, sap_debug_set_bwd_stages, sap_debug_set_fwd_form, sap_debug_set_bwd_form, SAP_MASK_SKIP, SAP_MASK_FULL, SAP_MASK_DIAG,
                  SAP_PASS_FWD, SAP_PASS_BWD, SAP_SCHED_RING, SAP_SCHED_BALANCED,
                  SAP_OP_SEND, SAP_OP_RECV, SAP_OP_COMPUTING, SAP_OP_COPY, SAP_T_Q, SAP_T_KV, SAP_T_O, SAP_T_DO, SAP_T_DQ, SAP_T_DKV)

__all__ = ["Stitched", "sap_attn_fwd_items", "sap_attn_bwd_items", "sap_axpy", "sap_attn_fwd_chunks", "sap_attn_bwd_begin", "sap_attn_bwd_chunks", "sap_attn_bwd_end", "Plan", "SapError", "sap_plan", "sap_attn_fwd", "sap_attn_fwd_partial", "sap_lse_merge", "sap_attn_bwd", "sap_attn_bwd_static",
           "sap_workspace_bytes", "sap_launch_count", "sap_debug_set_bwd_stages", "sap_debug_set_fwd_form", "sap_debug_set_bwd_form", "SAP_MASK_SKIP", "SAP_MASK_FULL", "SAP_MASK_DIAG",
           "SAP_PASS_FWD", "SAP_PASS_BWD", "SAP_SCHED_RING", "SAP_SCHED_BALANCED",
           "SAP_OP_SEND", "SAP_OP_RECV", "SAP_OP_COMPUTING", "SAP_OP_COPY", "SAP_T_Q", "SAP_T_KV", "SAP_T_O", "SAP_T_DO", "SAP_T_DQ", "SAP_T_DKV"]
