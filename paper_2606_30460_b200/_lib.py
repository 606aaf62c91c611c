"""Loads libsap_b200.so and declares the C ABI of include/sap.h for ctypes.  No fallback: a missing
library is an ImportError-class failure (RuntimeError), never a silent CPU path."""
from __future__ import annotations

import ctypes
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("SAP_B200_LIB", os.path.join(HERE, "libsap_b200.so"))  # override: instrumented builds

c_i32p = ctypes.POINTER(ctypes.c_int32)
c_f32p = ctypes.POINTER(ctypes.c_float)
vp = ctypes.c_void_p


class SapItem(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in ("q_chunk", "kv_chunk", "doc_lo", "doc_hi", "mask_kind", "step",
                                             "q_begin", "q_end", "kv_begin", "kv_end")]


# name -> (restype, argtypes); mirrors include/sap.h one to one
SIGNATURES = {
    "sap_plan_create": (ctypes.c_int, [vp, ctypes.c_int32, ctypes.c_int32, ctypes.POINTER(vp)]),
    "sap_plan_destroy": (None, [vp]),
    "sap_plan_n_items": (ctypes.c_int32, [vp]),
    "sap_plan_n_chunks": (ctypes.c_int32, [vp]),
    "sap_plan_n_tokens": (ctypes.c_int32, [vp]),
    "sap_plan_items": (ctypes.POINTER(SapItem), [vp]),
    "sap_plan_chunk_offsets": (c_i32p, [vp]),
    "sap_plan_kv_offsets": (c_i32p, [vp]),
    "sap_plan_kv_index": (c_i32p, [vp]),
    "sap_plan_kind_map": (ctypes.POINTER(ctypes.c_uint8), [vp]),
    "sap_plan_useful_pairs": (ctypes.c_int64, [vp]),
    "sap_plan_fwd_tiles": (ctypes.c_int64, [vp]),
    "sap_plan_schedule": (ctypes.c_int, [vp, ctypes.c_int32, vp, c_i32p]),
    "sap_plan_codegen": (ctypes.c_int32, [vp, vp, ctypes.c_int32, vp, ctypes.c_int32]),
    "sap_plan_codegen_bwd": (ctypes.c_int32, [vp, vp, ctypes.c_int32, vp, ctypes.c_int32]),
    "sap_plan_upload": (ctypes.c_int, [vp]),
    "sap_workspace_bytes": (ctypes.c_size_t, [vp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int]),
    "sap_attn_fwd": (ctypes.c_int, [vp, vp, vp, vp, vp, ctypes.c_int64, vp, vp, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                    ctypes.c_float, vp, ctypes.c_size_t, vp]),
    "sap_attn_fwd_partial": (ctypes.c_int, [vp, vp, vp, vp, vp, ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, vp, vp,
                                            ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_float, vp]),
    "sap_attn_fwd_items": (ctypes.c_int, [vp, vp, vp, vp, vp, ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, vp, vp,
                                          ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_float, vp]),
    "sap_lse_merge": (ctypes.c_int, [vp, vp, vp, vp, vp, ctypes.c_int, vp, ctypes.c_int64, ctypes.c_int,
                                     ctypes.c_int, ctypes.c_int64, ctypes.c_int64, vp]),
    "sap_attn_bwd": (ctypes.c_int, [vp, vp, vp, vp, vp, vp, vp, vp, ctypes.c_int64, vp, vp, vp, ctypes.c_int, ctypes.c_int,
                                    ctypes.c_int, ctypes.c_float, vp, ctypes.c_size_t, vp]),
    "sap_attn_bwd_static": (ctypes.c_int, [vp, vp, vp, vp, vp, vp, vp, vp, ctypes.c_int64, vp, vp, vp, ctypes.c_int, ctypes.c_int,
                                           ctypes.c_int, ctypes.c_float, vp]),
    "sap_attn_fwd_chunks": (ctypes.c_int, [vp, vp, vp, vp, vp, ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, vp, vp, ctypes.c_int,
                                           ctypes.c_int, ctypes.c_int, ctypes.c_float, vp]),
    "sap_attn_bwd_begin": (ctypes.c_int, [vp, vp, vp, ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, ctypes.c_int, ctypes.c_int,
                                          ctypes.c_int, vp, ctypes.c_size_t, vp]),
    "sap_attn_bwd_chunks": (ctypes.c_int, [vp, vp, vp, vp, vp, vp, vp, ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, vp, vp,
                                           ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_float, vp, ctypes.c_size_t, vp]),
    "sap_attn_bwd_items": (ctypes.c_int, [vp, vp, vp, vp, vp, vp, vp, ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, vp, vp,
                                          ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_float, vp, ctypes.c_size_t, vp]),
    "sap_axpy": (ctypes.c_int, [vp, ctypes.c_int, vp, ctypes.c_int, ctypes.c_int64, ctypes.c_float, ctypes.c_int, vp]),
    "sap_attn_bwd_end": (ctypes.c_int, [vp, ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, vp, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                        ctypes.c_float, vp, ctypes.c_size_t, vp]),
    "sap_stitched_granularity": (ctypes.c_int, [ctypes.c_int, ctypes.POINTER(ctypes.c_size_t)]),
    "sap_stitched_alloc": (ctypes.c_int, [ctypes.c_int32, ctypes.c_size_t, c_i32p, ctypes.c_int32, c_i32p, ctypes.POINTER(vp)]),
    "sap_stitched_ptr": (vp, [vp]),
    "sap_stitched_bytes": (ctypes.c_size_t, [vp]),
    "sap_stitched_owner": (ctypes.c_int32, [vp, ctypes.c_int32]),
    "sap_stitched_free": (None, [vp]),
    "sap_stitched_create_local": (ctypes.c_int, [ctypes.c_int32, ctypes.c_size_t, ctypes.c_int, ctypes.POINTER(ctypes.c_uint8),
                                                 ctypes.POINTER(vp)]),
    "sap_stitched_export_fd": (ctypes.c_int, [vp, ctypes.c_int32, ctypes.POINTER(ctypes.c_int)]),
    "sap_stitched_import_fd": (ctypes.c_int, [vp, ctypes.c_int32, ctypes.c_int]),
    "sap_strerror": (ctypes.c_char_p, [ctypes.c_int]),
    "sap_last_cuda_error": (ctypes.c_int, []),
    "sap_launch_count": (ctypes.c_int64, []),
    "sap_debug_tile_program": (ctypes.c_int32, [vp, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, vp, ctypes.c_int32, vp,
                                                ctypes.c_int32, c_i32p]),
    "sap_debug_set_bwd_stages": (ctypes.c_int, [ctypes.c_int]),
    "sap_debug_set_fwd_form": (ctypes.c_int, [ctypes.c_int]),
    "sap_debug_set_bwd_form": (ctypes.c_int, [ctypes.c_int]),
}

_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_30460_b200.build` "
                               "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)          # AttributeError if the symbol is not exported
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib
