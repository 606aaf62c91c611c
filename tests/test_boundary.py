"""Boundary behaviour that needs no GPU (SURVEY 8(b) error list): argument checks that the C ABI makes before it touches
the device, through raw ctypes calls with dummy non-null pointers."""
import ctypes

import numpy as np

from paper_2606_30460_b200 import _lib, sap_plan

DUMMY = ctypes.c_void_p(0x1000)   # non-null, 16-byte aligned, never dereferenced on these paths


def test_plan_mismatch_is_reported_before_anything_touches_the_device():
    plan = sap_plan([0, 700, 1800, 2048], 4)
    L = _lib.lib()
    # a plan built for 2048 tokens used with tensors of another length must not launch (it would read out of bounds)
    rc = L.sap_attn_fwd(DUMMY, DUMMY, DUMMY, DUMMY, plan.handle, 4096, DUMMY, DUMMY, 4, 4, 64, 0.125, None, 0, None)
    assert rc == 9 and b"plan mismatch" in L.sap_strerror(rc)
    rc = L.sap_attn_bwd(DUMMY, DUMMY, DUMMY, DUMMY, DUMMY, DUMMY, DUMMY, plan.handle, 1024, DUMMY, DUMMY, DUMMY, 4, 4, 64,
                        0.125, DUMMY, 1 << 30, None)
    assert rc == 9
    rc = L.sap_attn_fwd_partial(DUMMY, DUMMY, DUMMY, DUMMY, plan.handle, 2047, 0, 1, DUMMY, DUMMY, 4, 4, 64, 0.125, None)
    assert rc == 9
    rc = L.sap_attn_bwd_items(DUMMY, DUMMY, DUMMY, DUMMY, DUMMY, DUMMY, plan.handle, 0, 0, 1, DUMMY, DUMMY, 4, 4, 64, 0.125,
                              DUMMY, 1 << 30, None)
    assert rc == 9


def test_argument_errors_come_before_device_errors():
    plan = sap_plan([0, 2048], 4)
    L = _lib.lib()
    assert L.sap_attn_fwd(None, DUMMY, DUMMY, DUMMY, plan.handle, 2048, DUMMY, DUMMY, 4, 4, 64, 0.125, None, 0, None) == 1   # null pointer
    assert L.sap_attn_fwd(DUMMY, DUMMY, DUMMY, DUMMY, plan.handle, 2048, DUMMY, DUMMY, 4, 4, 96, 0.125, None, 0, None) == 4   # head_dim
    assert L.sap_attn_fwd(DUMMY, DUMMY, DUMMY, DUMMY, plan.handle, 2048, DUMMY, DUMMY, 6, 4, 64, 0.125, None, 0, None) == 4   # Hq % Hkv
    assert L.sap_attn_fwd(DUMMY, DUMMY, DUMMY, DUMMY, plan.handle, 2048, DUMMY, DUMMY, 4, 4, 64, 0.0, None, 0, None) == 1     # scale
    assert L.sap_axpy(DUMMY, 0, DUMMY, 0, 12, 1.0, 1, None) == 4    # n_elems % 8
    assert L.sap_axpy(None, 0, DUMMY, 0, 16, 1.0, 1, None) == 1
    for code in range(11):
        assert L.sap_strerror(code) != b"unknown status"


def test_workspace_size_formula():
    plan = sap_plan([0, 2048], 4)
    L = _lib.lib()
    need = L.sap_workspace_bytes(plan.handle, 8, 2, 128, 1)
    assert need == ((2048 * 8 * 4 + 255) // 256) * 256 + 2048 * 8 * 128 * 4
    assert L.sap_workspace_bytes(plan.handle, 8, 2, 128, 0) == 0
