"""Thin Python binding of include/sap.h: argument marshalling only (torch is used for device memory
and streams); every step of the hot path runs in the CUDA kernels behind the C ABI."""
from __future__ import annotations

import ctypes
from typing import Optional, Sequence

import numpy as np

from . import _lib

SAP_MASK_SKIP, SAP_MASK_FULL, SAP_MASK_DIAG = 0, 1, 2
SAP_PASS_FWD, SAP_PASS_BWD = 0, 1
SAP_SCHED_RING, SAP_SCHED_BALANCED = 0, 1
SAP_OP_SEND, SAP_OP_RECV, SAP_OP_COMPUTING, SAP_OP_COPY = 0, 1, 2, 3
SAP_T_Q, SAP_T_KV, SAP_T_O, SAP_T_DO, SAP_T_DQ, SAP_T_DKV = 0, 1, 2, 3, 4, 5


class SapError(RuntimeError):
    def __init__(self, status: int, where: str):
        L = _lib.lib()
        msg = L.sap_strerror(status).decode()
        extra = f" (cuda error {L.sap_last_cuda_error()})" if status == 7 else ""
        super().__init__(f"{where}: {msg}{extra}")
        self.status = status


def _check(status: int, where: str):
    if status != 0:
        raise SapError(status, where)


def _ptr(t) -> ctypes.c_void_p:
    return ctypes.c_void_p(0 if t is None else t.data_ptr())


def _stream(stream) -> ctypes.c_void_p:
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


class Plan:
    """sap_plan: host-side JIT planner result (items in ring order + compiled tile programs)."""

    def __init__(self, cu_seqlens: Sequence[int], n_chunks: int):
        cu = np.ascontiguousarray(np.asarray(cu_seqlens, dtype=np.int64).astype(np.int32))
        self._cu_host = cu
        self._h = ctypes.c_void_p(0)
        self._cu_dev = {}
        L = _lib.lib()
        _check(L.sap_plan_create(cu.ctypes.data_as(ctypes.c_void_p), len(cu) - 1, int(n_chunks),
                                 ctypes.byref(self._h)), "sap_plan_create")
        self.n_chunks = int(n_chunks)
        self.n_tokens = int(L.sap_plan_n_tokens(self._h))
        self.n_items = int(L.sap_plan_n_items(self._h))

    def __del__(self):
        h = getattr(self, "_h", None)
        try:
            if h is not None and h.value:
                _lib.lib().sap_plan_destroy(h)
                self._h = ctypes.c_void_p(0)
        except Exception:      # interpreter shutdown: module globals may already be gone
            pass

    @property
    def handle(self) -> ctypes.c_void_p:
        return self._h

    @property
    def items(self) -> np.ndarray:
        """int32 [n_items, 10] in sap_item_t field order."""
        p = _lib.lib().sap_plan_items(self._h)
        n = self.n_items
        if n == 0:
            return np.zeros((0, 10), dtype=np.int32)
        return np.ctypeslib.as_array(ctypes.cast(p, _lib.c_i32p), shape=(n, 10)).copy()

    def _arr(self, fn, n):
        return np.ctypeslib.as_array(fn(self._h), shape=(n,)).copy()

    @property
    def chunk_offsets(self) -> np.ndarray:
        return self._arr(_lib.lib().sap_plan_chunk_offsets, self.n_chunks + 1)

    @property
    def kv_offsets(self) -> np.ndarray:
        return self._arr(_lib.lib().sap_plan_kv_offsets, self.n_chunks + 1)

    @property
    def kv_index(self) -> np.ndarray:
        return self._arr(_lib.lib().sap_plan_kv_index, self.n_items) if self.n_items else np.zeros(0, np.int32)

    @property
    def kind_map(self) -> np.ndarray:
        P = self.n_chunks
        return self._arr(_lib.lib().sap_plan_kind_map, P * P).reshape(P, P)

    @property
    def useful_pairs(self) -> int:
        return int(_lib.lib().sap_plan_useful_pairs(self._h))

    @property
    def fwd_tiles(self) -> int:
        return int(_lib.lib().sap_plan_fwd_tiles(self._h))

    def schedule(self, policy: int = 1):
        """Compile Steps 2-3: (slots int32 [n_items, 2] = (rank, stage) per item, n_stages).  policy 0 = plain ring,
        1 = balanced (SAP_SCHED_BALANCED)."""
        slots = np.zeros((max(self.n_items, 1), 2), dtype=np.int32)
        n_stages = ctypes.c_int32(0)
        _check(_lib.lib().sap_plan_schedule(self._h, int(policy), slots.ctypes.data_as(ctypes.c_void_p),
                                            ctypes.byref(n_stages)), "sap_plan_schedule")
        return slots[:self.n_items], int(n_stages.value)

    def codegen(self, slots: np.ndarray, rank: int, backward: bool = False) -> np.ndarray:
        """Jitted code generation: int32 [n_codes, 5] = (stage, opcode, tensor, peer, item) of `rank` (sap_code_t),
        for the forward (sap_plan_codegen) or the backward pass (sap_plan_codegen_bwd)."""
        L = _lib.lib()
        fn = L.sap_plan_codegen_bwd if backward else L.sap_plan_codegen
        sl = np.ascontiguousarray(slots, dtype=np.int32)
        n = int(fn(self._h, sl.ctypes.data_as(ctypes.c_void_p), int(rank), None, 0))
        if n < 0:
            raise SapError(-n, "sap_plan_codegen")
        codes = np.zeros((max(n, 1), 5), dtype=np.int32)
        fn(self._h, sl.ctypes.data_as(ctypes.c_void_p), int(rank), codes.ctypes.data_as(ctypes.c_void_p), n)
        return codes[:n]

    def tile_program(self, kind: int, a: int = 0, b: int = 0):
        """Diagnostic: (tiles int32 [n,4], segs int32 [m,8]) of the compiled tile program `kind` (sap_debug_tile_program)."""
        L = _lib.lib()
        ns = ctypes.c_int32(0)
        nt = int(L.sap_debug_tile_program(self._h, int(kind), int(a), int(b), None, 0, None, 0, ctypes.byref(ns)))
        if nt < 0:
            raise SapError(-nt, "sap_debug_tile_program")
        tiles = np.zeros((max(nt, 1), 4), dtype=np.int32); segs = np.zeros((max(ns.value, 1), 8), dtype=np.int32)
        L.sap_debug_tile_program(self._h, int(kind), int(a), int(b), tiles.ctypes.data_as(ctypes.c_void_p), nt,
                                 segs.ctypes.data_as(ctypes.c_void_p), ns.value, ctypes.byref(ns))
        return tiles[:nt], segs[:ns.value]

    def upload(self):
        _check(_lib.lib().sap_plan_upload(self._h), "sap_plan_upload")

    def cu_seqlens_dev(self, device):
        import torch
        key = str(device)
        if key not in self._cu_dev:
            self._cu_dev[key] = torch.from_numpy(self._cu_host).to(device)
        return self._cu_dev[key]


def sap_plan(cu_seqlens: Sequence[int], n_chunks: int) -> Plan:
    return Plan(cu_seqlens, n_chunks)


def sap_workspace_bytes(plan: Plan, n_q_heads: int, n_kv_heads: int, head_dim: int, pass_: int) -> int:
    return int(_lib.lib().sap_workspace_bytes(plan.handle, n_q_heads, n_kv_heads, head_dim, pass_))


def _dims(q, k):
    N, Hq, d = q.shape
    return int(N), int(Hq), int(k.shape[1]), int(d)


def _require_cuda_bf16(*ts):
    import torch
    for t in ts:
        if type(t).__name__ == "ShardView":   # a shard addressed with global token rows (executor.ShardView)
            t = t._t
        if not (t.is_cuda and t.dtype == torch.bfloat16 and t.is_contiguous()):
            raise ValueError("expected contiguous CUDA bf16 tensors")


def sap_attn_fwd(q, k, v, cu_seqlens_dev, plan: Plan, out=None, lse=None, softmax_scale: Optional[float] = None,
                 stream=None):
    """out [N,Hq,d] bf16, lse [Hq,N] fp32 = sap_attn_fwd(...).  Asynchronous on `stream`."""
    import torch
    _require_cuda_bf16(q, k, v)
    N, Hq, Hkv, d = _dims(q, k)
    if out is None:
        out = torch.empty_like(q)
    if lse is None:
        lse = torch.empty((Hq, N), dtype=torch.float32, device=q.device)
    scale = float(d) ** -0.5 if softmax_scale is None else float(softmax_scale)
    _check(_lib.lib().sap_attn_fwd(_ptr(q), _ptr(k), _ptr(v), _ptr(cu_seqlens_dev), plan.handle, N, _ptr(out),
                                   _ptr(lse), Hq, Hkv, d, scale, None, 0, _stream(stream)), "sap_attn_fwd")
    return out, lse


def sap_attn_fwd_partial(q, k, v, cu_seqlens_dev, plan: Plan, item_begin: int, item_end: int,
                         softmax_scale: Optional[float] = None, stream=None):
    """Partial forward over plan items [item_begin, item_end): (out fp32 [N,Hq,d], lse fp32 [Hq,N])."""
    import torch
    _require_cuda_bf16(q, k, v)
    N, Hq, Hkv, d = _dims(q, k)
    out = torch.empty((N, Hq, d), dtype=torch.float32, device=q.device)
    lse = torch.empty((Hq, N), dtype=torch.float32, device=q.device)
    scale = float(d) ** -0.5 if softmax_scale is None else float(softmax_scale)
    _check(_lib.lib().sap_attn_fwd_partial(_ptr(q), _ptr(k), _ptr(v), _ptr(cu_seqlens_dev), plan.handle, N,
                                           int(item_begin), int(item_end), _ptr(out), _ptr(lse), Hq, Hkv, d, scale,
                                           _stream(stream)), "sap_attn_fwd_partial")
    return out, lse


def sap_attn_fwd_items(q, k, v, cu_seqlens_dev, plan: Plan, item_begin: int, item_end: int, out_f32, lse,
                       n_q_heads: int, n_kv_heads: int, head_dim: int, softmax_scale: Optional[float] = None, stream=None):
    """The forward `computing` instruction: partial forward of plan items [item_begin, item_end) into caller-provided
    buffers, touching only the Q tiles of those items.  Tensor arguments only need data_ptr() (the kernels index them
    with global token rows: see executor.ShardView)."""
    scale = float(head_dim) ** -0.5 if softmax_scale is None else float(softmax_scale)
    _check(_lib.lib().sap_attn_fwd_items(_ptr(q), _ptr(k), _ptr(v), _ptr(cu_seqlens_dev), plan.handle, plan.n_tokens,
                                         int(item_begin), int(item_end), _ptr(out_f32), _ptr(lse), int(n_q_heads),
                                         int(n_kv_heads), int(head_dim), scale, _stream(stream)), "sap_attn_fwd_items")


def sap_lse_merge(o_a, lse_a, o_b, lse_b, out_bf16: bool = False, row_begin: int = 0,
                  row_end: Optional[int] = None, o_out=None, lse_out=None, stream=None):
    import torch
    N, Hq, d = o_a.shape
    row_end = N if row_end is None else row_end
    if o_out is None:
        o_out = torch.zeros((N, Hq, d), dtype=torch.bfloat16 if out_bf16 else torch.float32, device=o_a.device)
    if lse_out is None:
        lse_out = torch.full((Hq, N), float("-inf"), dtype=torch.float32, device=o_a.device)
    _check(_lib.lib().sap_lse_merge(_ptr(o_a), _ptr(lse_a), _ptr(o_b), _ptr(lse_b), _ptr(o_out), int(out_bf16),
                                    _ptr(lse_out), N, Hq, d, int(row_begin), int(row_end), _stream(stream)),
           "sap_lse_merge")
    return o_out, lse_out


def sap_attn_bwd(dout, q, k, v, out, lse, cu_seqlens_dev, plan: Plan, softmax_scale: Optional[float] = None,
                 dq=None, dk=None, dv=None, workspace=None, stream=None):
    """dq [N,Hq,d], dk, dv [N,Hkv,d] bf16 = sap_attn_bwd(...).  Asynchronous on `stream`."""
    import torch
    _require_cuda_bf16(dout, q, k, v, out)
    N, Hq, Hkv, d = _dims(q, k)
    dq = torch.empty_like(q) if dq is None else dq
    dk = torch.empty_like(k) if dk is None else dk
    dv = torch.empty_like(v) if dv is None else dv
    need = sap_workspace_bytes(plan, Hq, Hkv, d, SAP_PASS_BWD)
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=q.device)
    scale = float(d) ** -0.5 if softmax_scale is None else float(softmax_scale)
    _check(_lib.lib().sap_attn_bwd(_ptr(dout), _ptr(q), _ptr(k), _ptr(v), _ptr(out), _ptr(lse),
                                   _ptr(cu_seqlens_dev), plan.handle, N, _ptr(dq), _ptr(dk), _ptr(dv), Hq, Hkv, d,
                                   scale, _ptr(workspace), workspace.numel(), _stream(stream)), "sap_attn_bwd")
    return dq, dk, dv


def sap_attn_bwd_static(dout, q, k, v, out, lse, cu_seqlens_dev, plan: Plan, dq, dk, dv, softmax_scale: Optional[float] = None,
                        stream=None):
    """sap_attn_bwd for callers that cannot allocate device memory where they need the gradients (a plug-in that is
    handed tensors but no allocator, code running where only a framework's pool may allocate): the workspace and the
    plan's tile program sit in a fixed array inside the library, so this binding allocates nothing either - dq, dk, dv
    must be passed in.  Problems whose workspace exceeds 16 MiB raise SapError (status 10).  One array per GPU is shared
    by all calls: keep them on one stream, or otherwise ordered; overlapping calls corrupt each other.  See sap.h."""
    _require_cuda_bf16(dout, q, k, v, out, dq, dk, dv)
    N, Hq, Hkv, d = _dims(q, k)
    scale = float(d) ** -0.5 if softmax_scale is None else float(softmax_scale)
    _check(_lib.lib().sap_attn_bwd_static(_ptr(dout), _ptr(q), _ptr(k), _ptr(v), _ptr(out), _ptr(lse), _ptr(cu_seqlens_dev),
                                          plan.handle, N, _ptr(dq), _ptr(dk), _ptr(dv), Hq, Hkv, d, scale, _stream(stream)),
           "sap_attn_bwd_static")
    return dq, dk, dv


def sap_launch_count() -> int:
    return int(_lib.lib().sap_launch_count())


def sap_debug_set_bwd_stages(mask: int) -> int:
    """Diagnostic: select the kernels sap_attn_bwd launches (1 = D pre-pass, 2 = dK/dV, 4 = dQ)."""
    return int(_lib.lib().sap_debug_set_bwd_stages(int(mask)))


def sap_debug_set_fwd_form(form: int) -> int:
    """Diagnostic: 0 = pair forward kernel when Hq/Hkv is even (default), 1 = always the one-head kernel."""
    return int(_lib.lib().sap_debug_set_fwd_form(int(form)))


def sap_debug_set_bwd_form(form: int) -> int:
    """Diagnostic: 0 = CTA-pair fused backward at head_dim 128 (default), 1 = always the one-CTA fused kernel."""
    return int(_lib.lib().sap_debug_set_bwd_form(int(form)))


# ---- per-rank launches: the same kernels restricted to the chunks one rank owns ----------------
def sap_attn_fwd_chunks(q, k, v, cu_seqlens_dev, plan: Plan, q_chunk_begin: int, q_chunk_end: int, out, lse,
                        softmax_scale: Optional[float] = None, stream=None):
    """Forward of q-chunks [q_chunk_begin, q_chunk_end): writes only those rows of out [N,Hq,d] / lse [Hq,N]."""
    _require_cuda_bf16(q, k, v, out)
    N, Hq, Hkv, d = _dims(q, k)
    scale = float(d) ** -0.5 if softmax_scale is None else float(softmax_scale)
    _check(_lib.lib().sap_attn_fwd_chunks(_ptr(q), _ptr(k), _ptr(v), _ptr(cu_seqlens_dev), plan.handle, N,
                                          int(q_chunk_begin), int(q_chunk_end), _ptr(out), _ptr(lse), Hq, Hkv, d, scale,
                                          _stream(stream)), "sap_attn_fwd_chunks")
    return out, lse


def sap_attn_bwd_begin(dout, out, plan: Plan, q_chunk_begin: int, q_chunk_end: int, n_kv_heads: int, workspace, stream=None):
    N, Hq, d = dout.shape
    _check(_lib.lib().sap_attn_bwd_begin(_ptr(dout), _ptr(out), plan.handle, int(N), int(q_chunk_begin), int(q_chunk_end),
                                         int(Hq), int(n_kv_heads), int(d), _ptr(workspace), workspace.numel(),
                                         _stream(stream)), "sap_attn_bwd_begin")


def sap_attn_bwd_chunks(dout, q, k, v, lse, cu_seqlens_dev, plan: Plan, kv_chunk_begin: int, kv_chunk_end: int, dk, dv,
                        workspace, softmax_scale: Optional[float] = None, stream=None):
    _require_cuda_bf16(dout, q, k, v, dk, dv)
    N, Hq, Hkv, d = _dims(q, k)
    scale = float(d) ** -0.5 if softmax_scale is None else float(softmax_scale)
    _check(_lib.lib().sap_attn_bwd_chunks(_ptr(dout), _ptr(q), _ptr(k), _ptr(v), _ptr(lse), _ptr(cu_seqlens_dev),
                                          plan.handle, N, int(kv_chunk_begin), int(kv_chunk_end), _ptr(dk), _ptr(dv), Hq, Hkv,
                                          d, scale, _ptr(workspace), workspace.numel(), _stream(stream)),
           "sap_attn_bwd_chunks")


def sap_attn_bwd_end(plan: Plan, q_chunk_begin: int, q_chunk_end: int, dq, n_kv_heads: int, workspace,
                     softmax_scale: Optional[float] = None, stream=None):
    N, Hq, d = dq.shape
    scale = float(d) ** -0.5 if softmax_scale is None else float(softmax_scale)
    _check(_lib.lib().sap_attn_bwd_end(plan.handle, int(N), int(q_chunk_begin), int(q_chunk_end), _ptr(dq), int(Hq),
                                       int(n_kv_heads), int(d), scale, _ptr(workspace), workspace.numel(),
                                       _stream(stream)), "sap_attn_bwd_end")


# ---- per-item launches: the backward `computing` instruction and the gradient COPY ----------------
def sap_attn_bwd_items(dout, q, k, v, lse, cu_seqlens_dev, plan: Plan, item_begin: int, item_end: int, dk, dv, workspace,
                       softmax_scale: Optional[float] = None, stream=None):
    """Fused backward of plan items [item_begin, item_end): dk / dv rows of the touched K/V tiles are written with the
    items' contribution, dQ contributions are added into the accumulator of `workspace`."""
    _require_cuda_bf16(dout, q, k, v, dk, dv)
    N, Hq, Hkv, d = _dims(q, k)
    scale = float(d) ** -0.5 if softmax_scale is None else float(softmax_scale)
    _check(_lib.lib().sap_attn_bwd_items(_ptr(dout), _ptr(q), _ptr(k), _ptr(v), _ptr(lse), _ptr(cu_seqlens_dev),
                                         plan.handle, N, int(item_begin), int(item_end), _ptr(dk), _ptr(dv), Hq, Hkv,
                                         d, scale, _ptr(workspace), workspace.numel(), _stream(stream)),
           "sap_attn_bwd_items")


def sap_axpy(dst, src, alpha: float = 1.0, accumulate: bool = True, stream=None):
    """dst = (dst if accumulate else 0) + alpha * src on the GPU; dst, src contiguous fp32 or bf16 CUDA tensors."""
    import torch
    if not (dst.is_cuda and src.is_cuda and dst.is_contiguous() and src.is_contiguous() and dst.numel() == src.numel()):
        raise ValueError("expected contiguous CUDA tensors of equal size")
    for t in (dst, src):
        if t.dtype not in (torch.float32, torch.bfloat16):
            raise ValueError("fp32 or bf16 only")
    _check(_lib.lib().sap_axpy(_ptr(dst), int(dst.dtype == torch.bfloat16), _ptr(src), int(src.dtype == torch.bfloat16),
                               dst.numel(), float(alpha), int(accumulate), _stream(stream)), "sap_axpy")
    return dst


class Stitched:
    """sap_stitched_alloc: one device address range of n_chunks * chunk_bytes bytes whose chunk c is memory of device
    devices[c] (SURVEY 8(f) NEXT-1 data plane).  `tensor(shape, dtype)` views the range as a torch tensor (the range
    stays alive as long as this object does: keep it)."""

    def __init__(self, n_chunks: int, chunk_bytes: int, devices: Optional[Sequence[int]] = None,
                 access_devices: Optional[Sequence[int]] = None):
        devices = [0] * n_chunks if devices is None else [int(d) for d in devices]
        access = sorted(set(devices)) if access_devices is None else [int(d) for d in access_devices]
        self.handle = ctypes.c_void_p()
        dev = (ctypes.c_int32 * len(devices))(*devices)
        acc = (ctypes.c_int32 * len(access))(*access)
        _check(_lib.lib().sap_stitched_alloc(int(n_chunks), int(chunk_bytes), dev, len(access), acc,
                                             ctypes.byref(self.handle)), "sap_stitched_alloc")
        self.ptr = int(_lib.lib().sap_stitched_ptr(self.handle))
        self.nbytes = int(_lib.lib().sap_stitched_bytes(self.handle))
        self.n_chunks, self.chunk_bytes, self.devices = int(n_chunks), int(chunk_bytes), devices

    @classmethod
    def create_local(cls, n_chunks: int, chunk_bytes: int, device: int, own: Sequence[bool]) -> "Stitched":
        """One process per GPU: reserve the whole range on `device`, create (exportable) and map the chunks with own[c];
        the others are mapped later with import_fd from their owners' export_fd descriptors."""
        self = cls.__new__(cls)
        self.handle = ctypes.c_void_p()
        mask = (ctypes.c_uint8 * int(n_chunks))(*[1 if o else 0 for o in own])
        _check(_lib.lib().sap_stitched_create_local(int(n_chunks), int(chunk_bytes), int(device), mask,
                                                    ctypes.byref(self.handle)), "sap_stitched_create_local")
        self.ptr = int(_lib.lib().sap_stitched_ptr(self.handle))
        self.nbytes = int(_lib.lib().sap_stitched_bytes(self.handle))
        self.n_chunks, self.chunk_bytes, self.devices = int(n_chunks), int(chunk_bytes), [int(device)] * int(n_chunks)
        return self

    def export_fd(self, chunk: int) -> int:
        fd = ctypes.c_int(-1)
        _check(_lib.lib().sap_stitched_export_fd(self.handle, int(chunk), ctypes.byref(fd)), "sap_stitched_export_fd")
        return int(fd.value)

    def import_fd(self, chunk: int, fd: int) -> None:
        _check(_lib.lib().sap_stitched_import_fd(self.handle, int(chunk), int(fd)), "sap_stitched_import_fd")

    @staticmethod
    def granularity(device: int = 0) -> int:
        g = ctypes.c_size_t()
        _check(_lib.lib().sap_stitched_granularity(int(device), ctypes.byref(g)), "sap_stitched_granularity")
        return int(g.value)

    def owner(self, chunk: int) -> int:
        return int(_lib.lib().sap_stitched_owner(self.handle, int(chunk)))

    def tensor(self, shape, dtype, device=None):
        import torch
        nbytes = int(np.prod(shape)) * torch.empty((), dtype=dtype).element_size()
        if nbytes > self.nbytes:
            raise ValueError(f"shape {tuple(shape)} needs {nbytes} bytes, the range has {self.nbytes}")
        typestr = {torch.bfloat16: "<u2", torch.float32: "<f4", torch.uint8: "|u1", torch.int32: "<i4"}[dtype]

        class _View:   # __cuda_array_interface__: torch wraps the memory, it does not own it
            __cuda_array_interface__ = {"shape": (nbytes // int(typestr[2]),), "typestr": typestr, "data": (self.ptr, False),
                                        "version": 2}
        t = torch.as_tensor(_View(), device=device if device is not None else f"cuda:{self.devices[0]}")
        if dtype == torch.bfloat16:
            t = t.view(torch.bfloat16)
        t = t.view(*shape)
        t._sap_stitched = self   # the tensor keeps the range alive
        return t

    def free(self):
        if getattr(self, "handle", None) is not None and self.handle:
            import torch
            torch.cuda.synchronize()   # no kernel may still be using the range when it is unmapped
            _lib.lib().sap_stitched_free(self.handle)
            self.handle = ctypes.c_void_p()

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass
