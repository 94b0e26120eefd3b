"""ctypes binding for libhx.so.  Names follow include/hx.h; no arithmetic happens here."""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libhx.so")

HX_OK, HX_ERR_INVALID_ARG, HX_ERR_UNSUPPORTED, HX_ERR_WORKSPACE, HX_ERR_CUDA, HX_ERR_NO_PAGES = range(6)

# every symbol include/hx.h declares (tests check that the library exports each one)
EXPORTS = [
    "hx_version", "hx_status_string", "hx_last_error", "hx_paged_cache_bytes", "hx_kv_ingest",
    "hx_kv_gather", "hx_decode_attention_workspace_bytes", "hx_decode_attention", "hx_pool_create",
    "hx_pool_shuffle", "hx_pool_alloc", "hx_pool_free", "hx_pool_num_free", "hx_pool_num_pages",
    "hx_pool_alloc_table", "hx_pool_destroy", "hx_decode_step_host", "hx_decode_plan_bytes", "hx_decode_plan",
    "hx_decode_attention_planned", "hx_decode_attention_chained",
    "hx_kv_ingest_stage", "hx_stage_overlap", "hx_kv_append", "hx_decode_attention_append",
    "hx_prefill_attention", "hx_decode_attention_overlapped", "hx_decode_step", "hx_shutdown",
    "hx_decode_attention_noalloc", "hx_decode_step_is_fused",
]

NOALLOC_SCRATCH_BYTES = 20 * 1024 * 1024      # HX_NOALLOC_SCRATCH_BYTES (include/hx.h)


class HxError(RuntimeError):
    def __init__(self, status: int, detail: str):
        self.status = status
        super().__init__(f"{status_string(status)}: {detail}")


class _CCache(C.Structure):
    _fields_ = [("k", C.c_void_p), ("v", C.c_void_p), ("layers", C.c_int32), ("num_pages", C.c_int32),
                ("kv_heads", C.c_int32), ("page_size", C.c_int32), ("head_dim", C.c_int32)]


class _CStepArgs(C.Structure):
    _fields_ = [
        ("q_host", C.c_void_p), ("out_host", C.c_void_p), ("q_dev", C.c_void_p), ("out_dev", C.c_void_p),
        ("cache", C.POINTER(_CCache)), ("layer", C.c_int32), ("q_heads", C.c_int32),
        ("block_table_dev", C.c_void_p), ("block_table_stride", C.c_int32),
        ("seq_lens_dev", C.c_void_p), ("batch", C.c_int32), ("max_seq_len", C.c_int32),
        ("sm_scale", C.c_float), ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
        ("src_k_host", C.POINTER(C.c_void_p)), ("src_v_host", C.POINTER(C.c_void_p)),
        ("src_k_dev", C.POINTER(C.c_void_p)), ("src_v_dev", C.POINTER(C.c_void_p)),
        ("ing_layers", C.c_int32), ("heads", C.c_int32), ("src_tp", C.c_int32), ("dst_tp", C.c_int32),
        ("dst_rank", C.c_int32),
        ("ing_block_table_host", C.c_void_p), ("ing_block_table_stride", C.c_int32),
        ("ing_cu_seqlens_host", C.c_void_p), ("ing_seq_lens_host", C.c_void_p),
        ("ing_block_table_dev", C.c_void_p), ("ing_cu_seqlens_dev", C.c_void_p), ("ing_seq_lens_dev", C.c_void_p),
        ("ing_batch", C.c_int32), ("ing_total_tokens", C.c_int32), ("ing_max_seq_len", C.c_int32),
        ("pull_src", C.c_int32), ("overlap_ingest", C.c_int32),
    ]


class _CStepDevArgs(C.Structure):
    _fields_ = [
        ("out", C.c_void_p), ("q", C.c_void_p), ("cache", C.POINTER(_CCache)), ("layer", C.c_int32), ("q_heads", C.c_int32),
        ("block_table", C.c_void_p), ("block_table_stride", C.c_int32), ("seq_lens", C.c_void_p),
        ("batch", C.c_int32), ("max_seq_len", C.c_int32), ("sm_scale", C.c_float),
        ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
        ("src_k", C.POINTER(C.c_void_p)), ("src_v", C.POINTER(C.c_void_p)),
        ("ing_layers", C.c_int32), ("heads", C.c_int32), ("src_tp", C.c_int32), ("dst_tp", C.c_int32), ("dst_rank", C.c_int32),
        ("ing_block_table", C.c_void_p), ("ing_block_table_stride", C.c_int32),
        ("ing_cu_seqlens", C.c_void_p), ("ing_seq_lens", C.c_void_p),
        ("ing_batch", C.c_int32), ("ing_total_tokens", C.c_int32), ("ing_max_seq_len", C.c_int32),
        ("overlap_ingest", C.c_int32),
        ("ev_ingest_begin", C.c_void_p), ("ev_ingest_end", C.c_void_p),
        ("ev_attention_begin", C.c_void_p), ("ev_attention_end", C.c_void_p),
    ]


_lib = None


def lib() -> C.CDLL:
    """Loads libhx.so (built in-tree by build.py).  Fails loudly when it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise ImportError(f"{_SO} not found: run `python -m paper_2502_07903_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(_SO)
        L.hx_version.restype = C.c_int
        L.hx_status_string.restype = C.c_char_p
        L.hx_status_string.argtypes = [C.c_int]
        L.hx_last_error.restype = C.c_char_p
        L.hx_paged_cache_bytes.restype = C.c_size_t
        L.hx_paged_cache_bytes.argtypes = [C.c_int32] * 5
        ing = [C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.c_int32, C.c_int32, C.c_int32, C.c_int32,
               C.c_int32, C.c_int32, C.POINTER(_CCache), C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p,
               C.c_int32, C.c_int32, C.c_int32, C.c_void_p]
        L.hx_kv_ingest.restype = C.c_int
        L.hx_kv_ingest.argtypes = ing
        L.hx_kv_gather.restype = C.c_int
        L.hx_kv_gather.argtypes = ing
        L.hx_decode_attention_workspace_bytes.restype = C.c_size_t
        L.hx_decode_attention_workspace_bytes.argtypes = [C.c_int32] * 6
        L.hx_decode_attention.restype = C.c_int
        L.hx_decode_attention.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(_CCache), C.c_int32, C.c_int32,
                                          C.c_void_p, C.c_int32, C.c_void_p, C.c_int32, C.c_int32, C.c_float,
                                          C.c_void_p, C.c_size_t, C.c_void_p]
        L.hx_pool_create.restype = C.c_int
        L.hx_pool_create.argtypes = [C.POINTER(C.c_void_p), C.c_int32]
        L.hx_pool_shuffle.restype = C.c_int
        L.hx_pool_shuffle.argtypes = [C.c_void_p, C.c_uint64]
        L.hx_pool_alloc.restype = C.c_int
        L.hx_pool_alloc.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
        L.hx_pool_free.restype = C.c_int
        L.hx_pool_free.argtypes = [C.c_void_p, C.c_void_p, C.c_int32]
        L.hx_pool_num_free.restype = C.c_int32
        L.hx_pool_num_free.argtypes = [C.c_void_p]
        L.hx_pool_num_pages.restype = C.c_int32
        L.hx_pool_num_pages.argtypes = [C.c_void_p]
        L.hx_pool_alloc_table.restype = C.c_int
        L.hx_pool_alloc_table.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_int32]
        L.hx_pool_destroy.restype = None
        L.hx_pool_destroy.argtypes = [C.c_void_p]
        L.hx_decode_plan_bytes.restype = C.c_size_t
        L.hx_decode_plan_bytes.argtypes = [C.c_int32] * 4
        L.hx_decode_plan.restype = C.c_int
        L.hx_decode_plan.argtypes = [C.c_void_p, C.c_size_t, C.POINTER(_CCache), C.c_int32, C.c_void_p, C.c_int32, C.c_void_p,
                                     C.c_int32, C.c_int32, C.c_void_p]
        L.hx_decode_attention_planned.restype = C.c_int
        L.hx_decode_attention_planned.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(_CCache), C.c_int32, C.c_int32, C.c_void_p,
                                                  C.c_size_t, C.c_int32, C.c_int32, C.c_float, C.c_void_p, C.c_size_t, C.c_void_p]
        L.hx_decode_attention_chained.restype = C.c_int
        L.hx_decode_attention_chained.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(_CCache), C.c_int32, C.c_int32, C.c_void_p,
                                                  C.c_size_t, C.c_int32, C.c_int32, C.c_float, C.c_void_p, C.c_size_t, C.c_int32,
                                                  C.c_void_p]
        L.hx_kv_ingest_stage.restype = C.c_int
        L.hx_kv_ingest_stage.argtypes = [C.POINTER(C.c_void_p), C.POINTER(C.c_void_p)] + [C.c_int32] * 9 + [
            C.POINTER(_CCache), C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_int32,
            C.c_void_p]
        L.hx_stage_overlap.restype = C.c_int
        L.hx_stage_overlap.argtypes = [C.c_int32] * 4 + [C.POINTER(C.c_int32)] * 3
        L.hx_kv_append.restype = C.c_int
        L.hx_kv_append.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(_CCache), C.c_int32, C.c_void_p, C.c_int32,
                                   C.c_void_p, C.c_int32, C.c_int32, C.c_void_p]
        L.hx_decode_attention_append.restype = C.c_int
        L.hx_decode_attention_append.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(_CCache),
                                                 C.c_int32, C.c_int32, C.c_void_p, C.c_int32, C.c_void_p, C.c_int32,
                                                 C.c_int32, C.c_float, C.c_void_p, C.c_size_t, C.c_void_p]
        L.hx_prefill_attention.restype = C.c_int
        L.hx_prefill_attention.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(_CCache), C.c_int32, C.c_int32,
                                           C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32,
                                           C.c_int32, C.c_int32, C.c_int32, C.c_float, C.c_void_p]
        L.hx_decode_attention_overlapped.restype = C.c_int
        L.hx_decode_attention_overlapped.argtypes = L.hx_decode_attention.argtypes[:-1] + [C.c_int32, C.c_void_p]
        L.hx_decode_attention_noalloc.restype = C.c_int
        L.hx_decode_attention_noalloc.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(_CCache), C.c_int32, C.c_int32,
                                                  C.c_void_p, C.c_int32, C.c_void_p, C.c_int32, C.c_int32, C.c_float,
                                                  C.c_void_p]
        L.hx_decode_step_host.restype = C.c_int
        L.hx_decode_step_host.argtypes = [C.POINTER(_CStepArgs), C.c_void_p]
        L.hx_decode_step.restype = C.c_int
        L.hx_decode_step.argtypes = [C.POINTER(_CStepDevArgs), C.c_void_p]
        L.hx_decode_step_is_fused.restype = C.c_int
        L.hx_decode_step_is_fused.argtypes = [C.POINTER(_CStepDevArgs), C.POINTER(C.c_int32)]
        L.hx_shutdown.restype = C.c_int
        _lib = L
    return _lib


def version() -> int:
    return int(lib().hx_version())


def status_string(status: int) -> str:
    return lib().hx_status_string(int(status)).decode()


def last_error() -> str:
    return lib().hx_last_error().decode()


def _check(status: int):
    if status != HX_OK:
        raise HxError(status, last_error())


def paged_cache_bytes(layers, num_pages, kv_heads, page_size, head_dim) -> int:
    return int(lib().hx_paged_cache_bytes(layers, num_pages, kv_heads, page_size, head_dim))


def _ptr(t) -> Optional[int]:
    """Raw address of a torch tensor / numpy array / int / None."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    if hasattr(t, "cuda_event"):               # torch.cuda.Event (already recorded once, so the handle exists)
        return t.cuda_event
    return t.ctypes.data


def _stream_ptr(stream) -> Optional[int]:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


class PagedCache:
    """One decode-TP rank's paged cache: k, v are device fp16 tensors
    [layers][num_pages][kv_heads][page_size][head_dim] owned by the caller (torch)."""

    def __init__(self, k, v):
        assert k.shape == v.shape and k.dim() == 5 and k.is_contiguous() and v.is_contiguous()
        self.k, self.v = k, v
        L, P, H, ps, D = k.shape
        self.c = _CCache(k.data_ptr(), v.data_ptr(), L, P, H, ps, D)

    @classmethod
    def empty(cls, layers, num_pages, kv_heads, head_dim, page_size=16, device="cuda"):
        import torch
        shape = (layers, num_pages, kv_heads, page_size, head_dim)
        return cls(torch.empty(shape, dtype=torch.float16, device=device),
                   torch.empty(shape, dtype=torch.float16, device=device))

    @property
    def ref(self):
        return C.byref(self.c)


def _ptr_array(tensors: Sequence):
    arr = (C.c_void_p * len(tensors))()
    for i, t in enumerate(tensors):
        arr[i] = _ptr(t)
    return arr


def _ingest(fn, src_k, src_v, layers, heads, head_dim, src_tp, dst_tp, dst_rank, dst: PagedCache,
            block_table, block_table_stride, cu_seqlens, seq_lens, batch, total_tokens, max_seq_len, stream):
    assert len(src_k) == src_tp and len(src_v) == src_tp
    _check(fn(_ptr_array(src_k), _ptr_array(src_v), layers, heads, head_dim, src_tp, dst_tp, dst_rank,
              dst.ref, _ptr(block_table), block_table_stride, _ptr(cu_seqlens), _ptr(seq_lens), batch,
              total_tokens, max_seq_len, _stream_ptr(stream)))


def kv_ingest(src_k, src_v, *, layers, heads, head_dim, src_tp, dst_tp, dst_rank, dst, block_table,
              block_table_stride, cu_seqlens, seq_lens, batch, total_tokens, max_seq_len, stream=None):
    """hx_kv_ingest (include/hx.h).  src_k / src_v: lists of src_tp device tensors (or None)."""
    _ingest(lib().hx_kv_ingest, src_k, src_v, layers, heads, head_dim, src_tp, dst_tp, dst_rank, dst,
            block_table, block_table_stride, cu_seqlens, seq_lens, batch, total_tokens, max_seq_len, stream)


def kv_gather(src_k, src_v, *, layers, heads, head_dim, src_tp, dst_tp, dst_rank, dst, block_table,
              block_table_stride, cu_seqlens, seq_lens, batch, total_tokens, max_seq_len, stream=None):
    """hx_kv_gather: exact inverse of kv_ingest (writes the shard tensors)."""
    _ingest(lib().hx_kv_gather, src_k, src_v, layers, heads, head_dim, src_tp, dst_tp, dst_rank, dst,
            block_table, block_table_stride, cu_seqlens, seq_lens, batch, total_tokens, max_seq_len, stream)


def kv_ingest_stage(src_k, src_v, *, src_layers, src_layer0, dst_layer0, layers, heads, head_dim, src_tp, dst_tp,
                    dst_rank, dst, block_table, block_table_stride, cu_seqlens, seq_lens, batch, total_tokens,
                    max_seq_len, stream=None):
    """hx_kv_ingest_stage (include/hx.h): `layers` layers, source layer src_layer0+c -> cache layer dst_layer0+c."""
    assert len(src_k) == src_tp and len(src_v) == src_tp
    _check(lib().hx_kv_ingest_stage(_ptr_array(src_k), _ptr_array(src_v), src_layers, src_layer0, dst_layer0, layers,
                                    heads, head_dim, src_tp, dst_tp, dst_rank, dst.ref, _ptr(block_table),
                                    block_table_stride, _ptr(cu_seqlens), _ptr(seq_lens), batch, total_tokens,
                                    max_seq_len, _stream_ptr(stream)))


def stage_overlap(src_first, src_count, dst_first, dst_count):
    """hx_stage_overlap -> (src_layer0, dst_layer0, layers)."""
    a, b, n = C.c_int32(), C.c_int32(), C.c_int32()
    _check(lib().hx_stage_overlap(src_first, src_count, dst_first, dst_count, C.byref(a), C.byref(b), C.byref(n)))
    return a.value, b.value, n.value


def kv_append(k_new, v_new, cache: PagedCache, *, layer, block_table, block_table_stride, seq_lens, batch,
              max_seq_len, stream=None):
    """hx_kv_append (include/hx.h): token n_i-1 of every request joins the paged cache."""
    _check(lib().hx_kv_append(_ptr(k_new), _ptr(v_new), cache.ref, layer, _ptr(block_table), block_table_stride,
                              _ptr(seq_lens), batch, max_seq_len, _stream_ptr(stream)))


def decode_attention_append(out, q, k_new, v_new, cache: PagedCache, *, layer, q_heads, block_table,
                            block_table_stride, seq_lens, batch, max_seq_len, sm_scale=0.0, workspace=None,
                            workspace_bytes=None, stream=None):
    """hx_decode_attention_append: hx_kv_append + hx_decode_attention in one launch."""
    if workspace_bytes is None:
        workspace_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    _check(lib().hx_decode_attention_append(_ptr(out), _ptr(q), _ptr(k_new), _ptr(v_new), cache.ref, layer, q_heads,
                                            _ptr(block_table), block_table_stride, _ptr(seq_lens), batch, max_seq_len,
                                            C.c_float(sm_scale), _ptr(workspace), workspace_bytes,
                                            _stream_ptr(stream)))


def prefill_attention(out, q, cache: PagedCache, *, layer, q_heads, block_table, block_table_stride, seq_lens,
                      q_lens, cu_q_lens, batch, total_q_tokens, max_q_len, max_seq_len, sm_scale=0.0, stream=None):
    """hx_prefill_attention (include/hx.h): causal paged attention of the last q_lens[i] tokens."""
    _check(lib().hx_prefill_attention(_ptr(out), _ptr(q), cache.ref, layer, q_heads, _ptr(block_table),
                                      block_table_stride, _ptr(seq_lens), _ptr(q_lens), _ptr(cu_q_lens), batch,
                                      total_q_tokens, max_q_len, max_seq_len, C.c_float(sm_scale),
                                      _stream_ptr(stream)))


def decode_attention_workspace_bytes(batch, q_heads, kv_heads, head_dim, max_seq_len, page_size=16) -> int:
    return int(lib().hx_decode_attention_workspace_bytes(batch, q_heads, kv_heads, head_dim, max_seq_len, page_size))


def decode_attention(out, q, cache: PagedCache, *, layer, q_heads, block_table, block_table_stride, seq_lens,
                     batch, max_seq_len, sm_scale=0.0, workspace=None, workspace_bytes=None, stream=None):
    """hx_decode_attention (include/hx.h).  All tensors are device tensors owned by the caller."""
    if workspace_bytes is None:
        workspace_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    _check(lib().hx_decode_attention(_ptr(out), _ptr(q), cache.ref, layer, q_heads, _ptr(block_table),
                                     block_table_stride, _ptr(seq_lens), batch, max_seq_len,
                                     C.c_float(sm_scale), _ptr(workspace), workspace_bytes, _stream_ptr(stream)))


def decode_attention_noalloc(out, q, cache: PagedCache, *, layer, q_heads, block_table, block_table_stride, seq_lens,
                             batch, max_seq_len, sm_scale=0.0, stream=None):
    """hx_decode_attention_noalloc (include/hx.h): decode_attention for a caller that has no device memory to spare
    for a workspace and no way to allocate one (a GPU already filled with KV pages, a plug-in without the host
    engine's allocator, a thread that must not cudaMalloc while a capture is open).  The scratch is a fixed
    NOALLOC_SCRATCH_BYTES array inside libhx, shared by every call on that GPU: calls must not overlap on the device,
    shapes that need more are refused (HxError, HX_ERR_WORKSPACE), and the first call on each GPU should happen at
    start-up, outside any stream capture.  Same result as decode_attention."""
    _check(lib().hx_decode_attention_noalloc(_ptr(out), _ptr(q), cache.ref, layer, q_heads, _ptr(block_table),
                                             block_table_stride, _ptr(seq_lens), batch, max_seq_len,
                                             C.c_float(sm_scale), _stream_ptr(stream)))


def decode_attention_overlapped(out, q, cache: PagedCache, *, layer, q_heads, block_table, block_table_stride, seq_lens,
                                batch, max_seq_len, behind_ingest, sm_scale=0.0, workspace=None, workspace_bytes=None,
                                stream=None):
    """hx_decode_attention_overlapped: with behind_ingest != 0 the caller states that the kernel directly before it on the
    stream is a launched hx_kv_ingest whose pages this call does not read; the attention then starts under it
    (see include/hx.h).  behind_ingest == 0: exactly decode_attention."""
    if workspace_bytes is None:
        workspace_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    _check(lib().hx_decode_attention_overlapped(_ptr(out), _ptr(q), cache.ref, layer, q_heads, _ptr(block_table),
                                                block_table_stride, _ptr(seq_lens), batch, max_seq_len,
                                                C.c_float(sm_scale), _ptr(workspace), workspace_bytes,
                                                int(behind_ingest), _stream_ptr(stream)))


def decode_plan_bytes(batch, kv_heads, max_seq_len, page_size=16) -> int:
    return int(lib().hx_decode_plan_bytes(batch, kv_heads, max_seq_len, page_size))


def decode_plan(plan, cache: PagedCache, *, q_heads, block_table, block_table_stride, seq_lens, batch, max_seq_len,
                plan_bytes=None, stream=None):
    """hx_decode_plan (include/hx.h): once per decode step; `plan` is a device byte tensor of >= decode_plan_bytes()."""
    if plan_bytes is None:
        plan_bytes = plan.numel() * plan.element_size()
    _check(lib().hx_decode_plan(_ptr(plan), plan_bytes, cache.ref, q_heads, _ptr(block_table), block_table_stride,
                                _ptr(seq_lens), batch, max_seq_len, _stream_ptr(stream)))


def decode_attention_planned(out, q, cache: PagedCache, *, layer, q_heads, plan, batch, max_seq_len, sm_scale=0.0,
                             workspace=None, workspace_bytes=None, plan_bytes=None, stream=None):
    """hx_decode_attention_planned: hx_decode_attention reading a plan instead of seq_lens / block_table."""
    if workspace_bytes is None:
        workspace_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    if plan_bytes is None:
        plan_bytes = plan.numel() * plan.element_size()
    _check(lib().hx_decode_attention_planned(_ptr(out), _ptr(q), cache.ref, layer, q_heads, _ptr(plan), plan_bytes, batch,
                                             max_seq_len, C.c_float(sm_scale), _ptr(workspace), workspace_bytes,
                                             _stream_ptr(stream)))


def decode_attention_chained(out, q, cache: PagedCache, *, layer, q_heads, plan, batch, max_seq_len, inputs_ready, sm_scale=0.0,
                             workspace=None, workspace_bytes=None, plan_bytes=None, stream=None):
    """hx_decode_attention_chained: hx_decode_attention_planned as a programmatic dependent of the preceding kernel."""
    if workspace_bytes is None:
        workspace_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    if plan_bytes is None:
        plan_bytes = plan.numel() * plan.element_size()
    _check(lib().hx_decode_attention_chained(_ptr(out), _ptr(q), cache.ref, layer, q_heads, _ptr(plan), plan_bytes, batch,
                                             max_seq_len, C.c_float(sm_scale), _ptr(workspace), workspace_bytes,
                                             int(inputs_ready), _stream_ptr(stream)))


def _fill_struct(a, kw):
    """Keyword names are the struct's field names; `cache` is a PagedCache; src_* are lists of tensors."""
    keep = []
    for name, ctype in a._fields_:
        if name not in kw:
            continue
        val = kw.pop(name)
        if name == "cache":
            a.cache = C.pointer(val.c)
        elif ctype is C.POINTER(C.c_void_p):
            arr = _ptr_array(val)
            keep.append(arr)
            setattr(a, name, arr)
        elif ctype is C.c_void_p:
            setattr(a, name, _ptr(val))
        else:
            setattr(a, name, val)
    assert not kw, f"unknown fields: {list(kw)}"
    return keep


def decode_step_host(**kw):
    """hx_decode_step_host: one whole decode step from HOST buffers (see hx_step_host_args)."""
    a = _CStepArgs()
    stream = kw.pop("stream", None)
    keep = _fill_struct(a, kw)
    _check(lib().hx_decode_step_host(C.byref(a), _stream_ptr(stream)))
    del keep


class DecodeStep:
    """hx_decode_step with its argument struct built once (the per-step host cost is then one ctypes call).
    Keyword names are hx_step_args' field names."""

    def __init__(self, **kw):
        self.a = _CStepDevArgs()
        self._keep = _fill_struct(self.a, dict(kw))
        self._refs = kw                      # keeps the tensors behind the raw pointers alive

    def __call__(self, stream=None):
        _check(lib().hx_decode_step(C.byref(self.a), _stream_ptr(stream)))

    def is_fused(self) -> bool:
        """hx_decode_step_is_fused: would this step run as the one fused kernel?  Enqueues nothing."""
        f = C.c_int32(0)
        _check(lib().hx_decode_step_is_fused(C.byref(self.a), C.byref(f)))
        return bool(f.value)


def decode_step(stream=None, **kw):
    """hx_decode_step (include/hx.h): ingest of the step's new prompts + attention over the active batch."""
    DecodeStep(**kw)(stream)


def shutdown():
    _check(lib().hx_shutdown())


class PagePool:
    """hx_page_pool: host free list of page ids (all-or-nothing allocation)."""

    def __init__(self, num_pages: int, shuffle_seed: Optional[int] = None):
        self._h = C.c_void_p()
        _check(lib().hx_pool_create(C.byref(self._h), num_pages))
        if shuffle_seed is not None:
            self.shuffle(shuffle_seed)

    def shuffle(self, seed: int):
        _check(lib().hx_pool_shuffle(self._h, seed))

    def alloc(self, n: int):
        import numpy as np
        ids = np.empty(n, dtype=np.int32)
        _check(lib().hx_pool_alloc(self._h, n, ids.ctypes.data))
        return ids

    def free(self, ids):
        import numpy as np
        ids = np.ascontiguousarray(ids, dtype=np.int32)
        _check(lib().hx_pool_free(self._h, ids.ctypes.data, ids.size))

    def alloc_table(self, seq_lens, stride: int, page_size: int = 16):
        import numpy as np
        seq_lens = np.ascontiguousarray(seq_lens, dtype=np.int32)
        bt = np.empty((len(seq_lens), stride), dtype=np.int32)
        _check(lib().hx_pool_alloc_table(self._h, seq_lens.ctypes.data, len(seq_lens), page_size,
                                         bt.ctypes.data, stride))
        return bt

    @property
    def num_free(self) -> int:
        return int(lib().hx_pool_num_free(self._h))

    @property
    def num_pages(self) -> int:
        return int(lib().hx_pool_num_pages(self._h))

    def close(self):
        if self._h:
            lib().hx_pool_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
