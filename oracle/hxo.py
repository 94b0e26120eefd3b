"""ctypes wrapper for oracle/hxo.c (argument marshalling only) + the float64 merge formula."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libhxo.so")
_SRC = os.path.join(_HERE, "hxo.c")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2, no intrinsics, no BLAS."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared",
                               "-o", _SO, _SRC, "-lm"])
    return _SO


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        L.hxo_half_to_double.restype = C.c_double
        L.hxo_half_to_double.argtypes = [C.c_uint16]
        L.hxo_max_threads.restype = C.c_int
        _lib = L
    return _lib


def max_threads() -> int:
    return int(lib().hxo_max_threads())


def _p(a, t=C.c_void_p):
    return C.cast(a.ctypes.data, t)


def half_to_double(bits: np.ndarray) -> np.ndarray:
    bits = np.ascontiguousarray(bits, dtype=np.uint16)
    out = np.empty(bits.shape, dtype=np.float64)
    lib().hxo_half_to_double_array(_p(bits), _p(out), C.c_int64(bits.size))
    return out


def _u16(a):
    a = np.asarray(a)
    if a.dtype == np.float16:
        a = a.view(np.uint16)
    assert a.dtype == np.uint16 and a.flags.c_contiguous
    return a


def _ingest(src_k, src_v, dst_k, dst_v, *, heads, src_tp, dst_tp, dst_rank, block_table,
            cu_seqlens, seq_lens, gather, threads):
    src_k = [_u16(a) for a in src_k]
    src_v = [_u16(a) for a in src_v]
    dst_k, dst_v = _u16(dst_k), _u16(dst_v)
    L, T, hs, D = src_k[0].shape
    Ld, P, hd, ps, Dd = dst_k.shape
    assert len(src_k) == src_tp == len(src_v) and hs == heads // src_tp
    assert (Ld, hd, Dd) == (L, heads // dst_tp, D) and dst_v.shape == dst_k.shape
    bt = np.ascontiguousarray(block_table, dtype=np.int32)
    cu = np.ascontiguousarray(cu_seqlens, dtype=np.int32)
    sl = np.ascontiguousarray(seq_lens, dtype=np.int32)
    PK = (C.c_void_p * src_tp)(*[a.ctypes.data for a in src_k])
    PV = (C.c_void_p * src_tp)(*[a.ctypes.data for a in src_v])
    rc = lib().hxo_kv_ingest(PK, PV, L, T, heads, D, src_tp, dst_tp, dst_rank, _p(dst_k), _p(dst_v),
                             P, ps, _p(bt), bt.shape[1], _p(cu), _p(sl), len(sl), int(gather),
                             int(threads))
    if rc:
        raise ValueError(f"hxo_kv_ingest: invalid arguments ({rc})")


def kv_ingest(src_k, src_v, dst_k, dst_v, *, heads, src_tp, dst_tp, dst_rank, block_table,
              cu_seqlens, seq_lens, threads=0):
    """Writes into dst_k / dst_v in place (only the valid slots of dst_rank's heads)."""
    _ingest(src_k, src_v, dst_k, dst_v, heads=heads, src_tp=src_tp, dst_tp=dst_tp,
            dst_rank=dst_rank, block_table=block_table, cu_seqlens=cu_seqlens, seq_lens=seq_lens,
            gather=0, threads=threads)


def kv_gather(src_k, src_v, dst_k, dst_v, *, heads, src_tp, dst_tp, dst_rank, block_table,
              cu_seqlens, seq_lens, threads=0):
    """Exact inverse: writes into the src_* shards in place from the paged cache."""
    _ingest(src_k, src_v, dst_k, dst_v, heads=heads, src_tp=src_tp, dst_tp=dst_tp,
            dst_rank=dst_rank, block_table=block_table, cu_seqlens=cu_seqlens, seq_lens=seq_lens,
            gather=1, threads=threads)


def kv_ingest_stage(src_k, src_v, dst_k, dst_v, *, heads, src_tp, dst_tp, dst_rank, src_layer0,
                    dst_layer0, count, block_table, cu_seqlens, seq_lens):
    """Pipeline-stage ingest (F3): `count` layers, source layer src_layer0+c -> cache layer
    dst_layer0+c.  Source and cache may hold different numbers of layers."""
    src_k = [_u16(a) for a in src_k]
    src_v = [_u16(a) for a in src_v]
    dst_k, dst_v = _u16(dst_k), _u16(dst_v)
    Ls, T, hs, D = src_k[0].shape
    Ld, P, hd, ps, Dd = dst_k.shape
    assert len(src_k) == src_tp == len(src_v) and hs == heads // src_tp
    assert (hd, Dd) == (heads // dst_tp, D) and dst_v.shape == dst_k.shape
    bt = np.ascontiguousarray(block_table, dtype=np.int32)
    cu = np.ascontiguousarray(cu_seqlens, dtype=np.int32)
    sl = np.ascontiguousarray(seq_lens, dtype=np.int32)
    PK = (C.c_void_p * src_tp)(*[a.ctypes.data for a in src_k])
    PV = (C.c_void_p * src_tp)(*[a.ctypes.data for a in src_v])
    rc = lib().hxo_kv_ingest_stage(PK, PV, Ls, src_layer0, Ld, dst_layer0, count, T, heads, D, src_tp,
                                   dst_tp, dst_rank, _p(dst_k), _p(dst_v), P, ps, _p(bt), bt.shape[1],
                                   _p(cu), _p(sl), len(sl))
    if rc:
        raise ValueError(f"hxo_kv_ingest_stage: invalid arguments ({rc})")


def kv_append(k_new, v_new, k, v, *, layer, block_table, seq_lens):
    """Append (F1): writes token n_i-1 of every request with n_i >= 1 into k / v in place."""
    k_new, v_new, k, v = _u16(k_new), _u16(v_new), _u16(k), _u16(v)
    B, Hkv, D = k_new.shape
    Ln, P, Hk, ps, Dk = k.shape
    assert (Hk, Dk) == (Hkv, D) and v.shape == k.shape and v_new.shape == k_new.shape
    bt = np.ascontiguousarray(block_table, dtype=np.int32)
    sl = np.ascontiguousarray(seq_lens, dtype=np.int32)
    assert len(sl) == B
    rc = lib().hxo_kv_append(_p(k_new), _p(v_new), _p(k), _p(v), layer, Ln, P, Hkv, ps, D, _p(bt),
                             bt.shape[1], _p(sl), B)
    if rc:
        raise ValueError("hxo_kv_append: invalid arguments")


def default_scale(head_dim: int) -> float:
    """(double)(float)(1/sqrt(D)): the constant both sides use (reading S2)."""
    return float(np.float32(1.0) / np.sqrt(np.float32(head_dim)))


def decode_attention(q, k, v, block_table, seq_lens, *, layer=0, sm_scale=None, threads=0):
    """q fp16 [B][Hq][D]; k, v fp16 [layers][P][Hkv][ps][D] -> float64 [B][Hq][D]."""
    q, k, v = _u16(q), _u16(k), _u16(v)
    B, Hq, D = q.shape
    Ln, P, Hkv, ps, Dk = k.shape
    assert Dk == D and v.shape == k.shape and 0 <= layer < Ln
    bt = np.ascontiguousarray(block_table, dtype=np.int32)
    sl = np.ascontiguousarray(seq_lens, dtype=np.int32)
    scale = default_scale(D) if sm_scale is None or sm_scale <= 0 else float(np.float32(sm_scale))
    out = np.empty((B, Hq, D), dtype=np.float64)
    rc = lib().hxo_decode_attention(_p(out), _p(q), _p(k), _p(v), layer, P, Hkv, ps, D, Hq, _p(bt),
                                    bt.shape[1], _p(sl), B, C.c_double(scale), int(threads))
    if rc:
        raise ValueError("hxo_decode_attention: invalid arguments")
    return out


def prefill_attention(q, k, v, block_table, seq_lens, q_lens, *, layer=0, sm_scale=None, threads=0):
    """Causal paged attention of the LAST q_lens[i] tokens of each request (F4).
    q fp16 [sum(q_lens)][Hq][D] packed by request -> float64 of the same shape."""
    q, k, v = _u16(q), _u16(k), _u16(v)
    Tq, Hq, D = q.shape
    Ln, P, Hkv, ps, Dk = k.shape
    assert Dk == D and v.shape == k.shape and 0 <= layer < Ln
    bt = np.ascontiguousarray(block_table, dtype=np.int32)
    sl = np.ascontiguousarray(seq_lens, dtype=np.int32)
    ql = np.ascontiguousarray(q_lens, dtype=np.int32)
    cu = np.zeros(len(ql) + 1, dtype=np.int32)
    np.cumsum(ql, out=cu[1:])
    assert cu[-1] == Tq and len(ql) == len(sl)
    scale = default_scale(D) if sm_scale is None or sm_scale <= 0 else float(np.float32(sm_scale))
    out = np.zeros((Tq, Hq, D), dtype=np.float64)
    rc = lib().hxo_prefill_attention(_p(out), _p(q), _p(k), _p(v), layer, P, Hkv, ps, D, Hq, _p(bt),
                                     bt.shape[1], _p(sl), _p(ql), _p(cu), len(sl), C.c_double(scale), int(threads))
    if rc:
        raise ValueError(f"hxo_prefill_attention: invalid arguments ({rc})")
    return out


def partial_attention(q_row, k, v, bt_row, g, t0, t1, *, layer=0, scale):
    q_row, k, v = _u16(q_row), _u16(k), _u16(v)
    _, P, Hkv, ps, D = k.shape
    bt_row = np.ascontiguousarray(bt_row, dtype=np.int32)
    m, l = C.c_double(), C.c_double()
    acc = np.empty(D, dtype=np.float64)
    lib().hxo_partial_attention(C.byref(m), C.byref(l), _p(acc), _p(q_row), _p(k), _p(v), layer, P,
                                Hkv, g, ps, D, _p(bt_row), t0, t1, C.c_double(scale))
    return m.value, l.value, acc


def merge_partials(parts):
    """Online-softmax merge in float64: m = max m_c; l = sum l_c e^{m_c-m}; acc likewise; out = acc/l.
    (FlashAttention identity, cited PAPER.md:L110.)"""
    m = max(p[0] for p in parts)
    l = sum(p[1] * np.exp(p[0] - m) for p in parts)
    acc = sum(p[2] * np.exp(p[0] - m) for p in parts)
    return acc / l
