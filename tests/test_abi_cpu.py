"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/hx.h declares,
the host page allocator behaves, and every invalid-argument class is rejected BEFORE any CUDA
call (so these run without a GPU; no compute call is made)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_2502_07903_b200 as hx
from paper_2502_07903_b200 import binding as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "hx.h")).read()
    declared = set(re.findall(r"\b(hx_[a-z_0-9]+)\s*\(", header))
    declared -= {"hx_page_pool"}
    assert declared == set(B.EXPORTS), declared ^ set(B.EXPORTS)
    L = hx.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert hx.version() == 135
    assert hx.status_string(0) == "HX_OK" and hx.status_string(5) == "HX_ERR_NO_PAGES"
    assert hx.status_string(77) == "HX_ERR_UNKNOWN"


def test_paged_cache_bytes():
    assert hx.paged_cache_bytes(80, 100, 4, 16, 128) == 80 * 100 * 4 * 16 * 128 * 2
    assert hx.paged_cache_bytes(0, 100, 4, 16, 128) == 0
    assert hx.paged_cache_bytes(2**31 - 1, 2**31 - 1, 2**31 - 1, 16, 128) == 0   # overflow


def test_pool_alloc_free_invariants():
    pool = hx.PagePool(64, shuffle_seed=7)
    pool2 = hx.PagePool(64, shuffle_seed=7)
    a = pool.alloc(10)
    assert np.array_equal(a, pool2.alloc(10))            # deterministic in the seed
    assert len(set(a.tolist())) == 10 and a.min() >= 0 and a.max() < 64
    assert pool.num_free == 54 and pool.num_pages == 64
    b = pool.alloc(54)
    assert set(a.tolist()) | set(b.tolist()) == set(range(64))
    with pytest.raises(hx.HxError) as e:
        pool.alloc(1)
    assert e.value.status == B.HX_ERR_NO_PAGES and pool.num_free == 0
    pool.free(a)
    assert pool.num_free == 10
    for bad in ([a[0]], [64], [-1], [b[0], b[0]]):       # double free, range, duplicate
        with pytest.raises(hx.HxError) as e:
            pool.free(bad)
        assert e.value.status == B.HX_ERR_INVALID_ARG and pool.num_free == 10
    pool.free(b)
    assert pool.num_free == 64
    assert hx.PagePool(0).num_free == 0


def test_pool_alloc_table_all_or_nothing():
    pool = hx.PagePool(10, shuffle_seed=1)
    bt = pool.alloc_table([17, 1, 0, 33], stride=4)
    assert (bt >= 0).sum(axis=1).tolist() == [2, 1, 0, 3] and pool.num_free == 4
    used = bt[bt >= 0]
    assert len(set(used.tolist())) == 6
    assert (bt[0, 2:] == -1).all() and (bt[2] == -1).all()
    with pytest.raises(hx.HxError) as e:
        pool.alloc_table([16 * 5], stride=8)
    assert e.value.status == B.HX_ERR_NO_PAGES and pool.num_free == 4
    with pytest.raises(hx.HxError) as e:
        pool.alloc_table([16 * 3], stride=2)             # row does not fit the stride
    assert e.value.status == B.HX_ERR_INVALID_ARG and pool.num_free == 4


class FakeCache:
    def __init__(self, layers=2, pages=8, heads=2, ps=16, D=128, k=0x1000, v=0x2000):
        self.c = B._CCache(k, v, layers, pages, heads, ps, D)

    @property
    def ref(self):
        return C.byref(self.c)


def _attn(cache=None, **over):
    kw = dict(layer=0, q_heads=4, block_table=0x3000, block_table_stride=4, seq_lens=0x4000, batch=2,
              max_seq_len=64, sm_scale=0.0, workspace=0x5000, workspace_bytes=1 << 30, stream=0)
    kw.update(over)
    out = kw.pop("out", 0x6000)
    q = kw.pop("q", 0x7000)
    hx.decode_attention(out, q, cache or FakeCache(), **kw)


@pytest.mark.parametrize("over,status", [
    (dict(out=0), B.HX_ERR_INVALID_ARG), (dict(q=0x7001), B.HX_ERR_INVALID_ARG),
    (dict(layer=2), B.HX_ERR_INVALID_ARG), (dict(layer=-1), B.HX_ERR_INVALID_ARG),
    (dict(q_heads=3), B.HX_ERR_INVALID_ARG), (dict(q_heads=6), B.HX_ERR_UNSUPPORTED),
    (dict(batch=-1), B.HX_ERR_INVALID_ARG), (dict(block_table_stride=3), B.HX_ERR_INVALID_ARG),
    (dict(block_table=0), B.HX_ERR_INVALID_ARG), (dict(seq_lens=0), B.HX_ERR_INVALID_ARG),
    (dict(sm_scale=float("nan")), B.HX_ERR_INVALID_ARG),
    (dict(cache=FakeCache(D=96)), B.HX_ERR_UNSUPPORTED), (dict(cache=FakeCache(ps=32)), B.HX_ERR_UNSUPPORTED),
    (dict(cache=FakeCache(k=0)), B.HX_ERR_INVALID_ARG), (dict(cache=FakeCache(v=0x2008)), B.HX_ERR_INVALID_ARG),
    (dict(cache=FakeCache(pages=0)), B.HX_ERR_INVALID_ARG),
])
def test_attention_rejects_invalid_arguments_without_launching(over, status):
    with pytest.raises(hx.HxError) as e:
        _attn(**over)
    assert e.value.status == status, str(e.value)
    assert hx.last_error()


def test_attention_workspace_check_and_empty_batch():
    need = hx.decode_attention_workspace_bytes(256, 64, 8, 128, 8192)
    assert need > 0 and need % 16 == 0
    with pytest.raises(hx.HxError) as e:
        _attn(cache=FakeCache(heads=8), q_heads=64, batch=256, max_seq_len=8192, block_table_stride=512,
              workspace_bytes=need - 1)
    assert e.value.status == B.HX_ERR_WORKSPACE
    with pytest.raises(hx.HxError) as e:
        _attn(cache=FakeCache(heads=8), q_heads=64, batch=256, max_seq_len=8192, block_table_stride=512,
              workspace=0, workspace_bytes=need)
    assert e.value.status == B.HX_ERR_WORKSPACE
    _attn(batch=0, out=0, q=0, block_table=0, seq_lens=0)          # HX_OK, nothing launched


def _ingest(fn=None, cache=None, src=None, **over):
    kw = dict(layers=2, heads=4, head_dim=128, src_tp=2, dst_tp=2, dst_rank=0, block_table=0x3000,
              block_table_stride=4, cu_seqlens=0x4000, seq_lens=0x5000, batch=2, total_tokens=100,
              max_seq_len=64, stream=0)
    kw.update(over)
    s = src if src is not None else [0x10000 * (r + 1) for r in range(kw["src_tp"])]
    (fn or hx.kv_ingest)(s, list(s), dst=cache or FakeCache(), **kw)


@pytest.mark.parametrize("over,status", [
    (dict(heads=5), B.HX_ERR_INVALID_ARG), (dict(heads=6, dst_tp=4), B.HX_ERR_INVALID_ARG),
    (dict(src_tp=8, src=[0x100] * 8), B.HX_ERR_UNSUPPORTED), (dict(dst_tp=8), B.HX_ERR_UNSUPPORTED),
    (dict(dst_rank=2), B.HX_ERR_INVALID_ARG), (dict(dst_rank=-1), B.HX_ERR_INVALID_ARG),
    (dict(layers=3), B.HX_ERR_INVALID_ARG), (dict(layers=-1), B.HX_ERR_INVALID_ARG),
    (dict(head_dim=64), B.HX_ERR_INVALID_ARG), (dict(cache=FakeCache(heads=4)), B.HX_ERR_INVALID_ARG),
    (dict(block_table_stride=3), B.HX_ERR_INVALID_ARG), (dict(max_seq_len=200), B.HX_ERR_INVALID_ARG),
    (dict(cu_seqlens=0), B.HX_ERR_INVALID_ARG), (dict(src=[0, 0x20000]), B.HX_ERR_INVALID_ARG),
    (dict(src=[0x10004, 0x20000]), B.HX_ERR_INVALID_ARG), (dict(cache=FakeCache(D=96), head_dim=96), B.HX_ERR_UNSUPPORTED),
])
@pytest.mark.parametrize("fn", ["kv_ingest", "kv_gather"])
def test_ingest_rejects_invalid_arguments_without_launching(fn, over, status):
    with pytest.raises(hx.HxError) as e:
        _ingest(fn=getattr(hx, fn), **over)
    assert e.value.status == status, str(e.value)


def test_ingest_unneeded_shard_may_be_null_and_empty_is_ok():
    # dst_rank 1 of dst_tp 2 with src_tp 2 needs only shard 1; batch == 0 returns OK before launch
    _ingest(src=[0, 0x20000], dst_rank=1, batch=0)
    _ingest(total_tokens=0, max_seq_len=0)
    _ingest(layers=0)


# ---------------------------------------------------------------- F3 / F1 entry points
def _stage(cache=None, src=None, **over):
    kw = dict(src_layers=3, src_layer0=1, dst_layer0=0, layers=2, heads=4, head_dim=128, src_tp=2, dst_tp=2,
              dst_rank=0, block_table=0x3000, block_table_stride=4, cu_seqlens=0x4000, seq_lens=0x5000, batch=2,
              total_tokens=100, max_seq_len=64, stream=0)
    kw.update(over)
    s = src if src is not None else [0x10000 * (r + 1) for r in range(kw["src_tp"])]
    hx.kv_ingest_stage(s, list(s), dst=cache or FakeCache(), **kw)


@pytest.mark.parametrize("over,status", [
    (dict(src_layer0=2), B.HX_ERR_INVALID_ARG), (dict(src_layer0=-1), B.HX_ERR_INVALID_ARG),
    (dict(dst_layer0=1), B.HX_ERR_INVALID_ARG), (dict(dst_layer0=-1), B.HX_ERR_INVALID_ARG),
    (dict(src_layers=-1), B.HX_ERR_INVALID_ARG), (dict(layers=-1), B.HX_ERR_INVALID_ARG),
    (dict(layers=3, src_layer0=0), B.HX_ERR_INVALID_ARG), (dict(heads=5), B.HX_ERR_INVALID_ARG),
    (dict(src=[0, 0x20000]), B.HX_ERR_INVALID_ARG),
])
def test_stage_ingest_rejects_invalid_arguments_without_launching(over, status):
    with pytest.raises(hx.HxError) as e:
        _stage(**over)
    assert e.value.status == status, str(e.value)
    _stage(layers=0)                                                   # nothing to move: OK, no launch
    _stage(batch=0)


def test_stage_overlap_host_helper():
    # prefill stages of 80 layers cut 27/27/26, decode stages 40/40 (Table 2 has PP=3 and PP=2)
    src = [(0, 27), (27, 27), (54, 26)]
    dst = [(0, 40), (40, 40)]
    covered = np.zeros((80,), dtype=int)
    for sf, sc in src:
        for df, dc in dst:
            a, b, n = hx.stage_overlap(sf, sc, df, dc)
            if n:
                assert sf + a == df + b and 0 <= a and a + n <= sc and 0 <= b and b + n <= dc
                covered[sf + a: sf + a + n] += 1
    assert (covered == 1).all()                                        # every layer moved exactly once
    assert hx.stage_overlap(0, 10, 10, 5) == (0, 0, 0)
    assert hx.stage_overlap(3, 4, 0, 100) == (0, 3, 4)
    with pytest.raises(hx.HxError):
        hx.stage_overlap(-1, 4, 0, 100)


def _append(cache=None, fused=False, **over):
    kw = dict(layer=0, block_table=0x3000, block_table_stride=4, seq_lens=0x4000, batch=2, max_seq_len=64, stream=0)
    kw.update(over)
    kn, vn = kw.pop("k_new", 0x8000), kw.pop("v_new", 0x9000)
    if fused:
        hx.decode_attention_append(kw.pop("out", 0x6000), kw.pop("q", 0x7000), kn, vn, cache or FakeCache(),
                                   q_heads=4, workspace=0x5000, workspace_bytes=1 << 30, **kw)
    else:
        hx.kv_append(kn, vn, cache or FakeCache(), **kw)


@pytest.mark.parametrize("fused", [False, True])
@pytest.mark.parametrize("over,status", [
    (dict(k_new=0), B.HX_ERR_INVALID_ARG), (dict(v_new=0x9004), B.HX_ERR_INVALID_ARG),
    (dict(layer=2), B.HX_ERR_INVALID_ARG), (dict(batch=-1), B.HX_ERR_INVALID_ARG),
    (dict(block_table=0), B.HX_ERR_INVALID_ARG), (dict(seq_lens=0), B.HX_ERR_INVALID_ARG),
    (dict(block_table_stride=3), B.HX_ERR_INVALID_ARG), (dict(cache=FakeCache(ps=8)), B.HX_ERR_UNSUPPORTED),
])
def test_append_rejects_invalid_arguments_without_launching(fused, over, status):
    with pytest.raises(hx.HxError) as e:
        _append(fused=fused, **over)
    assert e.value.status == status, str(e.value)
    _append(fused=fused, batch=0)


# ---------------------------------------------------------------- F4 entry point
def _prefill(cache=None, **over):
    kw = dict(layer=0, q_heads=4, block_table=0x3000, block_table_stride=4, seq_lens=0x4000, q_lens=0x4100,
              cu_q_lens=0x4200, batch=2, total_q_tokens=100, max_q_len=64, max_seq_len=64, sm_scale=0.0, stream=0)
    kw.update(over)
    out, q = kw.pop("out", 0x6000), kw.pop("q", 0x7000)
    hx.prefill_attention(out, q, cache or FakeCache(), **kw)


@pytest.mark.parametrize("over,status", [
    (dict(out=0), B.HX_ERR_INVALID_ARG), (dict(q=0x7004), B.HX_ERR_INVALID_ARG),
    (dict(layer=2), B.HX_ERR_INVALID_ARG), (dict(q_heads=3), B.HX_ERR_INVALID_ARG),
    (dict(q_heads=6), B.HX_ERR_UNSUPPORTED), (dict(batch=-1), B.HX_ERR_INVALID_ARG),
    (dict(q_lens=0), B.HX_ERR_INVALID_ARG), (dict(cu_q_lens=0), B.HX_ERR_INVALID_ARG),
    (dict(max_q_len=65), B.HX_ERR_INVALID_ARG), (dict(max_q_len=101, max_seq_len=200, block_table_stride=13), B.HX_ERR_INVALID_ARG),
    (dict(block_table_stride=3), B.HX_ERR_INVALID_ARG), (dict(sm_scale=float("nan")), B.HX_ERR_INVALID_ARG),
    (dict(cache=FakeCache(D=96)), B.HX_ERR_UNSUPPORTED), (dict(cache=FakeCache(ps=32)), B.HX_ERR_UNSUPPORTED),
])
def test_prefill_rejects_invalid_arguments_without_launching(over, status):
    with pytest.raises(hx.HxError) as e:
        _prefill(**over)
    assert e.value.status == status, str(e.value)
    _prefill(batch=0, out=0, q=0)                       # HX_OK, nothing launched
    _prefill(total_q_tokens=0, max_q_len=0)


def test_attention_overlapped_validates_like_attention():
    kw = dict(layer=0, q_heads=4, block_table=0x3000, block_table_stride=4, seq_lens=0x4000, batch=2,
              max_seq_len=64, sm_scale=0.0, workspace=0x5000, workspace_bytes=1 << 30, behind_ingest=1, stream=0)
    for over, status in [(dict(layer=2), B.HX_ERR_INVALID_ARG), (dict(q_heads=6), B.HX_ERR_UNSUPPORTED),
                         (dict(workspace=0), B.HX_ERR_WORKSPACE), (dict(block_table_stride=3), B.HX_ERR_INVALID_ARG),
                         (dict(behind_ingest=0, layer=2), B.HX_ERR_INVALID_ARG)]:
        with pytest.raises(hx.HxError) as e:
            hx.decode_attention_overlapped(0x6000, 0x7000, FakeCache(), **dict(kw, **over))
        assert e.value.status == status, str(e.value)
    hx.decode_attention_overlapped(0, 0, FakeCache(), **dict(kw, batch=0, block_table=0, seq_lens=0))   # HX_OK, no launch


# ---------------------------------------------------------------- whole-step entry points
def _step(**over):
    kw = dict(out=0x6000, q=0x7000, cache=FakeCache(heads=4), layer=0, q_heads=4, block_table=0x3000, block_table_stride=4,
              seq_lens=0x4000, batch=2, max_seq_len=64, sm_scale=0.0, workspace=0x5000, workspace_bytes=1 << 30,
              src_k=[0x10000, 0x20000], src_v=[0x30000, 0x40000], ing_layers=2, heads=4, src_tp=2, dst_tp=1, dst_rank=0,
              ing_block_table=0x8000, ing_block_table_stride=4, ing_cu_seqlens=0x9000, ing_seq_lens=0xA000, ing_batch=2,
              ing_total_tokens=100, ing_max_seq_len=64, overlap_ingest=1, stream=0)
    kw.update(over)
    hx.decode_step(**kw)


@pytest.mark.parametrize("over,status", [
    # an error in EITHER half is found before anything is enqueued (no CUDA call is made: this runs without a GPU)
    (dict(layer=2), B.HX_ERR_INVALID_ARG), (dict(q_heads=3), B.HX_ERR_INVALID_ARG), (dict(workspace=0), B.HX_ERR_WORKSPACE),
    (dict(out=0), B.HX_ERR_INVALID_ARG), (dict(block_table_stride=3), B.HX_ERR_INVALID_ARG),
    (dict(heads=5), B.HX_ERR_INVALID_ARG), (dict(dst_rank=1), B.HX_ERR_INVALID_ARG), (dict(ing_layers=3), B.HX_ERR_INVALID_ARG),
    (dict(src_k=[0, 0x20000]), B.HX_ERR_INVALID_ARG), (dict(ing_cu_seqlens=0), B.HX_ERR_INVALID_ARG),
    (dict(ing_max_seq_len=200), B.HX_ERR_INVALID_ARG), (dict(batch=-1), B.HX_ERR_INVALID_ARG), (dict(ing_batch=-1), B.HX_ERR_INVALID_ARG),
    # size limits of the attention launch are part of the dry run too (they used to surface only at launch time,
    # after the ingest half of an in-order step had been enqueued)
    (dict(cache=FakeCache(layers=80, pages=1 << 20, heads=4), overlap_ingest=0), B.HX_ERR_UNSUPPORTED),   # >= 2^31 cache rows
    (dict(block_table_stride=1 << 16, overlap_ingest=0), B.HX_ERR_UNSUPPORTED),                          # 2048 * stride * heads >= 2^28
])
def test_decode_step_validates_both_halves_before_it_enqueues(over, status):
    with pytest.raises(hx.HxError) as e:
        _step(**over)
    assert e.value.status == status, str(e.value)
    assert hx.last_error()


def test_decode_step_with_nothing_to_do_is_ok():
    _step(batch=0, ing_batch=0)                                       # HX_OK, nothing enqueued


def test_decode_step_host_validates_before_it_enqueues():
    kw = dict(q_host=0x100, out_host=0x200, q_dev=0x7000, out_dev=0x6000, cache=FakeCache(heads=4), layer=0, q_heads=4,
              block_table_dev=0x3000, block_table_stride=4, seq_lens_dev=0x4000, batch=2, max_seq_len=64, sm_scale=0.0,
              workspace=0x5000, workspace_bytes=1 << 30, src_k_host=[0x10000, 0x20000], src_v_host=[0x30000, 0x40000],
              src_k_dev=[0x50000, 0x60000], src_v_dev=[0x70000, 0x80000], ing_layers=2, heads=4, src_tp=2, dst_tp=1, dst_rank=0,
              ing_block_table_host=0x300, ing_block_table_stride=4, ing_cu_seqlens_host=0x400, ing_seq_lens_host=0x500,
              ing_block_table_dev=0x8000, ing_cu_seqlens_dev=0x9000, ing_seq_lens_dev=0xA000, ing_batch=2, ing_total_tokens=100,
              ing_max_seq_len=64, pull_src=0, overlap_ingest=1, stream=0)
    for over, status in [(dict(layer=5), B.HX_ERR_INVALID_ARG), (dict(q_host=0), B.HX_ERR_INVALID_ARG),
                         (dict(ing_seq_lens_host=0), B.HX_ERR_INVALID_ARG), (dict(heads=3), B.HX_ERR_INVALID_ARG),
                         (dict(workspace_bytes=16), B.HX_ERR_WORKSPACE), (dict(src_k_dev=[0, 0]), B.HX_ERR_INVALID_ARG)]:
        with pytest.raises(hx.HxError) as e:
            hx.decode_step_host(**dict(kw, **over))
        assert e.value.status == status, (over, str(e.value))


# ---------------------------------------------------------------- per-step plan
def test_plan_entry_points_reject_invalid_arguments_without_launching():
    need = hx.decode_plan_bytes(2, 2, 64)
    assert need > 0 and hx.decode_plan_bytes(-1, 2, 64) == 0
    pk = dict(q_heads=4, block_table=0x3000, block_table_stride=4, seq_lens=0x4000, batch=2, max_seq_len=64, plan_bytes=need, stream=0)
    for over, status in [(dict(plan_bytes=need - 1), B.HX_ERR_WORKSPACE), (dict(q_heads=3), B.HX_ERR_INVALID_ARG),
                         (dict(block_table=0), B.HX_ERR_INVALID_ARG), (dict(seq_lens=0), B.HX_ERR_INVALID_ARG),
                         (dict(block_table_stride=3), B.HX_ERR_INVALID_ARG), (dict(batch=-1), B.HX_ERR_INVALID_ARG)]:
        with pytest.raises(hx.HxError) as e:
            hx.decode_plan(0x9000, FakeCache(), **dict(pk, **over))
        assert e.value.status == status, (over, str(e.value))
    with pytest.raises(hx.HxError) as e:
        hx.decode_plan(0, FakeCache(), **pk)
    assert e.value.status == B.HX_ERR_INVALID_ARG
    hx.decode_plan(0, FakeCache(), **dict(pk, batch=0))                 # HX_OK, nothing launched
    ak = dict(layer=0, q_heads=4, plan=0x9000, plan_bytes=need, batch=2, max_seq_len=64, sm_scale=0.0, workspace=0x5000,
              workspace_bytes=1 << 30, stream=0)
    for over, status in [(dict(plan=0), B.HX_ERR_INVALID_ARG), (dict(plan=0x9004), B.HX_ERR_INVALID_ARG),
                         (dict(plan_bytes=16), B.HX_ERR_WORKSPACE), (dict(layer=2), B.HX_ERR_INVALID_ARG),
                         (dict(workspace=0), B.HX_ERR_WORKSPACE), (dict(q_heads=6), B.HX_ERR_UNSUPPORTED)]:
        with pytest.raises(hx.HxError) as e:
            hx.decode_attention_planned(0x6000, 0x7000, FakeCache(), **dict(ak, **over))
        assert e.value.status == status, (over, str(e.value))
    hx.decode_attention_planned(0, 0, FakeCache(), **dict(ak, batch=0))  # HX_OK, nothing launched
    for ready in (0, 1):                                                 # the chained launch validates like the planned one
        for over, status in [(dict(plan=0), B.HX_ERR_INVALID_ARG), (dict(plan_bytes=16), B.HX_ERR_WORKSPACE),
                             (dict(layer=2), B.HX_ERR_INVALID_ARG), (dict(workspace=0), B.HX_ERR_WORKSPACE)]:
            with pytest.raises(hx.HxError) as e:
                hx.decode_attention_chained(0x6000, 0x7000, FakeCache(), inputs_ready=ready, **dict(ak, **over))
            assert e.value.status == status, (ready, over, str(e.value))
        hx.decode_attention_chained(0, 0, FakeCache(), inputs_ready=ready, **dict(ak, batch=0))
