"""Pins for the oracle's NEXT-row functions: pipeline-stage ingest (F3) and
append of the decode step's token (F1), against things other than themselves.  CPU only."""
import numpy as np
import pytest
from scipy.special import softmax

import oracle
import workloads as W
from test_oracle_pins import dense_reference, numpy_ingest, small_case


# ---------------------------------------------------------------- F3: stage ingest
def _stage_case(S, R, L=6, seed_extra=0):
    heads, D, ps = 8, 16, 4
    lens = np.array([3, 4, 9, 16, 1], dtype=np.int32)
    c = W.IngestConfig(92, "t", L, heads, D, S, R, len(lens), "x")
    return W.make_ingest_inputs(c, lens=lens, bits=True, page_size=ps, seed_extra=seed_extra), heads, D, ps, lens


@pytest.mark.parametrize("S,R", [(1, 1), (4, 2), (2, 4), (8, 1)])
@pytest.mark.parametrize("src_cuts,dst_cuts", [([0, 6], [0, 6]), ([0, 2, 6], [0, 3, 6]), ([0, 1, 2, 5, 6], [0, 4, 6]),
                                               ([0, 6], [0, 1, 2, 3, 4, 5, 6])])
def test_stage_ingest_any_cut_equals_whole_model_ingest(S, R, src_cuts, dst_cuts):
    """layer j of the prefill replica goes to the GPU holding layer j of the decode
    replica.  Cut the L layers into prefill stages and, differently, into decode stages; moving
    every overlapping layer range stage pair by stage pair must build exactly the caches that the
    one-call ingest of the whole model builds (then sliced per decode stage)."""
    w, heads, D, ps, lens = _stage_case(S, R, seed_extra=S * 10 + R)
    L, P, hd = w["layers"], w["num_pages"], heads // R
    kw = dict(heads=heads, src_tp=S, dst_tp=R, block_table=w["block_table"], cu_seqlens=w["cu_seqlens"], seq_lens=lens)
    for qrank in range(R):
        whole_k = numpy_ingest(w["src_k"], heads, S, R, qrank, P, ps, w["block_table"], w["cu_seqlens"], lens)
        whole_v = numpy_ingest(w["src_v"], heads, S, R, qrank, P, ps, w["block_table"], w["cu_seqlens"], lens)
        for b0, b1 in zip(dst_cuts[:-1], dst_cuts[1:]):                 # one decode stage = one cache
            dk = np.full((b1 - b0, P, hd, ps, D), 0xDEAD, dtype=np.uint16)
            dv = np.full_like(dk, 0xDEAD)
            for a0, a1 in zip(src_cuts[:-1], src_cuts[1:]):             # one prefill stage = one set of shards
                lo, hi = max(a0, b0), min(a1, b1)
                if lo >= hi:
                    continue
                sk = [np.ascontiguousarray(a[a0:a1]) for a in w["src_k"]]
                sv = [np.ascontiguousarray(a[a0:a1]) for a in w["src_v"]]
                oracle.kv_ingest_stage(sk, sv, dk, dv, dst_rank=qrank, src_layer0=lo - a0, dst_layer0=lo - b0,
                                       count=hi - lo, **kw)
            assert np.array_equal(dk, whole_k[b0:b1]) and np.array_equal(dv, whole_v[b0:b1])


def test_stage_ingest_touches_only_the_named_layers_and_rejects_bad_ranges():
    w, heads, D, ps, lens = _stage_case(2, 2, L=3)
    P = w["num_pages"]
    dk = np.full((5, P, 4, ps, D), 0xDEAD, dtype=np.uint16)
    dv = np.full_like(dk, 0xDEAD)
    kw = dict(heads=heads, src_tp=2, dst_tp=2, dst_rank=1, block_table=w["block_table"],
              cu_seqlens=w["cu_seqlens"], seq_lens=lens)
    oracle.kv_ingest_stage(w["src_k"], w["src_v"], dk, dv, src_layer0=1, dst_layer0=3, count=2, **kw)
    assert (dk[:3] == 0xDEAD).all() and (dv[:3] == 0xDEAD).all()
    ref = numpy_ingest(w["src_k"], heads, 2, 2, 1, P, ps, w["block_table"], w["cu_seqlens"], lens)
    assert np.array_equal(dk[3:5], ref[1:3])
    assert not np.array_equal(dk[3], dk[4])                              # layers not collapsed onto one
    # K and V not swapped
    refv = numpy_ingest(w["src_v"], heads, 2, 2, 1, P, ps, w["block_table"], w["cu_seqlens"], lens)
    assert np.array_equal(dv[3:5], refv[1:3]) and not np.array_equal(dk[3:5], dv[3:5])
    for bad in (dict(src_layer0=2, dst_layer0=0, count=2), dict(src_layer0=0, dst_layer0=4, count=2),
                dict(src_layer0=-1, dst_layer0=0, count=1)):
        with pytest.raises(ValueError):
            oracle.kv_ingest_stage(w["src_k"], w["src_v"], dk, dv, **bad, **kw)
    # count = 0 is a no-op
    before = dk.copy()
    oracle.kv_ingest_stage(w["src_k"], w["src_v"], dk, dv, src_layer0=0, dst_layer0=0, count=0, **kw)
    assert np.array_equal(dk, before)


def test_stage_ingest_whole_range_equals_plain_ingest():
    w, heads, D, ps, lens = _stage_case(4, 2, L=2)
    P = w["num_pages"]
    a_k = np.full((2, P, 4, ps, D), 0xDEAD, dtype=np.uint16); a_v = np.full_like(a_k, 0xDEAD)
    b_k = a_k.copy(); b_v = a_v.copy()
    kw = dict(heads=heads, src_tp=4, dst_tp=2, dst_rank=0, block_table=w["block_table"],
              cu_seqlens=w["cu_seqlens"], seq_lens=lens)
    oracle.kv_ingest(w["src_k"], w["src_v"], a_k, a_v, **kw)
    oracle.kv_ingest_stage(w["src_k"], w["src_v"], b_k, b_v, src_layer0=0, dst_layer0=0, count=2, **kw)
    assert np.array_equal(a_k, b_k) and np.array_equal(a_v, b_v)


# ---------------------------------------------------------------- F1: append
def _append_case(seed=5, ps=4, Hkv=2, D=8, layers=3):
    lens = np.array([1, 4, 5, 8, 9, 0, 13], dtype=np.int32)           # page starts, page ends, empty
    q, k, v, bt, lens = small_case(seed, len(lens), Hkv * 2, Hkv, D, lens, ps, layers=layers)
    g = np.random.default_rng(seed + 1)
    k_new = g.integers(0, 65536, size=(len(lens), Hkv, D), dtype=np.uint16)
    v_new = g.integers(0, 65536, size=(len(lens), Hkv, D), dtype=np.uint16)
    return q, k.view(np.uint16).copy(), v.view(np.uint16).copy(), bt, lens, k_new, v_new


def test_append_writes_exactly_the_last_token_slot():
    """Independent numpy restatement (one token per step joins the cache): slot
    (n-1) mod ps of page bt[i][(n-1) div ps], every kv head, layer `layer` only; B*Hkv*D elements
    of each tensor change at most (exactly, counted by position), nothing when n = 0."""
    q, k, v, bt, lens, k_new, v_new = _append_case()
    layer, ps = 1, k.shape[3]
    k1, v1 = k.copy(), v.copy()
    oracle.kv_append(k_new, v_new, k1, v1, layer=layer, block_table=bt, seq_lens=lens)
    ek, ev = k.copy(), v.copy()
    for i, n in enumerate(lens):
        if n > 0:
            ek[layer, bt[i, (n - 1) // ps], :, (n - 1) % ps, :] = k_new[i]
            ev[layer, bt[i, (n - 1) // ps], :, (n - 1) % ps, :] = v_new[i]
    assert np.array_equal(k1, ek) and np.array_equal(v1, ev)
    # positions: run on two differently filled caches
    ka, kb = np.zeros_like(k), np.full_like(k, 0xFFFF)
    va, vb = np.zeros_like(v), np.full_like(v, 0xFFFF)
    oracle.kv_append(k_new, v_new, ka, va, layer=layer, block_table=bt, seq_lens=lens)
    oracle.kv_append(k_new, v_new, kb, vb, layer=layer, block_table=bt, seq_lens=lens)
    changed = (ka != 0) | (kb != 0xFFFF)
    assert int(changed.sum()) == int((lens > 0).sum()) * k.shape[2] * k.shape[4]
    assert not changed[0].any() and not changed[2].any()
    assert not np.array_equal(k1, v1)
    with pytest.raises(ValueError):
        oracle.kv_append(k_new, v_new, k1, v1, layer=3, block_table=bt, seq_lens=lens)


@pytest.mark.parametrize("S,R", [(1, 1), (2, 1), (4, 2)])
def test_ingest_of_n_minus_1_tokens_then_append_equals_ingest_of_n_tokens(S, R):
    """Consistency with the pinned ingest: the cache after prefill handed over n tokens equals the
    cache after it handed over n-1 and the decode step appended token n-1."""
    heads, D, ps, L = 4, 8, 4, 2
    lens = np.array([1, 4, 5, 8, 12], dtype=np.int32)
    c = W.IngestConfig(93, "t", L, heads, D, S, R, len(lens), "x")
    w = W.make_ingest_inputs(c, lens=lens, bits=True, page_size=ps)
    P, hd, cu = w["num_pages"], heads // R, w["cu_seqlens"]
    full = [np.concatenate(w[s], axis=2) for s in ("src_k", "src_v")]            # [L][T][heads][D]
    # the same prompts with their last token dropped
    keep = np.concatenate([np.arange(cu[i], cu[i + 1] - 1) for i in range(len(lens))]).astype(np.int64)
    lens_m = lens - 1
    cu_m = np.zeros(len(lens) + 1, dtype=np.int32); np.cumsum(lens_m, out=cu_m[1:])
    hs = heads // S
    sk_m = [np.ascontiguousarray(full[0][:, keep, r * hs:(r + 1) * hs]) for r in range(S)]
    sv_m = [np.ascontiguousarray(full[1][:, keep, r * hs:(r + 1) * hs]) for r in range(S)]
    for qrank in range(R):
        kw = dict(heads=heads, src_tp=S, dst_tp=R, dst_rank=qrank, block_table=w["block_table"])
        a_k = np.full((L, P, hd, ps, D), 0xDEAD, dtype=np.uint16); a_v = np.full_like(a_k, 0xDEAD)
        oracle.kv_ingest(w["src_k"], w["src_v"], a_k, a_v, cu_seqlens=cu, seq_lens=lens, **kw)
        b_k = np.full_like(a_k, 0xDEAD); b_v = np.full_like(a_k, 0xDEAD)
        oracle.kv_ingest(sk_m, sv_m, b_k, b_v, cu_seqlens=cu_m, seq_lens=lens_m, **kw)
        last = cu[1:] - 1
        for l in range(L):
            kn = np.ascontiguousarray(full[0][l, last, qrank * hd:(qrank + 1) * hd])
            vn = np.ascontiguousarray(full[1][l, last, qrank * hd:(qrank + 1) * hd])
            oracle.kv_append(kn, vn, b_k, b_v, layer=l, block_table=w["block_table"], seq_lens=lens)
        assert np.array_equal(a_k, b_k) and np.array_equal(a_v, b_v)


def test_attention_after_append_equals_dense_softmax_over_old_plus_new():
    q, k, v, bt, lens, _, _ = _append_case(seed=9, D=16)
    g = np.random.default_rng(77)
    Hkv, D, ps = k.shape[2], k.shape[4], k.shape[3]
    k_new = g.standard_normal((len(lens), Hkv, D)).astype(np.float16)
    v_new = g.standard_normal((len(lens), Hkv, D)).astype(np.float16)
    oracle.kv_append(k_new, v_new, k, v, layer=2, block_table=bt, seq_lens=lens)
    got = oracle.decode_attention(q, k.view(np.float16), v.view(np.float16), bt, lens, layer=2)
    # dense: the first n-1 cached tokens, then the new one, never reading the paged slot of token n-1
    scale = float(np.float32(1.0) / np.sqrt(np.float32(D)))
    kf, vf = k.view(np.float16), v.view(np.float16)
    for i, n in enumerate(lens):
        for h in range(q.shape[1]):
            gk = h // (q.shape[1] // Hkv)
            if n == 0:
                assert (got[i, h] == 0).all()
                continue
            t = np.arange(n - 1)
            Kd = np.concatenate([kf[2, bt[i, t // ps], gk, t % ps], k_new[i, gk][None]]).astype(np.float64)
            Vd = np.concatenate([vf[2, bt[i, t // ps], gk, t % ps], v_new[i, gk][None]]).astype(np.float64)
            np.testing.assert_allclose(got[i, h], softmax(Kd @ q[i, h].astype(np.float64) * scale) @ Vd, atol=1e-12)
    # and the generic dense pin still holds on the updated cache
    np.testing.assert_allclose(got, dense_reference(q, kf, vf, bt, lens, layer=2), atol=1e-12)


# ---------------------------------------------------------------- F4: causal paged prefill attention
def _prefill_case(seed, Hq, Hkv, D, lens, qlens, ps=4):
    lens = np.asarray(lens, dtype=np.int32)
    _, k, v, bt, lens = small_case(seed, len(lens), Hq, Hkv, D, lens, ps)
    qlens = np.asarray(qlens, dtype=np.int32)
    q = np.random.default_rng(seed + 100).standard_normal((int(qlens.sum()), Hq, D)).astype(np.float16)
    return q, k, v, bt, lens, qlens


def dense_causal(q, k, v, bt, lens, qlens):
    """Brute force with numpy/scipy only: gather the request's K/V densely, mask by position."""
    Tq, Hq, D = q.shape
    _, P, Hkv, ps, _ = k.shape
    G = Hq // Hkv
    scale = float(np.float32(1.0) / np.sqrt(np.float32(D)))
    out = np.zeros((Tq, Hq, D))
    row = 0
    for i, (n, m) in enumerate(zip(lens, qlens)):
        t = np.arange(n)
        Kd = k[0, bt[i, t // ps], :, t % ps].astype(np.float64)        # [n][Hkv][D]
        Vd = v[0, bt[i, t // ps], :, t % ps].astype(np.float64)
        for r in range(m):
            p = n - m + r
            for h in range(Hq):
                s = Kd[:p + 1, h // G] @ q[row, h].astype(np.float64) * scale
                out[row, h] = softmax(s) @ Vd[:p + 1, h // G]
            row += 1
    return out


@pytest.mark.parametrize("Hq,Hkv,D,lens,qlens", [
    (2, 2, 8, [5, 1, 9], [5, 1, 9]),            # whole-prompt prefill, MHA
    (4, 2, 16, [7, 12, 4], [3, 12, 0]),         # chunked / empty
    (8, 1, 8, [16, 17], [16, 2]),               # GQA, page boundaries
])
def test_prefill_equals_bruteforce_causal_dense(Hq, Hkv, D, lens, qlens):
    q, k, v, bt, lens, qlens = _prefill_case(21, Hq, Hkv, D, lens, qlens)
    got = oracle.prefill_attention(q, k, v, bt, lens, qlens)
    np.testing.assert_allclose(got, dense_causal(q, k, v, bt, lens, qlens), atol=1e-12)


def test_prefill_with_one_query_token_is_decode_attention():
    q, k, v, bt, lens, qlens = _prefill_case(22, 4, 2, 16, [1, 6, 13, 8], [1, 1, 1, 1])
    a = oracle.prefill_attention(q, k, v, bt, lens, qlens)
    b = oracle.decode_attention(q, k, v, bt, lens)              # q is [B][Hq][D] when every m_i = 1
    np.testing.assert_allclose(a, b, atol=1e-13)


def test_prefill_first_token_returns_v0_and_future_tokens_never_matter():
    q, k, v, bt, lens, qlens = _prefill_case(23, 2, 1, 8, [11, 6], [11, 6])
    base = oracle.prefill_attention(q, k, v, bt, lens, qlens)
    ps = k.shape[3]
    cu = np.concatenate([[0], np.cumsum(qlens)])
    for i in range(2):                                                    # position 0 sees only token 0
        v0 = v[0, bt[i, 0], 0, 0].astype(np.float64)
        np.testing.assert_array_equal(base[cu[i], 0], v0)
        np.testing.assert_array_equal(base[cu[i], 1], v0)
    # poison everything after position 4 of request 0: rows 0..4 must not change, later rows must
    k2, v2 = k.copy(), v.copy()
    for t in range(5, 11):
        k2[0, bt[0, t // ps], :, t % ps] = np.float16(3.0)
        v2[0, bt[0, t // ps], :, t % ps] = np.float16(-7.0)
    got = oracle.prefill_attention(q, k2, v2, bt, lens, qlens)
    np.testing.assert_array_equal(got[:5], base[:5])
    assert np.abs(got[5:11] - base[5:11]).max() > 1e-3
    np.testing.assert_array_equal(got[11:], base[11:])


def test_chunked_prefill_equals_tail_rows_of_whole_prefill_and_constant_v():
    q, k, v, bt, lens, qlens = _prefill_case(24, 4, 4, 8, [9, 14], [9, 14])
    whole = oracle.prefill_attention(q, k, v, bt, lens, qlens)
    ql2 = np.array([4, 5], dtype=np.int32)
    q2 = np.concatenate([q[5:9], q[9 + 9:9 + 14]])
    part = oracle.prefill_attention(q2, k, v, bt, lens, ql2)
    np.testing.assert_array_equal(part, np.concatenate([whole[5:9], whole[18:23]]))
    vc = np.broadcast_to(np.linspace(-1, 1, 8).astype(np.float16), v.shape).copy()
    np.testing.assert_allclose(oracle.prefill_attention(q, k, vc, bt, lens, qlens),
                               np.broadcast_to(vc[0, 0, 0, 0].astype(np.float64), whole.shape), atol=1e-14)
    with pytest.raises(ValueError):
        oracle.prefill_attention(q2, k, v, bt, lens, np.array([10, -1], dtype=np.int32))
