"""Pins for the oracle (oracle/hxo.c) against things other than itself: brute-force dense
numpy/scipy float64, closed forms, invariants, special cases (SURVEY.md §8(c) "pins").
CPU only.  A plausible mistake anywhere in the oracle (dropped term, wrong index, transposed
operand, wrong head map) fails at least one of these."""
import os

import numpy as np
import pytest
from scipy.special import softmax

import oracle
import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))


# ---------------------------------------------------------------- helpers (test-side only)
def dense_reference(q, k, v, bt, lens, layer=0, scale=None):
    """Brute force: gather each request's pages into dense [n][Hkv][D] float64 with numpy
    fancy indexing, then scipy softmax(q K^T * scale) V per head.  Independent of hxo.c."""
    B, Hq, D = q.shape
    _, P, Hkv, ps, _ = k.shape
    G = Hq // Hkv
    scale = float(np.float32(1.0) / np.sqrt(np.float32(D))) if scale is None else scale
    out = np.zeros((B, Hq, D))
    for i in range(B):
        n = int(lens[i])
        if n == 0:
            continue
        npg = (n + ps - 1) // ps
        pages = bt[i, :npg]
        Kd = k[layer][pages].astype(np.float64).transpose(0, 2, 1, 3).reshape(npg * ps, Hkv, D)[:n]
        Vd = v[layer][pages].astype(np.float64).transpose(0, 2, 1, 3).reshape(npg * ps, Hkv, D)[:n]
        for h in range(Hq):
            s = Kd[:, h // G, :] @ q[i, h].astype(np.float64) * scale
            out[i, h] = softmax(s) @ Vd[:, h // G, :]
    return out


def small_case(seed, B, Hq, Hkv, D, lens, ps, layers=1, spare=1.5):
    g = np.random.default_rng(seed)
    lens = np.asarray(lens, dtype=np.int32)
    need = int(((lens + ps - 1) // ps).sum())
    P = max(1, int(np.ceil(spare * need)) + 1)
    stride = max(1, int(((lens + ps - 1) // ps).max(initial=1)))
    bt = W.place_pages(lens, P, stride, g, ps)
    q = g.standard_normal((B, Hq, D)).astype(np.float16)
    k = g.standard_normal((layers, P, Hkv, ps, D)).astype(np.float16)
    v = g.standard_normal((layers, P, Hkv, ps, D)).astype(np.float16)
    return q, k, v, bt, lens


# ---------------------------------------------------------------- fp16 decode
def test_half_decode_all_patterns_vs_numpy():
    bits = np.arange(65536, dtype=np.uint16)
    got = oracle.half_to_double(bits)
    want = bits.view(np.float16).astype(np.float64)
    nan = np.isnan(want)
    assert np.array_equal(np.isnan(got), nan)
    assert np.array_equal(got[~nan], want[~nan])
    assert np.array_equal(np.signbit(got[~nan]), np.signbit(want[~nan]))  # -0 kept


# ---------------------------------------------------------------- attention: brute force
@pytest.mark.parametrize("B,Hq,Hkv,D,ps,lens", [
    (4, 4, 4, 64, 16, [17, 64, 100, 255]),          # BASELINE.json configs[0] shape
    (3, 4, 2, 8, 4, [1, 5, 70]),
    (2, 8, 1, 64, 16, [33, 16]),
    (4, 2, 2, 8, 4, [4, 3, 9, 1]),
    (1, 16, 2, 128, 16, [257]),
    (2, 3, 3, 16, 8, [15, 17]),
])
def test_paged_equals_dense_bruteforce(B, Hq, Hkv, D, ps, lens):
    q, k, v, bt, lens = small_case(1, B, Hq, Hkv, D, lens, ps, layers=2)
    for layer in (0, 1):
        got = oracle.decode_attention(q, k, v, bt, lens, layer=layer)
        want = dense_reference(q, k, v, bt, lens, layer=layer)
        np.testing.assert_allclose(got, want, rtol=0, atol=1e-12)


def test_fuzz_small_shapes():
    hyp = pytest.importorskip("hypothesis")
    from hypothesis import given, settings, strategies as st

    @settings(max_examples=40, deadline=None)
    @given(st.integers(0, 2**31), st.integers(1, 4), st.sampled_from([(1, 1), (2, 1), (4, 2), (4, 4), (3, 3)]),
           st.sampled_from([8, 64]), st.sampled_from([4, 16]), st.data())
    def run(seed, B, heads, D, ps, data):
        Hq, Hkv = heads
        lens = [data.draw(st.integers(1, 70)) for _ in range(B)]
        q, k, v, bt, lens = small_case(seed, B, Hq, Hkv, D, lens, ps)
        got = oracle.decode_attention(q, k, v, bt, lens)
        np.testing.assert_allclose(got, dense_reference(q, k, v, bt, lens), rtol=0, atol=1e-12)

    run()


def test_custom_scale_is_used():
    q, k, v, bt, lens = small_case(2, 2, 2, 2, 8, [9, 30], 4)
    got = oracle.decode_attention(q, k, v, bt, lens, sm_scale=0.37)
    want = dense_reference(q, k, v, bt, lens, scale=float(np.float32(0.37)))
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-12)
    assert np.abs(got - oracle.decode_attention(q, k, v, bt, lens)).max() > 1e-3


# ---------------------------------------------------------------- attention: closed forms
def test_constant_v_returns_v():
    q, k, v, bt, lens = small_case(3, 3, 4, 2, 64, [17, 64, 100], 16)
    vec = np.random.default_rng(0).standard_normal((2, 64)).astype(np.float16)
    v[:] = vec[None, None, :, None, :]
    got = oracle.decode_attention(q, k, v, bt, lens)
    want = np.repeat(vec.astype(np.float64), 2, axis=0)[None].repeat(3, 0)
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-13)


def test_single_token_returns_its_v_exactly():
    q, k, v, bt, lens = small_case(4, 3, 4, 2, 64, [1, 1, 1], 16)
    got = oracle.decode_attention(q, k, v, bt, lens)
    for i in range(3):
        for h in range(4):
            assert np.array_equal(got[i, h], v[0, bt[i, 0], h // 2, 0].astype(np.float64))


def test_zero_q_gives_mean_of_v():
    q, k, v, bt, lens = small_case(5, 2, 2, 2, 8, [23, 64], 4)
    q[:] = 0
    got = oracle.decode_attention(q, k, v, bt, lens)
    for i, n in enumerate(lens):
        pages = bt[i, :(n + 3) // 4]
        Vd = v[0][pages].astype(np.float64).transpose(0, 2, 1, 3).reshape(-1, 2, 8)[:n]
        np.testing.assert_allclose(got[i], Vd.mean(axis=0), rtol=0, atol=1e-13)


def test_empty_context_gives_zeros():
    q, k, v, bt, lens = small_case(6, 3, 2, 2, 8, [0, 5, 0], 4)
    got = oracle.decode_attention(q, k, v, bt, lens)
    assert np.array_equal(got[0], np.zeros((2, 8))) and np.array_equal(got[2], np.zeros((2, 8)))
    np.testing.assert_allclose(got, dense_reference(q, k, v, bt, lens), atol=1e-12)


def test_dominant_token_and_large_logits_stable():
    q, k, v, bt, lens = small_case(7, 2, 4, 4, 64, [100, 255], 16)
    q8 = (q.astype(np.float32) * 8).astype(np.float16)      # logit std ~ 8: near one-hot
    got = oracle.decode_attention(q8, k, v, bt, lens)
    assert np.isfinite(got).all()
    np.testing.assert_allclose(got, dense_reference(q8, k, v, bt, lens), rtol=0, atol=1e-12)
    # one dominant token: k_t = 30*q/|q|^2-ish -> output ~ v_t
    i, h, t = 1, 2, 77
    qq = q[i, h].astype(np.float64)
    k[0, bt[i, t // 16], h, t % 16] = (qq / (qq @ qq) * 8 * 60).astype(np.float16)  # score ~ 60
    got = oracle.decode_attention(q, k, v, bt, lens)
    np.testing.assert_allclose(got[i, h], v[0, bt[i, t // 16], h, t % 16].astype(np.float64), atol=1e-6)


# ---------------------------------------------------------------- attention: invariants
def test_page_permutation_invariance_bit_identical():
    q, k, v, bt, lens = small_case(8, 4, 4, 4, 64, [17, 64, 100, 255], 16)
    base = oracle.decode_attention(q, k, v, bt, lens)
    P = k.shape[1]
    perm = np.random.default_rng(9).permutation(P)          # new physical id of old page p
    k2, v2 = np.empty_like(k), np.empty_like(v)
    k2[:, perm], v2[:, perm] = k, v
    bt2 = np.where(bt >= 0, perm[np.clip(bt, 0, None)], -1).astype(np.int32)
    assert np.array_equal(base, oracle.decode_attention(q, k2, v2, bt2, lens))


def test_gqa_equals_mha_with_repeated_kv_heads():
    q, k, v, bt, lens = small_case(10, 3, 8, 2, 64, [17, 40, 100], 16)
    got = oracle.decode_attention(q, k, v, bt, lens)
    k_rep, v_rep = np.repeat(k, 4, axis=2), np.repeat(v, 4, axis=2)
    want = oracle.decode_attention(q, np.ascontiguousarray(k_rep), np.ascontiguousarray(v_rep), bt, lens)
    assert np.array_equal(got, want)
    np.testing.assert_allclose(got, dense_reference(q, k, v, bt, lens), atol=1e-12)


def test_split_merge_identity_random_splits():
    q, k, v, bt, lens = small_case(11, 2, 4, 2, 64, [100, 255], 16)
    full = oracle.decode_attention(q, k, v, bt, lens)
    scale = float(np.float32(1.0) / np.sqrt(np.float32(64)))
    g = np.random.default_rng(12)
    for i in range(2):
        for h in range(4):
            n = int(lens[i])
            cuts = np.sort(g.choice(np.arange(1, n), size=int(g.integers(1, 6)), replace=False))
            edges = [0, *cuts.tolist(), n]
            parts = [oracle.partial_attention(q[i, h], k, v, bt[i], h // 2, a, b, scale=scale)
                     for a, b in zip(edges[:-1], edges[1:])]
            np.testing.assert_allclose(oracle.merge_partials(parts), full[i, h], rtol=0, atol=1e-13)


def test_nan_poison_in_tail_slots_and_unowned_pages_is_harmless():
    q, k, v, bt, lens = small_case(13, 4, 4, 4, 64, [17, 64, 100, 255], 16)
    base = oracle.decode_attention(q, k, v, bt, lens)
    owned = np.zeros((k.shape[1], 16), dtype=bool)
    for i, n in enumerate(lens):
        for t in range(n):
            owned[bt[i, t // 16], t % 16] = True
    kb, vb = k.view(np.uint16).copy(), v.view(np.uint16).copy()
    mask = ~owned
    kb[0].transpose(0, 2, 1, 3)[mask] = 0x7E01
    vb[0].transpose(0, 2, 1, 3)[mask] = 0xFE55
    bt2 = bt.copy()
    got = oracle.decode_attention(q, kb.view(np.float16), vb.view(np.float16), bt2, lens)
    assert np.array_equal(got, base)


# ---------------------------------------------------------------- ingest
def numpy_ingest(src, heads, S, R, qrank, P, ps, bt, cu, lens):
    """Independent restatement via the logical view KV[l][i][t][h][d]: stitch the
    shards along heads, slice the rank's head range, then place token by token with numpy."""
    L, T, hs, D = src[0].shape
    full = np.concatenate(src, axis=2)                       # [L][T][heads][D], contiguous ranges (S4)
    hd = heads // R
    mine = full[:, :, qrank * hd:(qrank + 1) * hd, :]
    dst = np.full((L, P, hd, ps, D), 0xDEAD, dtype=np.uint16)
    for i, n in enumerate(lens):
        tok = cu[i] + np.arange(n)
        pages = bt[i, np.arange(n) // ps]
        slots = np.arange(n) % ps
        for j in range(hd):
            dst[:, pages, j, slots, :] = mine[:, tok, j, :]
    return dst


@pytest.mark.parametrize("S", [1, 2, 4, 8])
@pytest.mark.parametrize("R", [1, 2, 4, 8])
def test_ingest_matches_numpy_and_gather_roundtrips(S, R):
    heads, D, L, ps = 8, 16, 2, 4
    lens = np.array([1, 4, 5, 13, 16], dtype=np.int32)
    c = W.IngestConfig(90, "t", L, heads, D, S, R, len(lens), "x")
    w = W.make_ingest_inputs(c, lens=lens, bits=True, page_size=ps, seed_extra=S * 10 + R)
    P, hd, T = w["num_pages"], heads // R, w["total_tokens"]
    total_changed = 0
    rebuilt_k = [np.full_like(a, 0xBEEF) for a in w["src_k"]]
    rebuilt_v = [np.full_like(a, 0xBEEF) for a in w["src_v"]]
    for qrank in range(R):
        dk = np.full((L, P, hd, ps, D), 0xDEAD, dtype=np.uint16)
        dv = np.full((L, P, hd, ps, D), 0xDEAD, dtype=np.uint16)
        kw = dict(heads=heads, src_tp=S, dst_tp=R, dst_rank=qrank, block_table=w["block_table"],
                  cu_seqlens=w["cu_seqlens"], seq_lens=lens)
        oracle.kv_ingest(w["src_k"], w["src_v"], dk, dv, **kw)
        assert np.array_equal(dk, numpy_ingest(w["src_k"], heads, S, R, qrank, P, ps, w["block_table"], w["cu_seqlens"], lens))
        assert np.array_equal(dv, numpy_ingest(w["src_v"], heads, S, R, qrank, P, ps, w["block_table"], w["cu_seqlens"], lens))
        # sentinel count: everything not a valid slot is untouched (values are random 16-bit, so
        # count positions via a second run on a differently-filled destination)
        dk2 = np.full_like(dk, 0x1234)
        dv2 = np.full_like(dv, 0x1234)
        oracle.kv_ingest(w["src_k"], w["src_v"], dk2, dv2, **kw)
        changed = (dk != 0xDEAD) | (dk2 != 0x1234)
        total_changed += int(changed.sum())
        assert np.array_equal(dk[~changed], np.full(int((~changed).sum()), 0xDEAD, dtype=np.uint16))
        oracle.kv_gather(rebuilt_k, rebuilt_v, dk, dv, **kw)
    # every (layer, token, head, d) landed exactly once across ranks: L*T*heads*D for K
    assert total_changed == L * T * heads * D
    for r in range(S):
        assert np.array_equal(rebuilt_k[r], w["src_k"][r]) and np.array_equal(rebuilt_v[r], w["src_v"][r])


def test_ingest_multiset_preserved_and_k_v_not_swapped():
    c = W.CONFIGS["tiny_ingest"]
    w = W.make_ingest_inputs(c, bits=True)
    P = w["num_pages"]
    dk = np.zeros((1, P, 4, 16, 64), dtype=np.uint16)
    dv = np.zeros_like(dk)
    oracle.kv_ingest(w["src_k"], w["src_v"], dk, dv, heads=4, src_tp=2, dst_tp=1, dst_rank=0,
                     block_table=w["block_table"], cu_seqlens=w["cu_seqlens"], seq_lens=w["seq_lens"])
    mix = lambda a: int((a.astype(np.uint64) * np.uint64(0x9E3779B97F4A7C15) >> np.uint64(7)).sum(dtype=np.uint64))
    valid = np.zeros((P, 16), dtype=bool)
    for i, n in enumerate(w["seq_lens"]):
        for t in range(n):
            valid[w["block_table"][i, t // 16], t % 16] = True
    assert mix(np.concatenate([a.ravel() for a in w["src_k"]])) == mix(dk[0].transpose(0, 2, 1, 3)[valid])
    assert mix(np.concatenate([a.ravel() for a in w["src_v"]])) == mix(dv[0].transpose(0, 2, 1, 3)[valid])
    assert not np.array_equal(dk, dv)
    assert (dk[0].transpose(0, 2, 1, 3)[~valid] == 0).all()


def test_pure_paging_special_case_S1_R1():
    """S = R = 1: no regroup; a page tile is just 16 consecutive source rows, head-major."""
    c = W.IngestConfig(91, "t", 1, 2, 8, 1, 1, 2, "x")
    lens = np.array([16, 32], dtype=np.int32)
    w = W.make_ingest_inputs(c, lens=lens, bits=True)
    P = w["num_pages"]
    dk = np.zeros((1, P, 2, 16, 8), dtype=np.uint16)
    dv = np.zeros_like(dk)
    oracle.kv_ingest(w["src_k"], w["src_v"], dk, dv, heads=2, src_tp=1, dst_tp=1, dst_rank=0,
                     block_table=w["block_table"], cu_seqlens=w["cu_seqlens"], seq_lens=lens)
    src = w["src_k"][0][0]                                   # [T][2][8]
    assert np.array_equal(dk[0, w["block_table"][1, 1]], src[32:48].transpose(1, 0, 2))
    assert np.array_equal(dk[0, w["block_table"][0, 0]], src[0:16].transpose(1, 0, 2))


def test_ingest_then_attention_equals_dense_on_logical_kv():
    """End to end on the tiny config: shards -> paged cache (oracle ingest) -> oracle attention
    == dense softmax on the logical KV stitched from the shards."""
    c = W.CONFIGS["tiny_ingest"]
    w = W.make_ingest_inputs(c)
    P, lens, cu = w["num_pages"], w["seq_lens"], w["cu_seqlens"]
    dk = np.zeros((1, P, 4, 16, 64), dtype=np.uint16)
    dv = np.zeros_like(dk)
    oracle.kv_ingest(w["src_k"], w["src_v"], dk, dv, heads=4, src_tp=2, dst_tp=1, dst_rank=0,
                     block_table=w["block_table"], cu_seqlens=cu, seq_lens=lens)
    q = W.draw_fp16_normal((4, 4, 64), 1, W.configs.S_Q)
    got = oracle.decode_attention(q, dk.view(np.float16), dv.view(np.float16), w["block_table"], lens)
    Kl = np.concatenate(w["src_k"], axis=2).view(np.float16)[0].astype(np.float64)   # [T][4][64]
    Vl = np.concatenate(w["src_v"], axis=2).view(np.float16)[0].astype(np.float64)
    for i in range(4):
        for h in range(4):
            s = Kl[cu[i]:cu[i + 1], h] @ q[i, h].astype(np.float64) * 0.125
            np.testing.assert_allclose(got[i, h], softmax(s) @ Vl[cu[i]:cu[i + 1], h], atol=1e-12)


# ---------------------------------------------------------------- sizes (paper Table 1)
def test_kv_byte_counts_match_paper_table1():
    rows = {}
    for line in open(os.path.join(HERE, "golden", "table1_kv_bytes.txt")):
        if line.strip() and not line.startswith("#"):
            name, hidden, layers, per_layer, per_tok = line.split()
            rows[name] = tuple(map(int, (hidden, layers, per_layer, per_tok)))
    B_type = 2
    for name, (hidden, layers, per_layer, per_tok) in rows.items():
        assert 2 * hidden * B_type == per_layer and per_layer * layers == per_tok
    assert rows["opt30b"][3] == 48 * 56 * 128 * 2 * 2
    assert rows["llama70b_gqa"][3] == 80 * 8 * 128 * 2 * 2
    assert rows["llama70b_mha"][2] == 8 * rows["llama70b_gqa"][2]          # reading S16
    # workload byte accounting uses the same count
    a = W.make_attention_inputs(W.CONFIGS["tiny"])
    assert a["kv_bytes"] == 436 * 4 * 64 * 2 * 2


def test_workload_recipes_are_seeded_and_shaped():
    for name in ("opt30b_tp4", "llama70b_tp2", "llama70b_tp1"):
        c = W.CONFIGS[name]
        n1, n2 = W.attn_lengths(c), W.attn_lengths(c)
        assert np.array_equal(n1, n2) and len(n1) == c.batch
    n = W.attn_lengths(W.CONFIGS["opt30b_tp4"]); assert n.min() >= 512 and n.max() <= 2048
    n = W.attn_lengths(W.CONFIGS["llama70b_tp2"]); assert n.min() >= 64 and n.max() <= 4096
    n = W.attn_lengths(W.CONFIGS["llama70b_tp1"])
    assert ((n >= 128) & (n <= 1024)).sum() == 179 and ((n >= 4096) & (n <= 8192)).sum() == 77
    n = W.ingest_lengths(W.CONFIGS["llama70b_ingest"]); assert len(n) == 32 and n.min() >= 256 and n.max() <= 4096
