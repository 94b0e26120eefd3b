"""Seeded random shapes through the three kernels that carry the most scheduling logic — the decode attention's
work partition (unplanned, planned, chained), the fused decode step (attention + tile mover) and the persistent prefill
kernel — each against the oracle.  The shapes are drawn, not hand-picked: group sizes, head counts, both head sizes,
batches from 1 to a few hundred, contexts from 0 to a few thousand tokens, TP pairs, layers, chunked prefills."""
import numpy as np
import pytest

import workloads as W
from helpers import MAX_ABS_TOL, REL_L2_TOL, attn_errors, dev_u16, to_dev

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (no CPU fallback exists)")
    import paper_2502_07903_b200 as hx
    import oracle
    oracle.build()
    return hx, torch, oracle


def _draw_lens(g, B, hi):
    kind = g.integers(0, 4)
    if kind == 0:
        lens = g.integers(0, hi, size=B)
    elif kind == 1:                                            # heavy tail: a few long contexts among short ones
        lens = np.where(g.random(B) < 0.15, g.integers(hi // 2, hi, size=B), g.integers(0, max(2, hi // 16), size=B))
    elif kind == 2:                                            # page / tile boundaries
        lens = g.choice([0, 1, 15, 16, 17, 127, 128, 129, 255, 256, 257], size=B)
    else:
        lens = np.full(B, g.integers(1, hi))
    return lens.astype(np.int32)


@pytest.mark.parametrize("seed", range(10))
def test_fuzz_decode_attention_unplanned_planned_chained(env, seed):
    hx, torch, oracle = env
    g = W.rng(95, seed)
    G = int(g.choice([1, 2, 4, 8, 16])); Hkv = int(g.integers(1, 9)); D = int(g.choice([64, 128]))
    B = int(g.choice([1, 3, 17, 64, 200])); hi = int(g.choice([40, 600, 3000]))
    L = 2
    lens = _draw_lens(g, B, hi)
    c = W.AttnConfig(95, "fuzz", B, G * Hkv, Hkv, D, (hi + 15) // 16 + 1, "x")
    w = W.make_attention_inputs(c, lens=lens, layers=L, seed_extra=seed)
    cache = hx.PagedCache(to_dev(w["k"], torch), to_dev(w["v"], torch))
    bt, sl = torch.from_numpy(w["block_table"]).cuda(), torch.from_numpy(lens).cuda()
    mx = int(lens.max(initial=0))
    qd = to_dev(w["q"], torch)
    wsb = hx.decode_attention_workspace_bytes(B, G * Hkv, Hkv, D, mx)
    ws = torch.zeros(max(wsb, 16), dtype=torch.uint8, device="cuda")
    plan = torch.empty(max(hx.decode_plan_bytes(B, Hkv, mx), 16), dtype=torch.uint8, device="cuda")
    hx.decode_plan(plan, cache, q_heads=G * Hkv, block_table=bt, block_table_stride=bt.shape[1], seq_lens=sl, batch=B, max_seq_len=mx)
    for layer in range(L):
        ref = oracle.decode_attention(w["q"], w["k"], w["v"], w["block_table"], lens, layer=layer)
        outs = [torch.full_like(qd, float("nan")) for _ in range(4)]
        hx.decode_attention(outs[0], qd, cache, layer=layer, q_heads=G * Hkv, block_table=bt, block_table_stride=bt.shape[1],
                            seq_lens=sl, batch=B, max_seq_len=mx, workspace=ws, workspace_bytes=wsb)
        kw = dict(layer=layer, q_heads=G * Hkv, plan=plan, batch=B, max_seq_len=mx, workspace=ws, workspace_bytes=wsb)
        hx.decode_attention_planned(outs[1], qd, cache, **kw)
        hx.decode_attention_chained(outs[2], qd, cache, inputs_ready=1, **kw)
        hx.decode_attention_chained(outs[3], qd, cache, inputs_ready=0, **kw)
        torch.cuda.synchronize()
        got = outs[0].cpu().numpy()
        assert np.isfinite(got.astype(np.float32)).all(), (seed, G, Hkv, D, B, hi)
        max_abs, rel = attn_errors(got, ref)
        assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (seed, G, Hkv, D, B, hi, layer, max_abs, rel)
        for j in (1, 2, 3):                                   # same partition, same arithmetic: the same bits
            assert torch.equal(outs[j].view(torch.int16), outs[0].view(torch.int16)), (seed, j, layer)


@pytest.mark.parametrize("seed", range(8))
def test_fuzz_fused_decode_step(env, seed):
    hx, torch, oracle = env
    g = W.rng(96, seed)
    heads = int(g.choice([4, 8, 12, 16]))
    S = int(g.choice([s for s in (1, 2, 4, 8) if heads % s == 0])); R = int(g.choice([r for r in (1, 2, 4) if heads % r == 0]))
    q_rank = int(g.integers(0, R)); D = int(g.choice([64, 128])); layers = int(g.integers(1, 4))
    hd = heads // R
    G = int(g.choice([1, 2, 4]))
    ilens = _draw_lens(g, int(g.integers(1, 12)), int(g.choice([40, 700])))
    alens = np.maximum(_draw_lens(g, int(g.choice([1, 9, 60])), int(g.choice([100, 2500]))), 0)
    c = W.IngestConfig(96, "fuzz", layers, heads, D, S, R, len(ilens), "x")
    w = W.make_ingest_inputs(c, lens=ilens, bits=True, seed_extra=seed)
    P = w["num_pages"]
    apages = W.pages_for(alens)
    Pa = max(int(apages.sum()), 1)
    abt = np.full((len(alens), max(int(apages.max(initial=0)), 1)), -1, dtype=np.int32)
    perm = P + g.permutation(Pa).astype(np.int32)
    o = 0
    for i, n in enumerate(apages):
        abt[i, :n] = perm[o:o + n]
        o += n
    k0 = np.full((layers, P + Pa, hd, 16, D), 0xDEAD, dtype=np.uint16)
    v0 = np.full_like(k0, 0xDEAD)
    k0[:, P:] = W.draw_fp16_normal((layers, Pa, hd, 16, D), 96, 8, seed).view(np.uint16)
    v0[:, P:] = W.draw_fp16_normal((layers, Pa, hd, 16, D), 96, 9, seed).view(np.uint16)
    q = W.draw_fp16_normal((len(alens), hd * G, D), 96, 10, seed)
    layer_a = int(g.integers(0, layers))
    ref = oracle.decode_attention(q, k0.view(np.float16), v0.view(np.float16), abt, alens, layer=layer_a)
    ek, ev = k0.copy(), v0.copy()
    oracle.kv_ingest(w["src_k"], w["src_v"], ek, ev, heads=heads, src_tp=S, dst_tp=R, dst_rank=q_rank, block_table=w["block_table"],
                     cu_seqlens=w["cu_seqlens"], seq_lens=w["seq_lens"])
    cache = hx.PagedCache(to_dev(k0, torch), to_dev(v0, torch))
    qd = to_dev(q, torch)
    out = torch.full_like(qd, float("nan"))
    mx = int(alens.max(initial=0))
    wsb = hx.decode_attention_workspace_bytes(len(alens), hd * G, hd, D, mx)
    ws = torch.zeros(max(wsb, 16), dtype=torch.uint8, device="cuda")
    ibt = torch.from_numpy(w["block_table"]).cuda()
    hx.decode_step(out=out, q=qd, cache=cache, layer=layer_a, q_heads=hd * G, block_table=torch.from_numpy(abt).cuda(),
                   block_table_stride=abt.shape[1], seq_lens=torch.from_numpy(alens).cuda(), batch=len(alens), max_seq_len=mx,
                   sm_scale=0.0, workspace=ws, workspace_bytes=wsb, src_k=[to_dev(a, torch) for a in w["src_k"]],
                   src_v=[to_dev(a, torch) for a in w["src_v"]], ing_layers=layers, heads=heads, src_tp=S, dst_tp=R,
                   dst_rank=q_rank, ing_block_table=ibt, ing_block_table_stride=ibt.shape[1],
                   ing_cu_seqlens=torch.from_numpy(w["cu_seqlens"]).cuda(), ing_seq_lens=torch.from_numpy(w["seq_lens"]).cuda(),
                   ing_batch=len(ilens), ing_total_tokens=w["total_tokens"], ing_max_seq_len=int(ilens.max(initial=0)), overlap_ingest=1)
    torch.cuda.synchronize()
    tag = (seed, heads, S, R, q_rank, D, layers, G, list(ilens), len(alens))
    assert np.array_equal(dev_u16(cache.k), ek), tag
    assert np.array_equal(dev_u16(cache.v), ev), tag
    max_abs, rel = attn_errors(out.cpu().numpy(), ref)
    assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (tag, max_abs, rel)
    assert int(ws.view(torch.int32)[-4:].abs().sum()) == 0, tag


@pytest.mark.parametrize("seed", range(6))
def test_fuzz_prefill(env, seed):
    hx, torch, oracle = env
    g = W.rng(97, seed)
    G = int(g.choice([1, 2, 4, 8, 16])); Hkv = int(g.integers(1, 5)); D = int(g.choice([64, 128]))
    B = int(g.choice([1, 5, 20])); hi = int(g.choice([60, 500, 1200]))      # (the float64 oracle sets the size)
    lens = np.maximum(_draw_lens(g, B, hi), 1)
    mode = g.integers(0, 3)
    qlens = lens.copy() if mode == 0 else np.minimum(lens, g.integers(0, 300, size=B)).astype(np.int32) if mode == 1 else \
        np.where(g.random(B) < 0.5, lens, 1).astype(np.int32)
    c = W.AttnConfig(97, "fuzz", B, G * Hkv, Hkv, D, (hi + 15) // 16 + 1, "x")
    w = W.make_attention_inputs(c, lens=lens, seed_extra=seed)
    Tq = int(qlens.sum())
    if Tq == 0:
        qlens[0] = 1
        Tq = 1
    q = W.draw_fp16_normal((Tq, G * Hkv, D), 97, 40, seed)
    ref = oracle.prefill_attention(q, w["k"], w["v"], w["block_table"], lens, qlens)
    cache = hx.PagedCache(to_dev(w["k"], torch), to_dev(w["v"], torch))
    cu = np.zeros(B + 1, dtype=np.int32)
    np.cumsum(qlens, out=cu[1:])
    qd = to_dev(q, torch)
    out = torch.full_like(qd, float("nan"))
    bt = torch.from_numpy(w["block_table"]).cuda()
    hx.prefill_attention(out, qd, cache, layer=0, q_heads=G * Hkv, block_table=bt, block_table_stride=bt.shape[1],
                         seq_lens=torch.from_numpy(lens).cuda(), q_lens=torch.from_numpy(qlens).cuda(),
                         cu_q_lens=torch.from_numpy(cu).cuda(), batch=B, total_q_tokens=Tq, max_q_len=int(qlens.max()),
                         max_seq_len=int(lens.max()))
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert np.isfinite(got.astype(np.float32)).all(), (seed, G, Hkv, D, B, hi)
    max_abs, rel = attn_errors(got, ref)
    assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (seed, G, Hkv, D, B, hi, int(mode), max_abs, rel)
