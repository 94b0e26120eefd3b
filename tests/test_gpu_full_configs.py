"""Full-size BASELINE.json configs on the GPU, in the launch configuration bench.py times.
Attention: EVERY output row of configs[1], [2] and [4] against the float64 oracle, through hx_decode_attention and
through hx_decode_plan + hx_decode_attention_planned (bit-identical to each other); configs[4] also through
hx_decode_step with the step's handoff overlapped, as bench.py runs it.  Ingest: the whole 80-layer configs[3] call for both destination ranks,
layers 0 / 40 / 79 bit for bit against the oracle (element offsets past 2^31), every layer through the on-device
gather round trip, unowned pages intact."""
import numpy as np
import pytest

import workloads as W
from helpers import (MAX_ABS_TOL, REL_L2_TOL, attn_errors, dev_u16, oracle_ingest, run_gpu_attention, run_gpu_ingest,
                     to_dev)

pytestmark = [pytest.mark.gpu, pytest.mark.slow]


@pytest.fixture(scope="module")
def env():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (no CPU fallback exists)")
    import paper_2502_07903_b200 as hx
    import oracle
    oracle.build()
    return hx, torch, oracle


def _check_all_rows(name, got, ref, label):
    assert np.isfinite(got.astype(np.float32)).all(), (name, label)
    max_abs, rel_l2 = attn_errors(got, ref)
    assert max_abs <= MAX_ABS_TOL and rel_l2 <= REL_L2_TOL, (name, label, max_abs, rel_l2)
    worst = max(attn_errors(got[i], ref[i])[1] for i in range(len(got)))
    assert worst <= REL_L2_TOL, (name, label, worst)              # every single request too


@pytest.mark.parametrize("name", ["opt30b_tp4", "llama70b_tp2", "llama70b_tp1"])
def test_attention_full_config_every_row_unplanned_and_planned(env, name):
    hx, torch, oracle = env
    c = W.CONFIGS[name]
    w = W.make_attention_inputs(c)
    ref = oracle.decode_attention(w["q"], w["k"], w["v"], w["block_table"], w["seq_lens"])    # all B x Hq rows
    B, Hq, D = w["q"].shape
    cache = hx.PagedCache(to_dev(w["k"], torch), to_dev(w["v"], torch))
    qd = to_dev(w["q"], torch)
    bt = torch.from_numpy(w["block_table"]).cuda()
    sl = torch.from_numpy(w["seq_lens"]).cuda()
    mx = int(w["seq_lens"].max())
    wsb = hx.decode_attention_workspace_bytes(B, Hq, c.kv_heads, D, mx)
    ws = torch.zeros(wsb, dtype=torch.uint8, device="cuda")
    plan = torch.empty(hx.decode_plan_bytes(B, c.kv_heads, mx), dtype=torch.uint8, device="cuda")
    hx.decode_plan(plan, cache, q_heads=Hq, block_table=bt, block_table_stride=bt.shape[1], seq_lens=sl, batch=B, max_seq_len=mx)
    outs = {}
    for label in ("unplanned", "planned", "planned again", "unplanned again"):
        out = torch.full_like(qd, float("nan"))
        if label.startswith("planned"):
            hx.decode_attention_planned(out, qd, cache, layer=0, q_heads=Hq, plan=plan, batch=B, max_seq_len=mx, workspace=ws,
                                        workspace_bytes=wsb)
        else:
            hx.decode_attention(out, qd, cache, layer=0, q_heads=Hq, block_table=bt, block_table_stride=bt.shape[1],
                                seq_lens=sl, batch=B, max_seq_len=mx, workspace=ws, workspace_bytes=wsb)
        torch.cuda.synchronize()
        outs[label] = out.cpu().numpy()
        _check_all_rows(name, outs[label], ref, label)
    # same work partition, same arithmetic: the same bits with and without the plan, run to run
    for label in ("planned", "planned again", "unplanned again"):
        assert np.array_equal(outs[label].view(np.uint16), outs["unplanned"].view(np.uint16)), label


def test_config5_step_as_bench_runs_it(env):
    """configs[4] through hx_decode_step(overlap_ingest=1) — bench.py's timed call: the 16
    new 2048-token prompts land (prefill TP=4 -> decode TP=1) in pages the host allocator hands out while the
    attention runs over the 256-request batch.  Every output row and every page of the cache against the oracle."""
    hx, torch, oracle = env
    ca, ci = W.CONFIGS["llama70b_tp1"], W.CONFIGS["llama70b_tp1_ingest"]
    lens, ilens = W.attn_lengths(ca), W.ingest_lengths(ci)
    need, need_i = int(W.pages_for(lens).sum()), int(W.pages_for(ilens).sum())
    P = need + need_i + 256
    pool = hx.PagePool(P, shuffle_seed=11)
    bt_np = pool.alloc_table(lens, ca.max_pages)
    ibt_np = pool.alloc_table(ilens, 128)
    k_np = W.draw_fp16_normal((1, P, ca.kv_heads, 16, ca.head_dim), ca.cfg, W.configs.S_K, 77)
    v_np = W.draw_fp16_normal((1, P, ca.kv_heads, 16, ca.head_dim), ca.cfg, W.configs.S_V, 77)
    q_np = W.draw_fp16_normal((ca.batch, ca.q_heads, ca.head_dim), ca.cfg, W.configs.S_Q, 77)
    wi = W.make_ingest_inputs(ci, src_tp=4, bits=True)
    ref = oracle.decode_attention(q_np, k_np, v_np, bt_np, lens)
    ok, ov = k_np.view(np.uint16).copy(), v_np.view(np.uint16).copy()
    oracle.kv_ingest(wi["src_k"], wi["src_v"], ok, ov, heads=ci.heads, src_tp=4, dst_tp=1, dst_rank=0, block_table=ibt_np,
                     cu_seqlens=wi["cu_seqlens"], seq_lens=ilens)
    cache = hx.PagedCache(to_dev(k_np, torch), to_dev(v_np, torch))
    qd = to_dev(q_np, torch)
    out = torch.full_like(qd, float("nan"))
    mx = int(lens.max())
    wsb = hx.decode_attention_workspace_bytes(ca.batch, ca.q_heads, ca.kv_heads, ca.head_dim, mx)
    ws = torch.zeros(wsb, dtype=torch.uint8, device="cuda")
    sk = [to_dev(a, torch) for a in wi["src_k"]]
    sv = [to_dev(a, torch) for a in wi["src_v"]]
    if True:
        hx.decode_step(out=out, q=qd, cache=cache, layer=0, q_heads=ca.q_heads, block_table=torch.from_numpy(bt_np).cuda(),
                       block_table_stride=bt_np.shape[1], seq_lens=torch.from_numpy(lens).cuda(), batch=ca.batch,
                       max_seq_len=mx, sm_scale=0.0, workspace=ws, workspace_bytes=wsb, src_k=sk, src_v=sv, ing_layers=1,
                       heads=ci.heads, src_tp=4, dst_tp=1, dst_rank=0, ing_block_table=torch.from_numpy(ibt_np).cuda(),
                       ing_block_table_stride=128, ing_cu_seqlens=torch.from_numpy(wi["cu_seqlens"]).cuda(),
                       ing_seq_lens=torch.from_numpy(ilens).cuda(), ing_batch=len(ilens),
                       ing_total_tokens=wi["total_tokens"], ing_max_seq_len=2048, overlap_ingest=1)
        k_after = cache.k.clone()                       # enqueued on the caller's stream: ordered after BOTH kernels
        torch.cuda.synchronize()
    assert np.array_equal(dev_u16(k_after), ok) and np.array_equal(dev_u16(cache.v), ov)
    _check_all_rows("llama70b_tp1", out.cpu().numpy(), ref, "hx_decode_step, overlapped handoff")


def test_ingest_config4_all_80_layers_both_ranks(env):
    """configs[3] as bench.py runs it: ONE hx_kv_ingest call per destination rank over all 80 layers (23 GB of
    shards; element offsets reach 3.6e9 in the cache and 1.4e9 in a shard).  Ten layers - 0, 79 and eight drawn with a
    fixed seed - hold seeded host data and are compared bit for bit with the oracle, one layer at a time (SURVEY.md
    section 7, "22.8 GB"), so a layer permutation or offset error common to ingest and gather cannot hide; the
    other layers hold device-drawn 16-bit patterns and are checked by properties that hold at any size: the
    on-device gather of all 80 layers reproduces every shard exactly, and pages no prompt owns keep the fill."""
    hx, torch, oracle = env
    c = W.CONFIGS["llama70b_ingest"]
    w = W.make_ingest_inputs(c, layers=1)                  # lengths, cu_seqlens, block table (shared by all layers)
    L, T, P, S, R, D = c.layers, w["total_tokens"], w["num_pages"], c.src_tp, c.dst_tp, c.head_dim
    hs, hd = c.heads // S, c.heads // R
    checked = tuple(sorted({0, L - 1} | set(W.rng(c.cfg, 31).choice(np.arange(1, L - 1), size=8, replace=False).tolist())))
    assert len(checked) == 10
    host = {l: ([W.draw_u16_bits((1, T, hs, D), c.cfg, W.configs.S_SRCK, r, 7000 + l) for r in range(S)],
                [W.draw_u16_bits((1, T, hs, D), c.cfg, W.configs.S_SRCV, r, 7000 + l) for r in range(S)]) for l in checked}
    g = torch.Generator(device="cuda")
    g.manual_seed(4)
    sk = [torch.randint(-32768, 32767, (L, T, hs, D), dtype=torch.int16, device="cuda", generator=g) for _ in range(S)]
    sv = [torch.randint(-32768, 32767, (L, T, hs, D), dtype=torch.int16, device="cuda", generator=g) for _ in range(S)]
    for l in checked:
        for r in range(S):
            sk[r][l].copy_(torch.from_numpy(host[l][0][r][0].view(np.int16)))
            sv[r][l].copy_(torch.from_numpy(host[l][1][r][0].view(np.int16)))
    skh, svh = [t.view(torch.float16) for t in sk], [t.view(torch.float16) for t in sv]
    bt, cu, sl = (torch.from_numpy(w[k]).cuda() for k in ("block_table", "cu_seqlens", "seq_lens"))
    kw = dict(layers=L, heads=c.heads, head_dim=D, src_tp=S, dst_tp=R, block_table=bt, block_table_stride=bt.shape[1],
              cu_seqlens=cu, seq_lens=sl, batch=c.prompts, total_tokens=T, max_seq_len=int(w["seq_lens"].max()))
    fill = int(np.array([0xDEAD], dtype=np.uint16).view(np.int16)[0])
    owned = np.zeros(P, dtype=bool)
    owned[w["block_table"][w["block_table"] >= 0]] = True
    unowned = torch.from_numpy(np.flatnonzero(~owned)).cuda()
    gk = [torch.full_like(t, 0x0BAD) for t in sk]
    gv = [torch.full_like(t, 0x0BAD) for t in sv]
    for q in range(R):
        dk = torch.full((L, P, hd, 16, D), fill, dtype=torch.int16, device="cuda")
        dv = torch.full((L, P, hd, 16, D), fill, dtype=torch.int16, device="cuda")
        cache = hx.PagedCache(dk.view(torch.float16), dv.view(torch.float16))
        hx.kv_ingest(skh, svh, dst_rank=q, dst=cache, **kw)
        torch.cuda.synchronize()
        for l in checked:
            ok = np.full((1, P, hd, 16, D), 0xDEAD, dtype=np.uint16)
            ov = ok.copy()
            oracle.kv_ingest(host[l][0], host[l][1], ok, ov, heads=c.heads, src_tp=S, dst_tp=R, dst_rank=q,
                             block_table=w["block_table"], cu_seqlens=w["cu_seqlens"], seq_lens=w["seq_lens"])
            assert np.array_equal(dk[l].cpu().numpy().view(np.uint16), ok[0]), (q, l)
            assert np.array_equal(dv[l].cpu().numpy().view(np.uint16), ov[0]), (q, l)
        assert bool((dk[:, unowned] == fill).all()) and bool((dv[:, unowned] == fill).all()), q
        hx.kv_gather([t.view(torch.float16) for t in gk], [t.view(torch.float16) for t in gv], dst_rank=q, dst=cache, **kw)
        torch.cuda.synchronize()
        del dk, dv, cache
    for r in range(S):                                     # both ranks together rebuilt every shard, every layer
        assert torch.equal(gk[r], sk[r]) and torch.equal(gv[r], sv[r]), r


def test_ingest_config5_step_bit_exact(env):
    hx, torch, oracle = env
    c = W.CONFIGS["llama70b_tp1_ingest"]
    for S in (4, 1):
        w = W.make_ingest_inputs(c, src_tp=S)
        dk, dv = run_gpu_ingest(hx, torch, w, 0)
        ok, ov = oracle_ingest(oracle, w, 0)
        assert np.array_equal(dk, ok) and np.array_equal(dv, ov)


def test_prefill_bench_size_sampled_rows(env):
    """hx_prefill_attention at the size bench.py times (16 prompts x 2048 tokens, LLaMA-2-70B 64 q / 8 kv heads,
    ingested by hx_kv_ingest first: the cfg5 handoff prompts).  The oracle computes sampled (prompt, position)
    rows one by one — a row at position p is the one-query-token case of a context cut at p + 1 — then a sweep through
    one whole prompt (every 17th position: 121 rows x 64 heads that visit every in-page offset and every 128-token row
    tile; all 2048 rows cost the float64 oracle eight minutes, which the suite cannot afford); every output must be finite.  Per-row bound: REL_L2_TOL itself
    (a single row's error is bounded by P's fp16 rounding 2^-12 plus the output's 2^-11 = 7.3e-4)."""
    hx, torch, oracle = env
    from helpers import to_dev
    c = W.CONFIGS["llama70b_tp1_ingest"]
    w = W.make_ingest_inputs(c, src_tp=4)
    dk, dv = run_gpu_ingest(hx, torch, w, 0)                          # paged K/V as the decode rank holds it
    ok, ov = oracle_ingest(oracle, w, 0)
    assert np.array_equal(dk, ok) and np.array_equal(dv, ov)
    lens, cu = w["seq_lens"], w["cu_seqlens"]
    Hq, D, T = 64, 128, int(lens.sum())
    q = W.draw_fp16_normal((T, Hq, D), 5, 60)
    cache = hx.PagedCache(to_dev(dk, torch), to_dev(dv, torch))
    qd = to_dev(q, torch)
    out = torch.full_like(qd, float("nan"))
    bt = torch.from_numpy(w["block_table"]).cuda()
    sl = torch.from_numpy(lens).cuda()
    hx.prefill_attention(out, qd, cache, layer=0, q_heads=Hq, block_table=bt, block_table_stride=bt.shape[1],
                         seq_lens=sl, q_lens=sl, cu_q_lens=torch.from_numpy(cu).cuda(), batch=len(lens),
                         total_q_tokens=T, max_q_len=int(lens.max()), max_seq_len=int(lens.max()))
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert np.isfinite(got.astype(np.float32)).all()
    g = np.random.default_rng(11)
    reqs = g.integers(0, len(lens), size=48)
    poss = np.concatenate([[0, 1, 15, 16, 63, 64, 127, 128, 2047, 2046], g.integers(0, 2048, size=38)])
    rows = cu[reqs] + poss
    ref = oracle.prefill_attention(np.ascontiguousarray(q[rows]), ok.view(np.float16), ov.view(np.float16),
                                   np.ascontiguousarray(w["block_table"][reqs]), (poss + 1).astype(np.int32),
                                   np.ones(len(rows), dtype=np.int32))
    max_abs, rel_l2 = attn_errors(got[rows], ref)
    assert max_abs <= MAX_ABS_TOL and rel_l2 <= REL_L2_TOL, (max_abs, rel_l2)
    for j in range(len(rows)):
        _, r = attn_errors(got[rows[j]], ref[j])
        assert r <= REL_L2_TOL, (int(reqs[j]), int(poss[j]), r)
    # a sweep through one whole prompt: every 17th position (17 is coprime with the page size, so every in-page offset occurs)
    r0 = 5
    assert int(lens[r0]) == 2048
    sweep = np.arange(0, 2048, 17)
    srows = int(cu[r0]) + sweep
    ref_s = oracle.prefill_attention(np.ascontiguousarray(q[srows]), ok.view(np.float16), ov.view(np.float16),
                                     np.ascontiguousarray(np.repeat(w["block_table"][r0:r0 + 1], len(sweep), axis=0)),
                                     (sweep + 1).astype(np.int32), np.ones(len(sweep), dtype=np.int32))
    max_abs, rel_l2 = attn_errors(got[srows], ref_s)
    assert max_abs <= MAX_ABS_TOL and rel_l2 <= REL_L2_TOL, ("prompt sweep", max_abs, rel_l2)
    g64 = got[srows].astype(np.float64)
    row_rel = np.linalg.norm((g64 - ref_s).reshape(len(sweep), -1), axis=1) / np.linalg.norm(ref_s.reshape(len(sweep), -1), axis=1)
    assert row_rel.max() <= REL_L2_TOL, ("prompt sweep, worst row", int(sweep[row_rel.argmax()]), float(row_rel.max()))
