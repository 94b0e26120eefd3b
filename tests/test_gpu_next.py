"""GPU parity for the NEXT rows of SURVEY.md §8(f): pipeline-stage ingest (F3, bit-exact), append of
the step's token (F1, bit-exact), fused append-then-attend (cache bit-exact, output bit-identical to
append followed by attention, and within the north_star tolerances of the oracle), pull-mode ingest
from memory the GPU reaches over a link (F2: mapped pinned host memory stands in for a peer GPU)."""
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


def _sentinel_cache(hx, torch, shape, fill=0xDEAD):
    f = int(np.array([fill], dtype=np.uint16).view(np.int16)[0])
    dk = torch.full(shape, f, dtype=torch.int16, device="cuda").view(torch.float16)
    dv = torch.full(shape, f, dtype=torch.int16, device="cuda").view(torch.float16)
    return hx.PagedCache(dk, dv)


# ------------------------------------------------------------------ F3
@pytest.mark.parametrize("S,R,D", [(4, 2, 128), (1, 1, 64), (2, 4, 128)])
def test_stage_ingest_all_stage_pairs_bit_exact(env, S, R, D):
    """80-layer-like model cut 3/3/2 on the prefill side and 5/3 on the decode side (scaled to 8
    layers): every overlapping stage pair moved by hx_kv_ingest_stage == the oracle's stage ingest,
    and the union == the one-call hx_kv_ingest of the whole model."""
    hx, torch, oracle = env
    L, heads = 8, 8
    lens = np.array([1, 15, 16, 17, 33, 250], dtype=np.int32)
    c = W.IngestConfig(94, "t", L, heads, D, S, R, len(lens), "x")
    w = W.make_ingest_inputs(c, lens=lens, bits=True, seed_extra=S * 10 + R)
    P, hd = w["num_pages"], heads // R
    bt, cu, sl = (torch.from_numpy(w[k]).cuda() for k in ("block_table", "cu_seqlens", "seq_lens"))
    src_stages, dst_stages = [(0, 3), (3, 3), (6, 2)], [(0, 5), (5, 3)]
    for qrank in range(R):
        common = dict(heads=heads, head_dim=D, src_tp=S, dst_tp=R, dst_rank=qrank, block_table=bt,
                      block_table_stride=bt.shape[1], cu_seqlens=cu, seq_lens=sl, batch=len(lens),
                      total_tokens=w["total_tokens"], max_seq_len=int(lens.max()))
        whole = _sentinel_cache(hx, torch, (L, P, hd, 16, D))
        hx.kv_ingest([to_dev(a, torch) for a in w["src_k"]], [to_dev(a, torch) for a in w["src_v"]], layers=L,
                     dst=whole, **common)
        for df, dc in dst_stages:
            cache = _sentinel_cache(hx, torch, (dc, P, hd, 16, D))
            ok = np.full((dc, P, hd, 16, D), 0xDEAD, dtype=np.uint16)
            ov = np.full_like(ok, 0xDEAD)
            for sf, sc in src_stages:
                a, b, n = hx.stage_overlap(sf, sc, df, dc)
                if n == 0:
                    continue
                sk = [np.ascontiguousarray(x[sf:sf + sc]) for x in w["src_k"]]
                sv = [np.ascontiguousarray(x[sf:sf + sc]) for x in w["src_v"]]
                hx.kv_ingest_stage([to_dev(x, torch) for x in sk], [to_dev(x, torch) for x in sv], src_layers=sc,
                                   src_layer0=a, dst_layer0=b, layers=n, dst=cache, **common)
                oracle.kv_ingest_stage(sk, sv, ok, ov, heads=heads, src_tp=S, dst_tp=R, dst_rank=qrank, src_layer0=a,
                                       dst_layer0=b, count=n, block_table=w["block_table"], cu_seqlens=w["cu_seqlens"],
                                       seq_lens=lens)
            torch.cuda.synchronize()
            gk, gv = dev_u16(cache.k), dev_u16(cache.v)
            assert np.array_equal(gk, ok) and np.array_equal(gv, ov)
            assert np.array_equal(gk, dev_u16(whole.k)[df:df + dc]) and np.array_equal(gv, dev_u16(whole.v)[df:df + dc])


# ------------------------------------------------------------------ F1
def _append_inputs(cfgno, B, Hq, Hkv, D, lens, layers=2):
    c = W.AttnConfig(cfgno, "t", B, Hq, Hkv, D, 8, "x")
    w = W.make_attention_inputs(c, lens=np.asarray(lens, dtype=np.int32), layers=layers)
    k_new = W.draw_fp16_normal((B, Hkv, D), cfgno, 20)
    v_new = W.draw_fp16_normal((B, Hkv, D), cfgno, 21)
    return w, k_new, v_new


LENS = [1, 2, 15, 16, 17, 31, 32, 33, 255, 256, 257, 0, 1000, 48, 64, 700]


@pytest.mark.parametrize("G,Hkv,D", [(1, 4, 64), (8, 2, 128), (1, 14, 128), (4, 2, 64), (16, 1, 128)])
def test_append_and_fused_append_attention(env, G, Hkv, D):
    hx, torch, oracle = env
    B, Hq, layer = len(LENS), G * Hkv, 1
    w, k_new, v_new = _append_inputs(95, B, Hq, Hkv, D, LENS)
    lens = w["seq_lens"]
    # oracle: append then attention
    ok, ov = w["k"].view(np.uint16).copy(), w["v"].view(np.uint16).copy()
    oracle.kv_append(k_new, v_new, ok, ov, layer=layer, block_table=w["block_table"], seq_lens=lens)
    ref = oracle.decode_attention(w["q"], ok.view(np.float16), ov.view(np.float16), w["block_table"], lens, layer=layer)

    bt = torch.from_numpy(w["block_table"]).cuda()
    sl = torch.from_numpy(lens).cuda()
    qd, kn, vn = to_dev(w["q"], torch), to_dev(k_new, torch), to_dev(v_new, torch)
    ws_bytes = hx.decode_attention_workspace_bytes(B, Hq, Hkv, D, int(lens.max()))
    ws = torch.zeros(ws_bytes, dtype=torch.uint8, device="cuda")
    common = dict(layer=layer, block_table=bt, block_table_stride=bt.shape[1], seq_lens=sl, batch=B,
                  max_seq_len=int(lens.max()))
    # (1) two launches: hx_kv_append, then hx_decode_attention
    c1 = hx.PagedCache(to_dev(w["k"], torch), to_dev(w["v"], torch))
    hx.kv_append(kn, vn, c1, **common)
    out1 = torch.full_like(qd, float("nan"))
    hx.decode_attention(out1, qd, c1, q_heads=Hq, workspace=ws, **common)
    torch.cuda.synchronize()
    assert np.array_equal(dev_u16(c1.k), ok) and np.array_equal(dev_u16(c1.v), ov)        # bit-exact cache
    max_abs, rel = attn_errors(out1.cpu().numpy(), ref)
    assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (max_abs, rel)
    # (2) one launch: hx_decode_attention_append on a fresh copy of the old cache
    c2 = hx.PagedCache(to_dev(w["k"], torch), to_dev(w["v"], torch))
    out2 = torch.full_like(qd, float("nan"))
    hx.decode_attention_append(out2, qd, kn, vn, c2, q_heads=Hq, workspace=ws, **common)
    torch.cuda.synchronize()
    assert np.array_equal(dev_u16(c2.k), ok) and np.array_equal(dev_u16(c2.v), ov)        # bit-exact cache
    assert torch.equal(out1.view(torch.int16), out2.view(torch.int16))                   # same bits as (1)
    assert np.isfinite(out2.cpu().numpy().astype(np.float32)).all()


def test_fused_append_ignores_stale_slot_contents(env):
    """The slot of token n-1 holds NaN before the call (it was never written): the fused kernel must
    take the row from k_new/v_new, never from the page."""
    hx, torch, oracle = env
    B, Hq, Hkv, D = 6, 8, 1, 128
    lens = np.array([1, 5, 16, 17, 40, 129], dtype=np.int32)
    w, k_new, v_new = _append_inputs(96, B, Hq, Hkv, D, lens, layers=1)
    kb, vb = w["k"].view(np.uint16).copy(), w["v"].view(np.uint16).copy()
    for i, n in enumerate(lens):
        pg = w["block_table"][i, (n - 1) // 16]
        kb[0, pg, :, (n - 1) % 16:, :] = 0x7E00          # the new token's slot and the tail: NaN
        vb[0, pg, :, (n - 1) % 16:, :] = 0x7C00          # +Inf
    ok, ov = kb.copy(), vb.copy()
    oracle.kv_append(k_new, v_new, ok, ov, layer=0, block_table=w["block_table"], seq_lens=lens)
    ref = oracle.decode_attention(w["q"], ok.view(np.float16), ov.view(np.float16), w["block_table"], lens)
    cache = hx.PagedCache(to_dev(kb, torch), to_dev(vb, torch))
    bt, sl = torch.from_numpy(w["block_table"]).cuda(), torch.from_numpy(lens).cuda()
    qd = to_dev(w["q"], torch)
    out = torch.full_like(qd, float("nan"))
    ws = torch.zeros(hx.decode_attention_workspace_bytes(B, Hq, Hkv, D, 129), dtype=torch.uint8, device="cuda")
    hx.decode_attention_append(out, qd, to_dev(k_new, torch), to_dev(v_new, torch), cache, layer=0, q_heads=Hq,
                               block_table=bt, block_table_stride=bt.shape[1], seq_lens=sl, batch=B, max_seq_len=129,
                               workspace=ws)
    torch.cuda.synchronize()
    assert np.array_equal(dev_u16(cache.k), ok) and np.array_equal(dev_u16(cache.v), ov)
    got = out.cpu().numpy()
    assert np.isfinite(got.astype(np.float32)).all()
    max_abs, rel = attn_errors(got, ref)
    assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (max_abs, rel)


def test_decode_loop_append_attend_many_steps(env):
    """Eight decode steps of the cache life cycle (ingest -> [append+attend] x 8): after every step
    the cache equals the oracle's bit for bit and the output is within tolerance; contexts cross page
    boundaries during the loop."""
    hx, torch, oracle = env
    heads, D, Hq = 2, 128, 16
    lens0 = np.array([10, 15, 16, 30, 100], dtype=np.int32)
    B = len(lens0)
    c = W.IngestConfig(97, "t", 1, heads, D, 2, 1, B, "x")
    w = W.make_ingest_inputs(c, lens=lens0, spare=3.0)
    stride = 16
    bt_np = np.full((B, stride), -1, dtype=np.int32)
    bt_np[:, :w["block_table"].shape[1]] = w["block_table"]
    used = set(w["block_table"][w["block_table"] >= 0].tolist())
    free = [p for p in range(w["num_pages"]) if p not in used]
    P = w["num_pages"]
    cache = _sentinel_cache(hx, torch, (1, P, heads, 16, D), fill=0x7E00)
    ok = np.full((1, P, heads, 16, D), 0x7E00, dtype=np.uint16)
    ov = ok.copy()
    bt, cu, sl = torch.from_numpy(bt_np).cuda(), torch.from_numpy(w["cu_seqlens"]).cuda(), torch.from_numpy(lens0).cuda()
    hx.kv_ingest([to_dev(a, torch) for a in w["src_k"]], [to_dev(a, torch) for a in w["src_v"]], layers=1, heads=heads,
                 head_dim=D, src_tp=2, dst_tp=1, dst_rank=0, dst=cache, block_table=bt, block_table_stride=stride,
                 cu_seqlens=cu, seq_lens=sl, batch=B, total_tokens=w["total_tokens"], max_seq_len=int(lens0.max()))
    oracle.kv_ingest(w["src_k"], w["src_v"], ok, ov, heads=heads, src_tp=2, dst_tp=1, dst_rank=0, block_table=bt_np,
                     cu_seqlens=w["cu_seqlens"], seq_lens=lens0)
    ws = torch.zeros(hx.decode_attention_workspace_bytes(B, Hq, heads, D, 256), dtype=torch.uint8, device="cuda")
    lens = lens0.copy()
    for step in range(8):
        lens = lens + 1
        for i in range(B):                                   # a request that crossed a page boundary gets a page
            if (lens[i] - 1) % 16 == 0:
                bt_np[i, (lens[i] - 1) // 16] = free.pop()
        q = W.draw_fp16_normal((B, Hq, D), 97, 30, step)
        kn = W.draw_fp16_normal((B, heads, D), 97, 31, step)
        vn = W.draw_fp16_normal((B, heads, D), 97, 32, step)
        bt, sl = torch.from_numpy(bt_np).cuda(), torch.from_numpy(lens).cuda()
        out = torch.full((B, Hq, D), float("nan"), dtype=torch.float16, device="cuda")
        hx.decode_attention_append(out, to_dev(q, torch), to_dev(kn, torch), to_dev(vn, torch), cache, layer=0,
                                   q_heads=Hq, block_table=bt, block_table_stride=stride, seq_lens=sl, batch=B,
                                   max_seq_len=int(lens.max()), workspace=ws)
        torch.cuda.synchronize()
        oracle.kv_append(kn, vn, ok, ov, layer=0, block_table=bt_np, seq_lens=lens)
        ref = oracle.decode_attention(q, ok.view(np.float16), ov.view(np.float16), bt_np, lens)
        assert np.array_equal(dev_u16(cache.k), ok) and np.array_equal(dev_u16(cache.v), ov), step
        max_abs, rel = attn_errors(out.cpu().numpy(), ref)
        assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (step, max_abs, rel)


# ------------------------------------------------------------------ F2
def test_pull_mode_ingest_from_mapped_host_memory(env):
    """Pull-mode handoff: the ingest kernel reads the prefill shards through pointers into memory
    that is NOT this GPU's HBM.  A peer GPU is not available on the box; pinned host memory mapped
    into the device address space (UVA) is reached the same way, over a link, by the same loads."""
    hx, torch, oracle = env
    c = W.IngestConfig(98, "t", 2, 8, 128, 4, 2, 5, "x")
    lens = np.array([1, 16, 17, 100, 300], dtype=np.int32)
    w = W.make_ingest_inputs(c, lens=lens, bits=True)
    P = w["num_pages"]
    pin_k = [torch.from_numpy(a.view(np.int16)).pin_memory() for a in w["src_k"]]
    pin_v = [torch.from_numpy(a.view(np.int16)).pin_memory() for a in w["src_v"]]
    assert all(t.is_pinned() for t in pin_k + pin_v)
    bt, cu, sl = (torch.from_numpy(w[k]).cuda() for k in ("block_table", "cu_seqlens", "seq_lens"))
    for qrank in range(2):
        cache = _sentinel_cache(hx, torch, (2, P, 4, 16, 128))
        hx.kv_ingest(pin_k, pin_v, layers=2, heads=8, head_dim=128, src_tp=4, dst_tp=2, dst_rank=qrank, dst=cache,
                     block_table=bt, block_table_stride=bt.shape[1], cu_seqlens=cu, seq_lens=sl, batch=len(lens),
                     total_tokens=w["total_tokens"], max_seq_len=int(lens.max()))
        torch.cuda.synchronize()
        ok = np.full((2, P, 4, 16, 128), 0xDEAD, dtype=np.uint16)
        ov = ok.copy()
        oracle.kv_ingest(w["src_k"], w["src_v"], ok, ov, heads=8, src_tp=4, dst_tp=2, dst_rank=qrank,
                         block_table=w["block_table"], cu_seqlens=w["cu_seqlens"], seq_lens=lens)
        assert np.array_equal(dev_u16(cache.k), ok) and np.array_equal(dev_u16(cache.v), ov)


def test_decode_step_host_overlapped_handoff(env):
    """hx_decode_step_host(overlap_ingest=1): the new prompts' handoff runs on the library's side stream
    under the attention of an active batch whose pages are disjoint from it.  After the stream is
    synchronised both results are the oracle's: the new pages bit for bit, the batch's output within tolerance,
    staged and pull mode alike, twice in a row (the fork/join events are reused)."""
    hx, torch, oracle = env
    Hkv, D, Hq = 2, 128, 16
    ca = W.AttnConfig(99, "t", 6, Hq, Hkv, D, 64, "x")
    wa = W.make_attention_inputs(ca, lens=np.array([5, 100, 257, 600, 16, 1000], dtype=np.int32), spare=3.0)
    ci = W.IngestConfig(99, "t", 1, Hkv, D, 2, 1, 3, "x")
    ilens = np.array([33, 500, 128], dtype=np.int32)
    used = wa["block_table"][wa["block_table"] >= 0]
    wi = W.make_ingest_inputs(ci, lens=ilens)
    free = np.setdiff1d(np.arange(wa["num_pages"]), used)
    ibt = np.full((3, 32), -1, dtype=np.int32)
    o = 0
    for r, n in enumerate(ilens):
        k = (n + 15) // 16
        ibt[r, :k] = free[o:o + k]
        o += k
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    ref_out = oracle.decode_attention(wa["q"], wa["k"], wa["v"], wa["block_table"], wa["seq_lens"])
    ok, ov = wa["k"].view(np.uint16).copy(), wa["v"].view(np.uint16).copy()
    oracle.kv_ingest(wi["src_k"], wi["src_v"], ok, ov, heads=Hkv, src_tp=2, dst_tp=1, dst_rank=0, block_table=ibt,
                     cu_seqlens=wi["cu_seqlens"], seq_lens=ilens)
    for pull in (0, 1):
        cache = hx.PagedCache(to_dev(wa["k"], torch), to_dev(wa["v"], torch))
        qh, oh = pin(wa["q"]), torch.empty(wa["q"].shape, dtype=torch.float16).pin_memory()
        skh = [pin(a.view(np.int16)) for a in wi["src_k"]]; svh = [pin(a.view(np.int16)) for a in wi["src_v"]]
        skd = [torch.empty_like(a, device="cuda") for a in skh]; svd = [torch.empty_like(a, device="cuda") for a in svh]
        bth, cuh, slh = pin(ibt), pin(wi["cu_seqlens"]), pin(ilens)
        btd, cud, sld = (torch.empty_like(a, device="cuda") for a in (bth, cuh, slh))
        qd, od = torch.empty_like(qh, device="cuda"), torch.empty_like(oh, device="cuda")
        abt, asl = torch.from_numpy(wa["block_table"]).cuda(), torch.from_numpy(wa["seq_lens"]).cuda()
        wsb = hx.decode_attention_workspace_bytes(6, Hq, Hkv, D, 1000)
        ws = torch.zeros(wsb, dtype=torch.uint8, device="cuda")
        for rep in range(2):
            oh.zero_()
            hx.decode_step_host(q_host=qh, out_host=oh, q_dev=qd, out_dev=od, cache=cache, layer=0, q_heads=Hq,
                                block_table_dev=abt, block_table_stride=abt.shape[1], seq_lens_dev=asl, batch=6,
                                max_seq_len=1000, sm_scale=0.0, workspace=ws, workspace_bytes=wsb, src_k_host=skh,
                                src_v_host=svh, src_k_dev=skd, src_v_dev=svd, ing_layers=1, heads=Hkv, src_tp=2, dst_tp=1,
                                dst_rank=0, ing_block_table_host=bth, ing_block_table_stride=32, ing_cu_seqlens_host=cuh,
                                ing_seq_lens_host=slh, ing_block_table_dev=btd, ing_cu_seqlens_dev=cud, ing_seq_lens_dev=sld,
                                ing_batch=3, ing_total_tokens=wi["total_tokens"], ing_max_seq_len=500, pull_src=pull,
                                overlap_ingest=1)
            torch.cuda.current_stream().synchronize()          # the join makes the caller's stream cover the handoff
            assert np.array_equal(dev_u16(cache.k), ok) and np.array_equal(dev_u16(cache.v), ov), (pull, rep)
            max_abs, rel = attn_errors(oh.numpy(), ref_out)
            assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (pull, rep, max_abs, rel)


def test_decode_step_in_a_cuda_graph(env):
    """The calls only enqueue work and keep no per-call host state, so a whole decode step (ingest of new
    prompts, append + attention of the active batch) can be captured once in a CUDA graph and replayed; each
    replay sees the CURRENT contents of the device buffers.  Two replays with different inputs, both checked
    against the oracle."""
    hx, torch, oracle = env
    Hkv, D, Hq = 2, 128, 16
    ca = W.AttnConfig(87, "t", 5, Hq, Hkv, D, 64, "x")
    wa = W.make_attention_inputs(ca, lens=np.array([40, 100, 257, 600, 16], dtype=np.int32), spare=3.0)
    ci = W.IngestConfig(87, "t", 1, Hkv, D, 2, 1, 2, "x")
    ilens = np.array([33, 200], dtype=np.int32)
    used = wa["block_table"][wa["block_table"] >= 0]
    free = np.setdiff1d(np.arange(wa["num_pages"]), used)
    ibt = np.full((2, 16), -1, dtype=np.int32)
    o = 0
    for r, n in enumerate(ilens):
        k = (n + 15) // 16
        ibt[r, :k] = free[o:o + k]
        o += k
    cache = hx.PagedCache(to_dev(wa["k"], torch), to_dev(wa["v"], torch))
    B = 5
    qd = torch.empty((B, Hq, D), dtype=torch.float16, device="cuda")
    kn = torch.empty((B, Hkv, D), dtype=torch.float16, device="cuda")
    vn = torch.empty_like(kn)
    out = torch.empty_like(qd)
    wi0 = W.make_ingest_inputs(ci, lens=ilens)
    sk = [torch.empty(a.shape, dtype=torch.float16, device="cuda") for a in wi0["src_k"]]
    sv = [torch.empty(a.shape, dtype=torch.float16, device="cuda") for a in wi0["src_v"]]
    abt, asl = torch.from_numpy(wa["block_table"]).cuda(), torch.from_numpy(wa["seq_lens"]).cuda()
    ibt_d, icu, isl = torch.from_numpy(ibt).cuda(), torch.from_numpy(wi0["cu_seqlens"]).cuda(), torch.from_numpy(ilens).cuda()
    wsb = hx.decode_attention_workspace_bytes(B, Hq, Hkv, D, 600)
    ws = torch.zeros(wsb, dtype=torch.uint8, device="cuda")

    def step():
        hx.kv_ingest(sk, sv, layers=1, heads=Hkv, head_dim=D, src_tp=2, dst_tp=1, dst_rank=0, dst=cache, block_table=ibt_d,
                     block_table_stride=16, cu_seqlens=icu, seq_lens=isl, batch=2, total_tokens=int(ilens.sum()), max_seq_len=200)
        hx.decode_attention_append(out, qd, kn, vn, cache, layer=0, q_heads=Hq, block_table=abt, block_table_stride=abt.shape[1],
                                   seq_lens=asl, batch=B, max_seq_len=600, workspace=ws)

    step()                                          # warm-up outside capture (function attributes, tensor maps)
    torch.cuda.synchronize()
    cache.k.copy_(to_dev(wa["k"], torch)); cache.v.copy_(to_dev(wa["v"], torch))
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        step()
    ok, ov = wa["k"].view(np.uint16).copy(), wa["v"].view(np.uint16).copy()
    for rep in range(2):
        wi = W.make_ingest_inputs(ci, lens=ilens, seed_extra=10 + rep)
        q = W.draw_fp16_normal((B, Hq, D), 87, 70, rep)
        k1 = W.draw_fp16_normal((B, Hkv, D), 87, 71, rep)
        v1 = W.draw_fp16_normal((B, Hkv, D), 87, 72, rep)
        qd.copy_(to_dev(q, torch)); kn.copy_(to_dev(k1, torch)); vn.copy_(to_dev(v1, torch))
        for r in range(2):
            sk[r].copy_(to_dev(wi["src_k"][r], torch)); sv[r].copy_(to_dev(wi["src_v"][r], torch))
        g.replay()
        torch.cuda.synchronize()
        oracle.kv_ingest(wi["src_k"], wi["src_v"], ok, ov, heads=Hkv, src_tp=2, dst_tp=1, dst_rank=0, block_table=ibt,
                         cu_seqlens=wi["cu_seqlens"], seq_lens=ilens)
        oracle.kv_append(k1, v1, ok, ov, layer=0, block_table=wa["block_table"], seq_lens=wa["seq_lens"])
        ref = oracle.decode_attention(q, ok.view(np.float16), ov.view(np.float16), wa["block_table"], wa["seq_lens"])
        assert np.array_equal(dev_u16(cache.k), ok) and np.array_equal(dev_u16(cache.v), ov), rep
        max_abs, rel = attn_errors(out.cpu().numpy(), ref)
        assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (rep, max_abs, rel)


def test_attention_overlapped_with_the_ingest_before_it(env):
    """hx_decode_attention_overlapped right after hx_kv_ingest on one stream: the attention may start while the
    ingest is still landing (programmatic dependent launch).  The new prompts' pages are disjoint from the
    batch's, so both results must be the oracle's; a copy enqueued afterwards sees both finished.  Repeated so
    that the overlap really happens in some iterations."""
    hx, torch, oracle = env
    Hkv, D, Hq = 4, 128, 32
    ca = W.AttnConfig(86, "t", 8, Hq, Hkv, D, 256, "x")
    wa = W.make_attention_inputs(ca, lens=np.array([3000, 100, 257, 1600, 16, 2222, 900, 64], dtype=np.int32), spare=2.5)
    ci = W.IngestConfig(86, "t", 1, Hkv, D, 2, 1, 3, "x")
    ilens = np.array([1024, 2000, 128], dtype=np.int32)
    wi = W.make_ingest_inputs(ci, lens=ilens, bits=True)
    used = wa["block_table"][wa["block_table"] >= 0]
    free = np.setdiff1d(np.arange(wa["num_pages"]), used)
    ibt = np.full((3, 128), -1, dtype=np.int32)
    o = 0
    for r, n in enumerate(ilens):
        k = (n + 15) // 16
        ibt[r, :k] = free[o:o + k]
        o += k
    ref_out = oracle.decode_attention(wa["q"], wa["k"], wa["v"], wa["block_table"], wa["seq_lens"])
    ok, ov = wa["k"].view(np.uint16).copy(), wa["v"].view(np.uint16).copy()
    oracle.kv_ingest(wi["src_k"], wi["src_v"], ok, ov, heads=Hkv, src_tp=2, dst_tp=1, dst_rank=0, block_table=ibt,
                     cu_seqlens=wi["cu_seqlens"], seq_lens=ilens)
    sk = [to_dev(a, torch) for a in wi["src_k"]]; sv = [to_dev(a, torch) for a in wi["src_v"]]
    bt_i, cu_i, sl_i = torch.from_numpy(ibt).cuda(), torch.from_numpy(wi["cu_seqlens"]).cuda(), torch.from_numpy(ilens).cuda()
    abt, asl = torch.from_numpy(wa["block_table"]).cuda(), torch.from_numpy(wa["seq_lens"]).cuda()
    qd = to_dev(wa["q"], torch)
    wsb = hx.decode_attention_workspace_bytes(8, Hq, Hkv, D, 3000)
    ws = torch.zeros(wsb, dtype=torch.uint8, device="cuda")
    for rep in range(4):
        cache = hx.PagedCache(to_dev(wa["k"], torch), to_dev(wa["v"], torch))
        out = torch.full_like(qd, float("nan"))
        hx.kv_ingest(sk, sv, layers=1, heads=Hkv, head_dim=D, src_tp=2, dst_tp=1, dst_rank=0, dst=cache, block_table=bt_i,
                     block_table_stride=128, cu_seqlens=cu_i, seq_lens=sl_i, batch=3, total_tokens=int(ilens.sum()),
                     max_seq_len=2000)
        hx.decode_attention_overlapped(out, qd, cache, layer=0, q_heads=Hq, block_table=abt, block_table_stride=abt.shape[1],
                                       seq_lens=asl, batch=8, max_seq_len=3000, workspace=ws, behind_ingest=1)
        k_after = cache.k.clone()                    # stream-ordered after BOTH kernels
        torch.cuda.synchronize()
        assert np.array_equal(dev_u16(k_after), ok) and np.array_equal(dev_u16(cache.v), ov), rep
        max_abs, rel = attn_errors(out.cpu().numpy(), ref_out)
        assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (rep, max_abs, rel)
