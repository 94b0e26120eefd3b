"""GPU parity: the CUDA path (through the C-ABI binding) against the oracle, element by element,
on the same seeded inputs.  Ingest: bit-exact.  Attention: max-abs <= 2e-3 and relative-L2 <= 1e-3
(north_star; fp16 in, fp32 accumulate).  Run on the B200 box with `pytest -m gpu`."""
import numpy as np
import pytest

import workloads as W
from helpers import (MAX_ABS_TOL, REL_L2_TOL, attn_errors, oracle_ingest, run_gpu_attention,
                     run_gpu_ingest, to_dev)

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


def check_attn(env, w, label="", **kw):
    hx, torch, oracle = env
    got = run_gpu_attention(hx, torch, w, **kw)
    ref = oracle.decode_attention(w["q"] if "q" not in kw else kw["q"], w["k"], w["v"], w["block_table"],
                                  w["seq_lens"], layer=kw.get("layer", 0), sm_scale=kw.get("sm_scale"))
    assert np.isfinite(got.astype(np.float32)).all(), label
    max_abs, rel_l2 = attn_errors(got, ref)
    assert max_abs <= MAX_ABS_TOL and rel_l2 <= REL_L2_TOL, (label, max_abs, rel_l2)
    return got, ref


# ------------------------------------------------------------------ ingest (bit-exact)
def test_ingest_tiny_config_bit_exact(env):
    hx, torch, oracle = env
    w = W.make_ingest_inputs(W.CONFIGS["tiny_ingest"], bits=True)     # all 16-bit patterns
    dk, dv, gk, gv = run_gpu_ingest(hx, torch, w, 0, gather_back=True)
    ok, ov = oracle_ingest(oracle, w, 0)
    assert np.array_equal(dk, ok) and np.array_equal(dv, ov)
    for r in range(2):
        assert np.array_equal(gk[r], w["src_k"][r]) and np.array_equal(gv[r], w["src_v"][r])


@pytest.mark.parametrize("S", [1, 2, 4, 8])
@pytest.mark.parametrize("R", [1, 2, 4, 8])
@pytest.mark.parametrize("D", [64, 128])
def test_ingest_sweep_tp_pairs(env, S, R, D):
    hx, torch, oracle = env
    lens = np.array([1, 15, 16, 17, 31, 32, 33, 255, 256, 257, 0, 5], dtype=np.int32)
    c = W.IngestConfig(80, "sweep", 3, 8, D, S, R, len(lens), "x")
    w = W.make_ingest_inputs(c, lens=lens, bits=True, seed_extra=S * 100 + R * 10 + D)
    for q in range(R):
        dk, dv, gk, gv = run_gpu_ingest(hx, torch, w, q, gather_back=True)
        ok, ov = oracle_ingest(oracle, w, q)
        assert np.array_equal(dk, ok), (S, R, D, q)
        assert np.array_equal(dv, ov), (S, R, D, q)
        # gather rebuilds exactly the heads rank q owns; other positions keep the fill
        hs, hd = 8 // S, 8 // R
        for r in range(S):
            for j in range(hs):
                h = r * hs + j
                if q * hd <= h < (q + 1) * hd:
                    assert np.array_equal(gk[r][:, :, j], w["src_k"][r][:, :, j])
                    assert np.array_equal(gv[r][:, :, j], w["src_v"][r][:, :, j])
                else:
                    assert (gk[r][:, :, j] == 0x0BAD).all() and (gv[r][:, :, j] == 0x0BAD).all()


def test_ingest_odd_head_counts(env):
    hx, torch, oracle = env
    for heads, S, R in [(14, 2, 7), (56, 4, 4), (6, 3, 2), (12, 4, 3)]:
        lens = np.array([40, 3, 129], dtype=np.int32)
        c = W.IngestConfig(81, "odd", 2, heads, 128, S, R, 3, "x")
        w = W.make_ingest_inputs(c, lens=lens, bits=True, seed_extra=heads)
        for q in (0, R - 1):
            dk, dv = run_gpu_ingest(hx, torch, w, q)
            ok, ov = oracle_ingest(oracle, w, q)
            assert np.array_equal(dk, ok) and np.array_equal(dv, ov), (heads, S, R, q)


def test_ingest_empty_inputs(env):
    hx, torch, oracle = env
    c = W.IngestConfig(82, "empty", 1, 4, 128, 2, 1, 2, "x")
    w = W.make_ingest_inputs(c, lens=np.array([0, 0], dtype=np.int32), bits=True)
    dk, dv = run_gpu_ingest(hx, torch, w, 0)
    assert (dk == 0xDEAD).all() and (dv == 0xDEAD).all()


# ------------------------------------------------------------------ attention
def test_attention_tiny_config(env):
    w = W.make_attention_inputs(W.CONFIGS["tiny"])
    check_attn(env, w, "tiny")


@pytest.mark.parametrize("G,Hkv", [(1, 4), (2, 2), (4, 2), (8, 2), (16, 1), (1, 14), (8, 4)])
@pytest.mark.parametrize("D", [64, 128])
def test_attention_sweep_page_boundaries(env, G, Hkv, D):
    lens = np.array([1, 15, 16, 17, 31, 32, 33, 255, 256, 257, 1000, 2], dtype=np.int32)
    c = W.AttnConfig(70, "sweep", len(lens), G * Hkv, Hkv, D, 64, "x")
    w = W.make_attention_inputs(c, lens=lens, layers=2, seed_extra=G * 1000 + Hkv * 10 + D)
    check_attn(env, w, f"G={G} Hkv={Hkv} D={D}", layer=1)


def test_attention_custom_scale_and_empty_request(env):
    lens = np.array([0, 40, 0, 700], dtype=np.int32)
    c = W.AttnConfig(71, "scale", 4, 8, 1, 128, 64, "x")
    w = W.make_attention_inputs(c, lens=lens)
    got, _ = check_attn(env, w, "scale", sm_scale=0.05)
    assert (got[0] == 0).all() and (got[2] == 0).all()            # reading S11: zeros


def test_attention_single_token_is_bit_exact_v(env):
    hx, torch, _ = env
    lens = np.ones(5, dtype=np.int32)
    c = W.AttnConfig(72, "n1", 5, 8, 2, 128, 4, "x")
    w = W.make_attention_inputs(c, lens=lens)
    got = run_gpu_attention(hx, torch, w)
    for i in range(5):
        for h in range(8):
            assert np.array_equal(got[i, h].view(np.uint16), w["v"][0, w["block_table"][i, 0], h // 4, 0].view(np.uint16))


def test_attention_constant_v_and_zero_q(env):
    hx, torch, oracle = env
    c = W.AttnConfig(73, "cv", 3, 8, 1, 128, 64, "x")
    w = W.make_attention_inputs(c, lens=np.array([17, 300, 1000], dtype=np.int32))
    vec = W.draw_fp16_normal((128,), 73, 99)
    w["v"][:] = vec
    got = run_gpu_attention(hx, torch, w)
    assert np.abs(got.astype(np.float64) - vec.astype(np.float64)).max() <= 1e-3   # weights sum to 1
    w = W.make_attention_inputs(c, lens=np.array([17, 300, 1000], dtype=np.int32))
    check_attn(env, w, "q=0", q=np.zeros_like(w["q"]))


def test_attention_page_permutation_bit_identical(env):
    hx, torch, _ = env
    c = W.AttnConfig(74, "perm", 6, 16, 2, 128, 256, "x")
    w = W.make_attention_inputs(c, lens=np.array([17, 64, 100, 255, 2000, 4000], dtype=np.int32))
    base = run_gpu_attention(hx, torch, w)
    P = w["num_pages"]
    perm = W.rng(74, 50).permutation(P)
    w2 = dict(w)
    w2["k"], w2["v"] = np.empty_like(w["k"]), np.empty_like(w["v"])
    w2["k"][:, perm], w2["v"][:, perm] = w["k"], w["v"]
    w2["block_table"] = np.where(w["block_table"] >= 0, perm[np.clip(w["block_table"], 0, None)], -1).astype(np.int32)
    again = run_gpu_attention(hx, torch, w2)
    assert np.array_equal(base.view(np.uint16), again.view(np.uint16))
    assert np.array_equal(base.view(np.uint16), run_gpu_attention(hx, torch, w).view(np.uint16))   # run-to-run


def test_attention_nan_poison_is_harmless(env):
    hx, torch, _ = env
    c = W.AttnConfig(75, "poison", 5, 16, 2, 128, 64, "x")
    w = W.make_attention_inputs(c, lens=np.array([17, 64, 100, 255, 1], dtype=np.int32))
    base = run_gpu_attention(hx, torch, w)
    owned = np.zeros((w["num_pages"], 16), dtype=bool)
    for i, n in enumerate(w["seq_lens"]):
        for t in range(n):
            owned[w["block_table"][i, t // 16], t % 16] = True
    kb, vb = w["k"].view(np.uint16).copy(), w["v"].view(np.uint16).copy()
    kb[0].transpose(0, 2, 1, 3)[~owned] = 0x7E01      # NaN
    vb[0].transpose(0, 2, 1, 3)[~owned] = 0xFC00      # -inf
    w2 = dict(w, k=kb.view(np.float16), v=vb.view(np.float16))
    got = run_gpu_attention(hx, torch, w2)
    assert np.array_equal(got.view(np.uint16), base.view(np.uint16))


def test_attention_large_logits_stable(env):
    c = W.AttnConfig(76, "hot", 4, 8, 1, 128, 64, "x")
    w = W.make_attention_inputs(c, lens=np.array([100, 255, 777, 16], dtype=np.int32))
    q8 = (w["q"].astype(np.float32) * 8).astype(np.float16)
    check_attn(env, w, "8x logits", q=q8)


def test_ingest_then_attention_end_to_end_tiny(env):
    """configs[0] whole path: shards -> hx_kv_ingest -> hx_decode_attention vs oracle on the oracle's cache."""
    hx, torch, oracle = env
    w = W.make_ingest_inputs(W.CONFIGS["tiny_ingest"])
    dk, dv = run_gpu_ingest(hx, torch, w, 0, sentinel=0x7E01)
    ok, ov = oracle_ingest(oracle, w, 0, sentinel=0x7E01)
    assert np.array_equal(dk, ok) and np.array_equal(dv, ov)
    q = W.draw_fp16_normal((4, 4, 64), 1, W.configs.S_Q)
    wa = dict(q=q, k=dk.view(np.float16), v=dv.view(np.float16), block_table=w["block_table"],
              seq_lens=w["seq_lens"], num_pages=w["num_pages"])
    check_attn(env, wa, "tiny e2e")


def _planned(hx, torch, w, *, layer=0, sm_scale=0.0):
    """hx_decode_plan + hx_decode_attention_planned on a workload dict; returns fp16 numpy [B][Hq][D]."""
    B, Hq, D = w["q"].shape
    cache = hx.PagedCache(to_dev(w["k"], torch), to_dev(w["v"], torch))
    Hkv = cache.k.shape[2]
    qd = to_dev(w["q"], torch)
    out = torch.full_like(qd, float("nan"))
    bt = torch.from_numpy(w["block_table"]).cuda()
    sl = torch.from_numpy(np.ascontiguousarray(w["seq_lens"], dtype=np.int32)).cuda()
    mx = int(w["seq_lens"].max(initial=0))
    wsb = hx.decode_attention_workspace_bytes(B, Hq, Hkv, D, mx)
    ws = torch.zeros(max(wsb, 16), dtype=torch.uint8, device="cuda")
    plan = torch.full((max(hx.decode_plan_bytes(B, Hkv, mx), 16),), 0xAB, dtype=torch.uint8, device="cuda")
    hx.decode_plan(plan, cache, q_heads=Hq, block_table=bt, block_table_stride=bt.shape[1], seq_lens=sl, batch=B, max_seq_len=mx)
    bt.fill_(-7)                                    # the planned call must not need the table or the lengths any more
    sl.fill_(-7)
    hx.decode_attention_planned(out, qd, cache, layer=layer, q_heads=Hq, plan=plan, batch=B, max_seq_len=mx, sm_scale=sm_scale,
                                workspace=ws, workspace_bytes=wsb)
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.parametrize("G,Hkv,D", [(1, 4, 64), (8, 2, 128), (16, 1, 128), (1, 14, 128), (4, 2, 64), (8, 4, 128)])
def test_planned_attention_equals_unplanned_bit_for_bit(env, G, Hkv, D):
    """hx_decode_plan hoists what depends only on seq_lens and the block table out of the layer calls; the planned
    kernel uses the same work partition and arithmetic, so its output is the unplanned call's, bit for bit — page
    boundaries, empty contexts, a context of one token, two layers, custom scale."""
    hx, torch, oracle = env
    lens = np.array([1, 15, 16, 17, 0, 31, 32, 33, 255, 256, 257, 1000, 2, 0, 3000], dtype=np.int32)
    c = W.AttnConfig(78, "plan", len(lens), G * Hkv, Hkv, D, 256, "x")
    w = W.make_attention_inputs(c, lens=lens, layers=2, seed_extra=G * 100 + Hkv)
    for layer, scale in ((0, 0.0), (1, 0.07)):
        base = run_gpu_attention(hx, torch, w, layer=layer, sm_scale=scale)
        got = _planned(hx, torch, w, layer=layer, sm_scale=scale)
        assert np.array_equal(base.view(np.uint16), got.view(np.uint16)), (G, Hkv, D, layer)
        ref = oracle.decode_attention(w["q"], w["k"], w["v"], w["block_table"], lens, layer=layer, sm_scale=scale or None)
        max_abs, rel = attn_errors(got, ref)
        assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (G, Hkv, D, layer, max_abs, rel)
        assert (got[4] == 0).all() and (got[13] == 0).all()               # reading S11 through the plan's empty list


def test_one_plan_serves_every_layer_of_a_step(env):
    """The use the plan is for: one hx_decode_plan, then one planned call per layer, all against the oracle."""
    hx, torch, oracle = env
    lens = W.rng(79, 0).integers(1, 1500, size=40).astype(np.int32)
    c = W.AttnConfig(79, "plan", 40, 32, 4, 128, 128, "x")
    L = 5
    w = W.make_attention_inputs(c, lens=lens, layers=L)
    cache = hx.PagedCache(to_dev(w["k"], torch), to_dev(w["v"], torch))
    bt, sl = torch.from_numpy(w["block_table"]).cuda(), torch.from_numpy(lens).cuda()
    mx = int(lens.max())
    wsb = hx.decode_attention_workspace_bytes(40, 32, 4, 128, mx)
    ws = torch.zeros(wsb, dtype=torch.uint8, device="cuda")
    plan = torch.empty(hx.decode_plan_bytes(40, 4, mx), dtype=torch.uint8, device="cuda")
    hx.decode_plan(plan, cache, q_heads=32, block_table=bt, block_table_stride=bt.shape[1], seq_lens=sl, batch=40, max_seq_len=mx)
    qs = [W.draw_fp16_normal((40, 32, 128), 79, 5, l) for l in range(L)]
    outs = [torch.full((40, 32, 128), float("nan"), dtype=torch.float16, device="cuda") for _ in range(L)]
    for l in range(L):                                   # back to back, as a model's layer loop issues them
        hx.decode_attention_planned(outs[l], to_dev(qs[l], torch), cache, layer=l, q_heads=32, plan=plan, batch=40, max_seq_len=mx,
                                    workspace=ws, workspace_bytes=wsb)
    torch.cuda.synchronize()
    for l in range(L):
        ref = oracle.decode_attention(qs[l], w["k"], w["v"], w["block_table"], lens, layer=l)
        max_abs, rel = attn_errors(outs[l].cpu().numpy(), ref)
        assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (l, max_abs, rel)


def test_attention_batch_larger_than_one_launch(env):
    """B above the per-launch request limit (2048) goes out as several launches sharing one workspace."""
    g = W.rng(78, 0)
    lens = g.integers(0, 40, size=2100).astype(np.int32)
    lens[[0, 2047, 2048, 2099]] = [33, 17, 1, 16]
    c = W.AttnConfig(78, "bigB", len(lens), 8, 2, 64, 4, "x")
    check_attn(env, W.make_attention_inputs(c, lens=lens), "B=2100")


def test_attention_shared_pages_between_requests(env):
    """Two requests may point at the same physical pages (prefix sharing): attention only reads."""
    hx, torch, oracle = env
    c = W.AttnConfig(79, "shared", 3, 8, 1, 128, 8, "x")
    w = W.make_attention_inputs(c, lens=np.array([64, 64, 100], dtype=np.int32))
    w["block_table"][1, :4] = w["block_table"][0, :4]
    w["block_table"][2, :4] = w["block_table"][0, :4]
    got, ref = check_attn(env, w, "shared pages")
    assert not np.array_equal(got[0], got[1])            # different q, same KV


def test_attention_max_context_single_request(env):
    """One 8192-token request (512 pages, the cfg5 maximum) split over every worker of the grid."""
    c = W.AttnConfig(80, "long", 1, 8, 1, 128, 512, "x")
    check_attn(env, W.make_attention_inputs(c, lens=np.array([8192], dtype=np.int32)), "n=8192")


def test_ingest_on_side_stream_while_attention_runs(env):
    """Ingest into pages disjoint from the active batch may run on another stream."""
    hx, torch, oracle = env
    c = W.AttnConfig(81, "overlap", 16, 32, 4, 128, 128, "x")
    w = W.make_attention_inputs(c, lens=W.rng(81, 1).integers(500, 2000, size=16).astype(np.int32), spare=2.0)
    base = run_gpu_attention(hx, torch, w)
    used = set(w["block_table"][w["block_table"] >= 0].tolist())
    free = np.array([p for p in range(w["num_pages"]) if p not in used], dtype=np.int32)
    ci = W.IngestConfig(81, "ov", 1, 4, 128, 2, 1, 4, "x")
    wi = W.make_ingest_inputs(ci, lens=np.array([300, 200, 100, 17], dtype=np.int32), bits=True)
    need = W.pages_for(wi["seq_lens"])
    bt = np.full((4, int(need.max())), -1, dtype=np.int32)
    o = 0
    for i, k in enumerate(need):
        bt[i, :k] = free[o:o + k]; o += k
    from helpers import to_dev, dev_u16
    k, v = to_dev(w["k"], torch), to_dev(w["v"], torch)
    cache = hx.PagedCache(k, v)
    q = to_dev(w["q"], torch); out = torch.empty_like(q)
    btd = torch.from_numpy(w["block_table"]).cuda(); sl = torch.from_numpy(w["seq_lens"]).cuda()
    wsb = hx.decode_attention_workspace_bytes(16, 32, 4, 128, 2000)
    ws = torch.zeros(wsb, dtype=torch.uint8, device="cuda")
    sk = [to_dev(a, torch) for a in wi["src_k"]]; sv = [to_dev(a, torch) for a in wi["src_v"]]
    ibt = torch.from_numpy(bt).cuda(); icu = torch.from_numpy(wi["cu_seqlens"]).cuda(); isl = torch.from_numpy(wi["seq_lens"]).cuda()
    side = torch.cuda.Stream()
    torch.cuda.synchronize()
    for _ in range(3):
        with torch.cuda.stream(side):
            hx.kv_ingest(sk, sv, layers=1, heads=4, head_dim=128, src_tp=2, dst_tp=1, dst_rank=0, dst=cache, block_table=ibt,
                         block_table_stride=ibt.shape[1], cu_seqlens=icu, seq_lens=isl, batch=4, total_tokens=617, max_seq_len=300)
        hx.decode_attention(out, q, cache, layer=0, q_heads=32, block_table=btd, block_table_stride=btd.shape[1], seq_lens=sl,
                            batch=16, max_seq_len=2000, workspace=ws, workspace_bytes=wsb)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy().view(np.uint16), base.view(np.uint16))
    # and the ingested pages hold exactly what the oracle puts there
    ok = w["k"].view(np.uint16).copy(); ov = w["v"].view(np.uint16).copy()
    oracle.kv_ingest(wi["src_k"], wi["src_v"], ok, ov, heads=4, src_tp=2, dst_tp=1, dst_rank=0, block_table=bt,
                     cu_seqlens=wi["cu_seqlens"], seq_lens=wi["seq_lens"])
    assert np.array_equal(dev_u16(k), ok) and np.array_equal(dev_u16(v), ov)


def test_decode_step_host_matches_oracle(env):
    """hx_decode_step_host: host shards + host q in, host out back; ingest lands bit-exact and the
    attention over the freshly ingested pages matches the oracle (whole path, configs[0] shape)."""
    hx, torch, oracle = env
    from helpers import dev_u16
    wi = W.make_ingest_inputs(W.CONFIGS["tiny_ingest"])
    P, L, H, D = wi["num_pages"], 1, 4, 64
    lens = wi["seq_lens"]
    cache = hx.PagedCache(torch.zeros((L, P, H, 16, D), dtype=torch.float16, device="cuda"),
                          torch.zeros((L, P, H, 16, D), dtype=torch.float16, device="cuda"))
    q_np = W.draw_fp16_normal((4, 4, D), 1, W.configs.S_Q)
    pin = lambda a: torch.from_numpy(a).pin_memory()
    qh, oh = pin(q_np), torch.empty((4, 4, D), dtype=torch.float16).pin_memory()
    skh = [pin(a.view(np.int16)) for a in wi["src_k"]]; svh = [pin(a.view(np.int16)) for a in wi["src_v"]]
    skd = [torch.empty_like(a, device="cuda") for a in skh]; svd = [torch.empty_like(a, device="cuda") for a in svh]
    bth, cuh, slh = pin(wi["block_table"]), pin(wi["cu_seqlens"]), pin(lens)
    btd, cud, sld = (torch.empty_like(a, device="cuda") for a in (bth, cuh, slh))
    qd, od = torch.empty_like(qh, device="cuda"), torch.empty_like(oh, device="cuda")
    wsb = hx.decode_attention_workspace_bytes(4, 4, 4, D, 255)
    ws = torch.zeros(wsb, dtype=torch.uint8, device="cuda")
    # the active batch is the 4 prompts just ingested: its device block table / lengths are the staging copies
    hx.decode_step_host(q_host=qh, out_host=oh, q_dev=qd, out_dev=od, cache=cache, layer=0, q_heads=4,
                        block_table_dev=btd, block_table_stride=btd.shape[1], seq_lens_dev=sld, batch=4, max_seq_len=255,
                        sm_scale=0.0, workspace=ws, workspace_bytes=wsb, src_k_host=skh, src_v_host=svh, src_k_dev=skd,
                        src_v_dev=svd, ing_layers=1, heads=4, src_tp=2, dst_tp=1, dst_rank=0, ing_block_table_host=bth,
                        ing_block_table_stride=bth.shape[1], ing_cu_seqlens_host=cuh, ing_seq_lens_host=slh,
                        ing_block_table_dev=btd, ing_cu_seqlens_dev=cud, ing_seq_lens_dev=sld, ing_batch=4,
                        ing_total_tokens=wi["total_tokens"], ing_max_seq_len=255)
    torch.cuda.synchronize()
    ok = np.zeros((L, P, H, 16, D), dtype=np.uint16); ov = np.zeros_like(ok)
    oracle.kv_ingest(wi["src_k"], wi["src_v"], ok, ov, heads=4, src_tp=2, dst_tp=1, dst_rank=0,
                     block_table=wi["block_table"], cu_seqlens=wi["cu_seqlens"], seq_lens=lens)
    assert np.array_equal(dev_u16(cache.k), ok) and np.array_equal(dev_u16(cache.v), ov)
    ref = oracle.decode_attention(q_np, ok.view(np.float16), ov.view(np.float16), wi["block_table"], lens)
    max_abs, rel = attn_errors(oh.numpy(), ref)
    assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (max_abs, rel)
