"""The decode-side cache life cycle driven through the library's OWN allocator (SURVEY.md section 3.5, rows A1 -> A3 ->
A4-A8 -> free), and the ordering guarantees of the overlapped launches."""
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


@pytest.mark.slow
@pytest.mark.parametrize("overlap", [1, 0])
def test_cache_life_cycle_through_the_page_pool(env, overlap):
    """Five cfg5-shaped steps (64 q / 8 kv heads, D = 128, heavy-tailed contexts, new 2048-token prompts from a prefill
    TP = 4 group).  Every step: hx_pool_free of the requests that retired, hx_pool_alloc_table for the new prompts (the
    LIFO free list hands the retired pages straight back out: page REUSE), upload of their rows, hx_decode_step
    (ingest of the new prompts + attention over the active batch), then the new prompts replace the retired requests
    in the batch, so the NEXT step's attention reads what this step ingested.  After every step the whole cache equals
    the oracle's bit for bit and every output row is within tolerance."""
    hx, torch, oracle = env
    Hq, Hkv, D, S = 64, 8, 128, 4
    B, NEW, NLEN, STRIDE = 48, 4, 2048, 512
    g = W.rng(5, 40, overlap)
    lens = np.concatenate([g.integers(128, 1024, size=34, endpoint=True), g.integers(4096, 8192, size=14, endpoint=True)])
    g.shuffle(lens)
    lens = lens.astype(np.int32)
    need = int(W.pages_for(lens).sum())
    P = need + 2 * NEW * (NLEN // 16) + 64
    pool = hx.PagePool(P, shuffle_seed=3)
    bt_np = pool.alloc_table(lens, STRIDE)
    k_np = W.draw_fp16_normal((1, P, Hkv, 16, D), 5, 41, overlap)
    v_np = W.draw_fp16_normal((1, P, Hkv, 16, D), 5, 42, overlap)
    ok, ov = k_np.view(np.uint16).copy(), v_np.view(np.uint16).copy()
    cache = hx.PagedCache(to_dev(k_np, torch), to_dev(v_np, torch))
    wsb = hx.decode_attention_workspace_bytes(B, Hq, Hkv, D, 8192)
    ws = torch.zeros(wsb, dtype=torch.uint8, device="cuda")
    ci = W.IngestConfig(5, "life", 1, Hkv, D, S, 1, NEW, "x")
    ilens = np.full(NEW, NLEN, dtype=np.int32)
    seen_pages = set(bt_np[bt_np >= 0].tolist())
    reused = 0
    for step in range(5):
        # A1: the host allocator places the step's new prompts
        ibt_np = pool.alloc_table(ilens, NLEN // 16)
        new_pages = ibt_np[ibt_np >= 0]
        reused += len(seen_pages & set(new_pages.tolist()))
        seen_pages |= set(new_pages.tolist())
        assert not (set(new_pages.tolist()) & set(bt_np[bt_np >= 0].tolist()))          # disjoint from the active batch
        wi = W.make_ingest_inputs(ci, lens=ilens, src_tp=S, seed_extra=100 * overlap + step)
        q_np = W.draw_fp16_normal((B, Hq, D), 5, 43, overlap, step)
        qd = to_dev(q_np, torch)
        out = torch.full_like(qd, float("nan"))
        hx.decode_step(out=out, q=qd, cache=cache, layer=0, q_heads=Hq, block_table=torch.from_numpy(bt_np).cuda(),
                       block_table_stride=STRIDE, seq_lens=torch.from_numpy(lens).cuda(), batch=B, max_seq_len=int(lens.max()),
                       sm_scale=0.0, workspace=ws, workspace_bytes=wsb,
                       src_k=[to_dev(a, torch) for a in wi["src_k"]], src_v=[to_dev(a, torch) for a in wi["src_v"]],
                       ing_layers=1, heads=Hkv, src_tp=S, dst_tp=1, dst_rank=0, ing_block_table=torch.from_numpy(ibt_np).cuda(),
                       ing_block_table_stride=NLEN // 16, ing_cu_seqlens=torch.from_numpy(wi["cu_seqlens"]).cuda(),
                       ing_seq_lens=torch.from_numpy(ilens).cuda(), ing_batch=NEW, ing_total_tokens=NEW * NLEN,
                       ing_max_seq_len=NLEN, overlap_ingest=overlap)
        k_after, v_after = cache.k.clone(), cache.v.clone()      # on the caller's stream: after the join
        torch.cuda.synchronize()
        # the oracle's step.  overlap = 1 asserts that the attention does not read the new pages, so the order of the
        # two oracle calls does not matter; overlap = 0 is ingest first
        oracle.kv_ingest(wi["src_k"], wi["src_v"], ok, ov, heads=Hkv, src_tp=S, dst_tp=1, dst_rank=0, block_table=ibt_np,
                         cu_seqlens=wi["cu_seqlens"], seq_lens=ilens)
        ref = oracle.decode_attention(q_np, ok.view(np.float16), ov.view(np.float16), bt_np, lens)
        assert np.array_equal(dev_u16(k_after), ok) and np.array_equal(dev_u16(v_after), ov), step
        got = out.cpu().numpy()
        assert np.isfinite(got.astype(np.float32)).all(), step
        max_abs, rel = attn_errors(got, ref)
        assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (step, max_abs, rel)
        # the NEW oldest requests retire; the new prompts take their batch slots
        retire = np.arange(step * NEW, step * NEW + NEW) % B
        for j, i in enumerate(retire):
            pool.free(bt_np[i][bt_np[i] >= 0])
            bt_np[i] = -1
            bt_np[i, :NLEN // 16] = ibt_np[j]
            lens[i] = NLEN
    assert reused > 0, "the free list never handed a retired page back out"
    assert pool.num_free == P - int(W.pages_for(lens).sum())


def _long_ingest_setup(hx, torch, oracle, layers):
    """A handoff of 16 x 2048-token prompts over `layers` layers (~45 us per layer) next to a tiny active batch."""
    Hkv, D, Hq, S = 8, 128, 64, 4
    ilens = np.full(16, 2048, dtype=np.int32)
    T = int(ilens.sum())
    alens = np.array([40, 100, 17, 300], dtype=np.int32)
    P = 16 * 128 + int(W.pages_for(alens).sum()) + 32
    pool = hx.PagePool(P, shuffle_seed=9)
    abt = pool.alloc_table(alens, 32)
    ibt = pool.alloc_table(ilens, 128)
    g = torch.Generator(device="cuda")
    g.manual_seed(17)
    sk = [torch.randint(-32768, 32767, (layers, T, Hkv // S, D), dtype=torch.int16, device="cuda", generator=g) for _ in range(S)]
    sv = [torch.randint(-32768, 32767, (layers, T, Hkv // S, D), dtype=torch.int16, device="cuda", generator=g) for _ in range(S)]
    checked = (0, layers - 1)                                # the last layer's CTAs run last
    host = {}
    for l in checked:
        hk = [W.draw_u16_bits((1, T, Hkv // S, D), 5, 44, r, l) for r in range(S)]
        hv = [W.draw_u16_bits((1, T, Hkv // S, D), 5, 45, r, l) for r in range(S)]
        for r in range(S):
            sk[r][l].copy_(torch.from_numpy(hk[r][0].view(np.int16)))
            sv[r][l].copy_(torch.from_numpy(hv[r][0].view(np.int16)))
        host[l] = (hk, hv)
    k0 = W.draw_fp16_normal((1, P, Hkv, 16, D), 5, 46)
    v0 = W.draw_fp16_normal((1, P, Hkv, 16, D), 5, 47)
    q = W.draw_fp16_normal((len(alens), Hq, D), 5, 48)
    cu = np.zeros(17, dtype=np.int32)
    np.cumsum(ilens, out=cu[1:])
    expect = {}
    for l in checked:
        ek, ev = k0.view(np.uint16).copy(), v0.view(np.uint16).copy()
        oracle.kv_ingest(host[l][0], host[l][1], ek, ev, heads=Hkv, src_tp=S, dst_tp=1, dst_rank=0, block_table=ibt,
                         cu_seqlens=cu, seq_lens=ilens)
        expect[l] = (ek[0], ev[0])
    ref = oracle.decode_attention(q, k0, v0, abt, alens)     # the active batch lives in layer 0's pages, untouched
    return dict(Hkv=Hkv, D=D, Hq=Hq, S=S, ilens=ilens, T=T, alens=alens, P=P, abt=abt, ibt=ibt, sk=sk, sv=sv, k0=k0, v0=v0,
                q=q, cu=cu, expect=expect, ref=ref, checked=checked)


@pytest.mark.slow
def test_long_ingest_then_tiny_overlapped_attention_then_immediate_read(env):
    """include/hx.h promises that work enqueued after hx_decode_attention_overlapped is ordered after BOTH kernels.
    The hard case: an ingest that runs for more than a millisecond (32 layers, 4.3 GB of traffic), a tiny attention that
    would be done in microseconds, and a copy of the ingested pages enqueued right behind it.  The copy must hold the
    complete handoff (checked against the oracle on the first and the last layer, the last one being written last),
    and the attention's own result must be right; several repetitions."""
    hx, torch, oracle = env
    LAYERS = 32
    s = _long_ingest_setup(hx, torch, oracle, LAYERS)
    Hkv, D, Hq, S, P = s["Hkv"], s["D"], s["Hq"], s["S"], s["P"]
    skh, svh = [t.view(torch.float16) for t in s["sk"]], [t.view(torch.float16) for t in s["sv"]]
    ibt, cu, isl = torch.from_numpy(s["ibt"]).cuda(), torch.from_numpy(s["cu"]).cuda(), torch.from_numpy(s["ilens"]).cuda()
    abt, asl = torch.from_numpy(s["abt"]).cuda(), torch.from_numpy(s["alens"]).cuda()
    qd = to_dev(s["q"], torch)
    wsb = hx.decode_attention_workspace_bytes(4, Hq, Hkv, D, 300)
    ws = torch.zeros(wsb, dtype=torch.uint8, device="cuda")
    base_k = to_dev(s["k0"], torch).expand(LAYERS, -1, -1, -1, -1)
    base_v = to_dev(s["v0"], torch).expand(LAYERS, -1, -1, -1, -1)
    if True:
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for rep in range(4):
            cache = hx.PagedCache(base_k.contiguous(), base_v.contiguous())
            out = torch.full_like(qd, float("nan"))
            torch.cuda.synchronize()
            t0.record()
            hx.kv_ingest(skh, svh, layers=LAYERS, heads=Hkv, head_dim=D, src_tp=S, dst_tp=1, dst_rank=0, dst=cache,
                         block_table=ibt, block_table_stride=128, cu_seqlens=cu, seq_lens=isl, batch=16,
                         total_tokens=s["T"], max_seq_len=2048)
            if rep == 0:
                t1.record()      # only here, to show that the ingest is long: an event between the two launches takes
                                 # away their kernel-to-kernel adjacency; repetitions 1-3 are back to back
            hx.decode_attention_overlapped(out, qd, cache, layer=0, q_heads=Hq, block_table=abt, block_table_stride=32,
                                           seq_lens=asl, batch=4, max_seq_len=300, workspace=ws, workspace_bytes=wsb,
                                           behind_ingest=1)
            k_after = {l: cache.k[l].clone() for l in s["checked"]}      # the immediate read
            v_after = {l: cache.v[l].clone() for l in s["checked"]}
            torch.cuda.synchronize()
            if rep == 0:
                assert t0.elapsed_time(t1) >= 1.0, "the ingest is meant to run for >= 1 ms"
            for l in s["checked"]:
                assert np.array_equal(dev_u16(k_after[l]), s["expect"][l][0]), (rep, l)
                assert np.array_equal(dev_u16(v_after[l]), s["expect"][l][1]), (rep, l)
            max_abs, rel = attn_errors(out.cpu().numpy(), s["ref"])
            assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (rep, max_abs, rel)


def test_overlapped_attention_back_to_back_and_after_an_empty_ingest(env):
    """The overlapped launch may be a programmatic dependent ONLY directly behind a launched ingest kernel, and the caller
    says so explicitly (behind_ingest).  Behind another attention (same workspace: partial slots and arrival counters) or
    behind an hx_kv_ingest that launched nothing (batch == 0) the caller passes behind_ingest=0, and the call must behave
    exactly like hx_decode_attention - the library keeps no record of earlier calls that could say otherwise."""
    hx, torch, oracle = env
    Hq, Hkv, D = 32, 4, 128
    c = W.AttnConfig(88, "t", 24, Hq, Hkv, D, 256, "x")
    lens = W.rng(88, 1).integers(1, 3000, size=24).astype(np.int32)
    w = W.make_attention_inputs(c, lens=lens, layers=2)
    refs = [oracle.decode_attention(w["q"], w["k"], w["v"], w["block_table"], lens, layer=l) for l in (0, 1)]
    cache = hx.PagedCache(to_dev(w["k"], torch), to_dev(w["v"], torch))
    qd = to_dev(w["q"], torch)
    bt, sl = torch.from_numpy(w["block_table"]).cuda(), torch.from_numpy(lens).cuda()
    mx = int(lens.max())
    wsb = hx.decode_attention_workspace_bytes(24, Hq, Hkv, D, mx)
    ws = torch.zeros(wsb, dtype=torch.uint8, device="cuda")
    kw = dict(q_heads=Hq, block_table=bt, block_table_stride=bt.shape[1], seq_lens=sl, batch=24, max_seq_len=mx, workspace=ws,
              workspace_bytes=wsb)
    okw = dict(kw, behind_ingest=0)
    empty = torch.zeros(1, dtype=torch.int32, device="cuda")
    if True:
        outs = [torch.full_like(qd, float("nan")) for _ in range(6)]
        for j in range(0, 6, 2):                             # six launches back to back, alternating layers
            hx.decode_attention_overlapped(outs[j], qd, cache, layer=0, **okw)
            hx.decode_attention_overlapped(outs[j + 1], qd, cache, layer=1, **okw)
        torch.cuda.synchronize()
        for j, o in enumerate(outs):
            max_abs, rel = attn_errors(o.cpu().numpy(), refs[j % 2])
            assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (j, max_abs, rel)
        for j in range(2, 6):                                # same table, same inputs -> same bits
            assert torch.equal(outs[j].view(torch.int16), outs[j % 2].view(torch.int16)), j
        # an ingest of an empty batch launches nothing: the call behind it follows whatever ran before
        out = torch.full_like(qd, float("nan"))
        hx.decode_attention(outs[0], qd, cache, layer=1, **kw)
        hx.kv_ingest([empty.view(torch.float16)] * 2, [empty.view(torch.float16)] * 2, layers=1, heads=Hkv, head_dim=D, src_tp=2,
                     dst_tp=1, dst_rank=0, dst=cache, block_table=empty, block_table_stride=1, cu_seqlens=empty, seq_lens=empty,
                     batch=0, total_tokens=0, max_seq_len=0)
        hx.decode_attention_overlapped(out, qd, cache, layer=0, **okw)
        torch.cuda.synchronize()
        max_abs, rel = attn_errors(out.cpu().numpy(), refs[0])
        assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (max_abs, rel)


def _chain_setup(hx, torch, oracle, cfg_id, B, Hq, Hkv, D, L, hi):
    lens = W.rng(cfg_id, 1).integers(1, hi, size=B).astype(np.int32)
    lens[3] = 0                                                  # an empty context in the chain (reading S11)
    c = W.AttnConfig(cfg_id, "chain", B, Hq, Hkv, D, (hi + 15) // 16, "x")
    w = W.make_attention_inputs(c, lens=lens, layers=L)
    cache = hx.PagedCache(to_dev(w["k"], torch), to_dev(w["v"], torch))
    bt, sl = torch.from_numpy(w["block_table"]).cuda(), torch.from_numpy(lens).cuda()
    mx = int(lens.max())
    wsb = hx.decode_attention_workspace_bytes(B, Hq, Hkv, D, mx)
    ws = torch.zeros(wsb, dtype=torch.uint8, device="cuda")
    plan = torch.empty(hx.decode_plan_bytes(B, Hkv, mx), dtype=torch.uint8, device="cuda")
    hx.decode_plan(plan, cache, q_heads=Hq, block_table=bt, block_table_stride=bt.shape[1], seq_lens=sl, batch=B, max_seq_len=mx)
    qs = [W.draw_fp16_normal((B, Hq, D), cfg_id, 5, l) for l in range(L)]
    kw = dict(q_heads=Hq, plan=plan, batch=B, max_seq_len=mx, workspace=ws, workspace_bytes=wsb)
    return w, lens, cache, qs, kw


@pytest.mark.parametrize("ready", [1, 0])
def test_chained_layer_calls_equal_plain_planned_calls_bit_for_bit(env, ready):
    """hx_decode_attention_chained: the layer calls of a step launched as programmatic dependents of one another,
    sharing ONE workspace (partial slots, arrival counters).  inputs_ready = 1 lets call n+1 stream its first ranges
    while call n's last warps still merge, so every write of n+1 must wait for n: each layer's output must equal the
    plain planned call's bit for bit and the oracle within tolerance, over several repetitions of a 12-call chain."""
    hx, torch, oracle = env
    B, Hq, Hkv, D, L = 48, 32, 4, 128, 6
    w, lens, cache, qs, kw = _chain_setup(hx, torch, oracle, 91, B, Hq, Hkv, D, L, 2500)
    qd = [to_dev(q, torch) for q in qs]
    base = []
    for l in range(L):
        o = torch.full_like(qd[l], float("nan"))
        hx.decode_attention_planned(o, qd[l], cache, layer=l, **kw)
        torch.cuda.synchronize()
        base.append(o)
        ref = oracle.decode_attention(qs[l], w["k"], w["v"], w["block_table"], lens, layer=l)
        max_abs, rel = attn_errors(o.cpu().numpy(), ref)
        assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (l, max_abs, rel)
        assert (o[3] == 0).all()
    for rep in range(5):
        outs = [torch.full_like(qd[0], float("nan")) for _ in range(2 * L)]
        torch.cuda.synchronize()
        for j in range(2 * L):                               # nothing between the launches: they chain
            hx.decode_attention_chained(outs[j], qd[j % L], cache, layer=j % L, inputs_ready=ready, **kw)
        torch.cuda.synchronize()
        for j in range(2 * L):
            assert torch.equal(outs[j].view(torch.int16), base[j % L].view(torch.int16)), (ready, rep, j)


def test_chained_calls_sharing_one_output_buffer_and_behind_a_producer_kernel(env):
    """(a) inputs_ready = 1 with every call writing the SAME `out`: call n's late rows must not land over call n+1's, so
    after the chain `out` holds the last call's result exactly.  (b) inputs_ready = 0 directly behind the kernel that
    PRODUCES q (a device copy into q's buffer): the call must see the new q, whatever it overlapped."""
    hx, torch, oracle = env
    B, Hq, Hkv, D, L = 64, 16, 2, 128, 4
    w, lens, cache, qs, kw = _chain_setup(hx, torch, oracle, 92, B, Hq, Hkv, D, L, 1200)
    qd = [to_dev(q, torch) for q in qs]
    base = []
    for l in range(L):
        o = torch.full_like(qd[l], float("nan"))
        hx.decode_attention_planned(o, qd[l], cache, layer=l, **kw)
        base.append(o)
    torch.cuda.synchronize()
    for rep in range(5):
        out = torch.full_like(qd[0], float("nan"))
        n = 9 + rep
        for j in range(n):
            hx.decode_attention_chained(out, qd[j % L], cache, layer=j % L, inputs_ready=1, **kw)
        torch.cuda.synchronize()
        assert torch.equal(out.view(torch.int16), base[(n - 1) % L].view(torch.int16)), rep
    # (b): q arrives by a kernel enqueued directly before the call
    big = [q.repeat(64, 1, 1) for q in qd]                   # a copy long enough to still run when the next launch is ready
    qbuf = torch.zeros_like(big[0])
    for rep in range(3):
        outs = []
        for l in range(L):
            qbuf.copy_(big[l])                               # producer kernel (writes the q the next call reads)
            o = torch.full_like(qd[0], float("nan"))
            hx.decode_attention_chained(o, qbuf, cache, layer=l, inputs_ready=0, **kw)
            outs.append(o)
        torch.cuda.synchronize()
        for l in range(L):
            assert torch.equal(outs[l].view(torch.int16), base[l].view(torch.int16)), (rep, l)


def _fused_step_case(env, heads, S, R, q_rank, D, ilens, layers, seed, alens=(33, 100, 1, 700, 16), ing_layers=None,
                     pinned_src=False, expect_fused=None):
    """One hx_decode_step(overlap_ingest=1): the handoff (tile mover inside the attention kernel, handoff_tiles.cuh) lands
    in pages [0, P) of a sentinel-filled cache while the attention reads an active batch living in pages [P, P + Pa).
    Cache bit-exact against the oracle's ingest (sentinels intact), attention within tolerance."""
    hx, torch, oracle = env
    hd = heads // R
    G = 2
    c = W.IngestConfig(93, "fused", layers, heads, D, S, R, len(ilens), "x")
    w = W.make_ingest_inputs(c, lens=np.asarray(ilens, dtype=np.int32), bits=True, seed_extra=seed)
    P = w["num_pages"]
    alens = np.asarray(alens, dtype=np.int32)
    apages = W.pages_for(alens)
    Pa = int(apages.sum())
    abt = np.full((len(alens), int(apages.max())), -1, dtype=np.int32)
    perm = P + W.rng(93, 7, seed).permutation(Pa).astype(np.int32)
    o = 0
    for i, n in enumerate(apages):
        abt[i, :n] = perm[o:o + n]
        o += n
    k0 = np.full((layers, P + Pa, hd, 16, D), 0xDEAD, dtype=np.uint16)
    v0 = np.full_like(k0, 0xDEAD)
    k0[:, P:] = W.draw_fp16_normal((layers, Pa, hd, 16, D), 93, 8, seed).view(np.uint16)
    v0[:, P:] = W.draw_fp16_normal((layers, Pa, hd, 16, D), 93, 9, seed).view(np.uint16)
    q = W.draw_fp16_normal((len(alens), hd * G, D), 93, 10, seed)
    layer_a = layers - 1
    ref = oracle.decode_attention(q, k0.view(np.float16), v0.view(np.float16), abt, alens, layer=layer_a)
    ek, ev = k0.copy(), v0.copy()
    if ing_layers is None:
        ing_layers = layers
    if ing_layers > 0:                                     # ing_layers == 0: a handoff of no layers changes nothing
        oracle.kv_ingest(w["src_k"], w["src_v"], ek, ev, heads=heads, src_tp=S, dst_tp=R, dst_rank=q_rank, block_table=w["block_table"],
                         cu_seqlens=w["cu_seqlens"], seq_lens=w["seq_lens"])
    cache = hx.PagedCache(to_dev(k0, torch), to_dev(v0, torch))
    qd = to_dev(q, torch)
    out = torch.full_like(qd, float("nan"))
    mx = int(alens.max())
    wsb = hx.decode_attention_workspace_bytes(len(alens), hd * G, hd, D, mx)
    ws = torch.zeros(wsb, dtype=torch.uint8, device="cuda")
    ibt = torch.from_numpy(w["block_table"]).cuda()
    if pinned_src:       # pull mode (F2): the shards stay in pinned host memory, the GPU fetches them over the link
        place = lambda a: torch.from_numpy(a.view(np.int16)).pin_memory()
    else:
        place = lambda a: to_dev(a, torch)
    step = hx.DecodeStep(out=out, q=qd, cache=cache, layer=layer_a, q_heads=hd * G, block_table=torch.from_numpy(abt).cuda(),
                         block_table_stride=abt.shape[1], seq_lens=torch.from_numpy(alens).cuda(), batch=len(alens), max_seq_len=mx,
                         sm_scale=0.0, workspace=ws, workspace_bytes=wsb, src_k=[place(a) for a in w["src_k"]],
                         src_v=[place(a) for a in w["src_v"]], ing_layers=ing_layers, heads=heads, src_tp=S, dst_tp=R,
                         dst_rank=q_rank, ing_block_table=ibt, ing_block_table_stride=ibt.shape[1],
                         ing_cu_seqlens=torch.from_numpy(w["cu_seqlens"]).cuda(), ing_seq_lens=torch.from_numpy(w["seq_lens"]).cuda(),
                         ing_batch=len(ilens), ing_total_tokens=w["total_tokens"], ing_max_seq_len=int(max(ilens)), overlap_ingest=1)
    if expect_fused is not None:
        assert step.is_fused() == expect_fused, (heads, S, R, q_rank, D)
    for rep in range(2):                                   # twice: the kernel must leave its counters at zero
        step()
        k_after, v_after = cache.k.clone(), cache.v.clone()     # ordered after the one kernel that did both
        torch.cuda.synchronize()
        assert np.array_equal(dev_u16(k_after), ek), (heads, S, R, q_rank, D, rep)
        assert np.array_equal(dev_u16(v_after), ev), (heads, S, R, q_rank, D, rep)
        max_abs, rel = attn_errors(out.cpu().numpy(), ref)
        assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (heads, S, R, q_rank, D, rep, max_abs, rel)
    assert int(ws.view(torch.int32)[-4:].abs().sum()) == 0          # the two handoff counters are back at zero


@pytest.mark.parametrize("S", [1, 2, 4, 8])
@pytest.mark.parametrize("R", [1, 2, 4, 8])
@pytest.mark.parametrize("D", [64, 128])
def test_fused_step_handoff_tp_sweep_bit_exact(env, S, R, D):
    """Rows A2 + A3 as the fused step performs them (TMA tensor load of 16 token rows -> one bulk store per (page, head)
    tile): every (source TP, destination TP) pair, both head sizes, page-boundary prompt lengths, an empty prompt."""
    ilens = [1, 15, 16, 17, 31, 32, 33, 255, 256, 257, 0, 5]
    for q_rank in sorted({0, R - 1}):
        _fused_step_case(env, 8, S, R, q_rank, D, ilens, layers=3, seed=S * 100 + R * 10 + D + q_rank)


def test_fused_step_handoff_odd_heads_and_one_big_prompt(env):
    for heads, S, R in [(14, 2, 7), (56, 4, 4), (6, 3, 2), (12, 4, 2)]:
        _fused_step_case(env, heads, S, R, R - 1, 128, [40, 3, 129], layers=2, seed=heads)
    _fused_step_case(env, 8, 4, 1, 0, 128, [4099], layers=1, seed=5, alens=(900, 2000, 64, 3100, 31, 500, 7, 2048))


def test_fused_step_with_an_empty_handoff(env):
    """hx_decode_step(overlap_ingest=1) whose handoff moves nothing - every new prompt empty, or zero layers - is valid
    (hx_kv_ingest accepts both as no-ops): the cache keeps every bit, the attention result is unaffected."""
    _fused_step_case(env, 8, 2, 2, 1, 128, [0, 0, 0], layers=2, seed=11)
    _fused_step_case(env, 8, 4, 1, 0, 64, [0], layers=1, seed=12)
    _fused_step_case(env, 8, 2, 4, 3, 128, [40, 3, 129], layers=2, seed=13, ing_layers=0, expect_fused=False)


def test_fused_step_pulls_the_handoff_from_pinned_host_memory(env):
    """F2 inside the fused step: the source shards are NOT in this GPU's HBM (pinned host memory here, reached over PCIe;
    a peer GPU's memory is reached the same way over NVLink, tests/test_gpu_peer.py).  The step must still be the ONE
    fused kernel - the copy engines load each (page, head) tile through a tensor map over the remote shard and store it
    into its page - with the cache bit-exact and the attention within tolerance."""
    ilens = [1, 15, 16, 17, 31, 32, 33, 255, 256, 257, 0, 5]
    _fused_step_case(env, 8, 4, 2, 1, 128, ilens, layers=3, seed=31, pinned_src=True, expect_fused=True)
    _fused_step_case(env, 8, 1, 1, 0, 64, ilens, layers=2, seed=32, pinned_src=True, expect_fused=True)
    _fused_step_case(env, 8, 2, 8, 5, 128, [40, 3, 129], layers=2, seed=33, pinned_src=True, expect_fused=True)
    # and the ordinary case reports itself as fused, the 2100-request one (below) as not
    _fused_step_case(env, 8, 2, 2, 0, 128, [40, 3, 129], layers=2, seed=34, expect_fused=True)


def test_step_with_more_than_2048_requests_runs_in_order(env):
    """hx_decode_step(overlap_ingest=1) with an active batch above what one attention launch covers (2048): the fused
    kernel cannot take it, the library runs ingest then attention (two launches for the 2100 requests) in order.  Same
    checks as the fused case: cache bit-exact against the oracle's ingest, attention within tolerance."""
    alens = W.rng(93, 21).integers(0, 80, size=2100).astype(np.int32)
    alens[[0, 2047, 2048, 2099]] = [1, 79, 33, 16]
    _fused_step_case(env, 8, 2, 2, 1, 128, [40, 3, 129, 0, 16], layers=2, seed=21, alens=alens, expect_fused=False)


def test_layer_loop_of_chained_calls_in_a_cuda_graph(env):
    """A decode step's layer loop — one hx_decode_plan, then one hx_decode_attention_chained per layer — captured once in
    a CUDA graph (the programmatic launches become graph edges) and replayed with new queries: every layer of every
    replay must equal the plain planned call bit for bit."""
    hx, torch, oracle = env
    B, Hq, Hkv, D, L = 32, 32, 4, 128, 4
    w, lens, cache, qs, kw = _chain_setup(hx, torch, oracle, 94, B, Hq, Hkv, D, L, 1500)
    qbuf = [torch.empty((B, Hq, D), dtype=torch.float16, device="cuda") for _ in range(L)]
    outs = [torch.empty((B, Hq, D), dtype=torch.float16, device="cuda") for _ in range(L)]

    def loop():
        for l in range(L):
            hx.decode_attention_chained(outs[l], qbuf[l], cache, layer=l, inputs_ready=1, **kw)

    for l in range(L):
        qbuf[l].copy_(to_dev(qs[l], torch))
    loop()                                              # warm-up outside capture (function attributes, tensor maps)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        loop()
    for rep in range(3):
        qrep = [W.draw_fp16_normal((B, Hq, D), 94, 20 + rep, l) for l in range(L)]
        for l in range(L):
            qbuf[l].copy_(to_dev(qrep[l], torch))
            outs[l].fill_(float("nan"))
        g.replay()
        torch.cuda.synchronize()
        for l in range(L):
            base = torch.full_like(outs[l], float("nan"))
            hx.decode_attention_planned(base, qbuf[l], cache, layer=l, **kw)
            torch.cuda.synchronize()
            assert torch.equal(outs[l].view(torch.int16), base.view(torch.int16)), (rep, l)
            if rep == 0:
                ref = oracle.decode_attention(qrep[l], w["k"], w["v"], w["block_table"], lens, layer=l)
                max_abs, rel = attn_errors(outs[l].cpu().numpy(), ref)
                assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (l, max_abs, rel)
