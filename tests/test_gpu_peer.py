"""F2 as SURVEY.md section 8(f) wrote it: the handoff pulled from a PEER GPU's memory over NVLink (PAPER.md:L92 - the GPU that
holds layer j of the prefill replica sends to the GPU that holds layer j of the decode replica; PAPER.md:L110 - asynchronously,
overlapping compute).  Needs two GPUs in one process with peer access; every lease of this project so far had one GPU, so
these tests SKIP there (unmeasured on hardware) and run the day a 2-GPU box appears.  Shards live on
cuda:1, the paged cache and the kernels on cuda:0; nothing is staged: hx_kv_ingest and the fused hx_decode_step read the
shards through peer pointers."""
import numpy as np
import pytest

import workloads as W
from helpers import MAX_ABS_TOL, REL_L2_TOL, attn_errors, dev_u16

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env2():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (no CPU fallback exists)")
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs (peer memory over NVLink)")
    if not torch.cuda.can_device_access_peer(0, 1):
        pytest.skip("cuda:0 cannot access cuda:1 as a peer")
    import oracle
    import paper_2502_07903_b200 as hx
    oracle.build()
    torch.cuda.set_device(0)
    # torch enables peer access between two devices the first time it copies between them
    torch.zeros(1, device="cuda:1").to("cuda:0")
    torch.cuda.synchronize()
    return hx, torch, oracle


def _on_peer(a, torch):
    return torch.from_numpy(a.view(np.int16)).to("cuda:1").view(torch.float16)


def test_ingest_pulls_from_a_peer_gpu(env2):
    hx, torch, oracle = env2
    c = W.IngestConfig(97, "peer", 3, 8, 128, 4, 2, 6, "x")
    lens = np.array([1, 16, 17, 100, 300, 0], dtype=np.int32)
    w = W.make_ingest_inputs(c, lens=lens, bits=True)
    P = w["num_pages"]
    sk, sv = [_on_peer(a, torch) for a in w["src_k"]], [_on_peer(a, torch) for a in w["src_v"]]
    torch.cuda.synchronize("cuda:1")
    bt, cu, sl = (torch.from_numpy(w[k]).cuda() for k in ("block_table", "cu_seqlens", "seq_lens"))
    for qrank in range(2):
        shape = (3, P, 4, 16, 128)
        fill = int(np.array([0xDEAD], dtype=np.uint16).view(np.int16)[0])
        cache = hx.PagedCache(torch.full(shape, fill, dtype=torch.int16, device="cuda:0").view(torch.float16),
                              torch.full(shape, fill, dtype=torch.int16, device="cuda:0").view(torch.float16))
        hx.kv_ingest(sk, sv, layers=3, heads=8, head_dim=128, src_tp=4, dst_tp=2, dst_rank=qrank, dst=cache, block_table=bt,
                     block_table_stride=bt.shape[1], cu_seqlens=cu, seq_lens=sl, batch=len(lens),
                     total_tokens=w["total_tokens"], max_seq_len=int(lens.max()))
        torch.cuda.synchronize()
        ok = np.full(shape, 0xDEAD, dtype=np.uint16)
        ov = ok.copy()
        oracle.kv_ingest(w["src_k"], w["src_v"], ok, ov, heads=8, src_tp=4, dst_tp=2, dst_rank=qrank,
                         block_table=w["block_table"], cu_seqlens=w["cu_seqlens"], seq_lens=lens)
        assert np.array_equal(dev_u16(cache.k), ok) and np.array_equal(dev_u16(cache.v), ov), qrank


def test_fused_step_pulls_the_handoff_from_a_peer_gpu(env2):
    hx, torch, oracle = env2
    heads, S, R, D, layers = 8, 4, 1, 128, 2
    ilens = np.array([1, 15, 16, 17, 255, 256, 257, 0, 5], dtype=np.int32)
    w = W.make_ingest_inputs(W.IngestConfig(96, "peer", layers, heads, D, S, R, len(ilens), "x"), lens=ilens, bits=True)
    P = w["num_pages"]
    alens = np.array([33, 100, 1, 700, 16], dtype=np.int32)
    apages = W.pages_for(alens)
    Pa = int(apages.sum())
    abt = np.full((len(alens), int(apages.max())), -1, dtype=np.int32)
    perm = P + W.rng(96, 7).permutation(Pa).astype(np.int32)
    o = 0
    for i, n in enumerate(apages):
        abt[i, :n] = perm[o:o + n]
        o += n
    k0 = np.full((layers, P + Pa, heads, 16, D), 0xDEAD, dtype=np.uint16)
    v0 = np.full_like(k0, 0xDEAD)
    k0[:, P:] = W.draw_fp16_normal((layers, Pa, heads, 16, D), 96, 8).view(np.uint16)
    v0[:, P:] = W.draw_fp16_normal((layers, Pa, heads, 16, D), 96, 9).view(np.uint16)
    q = W.draw_fp16_normal((len(alens), heads * 2, D), 96, 10)
    ref = oracle.decode_attention(q, k0.view(np.float16), v0.view(np.float16), abt, alens, layer=1)
    ek, ev = k0.copy(), v0.copy()
    oracle.kv_ingest(w["src_k"], w["src_v"], ek, ev, heads=heads, src_tp=S, dst_tp=R, dst_rank=0, block_table=w["block_table"],
                     cu_seqlens=w["cu_seqlens"], seq_lens=w["seq_lens"])
    dev0 = lambda a: torch.from_numpy(a.view(np.int16)).to("cuda:0").view(torch.float16)
    cache = hx.PagedCache(dev0(k0), dev0(v0))
    qd = torch.from_numpy(q).to("cuda:0")
    out = torch.full_like(qd, float("nan"))
    wsb = hx.decode_attention_workspace_bytes(len(alens), heads * 2, heads, D, 700)
    ws = torch.zeros(wsb, dtype=torch.uint8, device="cuda:0")
    ibt = torch.from_numpy(w["block_table"]).cuda()
    step = hx.DecodeStep(out=out, q=qd, cache=cache, layer=1, q_heads=heads * 2, block_table=torch.from_numpy(abt).cuda(),
                         block_table_stride=abt.shape[1], seq_lens=torch.from_numpy(alens).cuda(), batch=len(alens), max_seq_len=700,
                         sm_scale=0.0, workspace=ws, workspace_bytes=wsb, src_k=[_on_peer(a, torch) for a in w["src_k"]],
                         src_v=[_on_peer(a, torch) for a in w["src_v"]], ing_layers=layers, heads=heads, src_tp=S, dst_tp=R,
                         dst_rank=0, ing_block_table=ibt, ing_block_table_stride=ibt.shape[1],
                         ing_cu_seqlens=torch.from_numpy(w["cu_seqlens"]).cuda(), ing_seq_lens=torch.from_numpy(w["seq_lens"]).cuda(),
                         ing_batch=len(ilens), ing_total_tokens=w["total_tokens"], ing_max_seq_len=int(ilens.max()), overlap_ingest=1)
    torch.cuda.synchronize("cuda:1")
    assert step.is_fused()
    step()
    torch.cuda.synchronize()
    assert np.array_equal(dev_u16(cache.k), ek) and np.array_equal(dev_u16(cache.v), ev)
    max_abs, rel = attn_errors(out.cpu().numpy(), ref)
    assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (max_abs, rel)
