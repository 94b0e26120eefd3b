"""Full-size BASELINE.json configs on the GPU, in the launch configuration bench.py times.
Attention: every output row of a sample of requests (shortest, longest, a spread) is computed by
the oracle one by one and compared; plus finite-ness of all rows.  Ingest: one whole layer of
config 4 compared bit for bit per destination rank, plus untouched-sentinel checks."""
import numpy as np
import pytest

import workloads as W
from helpers import MAX_ABS_TOL, REL_L2_TOL, attn_errors, oracle_ingest, run_gpu_attention, run_gpu_ingest

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


@pytest.mark.parametrize("name,nsample", [("opt30b_tp4", 12), ("llama70b_tp2", 16), ("llama70b_tp1", 10)])
def test_attention_full_config_sampled_rows(env, name, nsample):
    hx, torch, oracle = env
    c = W.CONFIGS[name]
    w = W.make_attention_inputs(c)
    got = run_gpu_attention(hx, torch, w)
    assert np.isfinite(got.astype(np.float32)).all()
    lens = w["seq_lens"]
    order = np.argsort(lens)
    pick = sorted(set(order[np.linspace(0, len(order) - 1, nsample).astype(int)].tolist()))
    ref = oracle.decode_attention(np.ascontiguousarray(w["q"][pick]), w["k"], w["v"],
                                  np.ascontiguousarray(w["block_table"][pick]), np.ascontiguousarray(lens[pick]))
    max_abs, rel_l2 = attn_errors(got[pick], ref)
    assert max_abs <= MAX_ABS_TOL and rel_l2 <= REL_L2_TOL, (name, max_abs, rel_l2)
    # worst single request also inside the relative bound
    for j, i in enumerate(pick):
        _, r = attn_errors(got[i], ref[j])
        assert r <= REL_L2_TOL, (name, i, r)


def test_ingest_config4_layers_bit_exact(env):
    hx, torch, oracle = env
    c = W.CONFIGS["llama70b_ingest"]
    w = W.make_ingest_inputs(c, layers=2)          # same lengths / TP pair / placement as the 80-layer run
    for q in range(c.dst_tp):
        dk, dv = run_gpu_ingest(hx, torch, w, q)
        ok, ov = oracle_ingest(oracle, w, q)
        assert np.array_equal(dk, ok) and np.array_equal(dv, ov)


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
    rows one by one — a row at position p is the one-query-token case of a context cut at p + 1 — and every
    output must be finite."""
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
        assert r <= 2 * REL_L2_TOL, (int(reqs[j]), int(poss[j]), r)
