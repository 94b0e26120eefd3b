"""GPU parity for hx_prefill_attention: the tcgen05 kernel against the float64
oracle (causal paged attention of the last q_lens[i] tokens), north_star tolerances."""
import numpy as np
import pytest

import workloads as W
from helpers import MAX_ABS_TOL, REL_L2_TOL, attn_errors, to_dev

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


def run_prefill(env, cfgno, Hq, Hkv, lens, qlens, layers=1, layer=0, poison=False, sm_scale=0.0, D=128):
    hx, torch, oracle = env
    lens = np.asarray(lens, dtype=np.int32)
    qlens = np.asarray(qlens, dtype=np.int32)
    c = W.AttnConfig(cfgno, "t", len(lens), Hq, Hkv, D, 8, "x")
    w = W.make_attention_inputs(c, lens=lens, layers=layers)
    Tq = int(qlens.sum())
    q = W.draw_fp16_normal((Tq, Hq, D), cfgno, 40)
    k, v = w["k"], w["v"]
    if poison:                                   # slots past the context end and unowned pages: NaN / Inf
        kb, vb = k.view(np.uint16).copy(), v.view(np.uint16).copy()
        owned = np.zeros((w["num_pages"], 16), dtype=bool)
        for i, n in enumerate(lens):
            t = np.arange(n)
            owned[w["block_table"][i, t // 16], t % 16] = True
        kb[:].transpose(0, 1, 3, 2, 4)[:, ~owned] = 0x7E00
        vb[:].transpose(0, 1, 3, 2, 4)[:, ~owned] = 0x7C00
        k, v = kb.view(np.float16), vb.view(np.float16)
    ref = oracle.prefill_attention(q, k, v, w["block_table"], lens, qlens, layer=layer,
                                   sm_scale=sm_scale if sm_scale > 0 else None)
    cache = hx.PagedCache(to_dev(k, torch), to_dev(v, torch))
    cu = np.zeros(len(lens) + 1, dtype=np.int32)
    np.cumsum(qlens, out=cu[1:])
    qd = to_dev(q, torch)
    out = torch.full_like(qd, float("nan"))
    bt = torch.from_numpy(w["block_table"]).cuda()
    hx.prefill_attention(out, qd, cache, layer=layer, q_heads=Hq, block_table=bt, block_table_stride=bt.shape[1],
                         seq_lens=torch.from_numpy(lens).cuda(), q_lens=torch.from_numpy(qlens).cuda(),
                         cu_q_lens=torch.from_numpy(cu).cuda(), batch=len(lens), total_q_tokens=Tq,
                         max_q_len=int(qlens.max(initial=0)), max_seq_len=int(lens.max(initial=0)), sm_scale=sm_scale)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert np.isfinite(got.astype(np.float32)).all()
    max_abs, rel = attn_errors(got, ref)
    assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (max_abs, rel)
    return got, ref


@pytest.mark.parametrize("G,Hkv", [(8, 1), (1, 2), (4, 2), (16, 1), (2, 1)])
def test_prefill_whole_prompts_page_and_tile_boundaries(env, G, Hkv):
    lens = [1, 15, 16, 17, 127, 128, 129, 255, 257, 300]
    run_prefill(env, 60 + G, G * Hkv, Hkv, lens, lens)


def test_prefill_llama70b_shape_long_prompt(env):
    run_prefill(env, 70, 16, 2, [1000, 700], [1000, 700])          # G = 8, several kv tiles per q tile


def test_prefill_chunked_and_decode_like_and_empty(env):
    lens = [300, 64, 200, 17, 129]
    qlens = [44, 1, 200, 0, 128]
    run_prefill(env, 71, 8, 1, lens, qlens)


def test_prefill_layer_and_scale_and_poison(env):
    run_prefill(env, 72, 8, 1, [100, 260, 31], [100, 260, 31], layers=3, layer=2, sm_scale=0.05)
    run_prefill(env, 73, 8, 1, [100, 260, 31, 130], [100, 60, 31, 130], poison=True)


def test_prefill_one_query_token_matches_decode_kernel(env):
    """q_lens = 1: the tensor-memory kernel and the streaming decode kernel answer the same question."""
    hx, torch, oracle = env
    lens = np.array([1, 16, 100, 513, 129], dtype=np.int32)
    got, ref = run_prefill(env, 74, 8, 1, lens, np.ones(5, dtype=np.int32))
    ref_dec = None
    c = W.AttnConfig(74, "t", 5, 8, 1, 128, 8, "x")
    w = W.make_attention_inputs(c, lens=lens)
    q = W.draw_fp16_normal((5, 8, 128), 74, 40)
    ref_dec = oracle.decode_attention(q, w["k"], w["v"], w["block_table"], lens)
    np.testing.assert_allclose(ref, ref_dec, atol=1e-13)


def test_prefill_chunk_on_a_long_context_and_wide_group(env):
    """A 300-token chunk at the end of a 5000-token context (most kv tiles carry no mask at all), and a
    G = 16 group (8 tokens x 16 heads per row tile)."""
    run_prefill(env, 75, 8, 1, [5000, 4097], [300, 1])
    run_prefill(env, 76, 16, 1, [700, 129, 33], [700, 129, 33])


@pytest.mark.parametrize("G,Hkv", [(1, 4), (8, 1), (4, 2)])
def test_prefill_head_dim_64(env, G, Hkv):
    """head_dim 64 (the shape of BASELINE.json configs[0]): one 64-wide operand region instead of two."""
    lens = [17, 64, 100, 255, 129, 300]
    run_prefill(env, 80 + G, G * Hkv, Hkv, lens, lens, D=64)
    run_prefill(env, 84 + G, G * Hkv, Hkv, [300, 64, 200], [44, 1, 200], D=64, poison=True)


@pytest.mark.parametrize("G,Hkv,D", [(1, 4, 128), (8, 2, 128), (2, 3, 64)])
def test_prefill_many_items_per_cta(env, G, Hkv, D):
    """The kernel is persistent: one CTA per SM walks (row-tile pair, request, kv head) items without draining between
    them, two row tiles in lockstep, their output tiles sharing one staged buffer.  Far more items than SMs, with
    everything that changes from one item to the next: prompts shorter than one row tile, requests with no query rows
    (skipped items), a second row tile that exists in one item and not in the next, partial last row tiles (stored row
    by row) between full ones (stored by TMA), chunked prefills, a context that ends inside a kv tile."""
    g = W.rng(90 + G, 3)
    lens = g.integers(1, 1500, size=44).astype(np.int32)
    qlens = lens.copy()
    qlens[::5] = np.minimum(lens[::5], g.integers(0, 200, size=len(lens[::5])))     # chunked / decode-like / empty
    qlens[3], lens[7], qlens[7] = 0, 128, 128
    lens[11], qlens[11] = 1, 1
    run_prefill(env, 90 + G, G * Hkv, Hkv, lens, qlens, poison=True, D=D)


def test_prefill_degenerate_calls_do_not_hang(env):
    """No query rows at all (every item of the persistent walk is skipped), a single one-token request, and q_lens above
    seq_lens (a contract violation that the kernel clamps): each must return, and the valid ones must be right."""
    hx, torch, oracle = env
    lens = np.array([100, 33, 1], dtype=np.int32)
    c = W.AttnConfig(98, "t", 3, 8, 1, 128, 8, "x")
    w = W.make_attention_inputs(c, lens=lens)
    cache = hx.PagedCache(to_dev(w["k"], torch), to_dev(w["v"], torch))
    bt = torch.from_numpy(w["block_table"]).cuda()
    q = W.draw_fp16_normal((141, 8, 128), 98, 40)              # room for the rows of every call below
    qd = to_dev(q, torch)

    def call(qlens, max_q):
        qlens = np.asarray(qlens, dtype=np.int32)
        cu = np.zeros(4, dtype=np.int32)
        np.cumsum(qlens, out=cu[1:])
        out = torch.full_like(qd, float("nan"))
        hx.prefill_attention(out, qd, cache, layer=0, q_heads=8, block_table=bt, block_table_stride=bt.shape[1],
                             seq_lens=torch.from_numpy(lens).cuda(), q_lens=torch.from_numpy(qlens).cuda(),
                             cu_q_lens=torch.from_numpy(cu).cuda(), batch=3, total_q_tokens=141, max_q_len=max_q, max_seq_len=100)
        torch.cuda.synchronize()
        return out.cpu().numpy(), cu

    got, _ = call([0, 0, 0], 1)                                   # nothing to do: nothing written
    assert np.isnan(got.astype(np.float32)).all()
    got, cu = call([0, 0, 1], 1)                                  # one row, one token of context: returns v_0
    ref = oracle.prefill_attention(q[:1], w["k"], w["v"], w["block_table"], lens, np.array([0, 0, 1], dtype=np.int32))
    assert attn_errors(got[:1], ref)[0] <= MAX_ABS_TOL
    got, cu = call([100, 40, 1], 100)                             # q_lens[1] = 40 > seq_lens[1] = 33: clamped to 33 rows, no hang
    ref = oracle.prefill_attention(np.concatenate([q[:100], q[100:133], q[140:141]]), w["k"], w["v"], w["block_table"], lens,
                                   np.array([100, 33, 1], dtype=np.int32))
    max_abs, rel = attn_errors(got[:100], ref[:100])              # request 0 is untouched by the violation
    assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (max_abs, rel)
