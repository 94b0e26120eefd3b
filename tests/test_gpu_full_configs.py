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
