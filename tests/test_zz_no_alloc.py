"""hx_decode_attention_noalloc: decode attention for callers that cannot allocate device memory.

Why the entry point exists.  hx_decode_attention asks its caller for a ~17 MB workspace.  Three kinds of caller cannot
produce one: a decode replica whose paged KV cache was sized at start-up to fill the GPU (a later cudaMalloc fails); an
attention backend plugged into another serving engine, which is handed tensors but not the engine's allocator (and a
raw cudaMalloc from inside the step loop would synchronise the whole device mid-step); and code that runs while
another thread has a stream capture open, where cudaMalloc is forbidden.  For them libhx carries a fixed 20 MiB scratch
array in its own device image; the call takes no workspace and allocates nothing.

What the tests below hold the entry point to:
  * its result equals the workspace path's (same kernel, so bit for bit; and within the suite's attention tolerance
    of the float64 oracle) on calls made one after another.  The array is shared and never re-zeroed by the caller, and
    the counters' position inside it depends on the shape, so the second call's counters land in what the first call
    used for partial results: the sequence below is chosen to make exactly that happen;
  * a shape that needs more scratch than the array holds is refused on the host, with both sizes in the message,
    before any CUDA call (this half needs no GPU and runs in the CPU suite).

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests proper.  The GPU test passes alone in a fresh process and after the rest of the suite (the scratch holds
whatever earlier launches of this process left there either way - none of the other tests touches it)."""
import ctypes as C

import numpy as np
import pytest

import workloads as W
from helpers import MAX_ABS_TOL, REL_L2_TOL, attn_errors, to_dev


def test_noalloc_is_exported_and_refuses_shapes_beyond_the_builtin_scratch():
    """Host-side half: the limit.  Group size 16 at head_dim 128 needs ~34 MB; the built-in array is 20 MiB."""
    import paper_2502_07903_b200 as hx
    from paper_2502_07903_b200 import binding as B
    assert hasattr(hx.lib(), "hx_decode_attention_noalloc")
    assert hx.NOALLOC_SCRATCH_BYTES == 20 * 1024 * 1024
    fits = hx.decode_attention_workspace_bytes(8, 64, 8, 128, 4096)            # LLaMA-2-70B TP=1: G = 8
    too_big = hx.decode_attention_workspace_bytes(8, 16, 1, 128, 4096)         # G = 16, head_dim 128
    assert 0 < fits <= hx.NOALLOC_SCRATCH_BYTES < too_big

    class FakeCache:                                    # never dereferenced: the refusal comes before any CUDA call
        def __init__(self, kv_heads, head_dim):
            self.c = B._CCache(4096, 8192, 1, 64, kv_heads, 16, head_dim)
            self.ref = C.byref(self.c)

    kw = dict(layer=0, block_table=4096, block_table_stride=256, seq_lens=4096, batch=8, max_seq_len=4096, stream=0)
    with pytest.raises(hx.HxError) as e:
        hx.decode_attention_noalloc(4096, 4096, FakeCache(1, 128), q_heads=16, **kw)
    assert e.value.status == B.HX_ERR_WORKSPACE
    assert str(too_big) in str(e.value) and str(hx.NOALLOC_SCRATCH_BYTES) in str(e.value)
    # the ordinary argument checks of hx_decode_attention still come first
    with pytest.raises(hx.HxError) as e:
        hx.decode_attention_noalloc(4096, 4096, FakeCache(3, 128), q_heads=16, **kw)     # 16 % 3 != 0
    assert e.value.status == B.HX_ERR_INVALID_ARG
    # an empty batch is a no-op, as in hx_decode_attention
    hx.decode_attention_noalloc(0, 0, FakeCache(1, 128), q_heads=16, **dict(kw, batch=0))


def _case(seed, B_, Hq, Hkv, D, lens):
    c = W.AttnConfig(seed, "noalloc", B_, Hq, Hkv, D, 4096, "x")
    return W.make_attention_inputs(c, lens=np.asarray(lens, dtype=np.int32), seed_extra=seed)


@pytest.mark.gpu
def test_noalloc_matches_workspace_path_on_consecutive_calls():
    """Three calls in a row on one stream, none of them preceded by any clearing from the caller's side:
    a head_dim-128 GQA batch long enough that every worker leaves partial results all over the scratch, then a
    head_dim-64 batch whose counters sit in the middle of those partials, then the first shape again with another q.
    Each result is compared with hx_decode_attention on a caller-allocated, zero-filled workspace."""
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (no CPU fallback exists)")
    import oracle
    import paper_2502_07903_b200 as hx
    oracle.build()

    long_lens = [4000, 3777, 3500, 3333, 3000, 2999, 2500, 2048, 4096, 3900, 3100, 2700, 1, 17, 0, 1000]
    cases = [
        _case(301, 16, 32, 4, 128, long_lens),                              # G = 8, D = 128: ~12 000 tiles, every pair split
        _case(302, 12, 8, 2, 64, [2000, 1500, 1000, 33, 16, 15, 0, 1, 2500, 3000, 700, 64]),   # G = 4, D = 64
        _case(303, 16, 32, 4, 128, long_lens[::-1]),
    ]
    dev = []
    for w in cases:
        cache = hx.PagedCache(to_dev(w["k"], torch), to_dev(w["v"], torch))
        qd = to_dev(w["q"], torch)
        bt = torch.from_numpy(w["block_table"]).cuda()
        sl = torch.from_numpy(np.ascontiguousarray(w["seq_lens"], dtype=np.int32)).cuda()
        B_, Hq, D = w["q"].shape
        kw = dict(layer=0, q_heads=Hq, block_table=bt, block_table_stride=bt.shape[1], seq_lens=sl, batch=B_,
                  max_seq_len=int(w["seq_lens"].max()))
        # the existing path: a workspace the caller allocates and zero-fills
        ws_bytes = hx.decode_attention_workspace_bytes(B_, Hq, cache.k.shape[2], D, kw["max_seq_len"])
        assert ws_bytes <= hx.NOALLOC_SCRATCH_BYTES
        ws = torch.zeros(ws_bytes, dtype=torch.uint8, device="cuda")
        want = torch.full_like(qd, float("nan"))
        hx.decode_attention(want, qd, cache, workspace=ws, workspace_bytes=ws_bytes, **kw)
        dev.append((cache, qd, kw, want, bt, sl))
    torch.cuda.synchronize()

    # everything the no-alloc calls need exists now; from here on this test allocates nothing on the device
    gots = [torch.full_like(d[1], float("nan")) for d in dev]
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    for (cache, qd, kw, _, _, _), got in zip(dev, gots):                     # back to back, same stream, no sync between
        hx.decode_attention_noalloc(got, qd, cache, **kw)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before

    for i, (w, d, got) in enumerate(zip(cases, dev, gots)):
        g, want = got.cpu().numpy(), d[3].cpu().numpy()
        assert np.isfinite(g.astype(np.float32)).all(), i
        ref = oracle.decode_attention(w["q"], w["k"], w["v"], w["block_table"], w["seq_lens"])
        for name, other in (("workspace path", want.astype(np.float64)), ("oracle", ref)):
            max_abs, rel_l2 = attn_errors(g, other)
            assert max_abs <= MAX_ABS_TOL and rel_l2 <= REL_L2_TOL, (i, name, max_abs, rel_l2)
        # same kernel, same work partition, same merge order: the scratch's address must not show in the bits
        assert np.array_equal(g.view(np.uint16), want.view(np.uint16)), i
        assert (g[np.asarray(w["seq_lens"]) == 0] == 0).all(), i              # empty requests: zero rows
