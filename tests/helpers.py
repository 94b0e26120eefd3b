"""Test-side helpers: upload workloads, call the C-ABI through the binding, compare with the oracle."""
import numpy as np


def to_dev(a, torch):
    if a.dtype == np.uint16:
        return torch.from_numpy(a.view(np.int16)).cuda().view(torch.float16)
    if a.dtype == np.float16:
        return torch.from_numpy(a).cuda()
    return torch.from_numpy(a).cuda()


def dev_u16(t):
    return t.cpu().view(__import__("torch").int16).numpy().view(np.uint16)


def run_gpu_attention(hx, torch, w, *, layer=0, sm_scale=0.0, q=None):
    """w: dict from workloads.make_attention_inputs.  Returns fp16 numpy [B][Hq][D]."""
    q_np = w["q"] if q is None else q
    B, Hq, D = q_np.shape
    k, v = to_dev(w["k"], torch), to_dev(w["v"], torch)
    cache = hx.PagedCache(k, v)
    qd = to_dev(q_np, torch)
    out = torch.full_like(qd, float("nan"))
    bt = torch.from_numpy(w["block_table"]).cuda()
    sl = torch.from_numpy(np.ascontiguousarray(w["seq_lens"], dtype=np.int32)).cuda()
    max_len = int(w["seq_lens"].max(initial=0))
    Hkv = k.shape[2]
    ws_bytes = hx.decode_attention_workspace_bytes(B, Hq, Hkv, D, max_len, k.shape[3])
    ws = torch.zeros(max(ws_bytes, 16), dtype=torch.uint8, device="cuda")
    hx.decode_attention(out, qd, cache, layer=layer, q_heads=Hq, block_table=bt,
                        block_table_stride=bt.shape[1], seq_lens=sl, batch=B, max_seq_len=max_len,
                        sm_scale=sm_scale, workspace=ws, workspace_bytes=ws_bytes)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def attn_errors(got_fp16, ref_f64):
    g = got_fp16.astype(np.float64)
    max_abs = float(np.abs(g - ref_f64).max(initial=0.0))
    den = float(np.linalg.norm(ref_f64.ravel()))
    rel_l2 = float(np.linalg.norm((g - ref_f64).ravel()) / den) if den > 0 else 0.0
    return max_abs, rel_l2


# north_star tolerances (fp16 in, fp32 accumulate): max-abs <= 2e-3, relative-L2 <= 1e-3
MAX_ABS_TOL = 2e-3
REL_L2_TOL = 1e-3


def run_gpu_ingest(hx, torch, w, dst_rank, *, sentinel=0xDEAD, gather_back=False):
    """w: dict from workloads.make_ingest_inputs.  Returns (dst_k, dst_v) uint16 numpy; with
    gather_back also the regathered shard lists."""
    L, heads, D, S, R = w["layers"], w["heads"], w["head_dim"], w["src_tp"], w["dst_tp"]
    hd = heads // R
    P, ps = w["num_pages"], w["page_size"]
    sk = [to_dev(a, torch) for a in w["src_k"]]
    sv = [to_dev(a, torch) for a in w["src_v"]]
    shape = (L, P, hd, ps, D)
    fill = np.array([sentinel], dtype=np.uint16).view(np.int16)[0]
    dk = torch.full(shape, int(fill), dtype=torch.int16, device="cuda").view(torch.float16)
    dv = torch.full(shape, int(fill), dtype=torch.int16, device="cuda").view(torch.float16)
    cache = hx.PagedCache(dk, dv)
    bt = torch.from_numpy(w["block_table"]).cuda()
    cu = torch.from_numpy(w["cu_seqlens"]).cuda()
    sl = torch.from_numpy(w["seq_lens"]).cuda()
    kw = dict(layers=L, heads=heads, head_dim=D, src_tp=S, dst_tp=R, dst_rank=dst_rank, dst=cache,
              block_table=bt, block_table_stride=bt.shape[1], cu_seqlens=cu, seq_lens=sl,
              batch=len(w["seq_lens"]), total_tokens=w["total_tokens"],
              max_seq_len=int(w["seq_lens"].max(initial=0)))
    hx.kv_ingest(sk, sv, **kw)
    torch.cuda.synchronize()
    res = (dev_u16(dk), dev_u16(dv))
    if gather_back:
        gk = [torch.full_like(a.view(torch.int16), 0x0BAD).view(torch.float16) for a in sk]
        gv = [torch.full_like(a.view(torch.int16), 0x0BAD).view(torch.float16) for a in sv]
        hx.kv_gather(gk, gv, **kw)
        torch.cuda.synchronize()
        res = res + ([dev_u16(a) for a in gk], [dev_u16(a) for a in gv])
    return res


def oracle_ingest(oracle, w, dst_rank, sentinel=0xDEAD):
    L, heads, D, R = w["layers"], w["heads"], w["head_dim"], w["dst_tp"]
    shape = (L, w["num_pages"], heads // R, w["page_size"], D)
    dk = np.full(shape, sentinel, dtype=np.uint16)
    dv = np.full(shape, sentinel, dtype=np.uint16)
    oracle.kv_ingest(w["src_k"], w["src_v"], dk, dv, heads=heads, src_tp=w["src_tp"], dst_tp=R,
                     dst_rank=dst_rank, block_table=w["block_table"], cu_seqlens=w["cu_seqlens"],
                     seq_lens=w["seq_lens"])
    return dk, dv
