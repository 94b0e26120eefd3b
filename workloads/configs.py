"""The five BASELINE.json configs as seeded numpy inputs. No method arithmetic."""
from __future__ import annotations

import dataclasses
import math
from concurrent.futures import ThreadPoolExecutor

import numpy as np

PAGE_SIZE = 16
SEED = 0

# rng streams
S_LEN, S_Q, S_K, S_V, S_PERM, S_SHUFFLE, S_ILEN, S_SRCK, S_SRCV = range(9)


def rng(cfg: int, stream: int, *extra: int) -> np.random.Generator:
    return np.random.default_rng(np.random.SeedSequence([SEED, cfg, stream, *extra]))


@dataclasses.dataclass(frozen=True)
class AttnConfig:
    cfg: int
    name: str
    batch: int
    q_heads: int        # local (per decode-TP rank) query heads
    kv_heads: int       # local kv heads
    head_dim: int
    max_pages: int      # block-table stride (max pages per request)
    lengths: str        # recipe name


@dataclasses.dataclass(frozen=True)
class IngestConfig:
    cfg: int
    name: str
    layers: int
    heads: int          # GLOBAL kv heads
    head_dim: int
    src_tp: int
    dst_tp: int
    prompts: int
    lengths: str


CONFIGS = {
    # cfg 1: tiny oracle case (BASELINE.json configs[0])
    "tiny": AttnConfig(1, "tiny", 4, 4, 4, 64, 16, "tiny"),
    "tiny_ingest": IngestConfig(1, "tiny_ingest", 1, 4, 64, 2, 1, 4, "tiny"),
    # cfg 2: OPT-30B decode TP=4 -> 14 heads per GPU (configs[1])
    "opt30b_tp4": AttnConfig(2, "opt30b_tp4", 64, 14, 14, 128, 128, "uniform_512_2048"),
    # cfg 3: LLaMA-2-70B decode TP=2 -> 32 q / 4 kv (configs[2])
    "llama70b_tp2": AttnConfig(3, "llama70b_tp2", 128, 32, 4, 128, 256, "lognormal_1024"),
    # cfg 4: ingest LLaMA-2-70B, prefill TP=4 -> decode TP=2 (configs[3])
    "llama70b_ingest": IngestConfig(4, "llama70b_ingest", 80, 8, 128, 4, 2, 32, "uniform_256_4096"),
    # cfg 5: LLaMA-2-70B TP=1 heavy-tailed decode + per-step ingest (configs[4])
    "llama70b_tp1": AttnConfig(5, "llama70b_tp1", 256, 64, 8, 128, 512, "heavy_tail"),
    "llama70b_tp1_ingest": IngestConfig(5, "llama70b_tp1_ingest", 1, 8, 128, 4, 1, 16, "fixed_2048"),
}


def attn_lengths(c: AttnConfig) -> np.ndarray:
    g = rng(c.cfg, S_LEN)
    if c.lengths == "tiny":
        n = np.array([17, 64, 100, 255])
    elif c.lengths == "uniform_512_2048":
        n = g.integers(512, 2048, size=c.batch, endpoint=True)
    elif c.lengths == "lognormal_1024":
        z = g.standard_normal(c.batch)
        n = np.clip(np.rint(np.exp(math.log(1024.0) + 0.6 * z)), 64, 4096)
    elif c.lengths == "heavy_tail":
        # "70% / 30%" read as fixed counts so the byte count is fixed
        n_short = int(round(0.7 * c.batch))
        short = g.integers(128, 1024, size=n_short, endpoint=True)
        long_ = g.integers(4096, 8192, size=c.batch - n_short, endpoint=True)
        n = np.concatenate([short, long_])
        rng(c.cfg, S_SHUFFLE).shuffle(n)
    else:
        raise ValueError(c.lengths)
    return n.astype(np.int32)


def ingest_lengths(c: IngestConfig) -> np.ndarray:
    g = rng(c.cfg, S_ILEN)
    if c.lengths == "tiny":
        n = np.array([17, 64, 100, 255])
    elif c.lengths == "uniform_256_4096":
        n = g.integers(256, 4096, size=c.prompts, endpoint=True)
    elif c.lengths == "fixed_2048":
        n = np.full(c.prompts, 2048)
    else:
        raise ValueError(c.lengths)
    return n.astype(np.int32)


def pages_for(lens: np.ndarray, page_size: int = PAGE_SIZE) -> np.ndarray:
    return (np.asarray(lens, dtype=np.int64) + page_size - 1) // page_size


def place_pages(lens, num_pages: int, stride: int, g: np.random.Generator,
                page_size: int = PAGE_SIZE, exclude=None):
    """Random page placement: a permutation of the pool handed out in request
    order. Returns block_table [B][stride] int32 (unused entries = -1)."""
    need = pages_for(lens, page_size)
    perm = g.permutation(num_pages)
    if exclude is not None:
        perm = perm[~np.isin(perm, np.asarray(exclude))]
    assert need.sum() <= perm.size, "pool too small"
    bt = np.full((len(lens), stride), -1, dtype=np.int32)
    o = 0
    for i, k in enumerate(need):
        assert k <= stride
        bt[i, :k] = perm[o:o + k]
        o += k
    return bt


def _fill_normal(out: np.ndarray, ss: np.random.SeedSequence, threads: int = 8):
    flat = out.reshape(-1)
    n = flat.size
    chunk = 1 << 22
    nchunks = (n + chunk - 1) // chunk
    kids = ss.spawn(nchunks)

    def work(j):
        a, b = j * chunk, min(n, (j + 1) * chunk)
        flat[a:b] = np.random.default_rng(kids[j]).standard_normal(b - a, dtype=np.float32).astype(np.float16)

    if nchunks == 1:
        work(0)
    else:
        with ThreadPoolExecutor(threads) as ex:
            list(ex.map(work, range(nchunks)))
    return out


def draw_fp16_normal(shape, cfg: int, stream: int, *extra: int) -> np.ndarray:
    """N(0,1) drawn in float32 and rounded to fp16, chunked so it is thread-parallel
    and independent of the thread count."""
    out = np.empty(shape, dtype=np.float16)
    return _fill_normal(out, np.random.SeedSequence([SEED, cfg, stream, *extra]))


def draw_u16_bits(shape, cfg: int, stream: int, *extra: int) -> np.ndarray:
    """Uniform 16-bit patterns (NaN payloads, -0, subnormals included) for bit-exact tests."""
    return rng(cfg, stream, *extra).integers(0, 65536, size=shape, dtype=np.uint16)


def make_attention_inputs(c: AttnConfig, *, layers: int = 1, spare: float = 1.25,
                          lens=None, page_size: int = PAGE_SIZE, seed_extra: int = 0):
    """q [B][Hq][D] fp16; paged k, v [layers][P][Hkv][ps][D] fp16 drawn directly in
    physical layout (all slots random); block table by random placement."""
    lens = attn_lengths(c) if lens is None else np.asarray(lens, dtype=np.int32)
    need = int(pages_for(lens, page_size).sum())
    num_pages = max(1, int(math.ceil(spare * need)))
    stride = max(c.max_pages, int(pages_for(lens, page_size).max(initial=1)))
    bt = place_pages(lens, num_pages, stride, rng(c.cfg, S_PERM, seed_extra), page_size)
    q = draw_fp16_normal((len(lens), c.q_heads, c.head_dim), c.cfg, S_Q, seed_extra)
    shape = (layers, num_pages, c.kv_heads, page_size, c.head_dim)
    k = draw_fp16_normal(shape, c.cfg, S_K, seed_extra)
    v = draw_fp16_normal(shape, c.cfg, S_V, seed_extra)
    return dict(cfg=c, seq_lens=lens, block_table=bt, num_pages=num_pages, q=q, k=k, v=v,
                page_size=page_size, layers=layers,
                kv_bytes=int(lens.astype(np.int64).sum()) * c.kv_heads * c.head_dim * 2 * 2)


def make_ingest_inputs(c: IngestConfig, *, layers=None, spare: float = 1.25, lens=None,
                       bits: bool = False, page_size: int = PAGE_SIZE, seed_extra: int = 0,
                       src_tp=None, dst_tp=None):
    """Source shards as a prefill TP group wrote them: S buffers [L][T][heads/S][D] for K and
    for V (prompts packed back to back on the token axis), plus lengths / cu_seqlens / block
    table. The paged destination is NOT built here (that is the method)."""
    L = c.layers if layers is None else layers
    S = c.src_tp if src_tp is None else src_tp
    R = c.dst_tp if dst_tp is None else dst_tp
    lens = ingest_lengths(c) if lens is None else np.asarray(lens, dtype=np.int32)
    T = int(lens.astype(np.int64).sum())
    cu = np.zeros(len(lens) + 1, dtype=np.int32)
    np.cumsum(lens, out=cu[1:])
    need = int(pages_for(lens, page_size).sum())
    num_pages = max(1, int(math.ceil(spare * need)))
    stride = max(1, int(pages_for(lens, page_size).max(initial=1)))
    bt = place_pages(lens, num_pages, stride, rng(c.cfg, S_PERM, 1000 + seed_extra), page_size)
    hs = c.heads // S
    shape = (L, T, hs, c.head_dim)
    if bits:
        src_k = [draw_u16_bits(shape, c.cfg, S_SRCK, r, seed_extra) for r in range(S)]
        src_v = [draw_u16_bits(shape, c.cfg, S_SRCV, r, seed_extra) for r in range(S)]
    else:
        src_k = [draw_fp16_normal(shape, c.cfg, S_SRCK, r, seed_extra).view(np.uint16) for r in range(S)]
        src_v = [draw_fp16_normal(shape, c.cfg, S_SRCV, r, seed_extra).view(np.uint16) for r in range(S)]
    return dict(cfg=c, layers=L, heads=c.heads, head_dim=c.head_dim, src_tp=S, dst_tp=R,
                seq_lens=lens, cu_seqlens=cu, total_tokens=T, block_table=bt, num_pages=num_pages,
                page_size=page_size, src_k=src_k, src_v=src_v,
                payload_bytes=2 * L * T * c.heads * c.head_dim * 2)
