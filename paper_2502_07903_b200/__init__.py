"""paper_2502_07903_b200 — thin Python binding over libhx (include/hx.h).

B200-native (sm_100a) decode-phase KV-cache path of HexGen-2 (arxiv 2502.07903):
`kv_ingest` (prefill-TP shards -> decode-TP paged cache) and `decode_attention`
(one-token MHA/GQA attention over the paged cache).  Argument marshalling only: every step
of the path runs in the CUDA kernels of csrc/.  There is no CPU fallback: importing
`binding` raises if libhx.so is missing.
"""
from .binding import (  # noqa: F401
    HxError, PagedCache, PagePool, lib, version, last_error, status_string,
    paged_cache_bytes, kv_ingest, kv_gather, decode_attention, decode_attention_workspace_bytes,
    decode_step_host, decode_plan_bytes, decode_plan, decode_attention_planned, decode_attention_chained, EXPORTS, kv_ingest_stage, stage_overlap, kv_append,
    decode_attention_append, prefill_attention, decode_attention_overlapped, decode_step, DecodeStep, shutdown,
    decode_attention_noalloc, NOALLOC_SCRATCH_BYTES,
)
