"""Seeded synthetic inputs for the hx decode-phase KV-cache path.

This module serves BOTH the oracle (oracle/) and the CUDA path
(paper_2502_07903_b200/): it draws lengths, page placements and random fp16
payloads. It holds none of the method's arithmetic: no attention, no softmax,
no head-regroup or page-scatter index math. Paged caches are drawn directly in
their physical layout (every slot random), so nothing here places a token.

Recipe: the paper's workloads are
samples of the Azure Conversation trace, which is not
available; BASELINE.json's length distributions stand in for it at the paper's
model shapes (OPT-30B, LLaMA-2-70B, fp16: PAPER.md:L142-L144, L254).
"""
from .configs import (  # noqa: F401
    CONFIGS, AttnConfig, IngestConfig, rng, attn_lengths, ingest_lengths,
    place_pages, draw_fp16_normal, draw_u16_bits, make_attention_inputs,
    make_ingest_inputs, pages_for,
)
