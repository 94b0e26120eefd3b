"""Python face of the hxo oracle (oracle/hxo.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this.  It never imports paper_2502_07903_b200 and shares no code with it.
Citations and the list of pins are in oracle/hxo.c's header.
"""
from .hxo import (  # noqa: F401
    build, lib, kv_ingest, kv_gather, decode_attention, partial_attention,
    half_to_double, max_threads, merge_partials, kv_ingest_stage, kv_append, prefill_attention,
)
