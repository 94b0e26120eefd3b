#!/usr/bin/env python
"""bench.py — one decode step of the hx KV-cache path on B200 (BASELINE.json configs[4]).

A "step" = the whole hot path over one batch: the host page
allocator frees last step's 16 prompts and allocates 16 new ones (2048 tokens each), their
block-table rows are uploaded, and ONE C-ABI call, hx_decode_step(overlap_ingest=1), lands their KV
(the hx_kv_ingest copy: prefill TP=4 -> decode TP=1, one layer) inside the SAME kernel that runs
hx_decode_attention over the fixed 256-request heavy-tailed batch (64 q / 8 kv heads, head_dim 128):
warps that have finished their attention range move the handoff's tiles with the copy engines.  The new
prompts' pages are disjoint from the batch's (the handoff is asynchronous "to enable
overlapping").  Inputs are seeded synthetic data (workloads/).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl hx|reference] [--oracle-table]

Prints ONE JSON line (rank 0).  `value` = (attention KV bytes + ingest read+write bytes) per
step x K / device time, inputs resident in HBM.  N > 1: independent replicas, one per GPU, no
collective on the data path ("replicas only"); value sums over ranks.  Without torchrun
(`WORLD_SIZE` unset) `--gpus N` re-executes itself under torch.distributed.run with N ranks.

Beside the contract keys (roofline, e2e, cpu_baseline, clocks, gpu_launches) the line carries:
`in_order` (the same step with both kernels on one stream, which also gives each kernel's time alone),
`overlapped_launch` (one stream, programmatic dependent launch), `cuda_graph` (the headline step replayed as a
CUDA graph), `e2e.*` (hx_decode_step_host from pinned host buffers) and `other_configs`: configs[1], [2]
(attention) and [3] (80-layer ingest) kernel-only, `prefill` (hx_prefill_attention against the tensor roofline),
`append_cfg5` (fused append + attention), `step_src_tp1` (the headline step with the handoff from a prefill TP=1 replica) and
`stream_peaks` (read-only / write-only HBM rates of the run).
`--oracle-table` prints the oracle's time per config at 1 thread and at all cores instead.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import socket
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402

METRIC = "decode-step KV bytes/s: paged decode-attention KV read + KV-ingest read+write (cfg5, 1 layer)"
UNIT = "GB/s"
NOMINAL_HBM_GBS = 8000.0
FALLBACK_HBM_GBS = 6650.0


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def measured_tensor_peak():
    """Dense bf16/fp16 tensor peak in TFLOP/s (burst figure: the prefill kernel is timed alone)."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["bf16_tflops"]), "measured (MEASURED_PEAKS.json bf16_tflops, cuBLAS 8192^3 burst)"
    except Exception:
        return 1590.0, "fallback (B200_PROFILING.md 1.59 PFLOP/s)"


def measured_tensor_peak_sustained():
    """The same under a seconds-long loop (the clocks sag under the power cap): for the back-to-back prefill figure."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["bf16_tflops_sustained"]), "measured (MEASURED_PEAKS.json bf16_tflops_sustained, cuBLAS 8192^3 looped for 4 s)"
    except Exception:
        return 1400.0, "fallback (B200_PROFILING.md 1.4 PFLOP/s sustained)"


def stream_peaks(torch, dev):
    """Read-only and write-only HBM stream rates of this GPU in this run: the attention kernel
    only reads, so it can exceed the copy figure.  torch ops over 4 GiB (context numbers, not the product)."""
    n = 1 << 30                                            # 4 GiB of float32
    x = torch.empty(n, dtype=torch.float32, device=dev)
    x.zero_()
    res = {}
    for name, fn in (("write_only_fill", lambda: x.zero_()), ("read_only_sum", lambda: x.sum())):
        med, mn = time_kernel(torch, fn, iters=5, warm=2)
        res[name + "_GBps"] = 4 * n / mn / 1e6
    del x
    return res


def prefill_extra(torch, hx, dev):
    """F4: hx_prefill_attention on the prefill that produced cfg5's new prompts: 16 prompts x
    2048 tokens, LLaMA-2-70B, one layer, K/V already in the paged cache.  Algorithmic flops = 4*D per causal
    (query, kv token) pair per q head; nothing padded or masked is counted."""
    res = {}
    peak, src = measured_tensor_peak()
    for name, (B, n, Hq, Hkv) in {"llama70b_tp1_16x2048": (16, 2048, 64, 8), "llama70b_prefill_tp4_16x2048": (16, 2048, 16, 2),
                                  "opt30b_tp4_16x2048": (16, 2048, 14, 14)}.items():
        D = 128
        pages = B * ((n + 15) // 16)
        k = torch.empty((1, pages, Hkv, 16, D), dtype=torch.float16, device=dev).normal_()
        v = torch.empty_like(k).normal_()
        cache = hx.PagedCache(k, v)
        g = torch.Generator(device=dev)
        g.manual_seed(7)
        bt = torch.randperm(pages, device=dev, generator=g).to(torch.int32).reshape(B, -1).contiguous()
        lens = torch.full((B,), n, dtype=torch.int32, device=dev)
        cu = torch.arange(B + 1, dtype=torch.int32, device=dev) * n
        q = torch.empty((B * n, Hq, D), dtype=torch.float16, device=dev).normal_()
        out = torch.empty_like(q)

        def fn():
            hx.prefill_attention(out, q, cache, layer=0, q_heads=Hq, block_table=bt, block_table_stride=bt.shape[1],
                                 seq_lens=lens, q_lens=lens, cu_q_lens=cu, batch=B, total_q_tokens=B * n, max_q_len=n,
                                 max_seq_len=n)
        med, mn = time_kernel(torch, fn, iters=10, warm=3)
        flops = B * Hq * (n * (n + 1) // 2) * 4 * D
        res[name] = {"ms_median": med, "ms_min": mn, "algorithmic_flops": flops, "TFLOPs": flops / med / 1e9,
                     "roofline": {"bound": "tensor", "achieved": flops / med / 1e9, "peak": peak, "unit": "TFLOP/s",
                                  "frac": flops / med / 1e9 / peak, "peak_source": src}}
        if name == "llama70b_tp1_16x2048":
            def fn_keep(out=out, q=q, cache=cache, bt=bt, lens=lens, cu=cu, B=B, n=n, Hq=Hq):     # (bound now: the loop rebinds the names)
                hx.prefill_attention(out, q, cache, layer=0, q_heads=Hq, block_table=bt, block_table_stride=bt.shape[1],
                                     seq_lens=lens, q_lens=lens, cu_q_lens=cu, batch=B, total_q_tokens=B * n, max_q_len=n,
                                     max_seq_len=n)
            keep = (fn_keep, flops)                               # for the sustained loop below (after the burst figures)
        del k, v, cache, q, out
    # the LLaMA-2-70B prefill again in a 0.5 s back-to-back loop, against the SUSTAINED cuBLAS figure (both sag with the clocks);
    # last, so that the heat it leaves does not sit in the burst figures above
    fn, flops = keep[0], keep[1]
    calls = 400
    sus = time_back_to_back(torch, fn, calls=calls, reps=1, warm=1)
    speak, ssrc = measured_tensor_peak_sustained()
    res["llama70b_tp1_16x2048"]["sustained"] = {"ms": sus, "TFLOPs": flops / sus / 1e9, "calls_back_to_back": calls, "peak": speak,
                                                "frac": flops / sus / 1e9 / speak, "peak_source": ssrc}
    del keep
    return res


def max_over_ranks(ms: float, world: int, device) -> float:
    """Multi-GPU numbers are the MAX over ranks of the device time (never wall clock)."""
    if world <= 1:
        return ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(bytes_per_step_per_rank: int, steps: int, world: int, ms_max: float) -> float:
    """Whole-job throughput in GB/s: every rank processes its own replica (weak scaling)."""
    return world * bytes_per_step_per_rank * steps / (ms_max * 1e-3) / 1e9


class ClockSampler:
    """nvidia-smi clocks / throttle reasons, sampled every 20 ms over the WHOLE run; stop() reports the samples that
    fell inside the timed window [mark_begin, mark_end] (and the whole run beside them)."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index: int):
        self.index, self.rows, self.proc, self.t0, self.t1 = index, [], None, None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "20"], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def mark_begin(self):
        self.t0 = time.time()

    def mark_end(self):
        self.t1 = time.time()

    @classmethod
    def _summary(cls, rows):
        sm = [float(r[1]) for r in rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        reasons = [n for j, n in enumerate(cls.NAMES) if any(len(r) > 4 + j and r[4 + j].startswith("Active") for r in rows)]
        return sm, reasons

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.1)
        self.proc.terminate()
        self.t.join(timeout=2)
        rows = [r for _, r in self.rows]
        mx = [float(r[2]) for r in rows if len(r) > 2 and r[2].replace(".", "").isdigit()]
        # a sample is attributed to the window if it was read inside it (+- one sampling period)
        win = [r for t, r in self.rows if self.t0 is not None and self.t0 - 0.02 <= t <= self.t1 + 0.04]
        sm_all, reasons_all = self._summary(rows)
        sm_win, reasons_win = self._summary(win)
        busy = [x for x in sm_all if x >= 0.5 * max(mx, default=0)]           # samples with the GPU clocked up
        return {"sm_mhz": float(np.median(sm_win)) if sm_win else (float(np.median(busy)) if busy else None),
                "sm_max_mhz": max(mx) if mx else None, "reasons": reasons_win if win else reasons_all,
                "samples": len(sm_all), "samples_in_timed_window": len(sm_win),
                "whole_run": {"sm_mhz_median": float(np.median(sm_all)) if sm_all else None, "reasons": reasons_all,
                              "seconds": (self.rows[-1][0] - self.rows[0][0]) if len(self.rows) > 1 else 0.0}}


NCU_TRAFFIC_FILE = os.path.join(ROOT, "profiles", "ncu_traffic.json")


def kernel_source_hash() -> str:
    """sha256 over the CUDA sources of the two hot kernels: ties an ncu capture to the tree it was taken on."""
    h = hashlib.sha256()
    for f in ("attention.cu", "handoff_tiles.cuh", "ingest.cu"):
        with open(os.path.join(ROOT, "paper_2502_07903_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def ncu_traffic():
    """dram read+write bytes per launch of the headline step's kernel from the committed ncu --set full capture — only if that capture
    was taken on THIS tree's kernels (profiles/ncu_traffic.json stores their source hash); else null, loudly."""
    try:
        with open(NCU_TRAFFIC_FILE) as f:
            d = json.load(f)
    except Exception:
        return None, "no profiles/ncu_traffic.json"
    if d.get("kernel_source_sha256") != kernel_source_hash():
        print("bench.py: WARNING: profiles/ncu_traffic.json was captured on other kernel sources; roofline.traffic = null",
              file=sys.stderr, flush=True)
        return None, "stale: profiles/ncu_traffic.json was captured on other kernel sources"
    return int(d["step_kernel_dram_bytes_per_launch"]), f"ncu --set full capture {d.get('capture')} (same kernel sources, not measured in this run)"


# ----------------------------------------------------------------------------------------------
def build_step_workload(torch, hx, seed_extra=0):
    """cfg5: resident 256-request cache + two alternating sets of 16 new prompts to ingest."""
    ca, ci = W.CONFIGS["llama70b_tp1"], W.CONFIGS["llama70b_tp1_ingest"]
    lens = W.attn_lengths(ca)
    need_attn = int(W.pages_for(lens).sum())
    ing_lens = W.ingest_lengths(ci)
    need_ing = int(W.pages_for(ing_lens).sum())
    num_pages = need_attn + 2 * need_ing + 512
    pool = hx.PagePool(num_pages, shuffle_seed=5)
    bt = pool.alloc_table(lens, ca.max_pages)                 # A1: random free-page list
    dev = torch.device("cuda")
    shape = (1, num_pages, ca.kv_heads, 16, ca.head_dim)
    g = torch.Generator(device=dev)
    g.manual_seed(1234 + seed_extra)
    k = torch.empty(shape, dtype=torch.float16, device=dev).normal_(generator=g)
    v = torch.empty(shape, dtype=torch.float16, device=dev).normal_(generator=g)
    q_np = W.draw_fp16_normal((ca.batch, ca.q_heads, ca.head_dim), ca.cfg, W.configs.S_Q, seed_extra)
    ing = W.make_ingest_inputs(ci, src_tp=4)
    st = dict(ca=ca, ci=ci, lens=lens, ing_lens=ing_lens, pool=pool, num_pages=num_pages,
              cache=hx.PagedCache(k, v), bt_host=bt, q_host=q_np, ing=ing,
              kv_bytes=int(lens.astype(np.int64).sum()) * ca.kv_heads * ca.head_dim * 4,
              ing_payload=ing["payload_bytes"])
    return st


def run_hx(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    import paper_2502_07903_b200 as hx

    torch.cuda.set_device(local_rank)
    torch.manual_seed(1234 + rank)                 # every device-side draw below (K/V/Q fills of the extras) is seeded
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    sampler = ClockSampler(local_rank)             # samples the whole run; the timed window is marked below
    sampler.start()
    st = build_step_workload(torch, hx, seed_extra=rank)
    ca, ci, ing = st["ca"], st["ci"], st["ing"]
    B, Hq, Hkv, D = ca.batch, ca.q_heads, ca.kv_heads, ca.head_dim
    max_len = int(st["lens"].max())
    cache = st["cache"]
    q = torch.from_numpy(st["q_host"]).to(dev)
    out = torch.empty_like(q)
    bt = torch.from_numpy(st["bt_host"]).to(dev)
    sl = torch.from_numpy(st["lens"]).to(dev)
    ws_bytes = hx.decode_attention_workspace_bytes(B, Hq, Hkv, D, max_len)
    ws = torch.zeros(max(ws_bytes, 16), dtype=torch.uint8, device=dev)
    # ingest sources resident in HBM (the prefill shards as they arrived)
    src_k = [torch.from_numpy(a.view(np.int16)).to(dev).view(torch.float16) for a in ing["src_k"]]
    src_v = [torch.from_numpy(a.view(np.int16)).to(dev).view(torch.float16) for a in ing["src_v"]]
    nI, TI = len(st["ing_lens"]), ing["total_tokens"]
    ing_stride = int(W.pages_for(st["ing_lens"]).max())
    ing_cu = torch.from_numpy(ing["cu_seqlens"]).to(dev)
    ing_sl = torch.from_numpy(ing["seq_lens"]).to(dev)
    ing_bt_dev = torch.empty((nI, ing_stride), dtype=torch.int32, device=dev)
    # the host runs ahead of the GPU: a ring of pinned row buffers, each reused only after the copy
    # that last read it has completed
    RING = 16
    ing_bt_pins = [torch.empty((nI, ing_stride), dtype=torch.int32).pin_memory() for _ in range(RING)]
    ring_ev = [None] * RING
    pool = st["pool"]
    prev = {"ids": None, "n": 0}

    def next_rows():
        """A1: free last step's prompts, allocate this step's (host), stage the new rows for upload."""
        if prev["ids"] is not None:
            pool.free(prev["ids"])
        rows = pool.alloc_table(st["ing_lens"], ing_stride)
        prev["ids"] = rows[rows >= 0]
        slot = prev["n"] % RING
        prev["n"] += 1
        if ring_ev[slot] is not None:
            ring_ev[slot].synchronize()
        pin = ing_bt_pins[slot]
        pin.numpy()[:] = rows
        return pin, slot

    # The rows of step n+1 are uploaded on a copy stream into the OTHER of two device row buffers while step n's kernels
    # run (as an engine's scheduler would: the allocation for the next step does not depend on this step's kernels).
    copy_stream = torch.cuda.Stream(device=dev)
    ing_bt_devs = [ing_bt_dev, torch.empty_like(ing_bt_dev)]
    buf_free = [None, None]                      # recorded on the main stream after the step that last read buffer i

    def upload_rows():
        pin, slot = next_rows()
        i = (prev["n"] - 1) & 1
        with torch.cuda.stream(copy_stream):
            if buf_free[i] is not None:
                copy_stream.wait_event(buf_free[i])
            ing_bt_devs[i].copy_(pin, non_blocking=True)
            ev = ring_ev[slot] or torch.cuda.Event()
            ev.record()
            ring_ev[slot] = ev
        torch.cuda.current_stream(dev).wait_event(ev)
        return i

    step_kw = dict(out=out, q=q, cache=cache, layer=0, q_heads=Hq, block_table=bt, block_table_stride=bt.shape[1],
                   seq_lens=sl, batch=B, max_seq_len=max_len, sm_scale=0.0, workspace=ws, workspace_bytes=ws_bytes,
                   src_k=src_k, src_v=src_v, ing_layers=1, heads=ci.heads, src_tp=4, dst_tp=1, dst_rank=0,
                   ing_block_table=ing_bt_dev, ing_block_table_stride=ing_stride, ing_cu_seqlens=ing_cu, ing_seq_lens=ing_sl,
                   ing_batch=nI, ing_total_tokens=TI, ing_max_seq_len=2048)
    # the headline step: ONE hx_decode_step call = one kernel (attention carrying the handoff)
    stepper = [hx.DecodeStep(overlap_ingest=1, **dict(step_kw, ing_block_table=b)) for b in ing_bt_devs]
    stepper_in_order = [hx.DecodeStep(overlap_ingest=0, **dict(step_kw, ing_block_table=b)) for b in ing_bt_devs]
    EV = ("ev_ingest_begin", "ev_ingest_end", "ev_attention_begin", "ev_attention_end")

    def step(which=stepper, events=None):
        i = upload_rows()
        for j, name in enumerate(EV):
            setattr(which[i].a, name, events[j].cuda_event if events else None)
        which[i]()
        ev = buf_free[i] or torch.cuda.Event()
        ev.record()
        buf_free[i] = ev

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def new_events(n):
        evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(n)]
        for row in evs:
            for e in row:
                e.record()                        # creates the handle the library records into
        return evs

    def timed_steps(which, with_events=True):
        for _ in range(max(args.warmup, 3)):
            step(which)
        barrier()
        ev = new_events(args.steps)
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        if which is stepper and not with_events:
            sampler.mark_begin()
        t0.record()
        for s_ in range(args.steps):
            step(which, ev[s_] if with_events else None)
        t1.record()
        barrier()
        if which is stepper and not with_events:
            sampler.mark_end()
        ing = [e[0].elapsed_time(e[1]) for e in ev]
        att = [e[2].elapsed_time(e[3]) for e in ev]
        return max_over_ranks(t0.elapsed_time(t1), world, dev), float(np.mean(ing)), float(np.mean(att)), float(np.min(att))

    # headline: in the overlapped step attention and handoff are ONE kernel, so the library's timing events bracket both.
    # The headline K steps carry no per-step events at all; the kernel is timed in a second pass of K steps.
    total_ms, _, _, _ = timed_steps(stepper, with_events=False)
    _, _, pair_ms, pair_min_ms = timed_steps(stepper)
    step_bytes = st["kv_bytes"] + 2 * st["ing_payload"]

    # ---- the same K steps with both kernels in order on one stream: each kernel's own CUDA-event time inside a step.
    # The roofline object below is the attention kernel's, from this timed region.
    ser_ms, ing_ms, att_ms, att_min_ms = timed_steps(stepper_in_order)
    ser_ing_ms, ser_att_ms = ing_ms, att_ms

    # ---- extra: single stream with hx_decode_attention_overlapped: the attention grid is a programmatic dependent of the
    # ingest kernel and starts while the handoff is still landing (disjoint pages)
    def step_pdl():
        i = upload_rows()
        hx.kv_ingest(src_k, src_v, layers=1, heads=ci.heads, head_dim=D, src_tp=4, dst_tp=1, dst_rank=0,
                     dst=cache, block_table=ing_bt_devs[i], block_table_stride=ing_stride, cu_seqlens=ing_cu,
                     seq_lens=ing_sl, batch=nI, total_tokens=TI, max_seq_len=2048)
        hx.decode_attention_overlapped(out, q, cache, layer=0, q_heads=Hq, block_table=bt, block_table_stride=bt.shape[1],
                                       seq_lens=sl, batch=B, max_seq_len=max_len, workspace=ws, workspace_bytes=ws_bytes,
                                       behind_ingest=1)
        ev = buf_free[i] or torch.cuda.Event()
        ev.record()
        buf_free[i] = ev

    barrier()
    for _ in range(3):
        step_pdl()
    barrier()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record()
    for _ in range(args.steps):
        step_pdl()
    p1.record()
    barrier()
    pdl_ms = max_over_ranks(p0.elapsed_time(p1), world, dev)

    # ---- extra: the headline step captured once in a CUDA graph (row upload + hx_decode_step: the fused kernel
    # becomes a graph edge) and replayed; two graphs alternate so that the host can stage step n+1's rows while step n runs
    main = torch.cuda.current_stream(dev)
    graphs = []
    cap = torch.cuda.Stream(device=dev)
    for st_ in stepper:
        for name in EV:
            setattr(st_.a, name, None)
    for gi in range(2):
        pin_g = torch.empty((nI, ing_stride), dtype=torch.int32).pin_memory()
        dev_g = torch.empty((nI, ing_stride), dtype=torch.int32, device=dev)
        pin_g.numpy()[:] = ing_bt_pins[0].numpy()
        gstep = hx.DecodeStep(overlap_ingest=1, **dict(step_kw, ing_block_table=dev_g))
        gr = torch.cuda.CUDAGraph()
        cap.wait_stream(main)
        with torch.cuda.graph(gr, stream=cap):
            dev_g.copy_(pin_g, non_blocking=True)
            gstep(stream=cap)
        graphs.append((gr, pin_g, torch.cuda.Event(), gstep))
    main.wait_stream(cap)

    def step_graph(n):
        gr, pin_g, ev, _ = graphs[n & 1]
        if prev["ids"] is not None:
            pool.free(prev["ids"])
        rows = pool.alloc_table(st["ing_lens"], ing_stride)
        prev["ids"] = rows[rows >= 0]
        if n >= 2:
            ev.synchronize()                         # this graph's previous replay has read its pinned rows
        pin_g.numpy()[:] = rows
        gr.replay()
        ev.record()

    barrier()
    for n in range(4):
        step_graph(n)
    barrier()
    g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    g0.record()
    for n in range(args.steps):
        step_graph(n)
    g1.record()
    barrier()
    graph_ms = max_over_ranks(g0.elapsed_time(g1), world, dev)

    # ---- e2e: the same step through hx_decode_step_host with HOST (pinned) buffers
    qh = torch.from_numpy(st["q_host"]).pin_memory()
    oh = torch.empty_like(qh).pin_memory()
    skh = [torch.from_numpy(a.view(np.int16)).pin_memory() for a in ing["src_k"]]
    svh = [torch.from_numpy(a.view(np.int16)).pin_memory() for a in ing["src_v"]]
    cu_h = torch.from_numpy(ing["cu_seqlens"]).pin_memory()
    sl_h = torch.from_numpy(ing["seq_lens"]).pin_memory()

    def step_e2e(pull, overlap=False):
        ing_bt_pin, _ = next_rows()                     # (the step synchronises below: no reuse hazard)
        hx.decode_step_host(
            pull_src=int(pull), overlap_ingest=int(overlap),
            q_host=qh, out_host=oh, q_dev=q, out_dev=out, cache=cache, layer=0, q_heads=Hq, block_table_dev=bt,
            block_table_stride=bt.shape[1], seq_lens_dev=sl, batch=B, max_seq_len=max_len, sm_scale=0.0,
            workspace=ws, workspace_bytes=ws_bytes, src_k_host=skh, src_v_host=svh, src_k_dev=src_k,
            src_v_dev=src_v, ing_layers=1, heads=ci.heads, src_tp=4, dst_tp=1, dst_rank=0,
            ing_block_table_host=ing_bt_pin, ing_block_table_stride=ing_stride, ing_cu_seqlens_host=cu_h,
            ing_seq_lens_host=sl_h, ing_block_table_dev=ing_bt_dev, ing_cu_seqlens_dev=ing_cu,
            ing_seq_lens_dev=ing_sl, ing_batch=nI, ing_total_tokens=TI, ing_max_seq_len=2048)
        torch.cuda.current_stream().synchronize()      # the step's result is read on the host
        return float(oh[0, 0, 0])

    def time_e2e(pull, overlap=False):
        for _ in range(3):
            step_e2e(pull, overlap)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            step_e2e(pull, overlap)
        e1.record()
        barrier()
        return max_over_ranks(e0.elapsed_time(e1), world, dev)

    # staged: cudaMemcpyAsync of the shards into HBM, then ingest (the headline e2e: the copy engine
    # drives PCIe a little better than SM loads do).  pull (F2): the ingest kernel reads the pinned
    # shards over the link itself (transfer + regroup + scatter fused); reported beside it.  The same
    # bytes cross the link either way.
    # overlap_ingest: the handoff (PCIe + ingest) runs on the library's side stream under the attention; the
    # step's attention does not read the pages it ingests (they are disjoint from the active batch).
    e2e_serial_ms = time_e2e(False)
    e2e_pull_ms = time_e2e(True)
    e2e_ms = time_e2e(False, overlap=True)
    e2e_pull_ov_ms = time_e2e(True, overlap=True)

    h2d = qh.numel() * 2 + sum(a.numel() * 2 for a in skh + svh) + nI * ing_stride * 4 + cu_h.numel() * 4 + sl_h.numel() * 4
    d2h = oh.numel() * 2
    peak, peak_src = measured_peak()
    att_gbs = st["kv_bytes"] / (att_ms * 1e-3) / 1e9
    ing_gbs = 2 * st["ing_payload"] / (ing_ms * 1e-3) / 1e9
    traffic, traffic_note = ncu_traffic()

    extra = {}
    if rank == 0 and not args.no_extra:
        extra = other_configs(torch, hx, dev, peak)
        # F1: the decode step's append, as its own launch and fused into the attention kernel
        kn = torch.empty((B, Hkv, D), dtype=torch.float16, device=dev).normal_()
        vn = torch.empty((B, Hkv, D), dtype=torch.float16, device=dev).normal_()
        akw = dict(layer=0, block_table=bt, block_table_stride=bt.shape[1], seq_lens=sl, batch=B, max_seq_len=max_len)

        def two_launches():
            hx.kv_append(kn, vn, cache, **akw)
            hx.decode_attention(out, q, cache, q_heads=Hq, workspace=ws, workspace_bytes=ws_bytes, **akw)

        def fused():
            hx.decode_attention_append(out, q, kn, vn, cache, q_heads=Hq, workspace=ws, workspace_bytes=ws_bytes, **akw)

        def alone():
            hx.decode_attention(out, q, cache, q_heads=Hq, workspace=ws, workspace_bytes=ws_bytes, **akw)
        m2, _ = time_kernel(torch, two_launches, iters=20)
        m1, _ = time_kernel(torch, fused, iters=20)
        m0, m0min = time_kernel(torch, alone, iters=20)
        extra["attention_cfg5_alone"] = {"ms_median": m0, "ms_min": m0min, "kv_GBps": st["kv_bytes"] / m0 / 1e6,
                                         "frac_of_measured": st["kv_bytes"] / m0 / 1e6 / peak,
                                         "timing": "one CUDA-event pair per call, nothing else on the GPU"}
        # SURVEY 8(d) reading (ii): the same step with the new prompts arriving from a prefill replica of TP = 1
        # (one shard holding all 8 kv heads) instead of TP = 4
        ing1 = W.make_ingest_inputs(ci, src_tp=1)
        sk1 = [torch.from_numpy(a.view(np.int16)).to(dev).view(torch.float16) for a in ing1["src_k"]]
        sv1 = [torch.from_numpy(a.view(np.int16)).to(dev).view(torch.float16) for a in ing1["src_v"]]
        stepper_s1 = [hx.DecodeStep(overlap_ingest=1, **dict(step_kw, src_k=sk1, src_v=sv1, src_tp=1, ing_block_table=b)) for b in ing_bt_devs]
        s1_ms, _, _, _ = timed_steps(stepper_s1, with_events=False)
        extra["step_src_tp1"] = {"ms_per_step": s1_ms / args.steps, "value": whole_job_value(step_bytes, args.steps, 1, s1_ms), "unit": UNIT,
                                 "note": "the headline step with the handoff from a prefill TP=1 replica (S=1 -> R=1) instead of TP=4"}
        del sk1, sv1, stepper_s1
        extra["prefill"] = prefill_extra(torch, hx, dev)
        extra["stream_peaks"] = stream_peaks(torch, dev)
        extra["append_cfg5"] = {"append_then_attention_ms": m2, "fused_append_attention_ms": m1,
                                "note": "hx_kv_append + hx_decode_attention (2 launches) vs hx_decode_attention_append (1 launch)"}
    clocks = sampler.stop()

    line = {
        "metric": METRIC, "value": whole_job_value(step_bytes, args.steps, world, total_ms), "unit": UNIT,
        "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f16 in / f32 accumulate",
        "data": "synthetic (seeded; BASELINE.json length mix stands in for the Azure Conversation trace)",
        "config": {"workload": "configs[4]: LLaMA-2-70B TP=1 decode (B=256, 64q/8kv, D=128, 179 ctx in [128,1024] + 77 in "
                               "[4096,8192], page 16, 1 layer) + per-step ingest of 16x2048-token prompts (prefill TP=4 -> decode TP=1)",
                   "step": "A1 host alloc/free + row upload, then ONE hx_decode_step(overlap_ingest=1) call = ONE kernel: decode "
                           "attention whose warps, once their range is done, move the handoff's (page, head) tiles (TMA load + bulk store)",
                   "tokens_in_cache": int(st["lens"].sum()), "attention_kv_bytes": st["kv_bytes"],
                   "ingest_payload_bytes": st["ing_payload"], "l2": "inputs larger than L2 (2.3 GB KV read per step vs 126 MB)",
                   "parallelism": "replicas only" if world > 1 else "1 GPU"},
        "clocks": clocks,
        "e2e": {"value": whole_job_value(step_bytes, args.steps, world, e2e_ms), "unit": UNIT,
                "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h), "ms_per_step": e2e_ms / args.steps,
                "path": "hx_decode_step_host(overlap_ingest=1): shards staged into HBM by cudaMemcpyAsync + ingest on the "
                        "library's side stream, under the attention of the active batch (disjoint pages)",
                "in_order_ms_per_step": e2e_serial_ms / args.steps,
                "in_order_value": whole_job_value(step_bytes, args.steps, world, e2e_serial_ms),
                "pull_mode_in_order_ms_per_step": e2e_pull_ms / args.steps,
                "pull_mode_overlapped_ms_per_step": e2e_pull_ov_ms / args.steps},
        "gpu_launches": int(args.steps * LAUNCHES_PER_STEP),
        "roofline": {"bound": "hbm", "kernel": "attn_handoff_kernel: THE kernel of the timed headline step (hx_decode_step, overlap_ingest=1): "
                                               "decode attention (in-kernel merge) whose warps also move the step's KV handoff; CUDA events "
                                               "around the kernel in a second pass of K steps (the headline K steps carry no events)",
                     "achieved": step_bytes / pair_ms / 1e6, "peak": peak, "unit": "GB/s", "frac": step_bytes / pair_ms / 1e6 / peak,
                     "peak_source": peak_src, "frac_of_nominal_8000": step_bytes / pair_ms / 1e6 / NOMINAL_HBM_GBS,
                     "traffic": traffic, "traffic_source": traffic_note, "algorithmic_bytes": step_bytes,
                     "algorithmic_bytes_note": "attention: sum n_i * 8 kv heads * 128 * 4 B read; handoff: payload read once + written once "
                                               "(DESIGN.md 6.1, 6.2)",
                     "ms": pair_ms, "ms_min": pair_min_ms,
                     "attention_alone_in_order_step": {"achieved": att_gbs, "frac": att_gbs / peak, "ms": att_ms, "ms_min": att_min_ms,
                                                       "algorithmic_bytes": st["kv_bytes"],
                                                       "note": "attn_stream_kernel behind the ingest kernel in hx_decode_step(overlap_ingest=0)"}},
        "step_pair": {"ms": pair_ms, "ms_min": pair_min_ms, "GBps": step_bytes / pair_ms / 1e6, "frac_of_measured": step_bytes / pair_ms / 1e6 / peak,
                      "note": "the ONE kernel of the headline step (attention + handoff), CUDA events around it; "
                              "bytes = attention KV read + ingest read + write"},
        "attention": {"kv_GBps": att_gbs, "tokens_per_s_one_layer": B / (att_ms * 1e-3),
                      "tokens_per_s_80_layers": B / (att_ms * 1e-3 * 80), "ms": att_ms},
        "ingest": {"traffic_GBps": ing_gbs, "payload_GBps": ing_gbs / 2, "frac": ing_gbs / peak,
                   "frac_of_nominal_8000": ing_gbs / NOMINAL_HBM_GBS, "ms": ing_ms,
                   "note": "hx_kv_ingest's kernel inside the K timed in-order steps (CUDA events around the kernel)"},
        "in_order": {"ms_per_step": ser_ms / args.steps, "value": whole_job_value(step_bytes, args.steps, world, ser_ms), "unit": UNIT,
                     "ingest_ms": ser_ing_ms, "attention_ms": ser_att_ms,
                     "ingest_traffic_GBps": 2 * st["ing_payload"] / ser_ing_ms / 1e6,
                     "ingest_frac_of_measured": 2 * st["ing_payload"] / ser_ing_ms / 1e6 / peak,
                     "attention_kv_GBps": st["kv_bytes"] / ser_att_ms / 1e6,
                     "note": "hx_decode_step(overlap_ingest=0): ingest then attention on one stream"},
        "overlapped_launch": {"ms_per_step": pdl_ms / args.steps, "value": whole_job_value(step_bytes, args.steps, world, pdl_ms),
                              "unit": UNIT, "note": "single stream; hx_decode_attention_overlapped starts under the ingest kernel "
                                                    "(programmatic dependent launch, disjoint pages)"},
        "cuda_graph": {"ms_per_step": graph_ms / args.steps, "value": whole_job_value(step_bytes, args.steps, world, graph_ms),
                       "unit": UNIT, "note": "the headline step (row upload + hx_decode_step) captured once and replayed"},
        "other_configs": extra,
    }
    if rank == 0:
        line["cpu_baseline"] = cpu_baseline(st) if world == 1 and not args.no_cpu else None
        print(json.dumps(line), flush=True)
    hx.shutdown()
    if world > 1:
        dist.destroy_process_group()


LAUNCHES_PER_STEP = 1          # hx_decode_step(overlap_ingest=1): the attention kernel carries the handoff (merge is in-kernel too)


def time_kernel(torch, fn, iters=20, warm=5):
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(iters)]
    for a, b in evs:
        a.record()
        fn()
        b.record()
    torch.cuda.synchronize()
    ts = [a.elapsed_time(b) for a, b in evs]
    return float(np.median(ts)), float(np.min(ts))


def time_back_to_back(torch, fn, calls=40, reps=5, warm=5):
    """One CUDA-event pair around `calls` back-to-back launches (as the layers of a model issue them), the
    stream synchronised on both sides; median over `reps`.  Returns ms per call."""
    for _ in range(warm):
        fn()
    ts = []
    for _ in range(reps):
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(calls):
            fn()
        b.record()
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b) / calls)
    return float(np.median(ts))


def other_configs(torch, hx, dev, peak, only=None):
    """Kernel-only numbers for configs[1], [2] (attention) and [3] (80-layer ingest), outside the
    timed step.  Cold L2: each timed call reads a different one of several cache copies.
    `only` (--kernel-only) restricts the run to one of them: a short command to put under ncu."""
    res = {}
    for name in ("opt30b_tp4", "llama70b_tp2", "llama70b_tp1"):
        if name != only and (only is not None or name == "llama70b_tp1"):
            continue
        c = W.CONFIGS[name]
        lens = W.attn_lengths(c)
        need = int(W.pages_for(lens).sum())
        P = int(need * 1.25)
        copies = max(2, int(np.ceil(4 * 126e6 / (need * c.kv_heads * 16 * c.head_dim * 4))))
        bt = torch.from_numpy(W.place_pages(lens, P, c.max_pages, W.rng(c.cfg, W.configs.S_PERM))).to(dev)
        shape = (copies, P, c.kv_heads, 16, c.head_dim)          # "layers" axis used as the copy axis
        k = torch.empty(shape, dtype=torch.float16, device=dev).normal_()
        v = torch.empty(shape, dtype=torch.float16, device=dev).normal_()
        cache = hx.PagedCache(k, v)
        q = torch.empty((c.batch, c.q_heads, c.head_dim), dtype=torch.float16, device=dev).normal_()
        out = torch.empty_like(q)
        sl = torch.from_numpy(lens).to(dev)
        mx = int(lens.max())
        wsb = hx.decode_attention_workspace_bytes(c.batch, c.q_heads, c.kv_heads, c.head_dim, mx)
        ws = torch.zeros(max(wsb, 16), dtype=torch.uint8, device=dev)
        state = {"i": 0}

        def fn():
            state["i"] = (state["i"] + 1) % copies
            hx.decode_attention(out, q, cache, layer=state["i"], q_heads=c.q_heads, block_table=bt,
                                block_table_stride=bt.shape[1], seq_lens=sl, batch=c.batch, max_seq_len=mx,
                                workspace=ws, workspace_bytes=wsb)
        plan = torch.empty(hx.decode_plan_bytes(c.batch, c.kv_heads, mx), dtype=torch.uint8, device=dev)
        hx.decode_plan(plan, cache, q_heads=c.q_heads, block_table=bt, block_table_stride=bt.shape[1], seq_lens=sl, batch=c.batch,
                       max_seq_len=mx)

        def fn_planned():
            state["i"] = (state["i"] + 1) % copies
            hx.decode_attention_planned(out, q, cache, layer=state["i"], q_heads=c.q_heads, plan=plan, batch=c.batch,
                                        max_seq_len=mx, workspace=ws, workspace_bytes=wsb)
        def fn_chained(ready):
            def f():
                state["i"] = (state["i"] + 1) % copies
                hx.decode_attention_chained(out, q, cache, layer=state["i"], q_heads=c.q_heads, plan=plan, batch=c.batch,
                                            max_seq_len=mx, workspace=ws, workspace_bytes=wsb, inputs_ready=ready)
            return f
        med, mn = time_kernel(torch, fn, iters=40)               # one event pair per call (adds ~2 us of event work)
        b2b = time_back_to_back(torch, fn)                       # one event pair around 40 calls: the layer-loop rate
        medp, mnp = time_kernel(torch, fn_planned, iters=40)
        b2bp = time_back_to_back(torch, fn_planned)
        b2bc1 = time_back_to_back(torch, fn_chained(1))          # layer calls as programmatic dependents of one another
        b2bc0 = time_back_to_back(torch, fn_chained(0))
        plan_ms, _ = time_kernel(torch, lambda: hx.decode_plan(plan, cache, q_heads=c.q_heads, block_table=bt,
                                                               block_table_stride=bt.shape[1], seq_lens=sl, batch=c.batch,
                                                               max_seq_len=mx), iters=10)
        kvb = int(lens.astype(np.int64).sum()) * c.kv_heads * c.head_dim * 4
        res[name] = {"kv_bytes": kvb,
                     "per_call_events": {"ms_median": med, "ms_min": mn, "kv_GBps": kvb / med / 1e6, "frac_of_measured": kvb / med / 1e6 / peak,
                                         "frac_of_nominal_8000": kvb / med / 1e6 / NOMINAL_HBM_GBS},
                     "back_to_back": {"ms": b2b, "kv_GBps": kvb / b2b / 1e6, "frac_of_measured": kvb / b2b / 1e6 / peak},
                     "planned_per_call_events": {"ms_median": medp, "ms_min": mnp, "kv_GBps": kvb / medp / 1e6,
                                                 "frac_of_measured": kvb / medp / 1e6 / peak,
                                                 "frac_of_nominal_8000": kvb / medp / 1e6 / NOMINAL_HBM_GBS},
                     "planned_back_to_back": {"ms": b2bp, "kv_GBps": kvb / b2bp / 1e6, "frac_of_measured": kvb / b2bp / 1e6 / peak},
                     "chained_back_to_back": {"ms": b2bc1, "kv_GBps": kvb / b2bc1 / 1e6, "frac_of_measured": kvb / b2bc1 / 1e6 / peak,
                                              "frac_of_nominal_8000": kvb / b2bc1 / 1e6 / NOMINAL_HBM_GBS,
                                              "inputs_ready_0_ms": b2bc0,
                                              "layer_loop": {"ms": b2bc0, "kv_GBps": kvb / b2bc0 / 1e6, "frac_of_measured": kvb / b2bc0 / 1e6 / peak,
                                                             "frac_of_nominal_8000": kvb / b2bc0 / 1e6 / NOMINAL_HBM_GBS,
                                                             "note": "inputs_ready=0: the only mode that is legal behind a kernel that writes q / this "
                                                                     "layer's K/V, i.e. in a real model's layer loop; THIS is the layer-loop figure"},
                                              "note": "hx_decode_attention_chained: each call a programmatic dependent of the one "
                                                      "before it.  ms / kv_GBps / frac_* at this level are inputs_ready=1 (streams under its "
                                                      "predecessor's tail, writes wait; the same q is reused and nothing runs between the calls): an "
                                                      "UPPER BOUND that needs PDL-aware producer kernels.  layer_loop = inputs_ready=0 (only launch + "
                                                      "set-up overlap)"},
                     "plan_ms": plan_ms, "tokens_per_s_one_layer": c.batch / (medp * 1e-3),
                     "timing": "per_call_events: one CUDA-event pair per call (SURVEY 8(d) protocol), median of 40; back_to_back: one event "
                               "pair around 40 calls; planned_*: hx_decode_plan once (plan_ms), then hx_decode_attention_planned per call, "
                               "as the layer loop of a decode step issues them",
                     "l2": f"rotating over {copies} cache copies"}
        del k, v, cache
    if only not in (None, "llama70b_ingest"):
        return res
    # configs[3]: 80-layer ingest, prefill TP=4 -> decode TP=2, both destination ranks
    c = W.CONFIGS["llama70b_ingest"]
    w1 = W.make_ingest_inputs(c, layers=1)
    T, P = w1["total_tokens"], w1["num_pages"]
    L = c.layers
    src_k = [torch.from_numpy(a.view(np.int16)).to(dev).view(torch.float16).expand(L, -1, -1, -1).contiguous() for a in w1["src_k"]]
    src_v = [torch.from_numpy(a.view(np.int16)).to(dev).view(torch.float16).expand(L, -1, -1, -1).contiguous() for a in w1["src_v"]]
    caches = [hx.PagedCache.empty(L, P, c.heads // c.dst_tp, c.head_dim, device=dev) for _ in range(c.dst_tp)]
    bt = torch.from_numpy(w1["block_table"]).to(dev)
    cu = torch.from_numpy(w1["cu_seqlens"]).to(dev)
    sl = torch.from_numpy(w1["seq_lens"]).to(dev)

    def fn():
        for r in range(c.dst_tp):
            hx.kv_ingest(src_k, src_v, layers=L, heads=c.heads, head_dim=c.head_dim, src_tp=c.src_tp, dst_tp=c.dst_tp,
                         dst_rank=r, dst=caches[r], block_table=bt, block_table_stride=bt.shape[1], cu_seqlens=cu,
                         seq_lens=sl, batch=c.prompts, total_tokens=T, max_seq_len=int(w1["seq_lens"].max()))
    med, mn = time_kernel(torch, fn, iters=10, warm=3)
    payload = 2 * L * T * c.heads * c.head_dim * 2
    res[c.name] = {"payload_bytes": payload, "traffic_bytes": 2 * payload, "ms_median": med, "ms_min": mn,
                   "traffic_GBps": 2 * payload / med / 1e6, "frac_of_measured": 2 * payload / med / 1e6 / peak,
                   "frac_of_nominal_8000": 2 * payload / med / 1e6 / NOMINAL_HBM_GBS,
                   "note": "both decode ranks (2 launches); 45+ GB moved per call, far above L2"}
    return res


# ---------------------------------------------------------------------------------------------- oracle legs
def oracle_sample(st, frac=0.5):
    """A bounded sample of the step for the CPU oracle: every 1/frac-th request of the batch (attention,
    host copy of the cache is NOT needed: the oracle gets its own seeded cache of the same shape)
    and 4 of the 16 ingest prompts."""
    ca = st["ca"]
    pick = np.arange(0, ca.batch, int(round(1 / frac)))
    lens = st["lens"][pick]
    c = W.AttnConfig(ca.cfg, "sample", len(pick), ca.q_heads, ca.kv_heads, ca.head_dim, ca.max_pages, "x")
    wa = W.make_attention_inputs(c, lens=lens, spare=1.0)
    ci = st["ci"]
    wi = W.make_ingest_inputs(ci, lens=st["ing_lens"][:4], src_tp=4)
    return wa, wi


def oracle_step(oracle, wa, wi):
    P = wi["num_pages"]
    dk = np.zeros((1, P, wi["heads"], 16, wi["head_dim"]), dtype=np.uint16)
    dv = np.zeros_like(dk)
    t0 = time.perf_counter()
    oracle.kv_ingest(wi["src_k"], wi["src_v"], dk, dv, heads=wi["heads"], src_tp=wi["src_tp"], dst_tp=1, dst_rank=0,
                     block_table=wi["block_table"], cu_seqlens=wi["cu_seqlens"], seq_lens=wi["seq_lens"])
    oracle.decode_attention(wa["q"], wa["k"], wa["v"], wa["block_table"], wa["seq_lens"])
    dt = time.perf_counter() - t0
    return dt, wa["kv_bytes"] + 2 * wi["payload_bytes"]


def cpu_baseline(st):
    import oracle
    oracle.build()
    wa, wi = oracle_sample(st)
    dt, nbytes = oracle_step(oracle, wa, wi)
    return {"value": nbytes / dt / 1e9, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle",
            "seconds": dt, "sample": f"every 2nd request of the cfg5 batch ({len(wa['seq_lens'])} requests, "
            f"{int(wa['seq_lens'].sum())} tokens, all 64 q heads) + ingest of 4 of the 16 prompts; float64 C oracle, OpenMP"}


def run_reference(args, rank):
    if rank != 0:
        return
    import oracle
    oracle.build()
    ca, ci = W.CONFIGS["llama70b_tp1"], W.CONFIGS["llama70b_tp1_ingest"]
    st = dict(ca=ca, ci=ci, lens=W.attn_lengths(ca), ing_lens=W.ingest_lengths(ci))
    wa, wi = oracle_sample(st, frac=1 / 16)        # smaller sample per step so K+W steps end in minutes
    for _ in range(args.warmup):
        oracle_step(oracle, wa, wi)
    times, nbytes = [], 0
    for _ in range(args.steps):
        dt, nbytes = oracle_step(oracle, wa, wi)
        times.append(dt)
    total = float(np.sum(times))
    val = nbytes * args.steps / total / 1e9
    sample = (f"every 16th request of the cfg5 batch ({len(wa['seq_lens'])} requests, {int(wa['seq_lens'].sum())} tokens) "
              f"+ ingest of 4 of the 16 prompts per step")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": total / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic (seeded)",
        "config": {"workload": "configs[4] (bounded sample per step, see cpu_baseline.sample)"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }), flush=True)


def oracle_table(args):
    """BASELINE.md section 5 / SURVEY section 8(d): the oracle as it stands, per config, at 1 thread and at all cores, on
    this box's host cores.  Attention configs run a bounded sample of requests at 1 thread (stated); the whole config
    at all cores.  configs[3] is one of its 80 layers (the oracle handles it one layer at a time)."""
    import oracle
    oracle.build()
    rows = []
    allc = oracle.max_threads()
    for name in ("tiny", "opt30b_tp4", "llama70b_tp2", "llama70b_tp1"):
        c = W.CONFIGS[name]
        w = W.make_attention_inputs(c, spare=1.0)
        for threads, frac in ((1, 1 if name == "tiny" else 8), (allc, 1)):
            pick = np.arange(0, c.batch, frac)
            t0 = time.perf_counter()
            oracle.decode_attention(np.ascontiguousarray(w["q"][pick]), w["k"], w["v"], np.ascontiguousarray(w["block_table"][pick]),
                                    np.ascontiguousarray(w["seq_lens"][pick]), threads=threads)
            dt = time.perf_counter() - t0
            nb = int(w["seq_lens"][pick].astype(np.int64).sum()) * c.kv_heads * c.head_dim * 4
            rows.append({"config": name, "threads": threads, "requests": len(pick), "of": c.batch, "seconds": dt,
                         "kv_GBps": nb / dt / 1e9, "tokens_per_s_one_layer": len(pick) / dt})
    for name, kw in (("tiny_ingest", {}), ("llama70b_ingest", {"layers": 1}), ("llama70b_tp1_ingest", {"src_tp": 4})):
        c = W.CONFIGS[name]
        w = W.make_ingest_inputs(c, **kw)
        for threads in (1, allc):
            for q in range(w["dst_tp"]):
                dk = np.zeros((w["layers"], w["num_pages"], w["heads"] // w["dst_tp"], 16, w["head_dim"]), dtype=np.uint16)
                dv = np.zeros_like(dk)
                t0 = time.perf_counter()
                oracle.kv_ingest(w["src_k"], w["src_v"], dk, dv, heads=w["heads"], src_tp=w["src_tp"], dst_tp=w["dst_tp"], dst_rank=q,
                                 block_table=w["block_table"], cu_seqlens=w["cu_seqlens"], seq_lens=w["seq_lens"], threads=threads)
                dt = time.perf_counter() - t0
                rows.append({"config": name, "threads": threads, "dst_rank": q, "layers": w["layers"], "seconds": dt,
                             "traffic_GBps": 2 * w["payload_bytes"] / w["dst_tp"] / dt / 1e9})
    print(json.dumps({"oracle_table": rows, "host_cores": os.cpu_count(), "oracle_max_threads": allc}), flush=True)


def free_port() -> int:
    with socket.socket() as s_:
        s_.bind(("127.0.0.1", 0))
        return s_.getsockname()[1]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="hx", choices=["hx", "reference"])
    ap.add_argument("--no-extra", action="store_true", help="skip the configs[1..3] kernel-only section")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--oracle-table", action="store_true", help="time the oracle per config at 1 thread and all cores, then exit")
    ap.add_argument("--kernel-only", default=None, choices=["opt30b_tp4", "llama70b_tp2", "llama70b_tp1", "llama70b_ingest", "prefill"],
                    help="time only this config's kernel (no step, no extras) and print a small JSON line: the command to profile")
    args = ap.parse_args()
    if args.oracle_table:
        oracle_table(args)
        return
    if args.impl == "reference":
        run_reference(args, int(os.environ.get("RANK", "0")))     # rank 0 alone works; n_gpus echoes --gpus
        return
    if "WORLD_SIZE" not in os.environ and args.gpus > 1:
        # a bare `python bench.py --gpus N`: start the N ranks ourselves (one process per GPU, replicas only)
        os.execv(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
                                  "--master-addr", "127.0.0.1", "--master-port", str(free_port()),
                                  os.path.abspath(__file__), *sys.argv[1:]])
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    from paper_2502_07903_b200.build import build
    build()
    if args.kernel_only:
        import torch
        import paper_2502_07903_b200 as hx
        torch.cuda.set_device(local_rank)
        torch.manual_seed(1234)
        dev = torch.device("cuda", local_rank)
        peak, _ = measured_peak()
        res = prefill_extra(torch, hx, dev) if args.kernel_only == "prefill" else other_configs(torch, hx, dev, peak, only=args.kernel_only)
        print(json.dumps({"kernel_only": args.kernel_only, "result": res}), flush=True)
        return
    run_hx(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
