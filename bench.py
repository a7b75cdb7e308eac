#!/usr/bin/env python
"""bench.py -- throughput of the paged-KV attention hot path on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A STEP is one pass of the whole hot path (rows a1..a4) over one batch of seeded
synthetic input:
    segment D  (BASELINE.json configs[4], the long-context decode the 70 %-of-HBM target is quoted on):
               mstar_kv_append of the 16 newest rows -> mstar_paged_attn_decode (split-K over 16 partitions
               + LSE combine) over 16 x 32768 tokens scattered in a 60 GiB pool;
    segment P  (configs[2], the prefill the 50 %-of-tensor-peak target is quoted on):
               mstar_kv_append of 8192 new rows -> mstar_paged_attn_prefill, causal over cached prefixes.
`value` is the decode metric (algorithmic K/V GB/s of segment D, inputs resident in HBM); the prefill
metric (TFLOP/s of segment P) rides in `prefill`.  `e2e` is the same decode metric with every per-step
input in pinned HOST memory, copied in and the output copied out inside the timed region (the K/V pool
is serving state and stays resident, like weights).  `roofline` / `roofline_prefill` are algorithmic
bytes (flops) over the CUDA-event duration of the kernel's launches against MEASURED_PEAKS.json.
`cpu_baseline` times the fp64 oracle on the host cores on a bounded sample of segment D.

Multi-GPU: the path does not shard across GPUs ("replicas only"): --gpus N runs N
independent replicas under torchrun, barrier + max-over-ranks timing, value = sum of the replicas' bytes
over the slowest replica's time ("scaling": "weak").
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "paged_decode_attn_GBps"
UNIT = "GB/s"
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}
# `traffic` of the roofline blocks: dram__bytes_read.sum + dram__bytes_write.sum per launch, read at run time from
# the committed summary of the `ncu --set full` capture (profiles/, one row per kernel of a whole step); valid for the
# full-size workloads only, None when the file or a row is missing.
NCU_SUMMARY = os.path.join("profiles", "r2_full_summary.csv")
_UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}


def load_ncu_traffic(path=None):
    """{'decode': bytes, 'prefill': bytes, 'source': file} from the summary CSV (header row, unit row, data rows)."""
    import csv
    path = os.path.join(ROOT, NCU_SUMMARY) if path is None else path
    out = {"decode": None, "prefill": None, "source": None}
    try:
        with open(path, newline="") as f:
            rows = list(csv.reader(f))
        head, units = rows[0], rows[1]
        ik, ir, iw = head.index("Kernel Name"), head.index("dram__bytes_read.sum"), head.index("dram__bytes_write.sum")

        def traffic(row):
            return float(row[ir]) * _UNIT[units[ir]] + float(row[iw]) * _UNIT[units[iw]]

        def first(sub):
            for r in rows[2:]:
                if sub in r[ik]:
                    return traffic(r)
            return None
        sk, cb = first("decode_splitk_kernel<128, 32, 8, 0, 4"), first("decode_combine_kernel")
        out["decode"] = None if sk is None or cb is None else int(sk + cb)
        pf = first("prefill_umma_kernel<16")
        out["prefill"] = None if pf is None else int(pf)
        out["source"] = os.path.relpath(path, ROOT)
    except Exception:
        pass
    return out


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            pk = json.load(f)
        return {"hbm_gbs": float(pk["hbm_gbs"]), "bf16_tflops": float(pk["bf16_tflops"]),
                "bf16_tflops_sustained": float(pk.get("bf16_tflops_sustained", pk["bf16_tflops"])),
                "source": "measured (MEASURED_PEAKS.json)"}
    except Exception:
        return dict(FALLBACK_PEAKS, source="fallback (B200_PROFILING.md)")


# ----------------------------------------------------------------------------- algorithmic work

def decode_bytes(b, nparts):
    """Algorithmic bytes of one decode call: K/V once, Q in, O out, tables, split-K partials write+read."""
    kv = b.kv_bytes_logical()
    S, Hq, D, p = b.num_seqs, b.num_q_heads, b.head_dim, b.page_size
    qo = 2 * S * Hq * D * 2
    tables = 4 * int(((b.seq_lens.astype(np.int64) + p - 1) // p).sum()) + 4 * S
    parts = 0 if nparts <= 1 else 2 * S * Hq * nparts * (D + 2) * 4
    return kv, kv + qo + tables + parts


def prefill_flops(b):
    """sum_s 4 Hq D (n_s P_s + n_s (n_s + 1) / 2): QK^T and PV, 2 flops per MAC, masked triangle excluded."""
    n = b.q_lens.astype(np.float64)
    P = b.seq_lens.astype(np.float64) - n
    return float((4.0 * b.num_q_heads * b.head_dim * (n * P + n * (n + 1) / 2)).sum())


def append_bytes(b):
    return 2 * 2 * b.total_q * b.num_kv_heads * b.head_dim * 2


def pack_step_inputs(torch, D, names):
    """Move the tensors D.<name> into one device buffer (256-byte aligned slices; D.<name> become views into it) and
    build its pinned host image.  Returns (device buffer, pinned host buffer, bytes of one upload)."""
    parts = [getattr(D, n) for n in names]
    offs, total = [], 0
    for t in parts:
        total = (total + 255) // 256 * 256
        offs.append(total)
        total += t.numel() * t.element_size()
    dev_buf = torch.zeros(total, dtype=torch.uint8, device=parts[0].device)
    for n, t, o in zip(names, parts, offs):
        view = dev_buf[o:o + t.numel() * t.element_size()].view(t.dtype).view(t.shape)
        view.copy_(t)
        setattr(D, n, view)
    host = dev_buf.cpu().pin_memory()
    return dev_buf, host, total


# ----------------------------------------------------------------------------- clocks

class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.004):
        super().__init__(daemon=True)
        self.index, self.period = index, period_s
        self.samples, self.reason_bits = [], 0
        self.max_mhz = None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self._stop_evt.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                self.reason_bits |= int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()
        if self.is_alive():
            self.join(timeout=2.0)

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        names = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
                 0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
                 0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}
        reasons = [n for bit, n in names.items() if self.reason_bits & bit and n != "gpu_idle"]
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz, "reasons": reasons,
                "samples": len(self.samples)}


# ----------------------------------------------------------------------------- distributed plumbing (replicas)

def dist_setup(n_gpus: int):
    """Returns (rank, world, local_rank, dist or None).  One process per GPU under torchrun."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world == 1:
        return 0, 1, 0, None
    import torch
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    backend = "nccl" if torch.cuda.is_available() else "gloo"
    if backend == "nccl":
        torch.cuda.set_device(local)
    dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world, local, dist


def max_over_ranks(dist, value: float, device) -> float:
    """Max of a per-rank scalar (device time in ms) over all ranks; identity for a single process."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(dist, value: float, device) -> float:
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


# ----------------------------------------------------------------------------- CPU oracle legs

def oracle_sample_batch(n_seqs: int):
    import workloads as W
    return W.config5_long_context(num_seqs=n_seqs, num_pages=max(4096, n_seqs * 1024 * 2))


def time_oracle_decode(b):
    """Wall seconds of the fp64 oracle (append + decode) on batch b, as it stands."""
    import oracle
    k, v = b.k_store.copy(), b.v_store.copy()
    t0 = time.perf_counter()
    oracle.kv_append(k, v, b.k_new, b.v_new, b.compact_slot_mapping)
    oracle.paged_decode(b.q, k, v, b.compact_block_table, b.seq_lens, b.scale)
    return time.perf_counter() - t0


def cpu_baseline(b):
    """The oracle as it stands on the host cores, on the decode batch the GPU was timed on."""
    import oracle
    time_oracle_decode(b)                      # warm-up (page-faults the buffers)
    dt = min(time_oracle_decode(b) for _ in range(2))
    return {"value": b.kv_bytes_logical() / dt / 1e9, "unit": UNIT, "cores": oracle.num_threads(),
            "kind": "oracle", "seconds": dt,
            "sample": "all %d sequences of configs[4] (32768 tokens, 32q/8kv heads, D 128, page 32), "
                      "append + decode, fp64, best of 2 after one warm-up" % b.num_seqs}


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    n_seqs = 1
    b = oracle_sample_batch(n_seqs)
    for _ in range(args.warmup):
        time_oracle_decode(b)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        time_oracle_decode(b)
    dt = (time.perf_counter() - t0) / max(args.steps, 1)
    val = b.kv_bytes_logical() / dt / 1e9
    sample = ("%d of the 16 sequences of configs[4] per step (32768 tokens, 32q/8kv, D 128, page 32), append + "
              "decode, fp64 oracle" % n_seqs)
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[4] long-context decode, bounded sample", "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ----------------------------------------------------------------------------- the CUDA arm

def other_workloads(torch, mstar, DeviceBatch, W, dev, flush, hbm_peak, iters=15, b_long=None, bf16_peak=1590.0):
    """configs[1] (BAGEL-like CFG-pair decode) and configs[3] (thinker + talker decode): median call time with a
    cold L2, GB/s on logical and on unique K/V bytes (shared prefix pages counted once), sequences per second."""
    ev = lambda: torch.cuda.Event(enable_timing=True)

    def prep(b):
        d = DeviceBatch(b, device=dev)
        d.append()
        S, Hq, Dh = b.num_seqs, b.num_q_heads, b.head_dim
        parts = mstar.decode_auto_partitions(S, b.num_kv_heads, b.max_seq_len)
        out = torch.empty((S, Hq, Dh), dtype=torch.bfloat16, device=dev)
        ws = torch.empty(mstar.decode_workspace_bytes(S, Hq, Dh, parts), dtype=torch.uint8, device=dev)
        call = lambda: mstar.paged_attn_decode(out, d.q_decode, d.pool, d.block_table, d.seq_lens, b.max_seq_len,
                                               float(b.scale), num_partitions=0, workspace=ws)
        return d, call, parts

    def median_ms(calls, streams=None):
        ts = []
        for _ in range(iters + 3):
            # cold L2 with clean lines: a 256 MB read (a fill would leave 126 MB of dirty lines whose write-back
            # the timed call then pays for).  No synchronize before the events: the read kernel is still running
            # while the host enqueues the call, so the timed interval holds GPU work, not host launch latency.
            _ = flush.view(torch.int64).sum()
            e0, e1 = ev(), ev()
            e0.record()
            if streams is None:
                for c in calls:
                    c()
            else:
                cur = torch.cuda.current_stream()
                for c, st in zip(calls, streams):
                    st.wait_stream(cur)
                    with torch.cuda.stream(st):
                        c()
                for st in streams:
                    cur.wait_stream(st)
            e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        ts = sorted(ts[3:])
        return ts[len(ts) // 2]

    def entry(b, ms, parts):
        lg, uq = b.kv_bytes_logical(), b.kv_bytes_unique()
        return {"seqs": b.num_seqs, "q_heads": b.num_q_heads, "kv_heads": b.num_kv_heads, "partitions": parts,
                "us": ms * 1e3, "kv_bytes_logical": lg, "kv_bytes_unique": uq,
                "GBps_logical": lg / (ms * 1e-3) / 1e9, "GBps_unique": uq / (ms * 1e-3) / 1e9,
                "frac_of_measured_hbm_unique": uq / (ms * 1e-3) / 1e9 / hbm_peak,
                "decode_tokens_per_s": b.num_seqs / (ms * 1e-3)}

    res = {"protocol": "one mstar_paged_attn_decode call (split-K + combine), num_partitions = 0 (balanced tile "
                       "ranges), L2 evicted by a 256 MB read before every call, CUDA events, median of %d" % iters}
    b2 = W.config2_bagel_cfg_decode()
    d2, c2, p2 = prep(b2)
    res["configs[1] BAGEL-like CFG-pair decode"] = entry(b2, median_ms([c2]), p2)
    del d2, c2
    bt, bk = W.config4_thinker(), W.config4_talker()
    dt, ct, pt = prep(bt)
    dk, ck, pk = prep(bk)
    res["configs[3] thinker decode"] = entry(bt, median_ms([ct]), pt)
    res["configs[3] talker decode"] = entry(bk, median_ms([ck]), pk)
    s_a, s_b = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)
    ms_both = median_ms([ct, ck], streams=[s_a, s_b])
    # the same two-stream step captured once and replayed as a CUDA graph (the decode calls only enqueue): a call
    # costs the host ~24 us through this binding, about a talker kernel, so the eager figure is partly host-bound
    graph, cap = torch.cuda.CUDAGraph(), torch.cuda.Stream(device=dev)
    with torch.cuda.stream(cap):
        with torch.cuda.graph(graph, stream=cap):
            s_a.wait_stream(cap)
            with torch.cuda.stream(s_a):
                ct()
            s_b.wait_stream(cap)
            with torch.cuda.stream(s_b):
                ck()
            cap.wait_stream(s_a)
            cap.wait_stream(s_b)
    torch.cuda.synchronize()
    ms_both_graph = median_ms([graph.replay])
    tot = bt.kv_bytes_logical() + bk.kv_bytes_logical()
    res["configs[3] thinker || talker (two streams)"] = {
        "us": ms_both * 1e3, "us_cuda_graph_replay": ms_both_graph * 1e3, "kv_bytes_logical": tot,
        "GBps_logical": tot / (ms_both * 1e-3) / 1e9,
        "frac_of_measured_hbm": tot / (ms_both * 1e-3) / 1e9 / hbm_peak,
        "frac_of_measured_hbm_cuda_graph_replay": tot / (ms_both_graph * 1e-3) / 1e9 / hbm_peak,
        "decode_tokens_per_s": (bt.num_seqs + bk.num_seqs) / (ms_both * 1e-3)}
    del graph
    del dk, ct, ck
    # shared-prefix cascade decode (mstar_paged_attn_decode_cascade, one call) against the plain
    # call on the same batch: configs[1] (5 % of the bytes shared) and 16 requests x {2, 3} CFG labels over a shared
    # context of 2048..6144 tokens (about 90 % of the logical bytes shared)
    def cascade_entry(b, n_br, shared):
        d = DeviceBatch(b, device=dev)
        d.append()
        S, Hq, Dh = b.num_seqs, b.num_q_heads, b.head_dim
        parts = mstar.decode_auto_partitions(S, b.num_kv_heads, b.max_seq_len)
        out = torch.empty((S, Hq, Dh), dtype=torch.bfloat16, device=dev)
        ws = torch.empty(mstar.decode_workspace_bytes(S, Hq, Dh, parts), dtype=torch.uint8, device=dev)
        wsc = torch.empty(mstar.decode_cascade_workspace_bytes(S, Hq, b.num_kv_heads, Dh, b.max_seq_len),
                          dtype=torch.uint8, device=dev)
        sh = torch.from_numpy(np.ascontiguousarray(shared, dtype=np.int32)).to(dev)
        ms_p = median_ms([lambda: mstar.paged_attn_decode(out, d.q_decode, d.pool, d.block_table, d.seq_lens,
                                                          b.max_seq_len, float(b.scale), num_partitions=0,
                                                          workspace=ws)])
        ms_c = median_ms([lambda: mstar.paged_attn_decode_cascade(out, d.q_decode, d.pool, d.block_table, d.seq_lens,
                                                                  sh, n_br, b.max_seq_len, float(b.scale),
                                                                  workspace=wsc)])
        lg, uq = b.kv_bytes_logical(), b.kv_bytes_unique()
        return {"seqs": S, "branches": n_br, "kv_bytes_logical": lg, "kv_bytes_unique": uq,
                "plain_us": ms_p * 1e3, "cascade_us": ms_c * 1e3, "cascade_over_plain": ms_c / ms_p,
                "plain_GBps_logical": lg / (ms_p * 1e-3) / 1e9, "cascade_GBps_unique": uq / (ms_c * 1e-3) / 1e9}

    res["cascade decode (SURVEY 8(f) rank 3): configs[1], CFG pairs sharing 256 tokens"] = cascade_entry(
        b2, 2, [256] * (b2.num_seqs // 2))
    for n_br in (2, 3):
        bc, shc = W.cfg_cascade_decode(n_branches=n_br)
        res["cascade decode (SURVEY 8(f) rank 3): 16 requests x %d labels over a shared context" % n_br] = \
            cascade_entry(bc, n_br, shc)
        del bc
    res["cascade decode note"] = ("one call: prefix streams (one consumer warp group per branch, the shared pages "
                                  "pass through shared memory once) + suffix streams + LSE combine; the plain call "
                                  "already fetches shared pages from HBM once when the branches' CTAs read them at "
                                  "the same time (126 MB L2), so the gain is L2 -> SM traffic and SM work")
    # the BAGEL-like denoise (flow) step, 4 requests x 3 CFG labels x 4096 latent tokens,
    # bidirectional block over the cached label context (causal = 0), appended to scratch pages first
    bf = W.flow_step_bagel()
    df = DeviceBatch(bf, device=dev)
    outf = torch.empty((bf.total_q, bf.num_q_heads, bf.head_dim), dtype=torch.bfloat16, device=dev)
    wsf = torch.empty(mstar.prefill_workspace_bytes(bf.num_seqs, bf.total_q, bf.num_q_heads, bf.head_dim),
                      dtype=torch.uint8, device=dev)

    def flow_call():
        mstar.kv_append(df.pool, df.k_new, df.v_new, df.slot_mapping)
        mstar.paged_attn_prefill(outf, df.q, df.cu_seqlens_q, df.pool, df.block_table, df.seq_lens, bf.max_q_len,
                                 bf.max_seq_len, float(bf.scale), causal=False, workspace=wsf)

    ms_f = median_ms([flow_call])
    n = bf.q_lens.astype(np.float64)
    fl = float((4.0 * bf.num_q_heads * bf.head_dim * n * bf.seq_lens.astype(np.float64)).sum())
    res["flow step (SURVEY 8(f) rank 1): 4 requests x 3 CFG labels x 4096 latent tokens, causal = 0"] = {
        "seqs": bf.num_seqs, "new_tokens": int(bf.q_lens[0]), "context": (bf.seq_lens - bf.q_lens).tolist(),
        "ms": ms_f, "flops": fl, "TFLOPs": fl / (ms_f * 1e-3) / 1e12,
        "note": "append of the block's K/V + prefill call; flops = sum 4 Hq D n (context + n)"}
    # page moves (offload / transfer): gather the thinker batch to contiguous rows and copy its
    # pages into the free half of its own pool
    dt2 = DeviceBatch(bt, device=dev)
    cu = np.zeros(bt.num_seqs + 1, dtype=np.int32)
    cu[1:] = np.cumsum(bt.seq_lens)
    cu_d = torch.from_numpy(cu).to(dev)
    kg = torch.empty((int(cu[-1]), bt.num_kv_heads, bt.head_dim), dtype=torch.bfloat16, device=dev)
    vg = torch.empty_like(kg)
    used = np.zeros(bt.num_pages, dtype=bool)
    used[bt.used_pages] = True
    src = torch.from_numpy(bt.used_pages.astype(np.int64)).to(dev)
    dstp = torch.from_numpy(np.flatnonzero(~used)[:len(bt.used_pages)].astype(np.int64)).to(dev)
    ms_g = median_ms([lambda: mstar.kv_gather(kg, vg, dt2.pool, dt2.block_table, dt2.seq_lens, cu_d)])
    ms_c = median_ms([lambda: mstar.kv_copy_pages(dt2.pool, dt2.pool, dstp, src)])
    gb = 2 * bt.kv_bytes_logical()
    cb = 2 * len(bt.used_pages) * 2 * bt.num_kv_heads * bt.page_size * bt.head_dim * 2
    res["page moves (SURVEY 8(f) rank 4) on the thinker pool"] = {
        "gather_us": ms_g * 1e3, "gather_GBps_read_plus_write": gb / (ms_g * 1e-3) / 1e9,
        "copy_pages_us": ms_c * 1e3, "copy_pages": int(len(bt.used_pages)),
        "copy_GBps_read_plus_write": cb / (ms_c * 1e-3) / 1e9,
        "frac_of_measured_copy_rate": cb / (ms_c * 1e-3) / 1e9 / hbm_peak}
    del dt2, kg, vg
    # the quantised pool.  Same batches, K/V as E4M3 codes with per-(page, head) scales written
    # by mstar_kv_append_fp8; one mstar_paged_attn_decode_fp8 call.  Bytes = one byte per element (+ the scales).
    from paper_2606_12688_b200.harness import DeviceBatchFp8

    def fp8_entry(b, parts_arg, seed):
        ks, vs = W.fp8_page_scales(seed, b.num_pages, b.num_kv_heads)
        d = DeviceBatchFp8(b, ks, vs, device=dev)
        d.quantise_store()
        d.append()
        S, Hq, Dh = b.num_seqs, b.num_q_heads, b.head_dim
        parts = parts_arg if parts_arg > 0 else mstar.decode_auto_partitions(S, b.num_kv_heads, b.max_seq_len)
        out = torch.empty((S, Hq, Dh), dtype=torch.bfloat16, device=dev)
        ws = torch.empty(mstar.decode_workspace_bytes(S, Hq, Dh, parts), dtype=torch.uint8, device=dev)
        call = lambda: mstar.paged_attn_decode_fp8(out, d.q_decode, d.pool, d.block_table, d.seq_lens, b.max_seq_len,
                                                   float(b.scale), num_partitions=parts_arg, workspace=ws)
        ms = median_ms([call])
        uq = b.kv_bytes_unique() // 2
        n_pages = int(sum((int(L) + b.page_size - 1) // b.page_size for L in b.seq_lens))
        byt = uq + n_pages * b.num_kv_heads * 8
        return {"seqs": S, "partitions": parts, "us": ms * 1e3, "kv_bytes_unique_fp8": uq,
                "bytes_with_scales": byt, "GBps": byt / (ms * 1e-3) / 1e9,
                "frac_of_measured_hbm": byt / (ms * 1e-3) / 1e9 / hbm_peak,
                "bf16_equivalent_GBps": b.kv_bytes_unique() / (ms * 1e-3) / 1e9,
                "decode_tokens_per_s": S / (ms * 1e-3)}

    def fp8_prefill_entry(b, causal, seed, peak_tf):
        """append_fp8 of the step's new rows + mstar_paged_attn_prefill_fp8 (expand + plan + tcgen05 kernel)."""
        ks, vs = W.fp8_page_scales(seed, b.num_pages, b.num_kv_heads)
        d = DeviceBatchFp8(b, ks, vs, device=dev)
        d.quantise_store()
        T, Hq, Dh = b.total_q, b.num_q_heads, b.head_dim
        from paper_2606_12688_b200.harness import bf16_tensor as _bt
        q = _bt(b.q, dev)
        cu = torch.from_numpy(b.cu_seqlens_q).to(dev)
        out = torch.empty((T, Hq, Dh), dtype=torch.bfloat16, device=dev)
        ws = torch.empty(mstar.prefill_fp8_workspace_bytes(b.num_seqs, T, Hq, b.num_kv_heads, b.page_size,
                                                           b.max_seq_len), dtype=torch.uint8, device=dev)

        def call():
            mstar.kv_append_fp8(d.pool, d.k_new, d.v_new, d.slot_mapping)
            mstar.paged_attn_prefill_fp8(out, q, cu, d.pool, d.block_table, d.seq_lens, b.max_q_len, b.max_seq_len,
                                         float(b.scale), workspace=ws, causal=causal)

        ms = median_ms([call])
        n = b.q_lens.astype(np.float64)
        Lf = b.seq_lens.astype(np.float64)
        fl = float((4.0 * Hq * Dh * (n * (Lf - n) + n * (n + 1) / 2)).sum()) if causal else \
            float((4.0 * Hq * Dh * n * Lf).sum())
        return {"seqs": b.num_seqs, "ms": ms, "flops": fl, "TFLOPs": fl / (ms * 1e-3) / 1e12,
                "frac_of_measured_bf16_burst": fl / (ms * 1e-3) / 1e12 / peak_tf,
                "note": "quantising append of the new rows + expand (codes -> exact bf16 scratch pool) + plan + "
                        "tcgen05 kernel with per-page scales; the MMAs are bf16 (kind::f16), so the bf16 peak applies"}

    res["fp8 pool (SURVEY 8(f) rank 4): configs[2] causal prefill"] = fp8_prefill_entry(W.config3_prefill(), True, 84,
                                                                                         bf16_peak)
    res["fp8 pool (SURVEY 8(f) rank 4): flow step, causal = 0"] = fp8_prefill_entry(bf, False, 85, bf16_peak)
    # SURVEY 8(f) rank 4, last clause: CUDA-graph-compatible sampling, 64 rows over a 151 936-entry vocabulary
    def sampling_entry(dtype, use_filters):
        Bs, Vs = 64, 151936
        g = torch.Generator(device=dev)
        g.manual_seed(5)
        lg = (torch.randn((Bs, Vs), device=dev, generator=g) * 3.0).to(dtype)
        seeds = torch.arange(Bs, dtype=torch.int64, device=dev) + 1000
        step = torch.zeros(1, dtype=torch.int64, device=dev)
        tk = torch.full((Bs,), 50 if use_filters else 0, dtype=torch.int32, device=dev)
        tp = torch.full((Bs,), 0.9 if use_filters else 1.0, dtype=torch.float32, device=dev)
        tt = torch.full((Bs,), 0.8, dtype=torch.float32, device=dev)
        tok = torch.empty(Bs, dtype=torch.int32, device=dev)
        ms = median_ms([lambda: mstar.sample_tokens(tok, lg, seeds, step, temperature=tt, top_k=tk, top_p=tp,
                                                    advance_step=True)])
        nbytes = Bs * Vs * lg.element_size()
        return {"rows": Bs, "vocab": Vs, "logits": str(dtype).split(".")[-1], "top_k": int(tk[0]),
                "top_p": float(tp[0]), "us": ms * 1e3, "tokens_per_s": Bs / (ms * 1e-3),
                "logit_bytes": nbytes, "GBps_one_read_of_the_logits": nbytes / (ms * 1e-3) / 1e9,
                "kernel": "cluster of 8 CTAs per row, the row read from HBM once and kept in shared memory"}

    res["sampling (SURVEY 8(f) rank 4): temperature only, fp32 logits"] = sampling_entry(torch.float32, False)
    res["sampling (SURVEY 8(f) rank 4): top-k 50 + top-p 0.9, fp32 logits"] = sampling_entry(torch.float32, True)
    res["sampling (SURVEY 8(f) rank 4): top-k 50 + top-p 0.9, bf16 logits"] = sampling_entry(torch.bfloat16, True)
    res["fp8 pool (SURVEY 8(f) rank 4): configs[1] decode"] = fp8_entry(b2, 0, 81)
    res["fp8 pool (SURVEY 8(f) rank 4): configs[3] thinker decode"] = fp8_entry(bt, 0, 82)
    if b_long is not None:
        res["fp8 pool (SURVEY 8(f) rank 4): configs[4] long-context decode, 16 partitions"] = fp8_entry(b_long, 16, 83)
    return res


def run_ours(args):
    import torch
    rank, world, local, dist = dist_setup(args.gpus)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback; use --impl reference "
                         "for the oracle timing)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    import paper_2606_12688_b200 as mstar
    from paper_2606_12688_b200.harness import DeviceBatch, bf16_tensor
    import workloads as W
    mstar.load_library()
    peaks = load_peaks()
    ncu_traffic = load_ncu_traffic()

    # ---- inputs (seeded, host-generated, uploaded once)
    free, _ = torch.cuda.mem_get_info()
    pool_pages = 491520 if free > 72 * (1 << 30) else 65536
    bd = W.config5_long_context(num_pages=pool_pages)
    bp = W.config3_prefill()
    D5 = DeviceBatch(bd, device=dev)
    # the per-step inputs of segment D live back to back in ONE device buffer (the batch's tensors are views into it),
    # so that the end-to-end step uploads them from pinned host memory with one copy, as a serving engine would
    step_dev, step_host, h2d = pack_step_inputs(torch, D5, ("q_decode", "k_new", "v_new", "slot_mapping", "block_table",
                                                           "seq_lens"))
    D3 = DeviceBatch(bp, device=dev)
    NPARTS = 16
    S5, Hq5, Dh = bd.num_seqs, bd.num_q_heads, bd.head_dim
    out5 = torch.empty((S5, Hq5, Dh), dtype=torch.bfloat16, device=dev)
    ws5 = torch.empty(mstar.decode_workspace_bytes(S5, Hq5, Dh, NPARTS), dtype=torch.uint8, device=dev)
    out3 = torch.empty((bp.total_q, bp.num_q_heads, bp.head_dim), dtype=torch.bfloat16, device=dev)
    ws3 = torch.empty(mstar.prefill_workspace_bytes(bp.num_seqs, bp.total_q, bp.num_q_heads, bp.head_dim),
                      dtype=torch.uint8, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2
    msl5, msl3, mql3 = bd.max_seq_len, bp.max_seq_len, bp.max_q_len
    sc5, sc3 = float(bd.scale), float(bp.scale)
    launches = [0]

    def seg_decode():
        mstar.kv_append(D5.pool, D5.k_new, D5.v_new, D5.slot_mapping); launches[0] += mstar.last_launch_count()
        mstar.paged_attn_decode(out5, D5.q_decode, D5.pool, D5.block_table, D5.seq_lens, msl5, sc5,
                                num_partitions=NPARTS, workspace=ws5); launches[0] += mstar.last_launch_count()

    def seg_prefill():
        mstar.kv_append(D3.pool, D3.k_new, D3.v_new, D3.slot_mapping); launches[0] += mstar.last_launch_count()
        mstar.paged_attn_prefill(out3, D3.q, D3.cu_seqlens_q, D3.pool, D3.block_table, D3.seq_lens, mql3, msl3,
                                 sc3, causal=True, workspace=ws3); launches[0] += mstar.last_launch_count()

    ev = lambda: torch.cuda.Event(enable_timing=True)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        seg_decode(); flush.fill_(1); seg_prefill()
    barrier()

    # ---- timed region: K steps, CUDA events per segment and per kernel group on the launching stream
    K = args.steps
    sampler = ClockSampler(local)
    sampler.start()
    launches[0] = 0
    marks = []
    t_wall0 = time.perf_counter()
    for _ in range(K):
        e = [ev() for _ in range(6)]
        e[0].record()
        mstar.kv_append(D5.pool, D5.k_new, D5.v_new, D5.slot_mapping); launches[0] += mstar.last_launch_count()
        e[1].record()
        mstar.paged_attn_decode(out5, D5.q_decode, D5.pool, D5.block_table, D5.seq_lens, msl5, sc5,
                                num_partitions=NPARTS, workspace=ws5); launches[0] += mstar.last_launch_count()
        e[2].record()
        flush.fill_(1)          # L2 flush between segments, outside the timed events
        e[3].record()
        mstar.kv_append(D3.pool, D3.k_new, D3.v_new, D3.slot_mapping); launches[0] += mstar.last_launch_count()
        e[4].record()
        mstar.paged_attn_prefill(out3, D3.q, D3.cu_seqlens_q, D3.pool, D3.block_table, D3.seq_lens, mql3, msl3,
                                 sc3, causal=True, workspace=ws3); launches[0] += mstar.last_launch_count()
        e[5].record()
        marks.append(e)
    barrier()
    wall_ms = (time.perf_counter() - t_wall0) * 1e3 / K
    sampler.stop()
    timed_launches = launches[0]
    t_app5 = sum(m[0].elapsed_time(m[1]) for m in marks) / K
    t_dec = sum(m[1].elapsed_time(m[2]) for m in marks) / K
    t_app3 = sum(m[3].elapsed_time(m[4]) for m in marks) / K
    t_pre = sum(m[4].elapsed_time(m[5]) for m in marks) / K
    t_segD = max_over_ranks(dist, t_app5 + t_dec, dev)
    t_segP = max_over_ranks(dist, t_app3 + t_pre, dev)
    t_dec_max = max_over_ranks(dist, t_dec, dev)
    t_pre_max = max_over_ranks(dist, t_pre, dev)

    kv_bytes, dec_bytes = decode_bytes(bd, NPARTS)
    flops = prefill_flops(bp)
    value = world * kv_bytes / (t_segD * 1e-3) / 1e9
    tokens_per_s = world * S5 / (t_segD * 1e-3)

    # ---- e2e: per-step inputs in pinned host memory, copied in; output copied out; same kernels
    h_out = torch.empty(out5.shape, dtype=out5.dtype).pin_memory()
    d2h = h_out.numel() * h_out.element_size()

    def e2e_step():
        step_dev.copy_(step_host, non_blocking=True)
        seg_decode()
        h_out.copy_(out5, non_blocking=True)

    for _ in range(3):
        e2e_step()
    barrier()
    e0, e1 = ev(), ev()
    e0.record()
    for _ in range(K):
        e2e_step()
    e1.record()
    barrier()
    t_e2e = max_over_ranks(dist, e0.elapsed_time(e1) / K, dev)
    e2e_value = world * kv_bytes / (t_e2e * 1e-3) / 1e9

    # ---- the serving-shaped decode configs (BAGEL CFG pairs, Qwen3-Omni thinker / talker): reported beside the
    # headline, outside the K timed steps; cold L2 (flush before every call), CUDA events, median of 15
    # ---- practical HBM-read ceiling: a read-only streaming kernel over 4 GiB of the K pool (K bytes
    # of random pages, the same memory the decode kernel streams), CUDA events, median of 7 after 2 warm-ups
    read_ceiling = None
    if rank == 0:
        from paper_2606_12688_b200 import bench_aux
        nbytes = min(4 << 30, D5.k_pool.numel() * 2)
        ts = []
        for _ in range(9):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            bench_aux.hbm_read_probe(D5.k_pool, nbytes)
            e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        ms_probe = sorted(ts[2:])[len(ts[2:]) // 2]
        read_ceiling = {"GBps": nbytes / (ms_probe * 1e-3) / 1e9, "bytes": nbytes, "ms": ms_probe,
                        "kernel": "bench_aux hbm_read_probe (16-byte read-only loads, 8 in flight per thread)"}

    other = None
    if rank == 0 and not args.no_other:
        other = other_workloads(torch, mstar, DeviceBatch, W, dev, flush, hbm_peak=peaks["hbm_gbs"], b_long=bd,
                                bf16_peak=peaks["bf16_tflops"])

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    clocks = sampler.summary()
    hbm_peak, tf_peak = peaks["hbm_gbs"], peaks["bf16_tflops"]
    dec_gbs = dec_bytes / (t_dec_max * 1e-3) / 1e9
    pre_tfs = flops / (t_pre_max * 1e-3) / 1e12
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K,
        "warmup": max(args.warmup, 3), "ms_per_step": t_segD + t_segP, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {
            "workload": "configs[4] long-context decode (a1 append 16 rows + a2 split-K x16 + a3 combine) then "
                        "configs[2] causal prefill over cached prefix (a1 append 8192 rows + a4)",
            "decode": {"seqs": S5, "seq_len": msl5, "q_heads": Hq5, "kv_heads": bd.num_kv_heads, "head_dim": Dh,
                       "page_size": bd.page_size, "pool_pages": pool_pages, "partitions": NPARTS,
                       "kv_bytes": kv_bytes},
            "prefill": {"seqs": bp.num_seqs, "new_tokens": int(bp.q_lens[0]), "prefix": (bp.seq_lens - bp.q_lens).tolist(),
                        "q_heads": bp.num_q_heads, "kv_heads": bp.num_kv_heads, "head_dim": bp.head_dim,
                        "page_size": bp.page_size, "flops": flops},
            "l2": "decode reads 2.1 GB per step (>> 126 MB L2); a 256 MB flush write runs before the prefill "
                  "segment, outside the timed events",
            "parallelism": "replicas" if world > 1 else "single GPU",
        },
        "ms_decode_segment": t_segD, "ms_prefill_segment": t_segP, "wall_ms_per_step": wall_ms,
        "decode_tokens_per_s": tokens_per_s,
        "prefill": {"metric": "paged_prefill_attn_TFLOPs", "value": world * flops / (t_segP * 1e-3) / 1e12,
                    "unit": "TFLOP/s", "ms": t_segP, "append_GBps": append_bytes(bp) / (t_app3 * 1e-3) / 1e9},
        "roofline": {"kernel": "decode_splitk_kernel + decode_combine_kernel (one mstar_paged_attn_decode call)",
                     "bound": "hbm", "achieved": dec_gbs, "peak": hbm_peak, "unit": "GB/s",
                     "frac": dec_gbs / hbm_peak,
                     "traffic": ncu_traffic["decode"] if pool_pages == 491520 else None,
                     "traffic_source": ncu_traffic["source"], "peak_source": peaks["source"],
                     "frac_of_nominal_8TBps": dec_gbs / 8000.0, "ms": t_dec_max, "bytes": dec_bytes,
                     "hbm_read_ceiling": read_ceiling,
                     "frac_of_read_ceiling": (dec_gbs / read_ceiling["GBps"]) if read_ceiling else None},
        "roofline_prefill": {"kernel": "prefill kernel (one mstar_paged_attn_prefill call)", "bound": "tensor",
                             "achieved": pre_tfs, "peak": tf_peak, "unit": "TFLOP/s", "frac": pre_tfs / tf_peak,
                             "traffic": ncu_traffic["prefill"], "traffic_source": ncu_traffic["source"],
                             "peak_source": peaks["source"] + ", burst",
                             "frac_of_sustained": pre_tfs / peaks["bf16_tflops_sustained"],
                             "frac_of_nominal_2250": pre_tfs / 2250.0, "ms": t_pre_max, "flops": flops},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms": t_e2e, "note": "segment D with q, new K/V rows, slot mapping, block table and seq_lens (packed, one upload) in "
                                     "pinned host memory; the K/V pool is resident serving state.  Steps run back to "
                                     "back (a step reads 17x the L2 in K/V); the upload leaves the step's inputs in L2, "
                                     "whereas `value` is timed behind an L2 flush with cold metadata"},
        "gpu_launches": timed_launches,
        "clocks": clocks,
    }
    if other is not None:
        line["other_workloads"] = other
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(bd)
    elif not args.no_cpu_baseline:
        line["cpu_baseline"] = {"value": None, "unit": UNIT, "cores": None, "kind": "oracle",
                                "sample": "reported at N=1 only"}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


def run_sustained(args):
    """--sustained: each kernel of the path launched back to back for a few seconds while NVML samples board power,
    SM clock and throttle reasons, next to a cuBLAS bf16 GEMM and a device copy under the same regime.  Not the bench
    line: it shows which limit (power cap, clock) the measured rates sit under.  One JSON object on stdout."""
    import pynvml as nv
    import torch
    import paper_2606_12688_b200 as mstar
    import workloads as W
    from paper_2606_12688_b200.harness import DeviceBatch
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    mstar.load_library()
    nv.nvmlInit()
    h = nv.nvmlDeviceGetHandleByIndex(0)
    out = {"mode": "sustained", "seconds_per_kernel": args.sustained,
           "power_limit_w": nv.nvmlDeviceGetEnforcedPowerLimit(h) / 1e3,
           "sm_max_mhz": int(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)), "kernels": {}}
    names = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
             0x80: "hw_power_brake_slowdown"}

    def sustained(name, call, work, unit):
        stop, samples = threading.Event(), []

        def sampler():
            while not stop.is_set():
                samples.append((nv.nvmlDeviceGetPowerUsage(h) / 1e3, nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM),
                                nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)))
                time.sleep(0.02)
        th = threading.Thread(target=sampler, daemon=True)
        call()
        torch.cuda.synchronize()
        th.start()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0, n = time.time(), 0
        e0.record()
        while time.time() - t0 < args.sustained:
            for _ in range(50):
                call()
            n += 50
            torch.cuda.synchronize()
        e1.record()
        torch.cuda.synchronize()
        stop.set()
        th.join()
        smp = samples[len(samples) // 3:] or samples
        bits = 0
        for x in smp:
            bits |= x[2]
        us = e0.elapsed_time(e1) * 1e3 / n
        out["kernels"][name] = {"us_per_call": us, "rate": work / (us * 1e-6), "unit": unit,
                                "power_w_median": float(np.median([x[0] for x in smp])),
                                "sm_mhz_median": float(np.median([x[1] for x in smp])),
                                "reasons": [v for k, v in names.items() if bits & k]}

    def prefill_call(b, causal):
        d = DeviceBatch(b, device=dev)
        d.append()
        o = torch.empty((b.total_q, b.num_q_heads, b.head_dim), dtype=torch.bfloat16, device=dev)
        ws = torch.empty(mstar.prefill_workspace_bytes(b.num_seqs, b.total_q, b.num_q_heads, b.head_dim),
                         dtype=torch.uint8, device=dev)
        return lambda: mstar.paged_attn_prefill(o, d.q, d.cu_seqlens_q, d.pool, d.block_table, d.seq_lens, b.max_q_len,
                                                b.max_seq_len, float(b.scale), causal=causal, workspace=ws)

    b3 = W.config3_prefill()
    sustained("prefill configs[2] (plan + attention)", prefill_call(b3, True), prefill_flops(b3) / 1e12, "TFLOP/s")
    bf = W.flow_step_bagel()
    n, L = bf.q_lens.astype(np.float64), bf.seq_lens.astype(np.float64)
    sustained("prefill flow step, causal = 0", prefill_call(bf, False),
              float((4.0 * bf.num_q_heads * bf.head_dim * n * L).sum()) / 1e12, "TFLOP/s")
    a = torch.randn(8192, 8192, device=dev, dtype=torch.bfloat16)
    bm = torch.randn(8192, 8192, device=dev, dtype=torch.bfloat16)
    c = torch.empty(8192, 8192, device=dev, dtype=torch.bfloat16)
    sustained("cuBLAS bf16 GEMM 8192^3", lambda: torch.matmul(a, bm, out=c), 2 * 8192.0 ** 3 / 1e12, "TFLOP/s")
    del a, bm, c
    x = torch.empty(1 << 30, dtype=torch.uint8, device=dev)
    y = torch.empty_like(x)
    sustained("device copy 1 GiB", lambda: y.copy_(x), 2 * float(1 << 30) / 1e9, "GB/s read + write")
    del x, y
    b2 = W.config2_bagel_cfg_decode()
    d2 = DeviceBatch(b2, device=dev)
    d2.append()
    sustained("decode configs[1] (warm L2)", lambda: d2.decode(num_partitions=0), b2.kv_bytes_unique() / 1e9,
              "GB/s of unique K/V")
    print(json.dumps(out))
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other", action="store_true", help="skip the configs[1] / configs[3] decode timings")
    ap.add_argument("--sustained", type=float, default=0.0, metavar="SECONDS",
                    help="instead of the bench line: power / clock of each kernel launched back to back for SECONDS")
    args = ap.parse_args(argv)
    if args.impl == "reference":
        return run_reference(args)
    if args.sustained > 0:
        return run_sustained(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # plain `python bench.py --gpus N`: become N ranks (one per GPU) under torchrun on this node
        return respawn_under_torchrun(args.gpus, sys.argv[1:] if argv is None else list(argv))
    return run_ours(args)


def torchrun_command(n_gpus: int, argv, port=None):
    """The command line `python bench.py --gpus N` turns itself into when it is not already under torchrun."""
    if port is None:
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(n_gpus),
            "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *argv]


def respawn_under_torchrun(n_gpus: int, argv):
    import subprocess
    return subprocess.call(torchrun_command(n_gpus, argv))


if __name__ == "__main__":
    sys.exit(main())
