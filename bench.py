#!/usr/bin/env python
"""bench.py — throughput of UltraQuant's hot path on B200 (driver contract: see README/DESIGN.md).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2|3|5|1]

One STEP = one pass of the whole hot path over one decode batch:
  uq_rotate_quantize_append  (1 new K/V token per sequence: rotate, scale, encode, paged store;
                              plus the step's queries: rotate + FP8 cast)
  uq_decode_attention        (paged split-K FP8 x FP4 attention over the whole context)
  uq_merge_splits            (split partials -> bf16 output)
Workload (default): BASELINE.json configs[1] — Qwen3-235B-shaped layer, 64 Q / 4 KV heads,
head_dim 128, batch 32, every sequence at 32,768 tokens, page_size 16, random block tables,
K,V bf16 ~ N(0,1) with 3 K channels x8 (seed 1).  The cache is prefilled to 32,767 tokens per
sequence through uq_rotate_quantize_append; every timed step appends token 32,768 (into the
same slot each step, so the context stays at exactly 32,768) and decodes over 32,768 tokens.

Metric = BASELINE.json's "decode-attention HBM GB/s": algorithmic bytes the step must move
(136 B per (token, kv_head) of K+V codes and scales, block tables, Q, O, split partials, the
appended rows — SURVEY.md §8(d)) divided by the device time of the step.  us/step and the
fractions of the nominal 8 TB/s and of the measured copy peak ride along in the same line.

--impl reference times the float64 CPU oracle (oracle/) on the same metric and config; it and
the cpu_baseline leg are the only places this file touches oracle/.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np
import torch

METRIC = "decode_attention_hbm_gbps"
UNIT = "GB/s"
NOMINAL_HBM_GBS = 8000.0          # BASELINE.json north_star: "the B200's ~8 TB/s peak"
FALLBACK_HBM_GBS = 6650.0         # /opt/skills/guides/B200_PROFILING.md fallback



def _source_key() -> str:
    """sha256 (first 16 hex digits) over the CUDA sources the library is built from, in name order: identifies the
    BUILD a profile was taken of (the GPU box has no .git, so a commit id is not available at run time)."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2606_20474_b200", "csrc")
    for fn in sorted(os.listdir(d)):
        if fn.endswith((".cu", ".cuh")):
            h.update(fn.encode()); h.update(open(os.path.join(d, fn), "rb").read())
    return h.hexdigest()[:16]


def _ncu_traffic(kernel: str, workload_key: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` from the `ncu --set full` capture recorded
    in profiles/ncu_traffic.json — only if that capture was taken of THIS build (same source key); else None."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.json")) as f:
            tab = json.load(f)
    except Exception:
        return None
    key = _source_key()
    for e in tab.get("captures", []):
        if e.get("source_key") == key and e.get("kernel") == kernel and e.get("workload") == workload_key:
            return int(e["dram_bytes_read"]) + int(e["dram_bytes_write"])
    return None


# ----------------------------------------------------------------------------- helpers
def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy read+write)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s; MEASURED_PEAKS.json absent)"


KV_FORMAT = "fp4"                 # --kv: fp4 = UltraQuant (the product); fp8 / bf16 = the paper's comparison caches
HEAD_DIM = 128                    # --head-dim: the config's shape at another head size (64 / 256)


def _workload(idx: int, rank: int):
    import dataclasses

    from paper_2606_20474_b200 import workloads as W
    wl = W.make_config(idx, peaked_frac=0.0, head_dim=HEAD_DIM)
    if rank:
        wl = dataclasses.replace(wl, seed=wl.seed + 1000 * rank)   # other values, same structure
    return wl


def step_bytes(wl, num_splits: int, ctx_after: np.ndarray, new_per_seq: int):
    """Algorithmic bytes of one step; returns (total, decode_kernel_only)."""
    d, Hq, Hkv, B = wl.head_dim, wl.num_q_heads, wl.num_kv_heads, wl.batch
    per_tok = 2 * (d // 2 + d // 32)                                 # 136 B
    if KV_FORMAT == "fp8":
        per_tok = 2 * d                                              # comparison cache: one E4M3 byte per element
    elif KV_FORMAT == "bf16":
        per_tok = 4 * d
    elif KV_FORMAT == "tq":
        per_tok = 2432 // 16                                         # Ultra-TQ record: 152 B per (token, kv head)
    tokens = int(ctx_after.astype(np.int64).sum())
    pages = int(((ctx_after.astype(np.int64) + wl.page_size - 1) // wl.page_size).sum())
    kv = tokens * Hkv * per_tok
    bt = 4 * pages
    q8 = B * Hq * d
    partials = B * Hq * num_splits * (4 * d + 8)
    decode = kv + bt + q8 + partials                                 # decode kernel: read KV, tables, Q; write partials
    merge = partials + B * Hq * d * 2                                # read partials, write bf16 O
    n_new = B * new_per_seq
    append = n_new * Hkv * (2 * d * 2 + per_tok) + B * Hq * (2 * d + d)   # read bf16 K,V rows + Q; write records + q_fp8
    return decode + merge + append, decode


def max_over_ranks(values, world: int, device="cpu"):
    """MAX over ranks of a list of per-rank timings (the contract's "max over ranks"); the data path
    itself has no collective.  Works with any initialised backend (NCCL on GPUs, gloo in the CPU test)."""
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world > 1:
        torch.distributed.all_reduce(t, op=torch.distributed.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def whole_job_value(bytes_per_rank: int, world: int, ms_per_step: float) -> float:
    """Aggregate GB/s of `world` replicas that each move bytes_per_rank per step (weak scaling)."""
    return world * bytes_per_rank / (ms_per_step * 1e-3) / 1e9


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed regions run."""

    def __init__(self, index: int, period_s: float = 0.005):
        super().__init__(daemon=True)
        self.period = period_s
        self.samples = []            # (window label or None/False, sm_mhz, reasons bitmask)
        self.busy = False            # label of the timed window being sampled (True = the default one)
        self._stop_evt = threading.Event()
        self.ok = False
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:     # no NVML: the line says so instead of inventing clocks
            self.err = repr(e)

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self._stop_evt.is_set():
            try:
                mhz = int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                reasons = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                self.samples.append((self.busy, mhz, reasons))
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()

    def summary(self, label=None):
        """Clocks over the samples of one labelled window (label given) or of every timed window except 'sustain'."""
        if not self.ok:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml_unavailable"]}
        nv = self.nv
        if label is not None:
            busy = [s for s in self.samples if s[0] == label]
        else:
            busy = [s for s in self.samples if s[0] and s[0] != "sustain"] or self.samples
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake_slowdown",
        }
        seen = set()
        for _, _, r in busy:
            for bit, nm in names.items():
                if r & bit:
                    seen.add(nm)
        return {"sm_mhz": (statistics.median([s[1] for s in busy]) if busy else None),
                "sm_max_mhz": self.max_mhz, "reasons": sorted(seen), "samples": len(busy)}


# ----------------------------------------------------------------------------- our arm
def fill_cache(uq, W, cfg, wl, lens, device, chunk_tokens=1 << 16):
    """Prefill through uq_rotate_quantize_append (bulk appends); shared prefix written once."""
    fmt = {"fp8": uq.KV_FP8_E4M3, "bf16": uq.KV_BF16, "tq": uq.KV_ULTRA_TQ}.get(KV_FORMAT)
    cache = uq.alloc_cache(cfg, wl.num_pages, device) if fmt is None else uq.alloc_baseline_cache(cfg, fmt, wl.num_pages, device)
    bt_dev = torch.from_numpy(wl.block_tables).to(device)
    B = wl.batch

    def put(b_gen, b_tab, start, n_total):
        done = 0
        while done < n_total:
            n = min(chunk_tokens, n_total - done)
            k, v = W.gen_kv(wl, b_gen, done, done + n, device)
            before = np.zeros(B, np.int32); before[b_tab] = start + done
            cu = np.zeros(B + 1, np.int32); cu[b_tab + 1:] = n
            if fmt is None:
                uq.rotate_quantize_append(cfg, k, v, torch.from_numpy(cu).to(device),
                                          torch.from_numpy(before).to(device), bt_dev, cache)
            elif fmt == uq.KV_ULTRA_TQ:
                uq.tq_append(cfg, W.TQ_CODEBOOK, k, v, torch.from_numpy(cu).to(device), torch.from_numpy(before).to(device),
                             bt_dev, cache)
            else:
                uq.baseline_append(cfg, fmt, k, v, torch.from_numpy(cu).to(device), torch.from_numpy(before).to(device),
                                   bt_dev, cache)
            done += n

    if wl.prefix_len:
        put(-1, 0, 0, wl.prefix_len)
    for b in range(B):
        put(b, b, wl.prefix_len, int(lens[b]) - wl.prefix_len)
    torch.cuda.synchronize()
    return cache, bt_dev


def run_ours(args, rank, world, local_rank):
    import paper_2606_20474_b200 as uq
    from paper_2606_20474_b200 import workloads as W

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the hot path has no CPU fallback")
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    wl = _workload(args.config, rank)
    # the timed step appends ONE token per sequence right before the decode: the promise of UQ_FLAG_SMALL_APPEND_AHEAD
    cfg = uq.UQConfig(num_q_heads=wl.num_q_heads, num_kv_heads=wl.num_kv_heads, head_dim=wl.head_dim,
                      flags=0 if args.no_early else uq.FLAG_SMALL_APPEND_AHEAD)
    B, Hq, Hkv, d = wl.batch, wl.num_q_heads, wl.num_kv_heads, wl.head_dim

    # context AFTER the step's append = the config's lengths; the cache holds one token less
    ctx_after = wl.ctx_lens.astype(np.int32)
    ctx_before = ctx_after - 1
    cache, bt_dev = fill_cache(uq, W, cfg, wl, ctx_before, dev)
    S = args.splits or uq.suggest_num_splits(cfg, B, int(ctx_after.mean()))
    bufs = uq.StepBuffers(cfg, B, S, dev)

    # a small ring of per-step inputs (different values each step)
    n_in = 4
    qs = [W.gen_q(wl, dev, step=i) for i in range(n_in)]
    wl1 = wl if wl.new_tokens == 1 else __import__("dataclasses").replace(wl, new_tokens=1)
    kvs = [W.gen_new_kv(wl1, i, dev) for i in range(n_in)]
    cu_dev = torch.arange(B + 1, dtype=torch.int32, device=dev)
    before_dev = torch.from_numpy(ctx_before).to(dev)
    after_dev = torch.from_numpy(ctx_after).to(dev)
    stream = torch.cuda.current_stream()

    # one CUDA graph per entry of the input ring (uq.StepGraph: the step's three kernels, one launch for the host)
    step_graphs = None
    if args.graph:
        step_graphs = [uq.StepGraph(cfg, bufs, qs[j], kvs[j][0], kvs[j][1], cu_dev, before_dev, after_dev, bt_dev, cache)
                       for j in range(n_in)]

    # --shared-prefix 1 (configs with a shared prefix): the prefix through uq_decode_prefix_attention (8 or 16 sequences
    # per prefix tile), the private suffixes through uq_decode_attention, uq_merge_splits2 over both sets of partials
    pbufs, pfx = None, 0
    if args.shared_prefix and wl.prefix_len >= 128:
        pfx = (int(wl.prefix_len) // 128) * 128
        pbufs = uq.PrefixBuffers(cfg, B, uq.suggest_prefix_splits(cfg, B, pfx), dev)
        pbufs.suffix_lens.copy_(torch.from_numpy((ctx_after - pfx).astype(np.int32)))
        # slots of the suffix call: the suffix lengths are far more skewed than the whole lengths (config 4: mean 16.5k,
        # maximum 98k), and the balanced schedule lengthens every CTA's range until the longest item fits into S - 1
        # of them — so S follows from the longest suffix, which the host knows (uq_suggest_num_splits_max)
        suf = (ctx_after - pfx).astype(np.int64)
        S_suffix = args.splits or uq.suggest_num_splits_max(cfg, B, max(1, int(suf.mean())), int(suf.max()))
        bufs_sp = uq.StepBuffers(cfg, B, S_suffix, dev)

    fmt = {"fp8": uq.KV_FP8_E4M3, "bf16": uq.KV_BF16, "tq": uq.KV_ULTRA_TQ}.get(KV_FORMAT)
    q_rot = torch.empty_like(qs[0]) if fmt == uq.KV_ULTRA_TQ else None

    def step(i):
        if fmt == uq.KV_ULTRA_TQ:                        # Alg. 2: append + rotated bf16 query, codebook decode, merge
            k_new, v_new = kvs[i % n_in]
            uq.tq_append(cfg, W.TQ_CODEBOOK, k_new, v_new, cu_dev, before_dev, bt_dev, cache, q=qs[i % n_in], q_rot=q_rot,
                         stream=stream)
            uq.tq_decode_attention(cfg, W.TQ_CODEBOOK, q_rot, cache, bt_dev, after_dev, S, bufs.partial_acc, bufs.partial_ml,
                                   stream=stream)
            uq.merge_splits(cfg, bufs.partial_acc, bufs.partial_ml, bufs.out, stream=stream)
            return bufs.out
        if fmt is not None:                              # comparison cache: append, decode, merge over FP8 / BF16 KV
            k_new, v_new = kvs[i % n_in]
            return uq.baseline_decode_step(cfg, fmt, bufs, qs[i % n_in], k_new, v_new, cu_dev, before_dev, after_dev,
                                           bt_dev, cache, stream=stream)
        if pbufs is not None:
            k_new, v_new = kvs[i % n_in]
            uq.rotate_quantize_append(cfg, k_new, v_new, cu_dev, before_dev, bt_dev, cache, q=qs[i % n_in],
                                      q_fp8=bufs_sp.q_fp8, stream=stream)
            return uq.decode_attention_shared_prefix(cfg, bufs_sp, pbufs, cache, bt_dev, pfx, stream=stream)
        if step_graphs is not None:
            return step_graphs[i % n_in].launch()
        k_new, v_new = kvs[i % n_in]
        return uq.decode_step(cfg, bufs, qs[i % n_in], k_new, v_new, cu_dev, before_dev, after_dev,
                              bt_dev, cache, stream=stream)

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local_rank)
    sampler.start()

    # ---- device-resident timing: W warm-up, then exactly K steps between two events
    for i in range(max(args.warmup, 3)):
        step(i)
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.busy = True
    ev0.record(stream)
    for i in range(args.steps):
        step(i)
    ev1.record(stream)
    barrier()
    sampler.busy = False
    ms_total = ev0.elapsed_time(ev1)

    # ---- the spread over steps: the same K steps (at most 200) with an event after every step.  (An event between two
    # steps ends the programmatic overlap of merge(i) with append(i+1), so these are a little longer than ms_per_step.)
    n_sp = min(args.steps, 200)
    sp_ev = [torch.cuda.Event(enable_timing=True) for _ in range(n_sp + 1)]
    sampler.busy = True
    sp_ev[0].record(stream)
    for i in range(n_sp):
        step(i)
        sp_ev[i + 1].record(stream)
    barrier()
    sampler.busy = False
    step_ms = [a.elapsed_time(b) for a, b in zip(sp_ev[:-1], sp_ev[1:])]

    # ---- the same steps once more with an event on both sides of every decode launch (the dominant kernel's
    # duration for the roofline; an event between two launches ends their programmatic overlap, so this pass
    # is not the one `value` is taken from)
    # (at most 50 steps: on the long configs a second full-length pass runs into sw_power_cap and times the cap)
    n_inst = min(args.steps, 50)
    dec_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
              for _ in range(n_inst)]
    sampler.busy = True
    for i in range(n_inst):
        k_new, v_new = kvs[i % n_in]
        if fmt == uq.KV_ULTRA_TQ:
            uq.tq_append(cfg, W.TQ_CODEBOOK, k_new, v_new, cu_dev, before_dev, bt_dev, cache, q=qs[i % n_in], q_rot=q_rot,
                         stream=stream)
            dec_ev[i][0].record(stream)
            uq.tq_decode_attention(cfg, W.TQ_CODEBOOK, q_rot, cache, bt_dev, after_dev, S, bufs.partial_acc, bufs.partial_ml,
                                   stream=stream)
            dec_ev[i][1].record(stream)
            uq.merge_splits(cfg, bufs.partial_acc, bufs.partial_ml, bufs.out, stream=stream)
            continue
        if fmt is not None:
            fp8 = fmt == uq.KV_FP8_E4M3
            uq.baseline_append(cfg, fmt, k_new, v_new, cu_dev, before_dev, bt_dev, cache, q=qs[i % n_in] if fp8 else None,
                               q_out=bufs.q_fp8 if fp8 else None, stream=stream)
            dec_ev[i][0].record(stream)
            uq.baseline_decode_attention(cfg, fmt, bufs.q_fp8 if fp8 else qs[i % n_in], cache, bt_dev, after_dev, S,
                                         bufs.partial_acc, bufs.partial_ml, stream=stream)
            dec_ev[i][1].record(stream)
            uq.merge_splits(cfg, bufs.partial_acc, bufs.partial_ml, bufs.out, stream=stream)
            continue
        uq.rotate_quantize_append(cfg, k_new, v_new, cu_dev, before_dev, bt_dev, cache,
                                  q=qs[i % n_in], q_fp8=bufs.q_fp8, stream=stream)
        dec_ev[i][0].record(stream)
        uq.decode_attention(cfg, bufs.q_fp8, cache, bt_dev, after_dev, S, bufs.partial_acc,
                            bufs.partial_ml, stream=stream)
        dec_ev[i][1].record(stream)
        uq.merge_splits(cfg, bufs.partial_acc, bufs.partial_ml, bufs.out, stream=stream)
    barrier()
    sampler.busy = False
    dec_ms = [a.elapsed_time(b) for a, b in dec_ev]
    # --shared-prefix 1: the two decode kernels of the step timed one by one as well (events between the launches)
    sp_kernels = None
    if pbufs is not None:
        n_sp = min(n_inst, 20)
        ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(n_sp)]
        for i in range(n_sp):
            k_new, v_new = kvs[i % n_in]
            uq.rotate_quantize_append(cfg, k_new, v_new, cu_dev, before_dev, bt_dev, cache, q=qs[i % n_in],
                                      q_fp8=bufs_sp.q_fp8, stream=stream)
            uq.decode_attention_shared_prefix(cfg, bufs_sp, pbufs, cache, bt_dev, pfx, stream=stream,
                                              mark=lambda j, e=ev[i]: e[j].record(stream))
        barrier()
        sp_kernels = {"prefix_kernel_us": round(statistics.fmean(e[0].elapsed_time(e[1]) for e in ev) * 1e3, 2),
                      "suffix_kernel_us": round(statistics.fmean(e[1].elapsed_time(e[2]) for e in ev) * 1e3, 2),
                      "launches": n_sp}

    # ---- sustained: back-to-back steps for at least --sustain seconds between two events (north_star: "sustaining
    # >= 70 % of B200 HBM peak"), with its own clock record — a 2 ms burst runs at boost clock, seconds of
    # full-bandwidth load run under the 1 kW power cap
    sustained = None
    if args.sustain > 0:
        est = max_over_ranks([ms_total / args.steps], world, dev)[0]
        n_sus = max(args.steps, int(args.sustain * 1e3 / max(est, 1e-3)) + 1)
        for i in range(3):
            step(i)
        barrier()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        sampler.busy = "sustain"
        s0.record(stream)
        for i in range(n_sus):
            step(i)
        s1.record(stream)
        barrier()
        sampler.busy = False
        sustained = (n_sus, s0.elapsed_time(s1))
        time.sleep(0.5)                                # let the part cool off before the end-to-end leg

    # ---- end-to-end through the public host-buffer API: H2D of the step's inputs, D2H of O
    # one pinned staging block per entry of the input ring (the caller's own buffers: it writes a step's inputs
    # there), uploaded in a single copy per step
    stages = []
    for j in range(n_in if fmt is None else 0):
        st = uq.HostStage(cfg, B, int(kvs[j][0].shape[0]), int(bt_dev.shape[1]), dev)
        st.h["q"].copy_(qs[j].cpu()); st.h["k_new"].copy_(kvs[j][0].cpu()); st.h["v_new"].copy_(kvs[j][1].cpu())
        st.h["cu_new"].copy_(cu_dev.cpu()); st.h["seq_lens_before"].copy_(before_dev.cpu())
        st.h["seq_lens_after"].copy_(after_dev.cpu()); st.h["block_tables"].copy_(bt_dev.cpu())
        stages.append(st)
    out_host = torch.empty((B, Hq, d), dtype=torch.bfloat16).pin_memory()

    # the host step (one H2D copy, three kernels, one D2H copy) captured once per staging block as a CUDA graph: a
    # step costs the host one graph launch
    graphs = [uq.HostStepGraph(cfg, bufs, st, cache, out_host, tables=False) for st in stages]
    ms_e2e = 0.0

    def step_host(i):
        graphs[i % n_in].launch()
        stream.synchronize()           # the caller reads O before it can issue the next step

    h2d = stages[0].step_nbytes if stages else 0   # the step's own inputs as they are copied (fields 256-byte aligned)
    d2h = out_host.numel() * out_host.element_size()
    if stages:
        for i in range(max(args.warmup, 3)):
            step_host(i)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        sampler.busy = True
        e0.record(stream)
        for i in range(args.steps):
            step_host(i)
        e1.record(stream)
        barrier()
        sampler.busy = False
        ms_e2e = e0.elapsed_time(e1)
    sampler.stop()

    # ---- reduce over ranks: max time, summed bytes
    total_b, decode_b = step_bytes(wl, S, ctx_after, 1)
    red = max_over_ranks([ms_total, ms_e2e, statistics.fmean(dec_ms), statistics.median(dec_ms), min(dec_ms),
                          statistics.median(step_ms), min(step_ms), sustained[1] if sustained else 0.0], world, dev)
    ms_total, ms_e2e, dec_ms_mean, dec_ms_med, dec_ms_min, step_ms_med, step_ms_min, ms_sus = red
    ms_step = ms_total / args.steps
    value = whole_job_value(total_b, world, ms_step)
    e2e_value = whole_job_value(total_b, world, ms_e2e / args.steps) if ms_e2e > 0 else 0.0
    peak, peak_src = _peaks()
    achieved = decode_b / (dec_ms_mean * 1e-3) / 1e9
    line = {
        "metric": METRIC, "value": round(value, 1), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": round(ms_step, 5),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": {"fp4": "fp8xfp4->f32", "fp8": "fp8xfp8->f32", "bf16": "bf16xbf16->f32", "tq": "bf16xbf16->f32 (codebook / uniform 4-bit dequantised on read)"}[KV_FORMAT],
        "data": "synthetic", "impl": "ours",
        **({"kv_format": KV_FORMAT + " (comparison cache, PAPER.md:163 - not the headline metric; e2e not measured)"}
           if fmt is not None else {}),
        "config": {"workload": f"BASELINE.json configs[{args.config - 1}] {wl.name}: batch {B}, "
                               f"{Hq} Q / {Hkv} KV heads, head_dim {d}, ctx {int(ctx_after.min())}"
                               f"..{int(ctx_after.max())} tokens, page_size {wl.page_size}, random block tables; "
                               "step = append 1 token/seq + rotate/FP8 Q + split-K decode + merge",
                   "batch_per_gpu": B, "tokens_per_gpu": int(ctx_after.astype(np.int64).sum()),
                   "num_splits": S, "parallelism": f"replica x{world} (sequences sharded, no collective)",
                   "l2": f"KV working set {wl.kv_bytes_per_step() / 1e6:.0f} MB per step >> 126 MB L2 (no flush needed)"},
        "us_per_step": round(ms_step * 1e3, 2),
        "us_per_step_spread": {"median": round(step_ms_med * 1e3, 2), "min": round(step_ms_min * 1e3, 2), "steps": n_sp,
                               "note": "one event per step (ends the overlap of merge(i) with append(i+1))"},
        "decode_kernel_us": round(dec_ms_mean * 1e3, 2),
        "decode_kernel_us_spread": {"median": round(dec_ms_med * 1e3, 2), "min": round(dec_ms_min * 1e3, 2), "launches": n_inst},
        "bytes_per_step": total_b,
        **({"shared_prefix_kernels": sp_kernels} if sp_kernels else {}),
        **({"shared_prefix": {
            "note": "bytes_per_step / value / roofline count LOGICAL bytes; the prefix pages are named by every block "
                    "table and read from HBM once per step (L2 serves the rest), so the fractions of the HBM peak can "
                    "exceed what HBM alone delivers",
            "prefix_tokens": int(wl.prefix_len), "shared_prefix_decode": bool(args.shared_prefix),
            "physical_kv_bytes_per_step": int((int(ctx_after.astype(np.int64).sum()) - (B - 1) * int(wl.prefix_len))
                                              * Hkv * 136)}} if wl.prefix_len else {}),
        "frac_of_nominal_8TBs": round(value / world / NOMINAL_HBM_GBS, 4),
        "frac_of_measured_peak": round(value / world / peak, 4),
        "e2e": {"value": round(e2e_value, 1), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                "d2h_bytes_per_step": int(d2h), "us_per_step": round(ms_e2e / args.steps * 1e3, 2),
                "note": "uq.HostStepGraph (one CUDA-graph launch per step): host pinned Q/K_new/V_new/lens -> device (one staged copy), three kernels, O -> host, sync every step; "
                        "the FP4 cache is resident state and so are the block tables (uploaded when they change: a sequence "
                        "crosses a page boundary every 16th step; they do not change between the timed steps)",
                "block_table_bytes": int(stages[0].nbytes - stages[0].step_nbytes) if stages else 0},
        "gpu_launches": (4 if pbufs is not None else 3) * args.steps,
        "clocks": sampler.summary(),
        **({"sustained": {
            "value": round(whole_job_value(total_b, world, ms_sus / sustained[0]), 1), "unit": UNIT,
            "us_per_step": round(ms_sus / sustained[0] * 1e3, 2), "steps": sustained[0], "seconds": round(ms_sus * 1e-3, 3),
            "frac_of_nominal_8TBs": round(whole_job_value(total_b, world, ms_sus / sustained[0]) / world / NOMINAL_HBM_GBS, 4),
            "frac_of_measured_peak": round(whole_job_value(total_b, world, ms_sus / sustained[0]) / world / peak, 4),
            "clocks": sampler.summary("sustain"),
            "note": "the same step, back to back for at least --sustain seconds between two CUDA events"}} if sustained else {}),
        "roofline": {"bound": "hbm", "kernel": "uq::decode_kernel" if fmt is None else "uq::decode_cmp_kernel", "achieved": round(achieved, 1),
                     "peak": peak, "unit": "GB/s", "frac": round(achieved / peak, 4),
                     "frac_of_nominal_8TBs": round(achieved / NOMINAL_HBM_GBS, 4),
                     "traffic": _ncu_traffic("decode_kernel" if fmt is None else "decode_cmp_kernel",
                                             f"cfg{args.config}" + (f"_d{d}" if d != 128 else "") + (f"_{KV_FORMAT}" if fmt else "")),
                     "algorithmic_bytes": decode_b,
                     "source_key": _source_key(),
                     "peak_source": peak_src,
                     "timing": "CUDA events around every uq_decode_attention launch, mean over a second pass of the same K steps "
                               "(at most 50; events between launches would end the programmatic overlap of the timed pass)"},
    }
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(args.config, budget_s=args.cpu_budget)
    return line


# ----------------------------------------------------------------------------- oracle legs
def _oracle_sample(idx: int, n_seq: int, length: int):
    """Oracle inputs for the first n_seq sequences of config idx truncated to `length` tokens:
    logical cache arrays of the context minus one token, the step's new K/V row and query."""
    import dataclasses

    import oracle
    from paper_2606_20474_b200 import workloads as W     # input generator only (no arithmetic)
    wl = _workload(idx, 0)
    wl1 = wl if wl.new_tokens == 1 else dataclasses.replace(wl, new_tokens=1)
    q = W.gen_q(wl, "cpu", step=0).view(torch.uint16).numpy()
    k_new, v_new = W.gen_new_kv(wl1, 0, "cpu")
    k_new, v_new = k_new.view(torch.uint16).numpy(), v_new.view(torch.uint16).numpy()
    seqs = []
    for b in range(n_seq):
        L = min(int(wl.ctx_lens[b]), length)
        k, v = W.seq_kv(wl, b, L - 1, "cpu")
        arrays = oracle.encode_kv(k.view(torch.uint16).numpy(), v.view(torch.uint16).numpy())
        seqs.append((L, arrays))
    return wl, q, k_new, v_new, seqs


def _oracle_step(oracle, wl, q, k_new, v_new, seqs):
    """One hot-path step on the CPU oracle for the sample: append 1 token, encode Q, attend."""
    nbytes = 0
    per_tok = 2 * (wl.head_dim // 2 + wl.head_dim // 32)
    for b, (L, arrays) in enumerate(seqs):
        new = oracle.encode_kv(k_new[b:b + 1], v_new[b:b + 1])
        full = [np.concatenate([a, n], axis=0) for a, n in zip(arrays, new)]
        q8 = oracle.encode_q(q[b])
        oracle.attention(q8, *full, wl.num_q_heads, wl.num_kv_heads)
        nbytes += L * wl.num_kv_heads * per_tok + 4 * ((L + 15) // 16) + wl.num_q_heads * wl.head_dim * 3
    return nbytes


def cpu_baseline(idx: int, budget_s: float = 15.0):
    import oracle
    oracle.build()
    cores = oracle.num_threads()
    # size the sample: one short probe, then whole sequences up to the budget
    wl, q, k_new, v_new, seqs = _oracle_sample(idx, 1, 2048)
    t0 = time.perf_counter(); _oracle_step(oracle, wl, q, k_new, v_new, seqs); probe = time.perf_counter() - t0
    tok_per_s = 2048 / max(probe, 1e-6)
    full_len = int(wl.ctx_lens[0])
    want_tokens = max(2048, int(tok_per_s * budget_s))
    n_seq = max(1, min(wl.batch, want_tokens // full_len))
    length = full_len if want_tokens >= full_len else (want_tokens // 16) * 16
    wl, q, k_new, v_new, seqs = _oracle_sample(idx, n_seq, length)
    t0 = time.perf_counter()
    nbytes = _oracle_step(oracle, wl, q, k_new, v_new, seqs)
    dt = time.perf_counter() - t0
    # the same oracle on ONE core ("timed on 1 core and on all cores"), on a sample sized for ~budget/3
    one = None
    try:
        oracle.set_num_threads(1)
        len1 = int(min(full_len, max(1024, (int(tok_per_s / max(cores, 1) * budget_s / 3) // 16) * 16)))
        wl1, q1, k1, v1, seqs1 = _oracle_sample(idx, 1, len1)
        t0 = time.perf_counter()
        nb1 = _oracle_step(oracle, wl1, q1, k1, v1, seqs1)
        dt1 = time.perf_counter() - t0
        one = {"value": round(nb1 / dt1 / 1e9, 5), "unit": UNIT, "cores": 1, "seconds": round(dt1, 3),
               "sample": f"sequence 0 of config {idx} truncated to {seqs1[0][0]} tokens"}
    finally:
        oracle.set_num_threads(cores)
    return {"value": round(nbytes / dt / 1e9, 5), "unit": UNIT, "cores": cores, "kind": "oracle",
            "seconds": round(dt, 3),
            "sample": f"{n_seq} of {wl.batch} sequences of config {idx}, {seqs[0][0]} tokens each "
                      f"(append 1 token + Q encode + float64 attention, all {wl.num_q_heads} heads)",
            "one_core": one,
            "quant_error_vs_bf16": _quant_error_context(oracle, idx)}


def _quant_error_context(oracle, idx: int, length: int = 4096):
    """Context only (north_star): the method's own error — the oracle's attention over the FP4 / FP8-quantised
    values against float64 attention over the unquantised bf16 Q, K, V — on sequence 0 truncated to `length` tokens."""
    from paper_2606_20474_b200 import workloads as W     # input generator only (no arithmetic)
    wl = _workload(idx, 0)
    L = min(int(wl.ctx_lens[0]), length)
    k, v = W.seq_kv(wl, 0, L, "cpu")
    q = W.gen_q(wl, "cpu", step=0)[0]
    arrays = oracle.encode_kv(k.view(torch.uint16).numpy(), v.view(torch.uint16).numpy())
    out_q = oracle.attention(oracle.encode_q(q.view(torch.uint16).numpy()), *arrays, wl.num_q_heads, wl.num_kv_heads)
    out_d = oracle.attention_dense(q.double().numpy(), k.double().numpy(), v.double().numpy())
    return {"rel_fro": round(float(np.linalg.norm(out_q - out_d) / np.linalg.norm(out_d)), 5),
            "max_abs": round(float(np.abs(out_q - out_d).max()), 5),
            "sample": f"sequence 0 of config {idx}, first {L} tokens, all {wl.num_q_heads} heads",
            "note": "synthetic N(0,1) inputs: an output row is a near-uniform average of random values, so the relative "
                    "figure is the quantisers' own noise (4-bit V: 0.125 relative RMS per element, plus the score "
                    "noise of 4-bit K and FP8 Q) undamped by any signal; context, not a parity figure"}


def run_reference(args):
    """The reference arm for this tier is the oracle as it stands, on the host cores."""
    import oracle
    oracle.build()
    cores = oracle.num_threads()
    W_, K_ = max(args.warmup, 0), args.steps
    wl, q, k_new, v_new, seqs = _oracle_sample(args.config, 1, 1024)
    t0 = time.perf_counter(); _oracle_step(oracle, wl, q, k_new, v_new, seqs); probe = time.perf_counter() - t0
    tok_per_s = 1024 / max(probe, 1e-6)
    per_step_s = max(0.05, min(10.0, args.ref_budget / max(1, W_ + K_)))
    full_len = int(wl.ctx_lens[0])
    length = int(min(full_len, max(256, (int(tok_per_s * per_step_s) // 16) * 16)))
    wl, q, k_new, v_new, seqs = _oracle_sample(args.config, 1, length)
    for _ in range(W_):
        _oracle_step(oracle, wl, q, k_new, v_new, seqs)
    t0 = time.perf_counter()
    nbytes = 0
    for _ in range(K_):
        nbytes += _oracle_step(oracle, wl, q, k_new, v_new, seqs)
    dt = time.perf_counter() - t0
    value = nbytes / dt / 1e9
    sample = (f"per step: 1 of {wl.batch} sequences of config {args.config} truncated to {seqs[0][0]} tokens "
              f"(append 1 token + Q encode + float64 attention, all {wl.num_q_heads} heads)")
    return {"metric": METRIC, "value": round(value, 5), "unit": UNIT, "n_gpus": args.gpus, "steps": K_,
            "warmup": W_, "ms_per_step": round(dt / K_ * 1e3, 3), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "impl": "reference",
            "config": {"workload": f"BASELINE.json configs[{args.config - 1}] {wl.name} (bounded sample: {sample})"},
            "cpu_baseline": {"value": round(value, 5), "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": round(value, 5), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


# ----------------------------------------------------------------------------- bulk append
def run_bulk_append(args):
    """Not the headline metric: prefill-sized quantize-on-append of one sequence of the chosen config (32,768
    new tokens x Hkv heads per call by default), algorithmic bytes = 2 * 256 B read + 136 B written per
    (token, kv head), CUDA events over K calls."""
    import paper_2606_20474_b200 as uq
    from paper_2606_20474_b200 import workloads as W
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the hot path has no CPU fallback")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    wl = _workload(args.config, 0)
    cfg = uq.UQConfig(num_q_heads=wl.num_q_heads, num_kv_heads=wl.num_kv_heads)
    n = min(args.bulk_append, int(wl.ctx_lens[0]))
    nseq = max(1, min(args.bulk_seqs, wl.batch))           # sequences that receive n new tokens each in one call
    cache = uq.alloc_cache(cfg, wl.num_pages, dev)
    bt = torch.from_numpy(wl.block_tables).to(dev)
    src_bytes = 2 * nseq * n * wl.num_kv_heads * 2 * wl.head_dim
    # the source rows of consecutive calls come from `rot` different buffers, together larger than L2 (126 MB), so a
    # call never finds its inputs in L2 from the call before
    rot = max(2, -(-300_000_000 // src_bytes))
    srcs = []
    for r in range(rot):
        kv = [W.gen_kv(wl, b, 0, n, dev) for b in range(nseq)] if r == 0 else None
        if r == 0:
            k0, v0 = torch.cat([a for a, _ in kv]), torch.cat([a for _, a in kv])
            srcs.append((k0, v0))
        else:
            srcs.append((k0.roll(r, 0).contiguous(), v0.roll(r, 0).contiguous()))
    before = torch.zeros(wl.batch, dtype=torch.int32, device=dev)
    cu = np.zeros(wl.batch + 1, np.int32)
    cu[1:nseq + 1] = n * np.arange(1, nseq + 1); cu[nseq + 1:] = n * nseq
    cu = torch.from_numpy(cu).to(dev)
    stream = torch.cuda.current_stream()
    for i in range(max(args.warmup, 3)):
        uq.rotate_quantize_append(cfg, srcs[i % rot][0], srcs[i % rot][1], cu, before, bt, cache, stream=stream)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for i in range(args.steps):
        uq.rotate_quantize_append(cfg, srcs[i % rot][0], srcs[i % rot][1], cu, before, bt, cache, stream=stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    nbytes = nseq * n * wl.num_kv_heads * (2 * 2 * wl.head_dim + 136)
    peak, peak_src = _peaks()
    gbs = nbytes / (ms * 1e-3) / 1e9
    return {"metric": "bulk_append_hbm_gbps", "value": round(gbs, 1), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": round(ms, 5), "higher_is_better": True, "dtype": "f32/f64->fp4",
            "data": "synthetic", "impl": "ours",
            "config": {"workload": f"bulk quantize-on-append, {nseq} x {n} tokens x {wl.num_kv_heads} kv heads of {wl.name} "
                                   f"per call; source rows {src_bytes / 1e6:.1f} MB per call, {rot} source buffers in "
                                   "rotation (together > L2)"},
            "bytes_per_step": nbytes, "gpu_launches": args.steps,
            "roofline": {"bound": "hbm", "kernel": "uq::append_bulk_kernel", "achieved": round(gbs, 1), "peak": peak,
                         "unit": "GB/s", "frac": round(gbs / peak, 4),
                         "traffic": _ncu_traffic("append_bulk_kernel", f"cfg{args.config}_bulk{n}x{nseq}"),
                         "algorithmic_bytes": nbytes, "peak_source": peak_src}}


# ----------------------------------------------------------------------------- calibration
def run_calibrate(args):
    """Not the headline metric: uq_calibrate_c (Eq.(2)) over VECTORS synthetic keys of the chosen config
    and the 56 constants 0.100 .. 0.320 in steps of 0.004, power-of-two scale; CUDA events over K calls.  Bound: the
    float64 pipe.  Counted float64 operations per (vector, constant): 128 elements x (7 ladder compares + 2 products
    + 2 additions) = 1408, plus per vector and pass of 8 constants the rotation (7 x 128 additions + 128 products)
    and the group maxima (128 compares): 1152 / 8 = 144 per (vector, constant).  Peak: 64 float64 lanes per SM x
    SM count x the SM clock (one operation per lane and cycle)."""
    import paper_2606_20474_b200 as uq
    from paper_2606_20474_b200 import workloads as W
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the hot path has no CPU fallback")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    wl = _workload(args.config, 0)
    cfg = uq.UQConfig(num_q_heads=wl.num_q_heads, num_kv_heads=wl.num_kv_heads)
    n_tok = max(1, min(args.calibrate // wl.num_kv_heads, int(wl.ctx_lens[0])))
    k, _ = W.gen_kv(wl, 0, 0, n_tok, dev)
    x = k.reshape(-1, wl.head_dim).contiguous()
    cs = torch.arange(0.100, 0.322, 0.004, dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream()
    for _ in range(max(args.warmup, 3)):
        sq, nrm = uq.calibrate_c(cfg, x, cs, rotate=True, pow2_scale=True, stream=stream)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        sq, nrm = uq.calibrate_c(cfg, x, cs, rotate=True, pow2_scale=True, stream=stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    evals = x.shape[0] * cs.shape[0]
    ops = evals * (1408 + 144)
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    peak = 64 * sms * 1.965e9 / 1e12
    best = float(cs[int(torch.argmin(sq).item())])
    return {"metric": "calibrate_vector_constant_evals_per_s", "value": round(evals / (ms * 1e-3) / 1e9, 3), "unit": "G/s",
            "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": round(ms, 5),
            "higher_is_better": True, "dtype": "f64", "data": "synthetic", "impl": "ours",
            "config": {"workload": f"uq_calibrate_c: {x.shape[0]} rotated key vectors of {wl.name} x {cs.shape[0]} "
                                   "constants (0.100 .. 0.320), power-of-two scale"},
            "argmin_c": round(best, 3), "rel_mse_at_argmin": float(sq.min().item() / nrm.item()), "gpu_launches": args.steps,
            "roofline": {"bound": "alu", "kernel": "uq::calib_kernel", "achieved": round(ops / (ms * 1e-3) / 1e12, 3),
                         "peak": round(peak, 2), "unit": "Tfp64op/s", "frac": round(ops / (ms * 1e-3) / 1e12 / peak, 4),
                         "traffic": None, "peak_source": "64 float64 lanes per SM x SMs x 1.965 GHz (DESIGN.md 5.4)"}}


# ----------------------------------------------------------------------------- main
def dump_trace(path: str) -> None:
    """--trace: the [tile][16 events] clock64 tables a -DUQ_TRACE build of libuq.so keeps for one CTA of the decode kernel
    and one of the shared-prefix kernel (event numbers: the comments at TRD / TRP in csrc/).  Rows of zeros are left out."""
    import ctypes

    import paper_2606_20474_b200 as uq
    lib = ctypes.CDLL(uq.library_path())
    with open(path, "w") as f:
        for name in ("decode", "prefix"):
            try:
                fn = getattr(lib, "uq_debug_trace_read_" + name)
            except AttributeError:
                f.write(f"# {name}: libuq.so was not built with -DUQ_TRACE\n")
                continue
            buf = np.zeros(256 * 16, np.uint64)
            rc = fn(buf.ctypes.data_as(ctypes.c_void_p), ctypes.c_size_t(buf.nbytes))
            t = buf.reshape(256, 16)
            f.write(f"# {name} kernel, traced CTA: clock64 per (tile, event 0..15), cudaMemcpyFromSymbol rc={rc}\n")
            for i, row in enumerate(t):
                if row.any():
                    f.write(f"{i} " + " ".join(str(int(v)) for v in row) + "\n")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, choices=[1, 2, 3, 4, 5],
                    help="BASELINE.json config number (1-based); 2 is the one the metric is quoted on")
    ap.add_argument("--splits", type=int, default=0, help="num_splits override (0 = uq_suggest_num_splits)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--shared-prefix", type=int, default=0, choices=[0, 1],
                    help="1 (config 4): the timed step decodes the shared prefix with uq_decode_prefix_attention")
    ap.add_argument("--graph", type=int, default=0, choices=[0, 1],
                    help="1: the timed steps are launches of uq.StepGraph (one CUDA graph per step)")
    ap.add_argument("--bulk-seqs", type=int, default=1, metavar="S",
                    help="with --bulk-append: sequences that receive TOKENS new tokens each in one call")
    ap.add_argument("--bulk-append", type=int, default=0, metavar="TOKENS",
                    help="instead of the decode step, time bulk quantize-on-append of TOKENS new tokens per call")
    ap.add_argument("--calibrate", type=int, default=0, metavar="VECTORS",
                    help="instead of the decode step, time uq_calibrate_c over VECTORS key vectors and 56 constants")
    ap.add_argument("--trace", default="", metavar="FILE",
                    help="debug builds only (UQ_NVCC_EXTRA=-DUQ_TRACE python -m paper_2606_20474_b200.build): after the run, write "
                         "the per-tile clock64 tables of the traced CTAs (decode kernel, shared-prefix kernel) to FILE as text")
    ap.add_argument("--no-early", action="store_true",
                    help="do not set UQ_FLAG_SMALL_APPEND_AHEAD (the decode kernel then waits for the append before it reads anything)")
    ap.add_argument("--kv", default="fp4", choices=["fp4", "fp8", "bf16", "tq"],
                    help="fp4: UltraQuant (default).  fp8 / bf16 / tq: the same step over the paper's comparison caches "
                         "(tq = Ultra-TQ, the codebook encoding of Algorithm 2)")
    ap.add_argument("--head-dim", type=int, default=128, choices=[64, 128, 256],
                    help="run the config's shape at another head size (the decode step only)")
    ap.add_argument("--sustain", type=float, default=2.0, metavar="SECONDS",
                    help="also time back-to-back steps for at least SECONDS (own clock record); 0 = skip")
    ap.add_argument("--cpu-budget", type=float, default=15.0, help="seconds of oracle work for cpu_baseline")
    ap.add_argument("--ref-budget", type=float, default=90.0, help="seconds for the whole --impl reference run")
    args = ap.parse_args()

    global HEAD_DIM, KV_FORMAT
    HEAD_DIM = args.head_dim
    KV_FORMAT = args.kv
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.bulk_append > 0:
        if rank == 0:
            print(json.dumps(run_bulk_append(args)), flush=True)
        return 0
    if args.calibrate > 0:
        if rank == 0:
            print(json.dumps(run_calibrate(args)), flush=True)
        return 0
    if args.impl == "reference":
        if rank == 0:
            print(json.dumps(run_reference(args)), flush=True)
        return 0

    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        torch.cuda.set_device(local_rank)
        torch.distributed.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    try:
        line = run_ours(args, rank, world, local_rank)
        if rank == 0:
            print(json.dumps(line), flush=True)
            if args.trace:
                dump_trace(args.trace)
    finally:
        if world > 1:
            torch.distributed.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
