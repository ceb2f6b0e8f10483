"""Seeded synthetic workloads shaped like BASELINE.json's five configs.

This module only GENERATES INPUTS (shapes, lengths, block tables, bf16 K/V/Q values).  It
holds none of the method's arithmetic (no rotation, no quantiser, no attention) and is the
one module both the CUDA path's callers and the oracle's tests may import.

Recipe: values are torch.randn in fp32 on the requested device
from a torch.Generator seeded per (config seed, sequence, 4096-token chunk), multiplied by a
per-(kv_head, channel) scale that carries the config's outlier structure, then cast to bf16.
Lengths, permutations and channel choices come from numpy.random.default_rng(seed).  The
paper's own workloads (production agent traces, SWE-bench, RULER, ... — PAPER.md:51,138,153)
are not available; these tensors take their shapes and value structure and stand in for them.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np
import torch

CHUNK = 4096          # tokens per generator chunk (fixed so every caller sees the same values)
PAGE = 16

# Input of the Ultra-TQ comparison path (Alg. 2 "Require: codebook C_K"): a 16-level codebook for the
# coordinates of a 32-channel block scaled to unit l2 norm — the textbook 16-level Lloyd-Max levels of N(0, 1)
# divided by sqrt(32).  The paper's own codebook is calibrated on captured activations (out of scope): this table is
# data handed to both the CUDA path and the oracle, like every other input.
_LM16 = (0.1284, 0.3881, 0.6568, 0.9424, 1.256, 1.618, 2.069, 2.733)
TQ_CODEBOOK = tuple([-v / 32 ** 0.5 for v in reversed(_LM16)] + [v / 32 ** 0.5 for v in _LM16])


@dataclasses.dataclass
class Workload:
    name: str
    seed: int
    batch: int
    num_q_heads: int
    num_kv_heads: int
    head_dim: int
    page_size: int
    ctx_lens: np.ndarray            # int32 [B] tokens in the cache BEFORE the timed step's append
    new_tokens: int                 # tokens appended per sequence inside the timed step (0 or 1)
    prefix_len: int                 # tokens shared by every sequence (same physical pages)
    block_tables: np.ndarray        # int32 [B, max_pages]
    num_pages: int                  # physical pages the cache must hold
    k_chan_scale: np.ndarray        # float32 [Hkv, d]
    v_chan_scale: np.ndarray        # float32 [Hkv, d]
    peaked_frac: float = 0.0        # fraction of (b, q_head) rows given a peaked query
    note: str = ""

    @property
    def group(self) -> int:
        return self.num_q_heads // self.num_kv_heads

    @property
    def max_pages(self) -> int:
        return int(self.block_tables.shape[1])

    @property
    def total_tokens(self) -> int:
        return int(self.ctx_lens.astype(np.int64).sum()) + self.batch * self.new_tokens

    def kv_bytes_per_step(self) -> int:
        """Algorithmic KV bytes one decode step reads: 136 B per (token, kv_head) at d=128
        (0.5 B/elem + 1 B per 32 elems, K and V — PAPER.md:98)."""
        per = 2 * (self.head_dim // 2 + self.head_dim // 32)
        return self.total_tokens * self.num_kv_heads * per


def _chunk_seed(seed: int, seq: int, chunk: int) -> int:
    return (seed * 1_000_003 + (seq + 1) * 40_009 + chunk) % (2**31 - 1)


def gen_kv_chunk(wl: Workload, seq: int, chunk: int, device="cpu"):
    """bf16 K, V of shape [CHUNK, Hkv, d] for tokens [chunk*CHUNK, (chunk+1)*CHUNK) of sequence
    `seq` (seq = -1 is the shared prefix).  Position-addressed, so any caller regenerates the
    same values."""
    dev = torch.device(device)
    g = torch.Generator(device=dev)
    g.manual_seed(_chunk_seed(wl.seed, seq, chunk))
    shape = (CHUNK, wl.num_kv_heads, wl.head_dim)
    k = torch.randn(shape, generator=g, device=dev, dtype=torch.float32)
    v = torch.randn(shape, generator=g, device=dev, dtype=torch.float32)
    k = k * torch.from_numpy(wl.k_chan_scale).to(dev)
    v = v * torch.from_numpy(wl.v_chan_scale).to(dev)
    return k.to(torch.bfloat16), v.to(torch.bfloat16)


def gen_kv(wl: Workload, seq: int, t0: int, t1: int, device="cpu"):
    """bf16 K, V [t1-t0, Hkv, d] for private tokens t0..t1-1 of `seq` (positions counted from
    the start of that sequence's own stream; the shared prefix is seq = -1)."""
    ks, vs = [], []
    t = t0
    while t < t1:
        c = t // CHUNK
        lo = t - c * CHUNK
        hi = min(t1 - c * CHUNK, CHUNK)
        k, v = gen_kv_chunk(wl, seq, c, device)
        ks.append(k[lo:hi])
        vs.append(v[lo:hi])
        t = c * CHUNK + hi
    if not ks:
        shape = (0, wl.num_kv_heads, wl.head_dim)
        z = torch.zeros(shape, dtype=torch.bfloat16, device=device)
        return z, z.clone()
    return torch.cat(ks), torch.cat(vs)


def seq_kv(wl: Workload, b: int, length: int, device="cpu"):
    """bf16 K, V [length, Hkv, d] of the logical sequence b: shared prefix then its own stream."""
    p = min(wl.prefix_len, length)
    kp, vp = gen_kv(wl, -1, 0, p, device)
    ks, vs = gen_kv(wl, b, 0, length - p, device)
    return torch.cat([kp, ks]), torch.cat([vp, vs])


def gen_q(wl: Workload, device="cpu", step: int = 0):
    """bf16 Q [B, Hq, d] ~ N(0,1).  With wl.peaked_frac > 0 a seeded subset of (b, h) rows is
    replaced by alpha * K[b, t*, h // G] (alpha = 0.5 or 4) so that a dominant token exists and
    outputs are O(1) — the rows on which the 1e-2 relative tolerance does the checking."""
    dev = torch.device(device)
    g = torch.Generator(device=dev)
    g.manual_seed(_chunk_seed(wl.seed, 10_000 + step, 7))
    q = torch.randn((wl.batch, wl.num_q_heads, wl.head_dim), generator=g, device=dev,
                    dtype=torch.float32)
    if wl.peaked_frac > 0:
        rng = np.random.default_rng(wl.seed + 77 + step)
        n_rows = wl.batch * wl.num_q_heads
        n_pk = max(1, int(round(wl.peaked_frac * n_rows)))
        rows = rng.choice(n_rows, size=min(n_pk, n_rows), replace=False)
        for i, r in enumerate(rows):
            b, h = divmod(int(r), wl.num_q_heads)
            L = int(wl.ctx_lens[b])
            if L == 0:
                continue
            t = int(rng.integers(0, L))
            alpha = 0.5 if i % 2 == 0 else 4.0
            if t < wl.prefix_len:
                k, _ = gen_kv(wl, -1, t, t + 1, device)
            else:
                k, _ = gen_kv(wl, b, t - wl.prefix_len, t - wl.prefix_len + 1, device)
            q[b, h] = alpha * k[0, h // wl.group].to(torch.float32)
    return q.to(torch.bfloat16)


def gen_new_kv(wl: Workload, step: int, device="cpu"):
    """bf16 K, V [B * new_tokens, Hkv, d] appended in timed step `step` (config 4)."""
    dev = torch.device(device)
    g = torch.Generator(device=dev)
    g.manual_seed(_chunk_seed(wl.seed, 20_000 + step, 11))
    shape = (wl.batch * wl.new_tokens, wl.num_kv_heads, wl.head_dim)
    k = torch.randn(shape, generator=g, device=dev, dtype=torch.float32)
    v = torch.randn(shape, generator=g, device=dev, dtype=torch.float32)
    k = k * torch.from_numpy(wl.k_chan_scale).to(dev)
    v = v * torch.from_numpy(wl.v_chan_scale).to(dev)
    return k.to(torch.bfloat16), v.to(torch.bfloat16)


# ----------------------------------------------------------------------------- configs
def _tables(rng, ctx_lens, prefix_len, page, extra_tokens, permute=True):
    """Physical page assignment: the prefix's pages are 0..P-1 and head every table; each
    sequence's private pages are drawn from a random permutation of the rest."""
    B = len(ctx_lens)
    assert prefix_len % page == 0
    n_prefix = prefix_len // page
    need = [max(0, -(-(int(L) + extra_tokens - prefix_len) // page)) for L in ctx_lens]
    n_private = int(sum(need))
    num_pages = n_prefix + n_private
    order = np.arange(n_prefix, num_pages, dtype=np.int64)
    if permute:
        order = rng.permutation(order)
    max_pages = n_prefix + (max(need) if need else 0)
    max_pages = max(max_pages, 1)
    bt = np.zeros((B, max_pages), np.int32)
    pos = 0
    for b in range(B):
        bt[b, :n_prefix] = np.arange(n_prefix)
        bt[b, n_prefix:n_prefix + need[b]] = order[pos:pos + need[b]]
        pos += need[b]
    return bt, max(num_pages, 1)


def make_config(idx: int, scale: float = 1.0, peaked_frac: float | None = None, head_dim: int = 128) -> Workload:
    """BASELINE.json config `idx` (1-5).  scale < 1 shrinks batch and context for CPU-sized
    parity cases while keeping the structure (ragged lengths, shared prefix, outliers).
    head_dim other than 128 (64, 256: the other head sizes the paper validates) keeps
    everything else of the config."""
    seed = idx - 1
    rng = np.random.default_rng(seed)
    d, page = int(head_dim), PAGE

    def sc(n, lo=1):
        return max(lo, int(round(n * scale)))

    ones = None
    if idx == 1:
        B, Hq, Hkv = 1, 8, 1
        ctx = np.array([sc(1024, 16)], np.int32)
        ks = np.ones((Hkv, d), np.float32)
        ks[:, rng.choice(d, 4, replace=False)] = 10.0
        vs = np.ones((Hkv, d), np.float32)
        bt, npg = _tables(rng, ctx, 0, page, 0, permute=False)   # identity block table
        name, new, prefix = "cfg1_tiny", 0, 0
    elif idx == 2:
        B, Hq, Hkv = sc(32), 64, 4
        ctx = np.full(B, sc(32768, 16), np.int32)
        ks = np.ones((Hkv, d), np.float32)
        ks[:, rng.choice(d, 3, replace=False)] = 8.0               # "2% of K channels" of 128
        vs = np.ones((Hkv, d), np.float32)
        bt, npg = _tables(rng, ctx, 0, page, 0)
        name, new, prefix = "cfg2_qwen3_235b_32k", 0, 0
    elif idx == 3:
        B, Hq, Hkv = sc(64), 48, 8
        ctx = rng.integers(sc(16384, 16), sc(65536, 32) + 1, size=B).astype(np.int32)
        ks = np.exp(0.5 * rng.standard_normal((Hkv, d))).astype(np.float32)
        vs = np.exp(0.5 * rng.standard_normal((Hkv, d))).astype(np.float32)
        bt, npg = _tables(rng, ctx, 0, page, 0)
        name, new, prefix = "cfg3_wide_kv_ragged", 0, 0
    elif idx == 4:
        B, Hq, Hkv = sc(256), 64, 4
        prefix = (sc(30000, 16) // page) * page
        suf = np.minimum(np.rint(np.exp(math.log(10000 * scale) + 1.0 * rng.standard_normal(B))),
                         sc(98000)).astype(np.int64)
        suf = np.maximum(suf, 1)
        ctx = (prefix + suf).astype(np.int32)
        ks = np.ones((Hkv, d), np.float32)
        vs = np.ones((Hkv, d), np.float32)
        bt, npg = _tables(rng, ctx, prefix, page, 64)              # room for 64 appended tokens
        name, new = "cfg4_agent_trace_shared_prefix", 1
    elif idx == 5:
        B, Hq, Hkv = sc(8), 64, 4
        ctx = np.full(B, sc(262144, 16), np.int32)
        ks = np.ones((Hkv, d), np.float32)
        ks[:, rng.choice(d, 1, replace=False)] = 16.0
        vs = np.ones((Hkv, d), np.float32)
        bt, npg = _tables(rng, ctx, 0, page, 0)
        name, new, prefix = "cfg5_long_context", 0, 0
    else:
        raise ValueError(f"unknown config {idx}")
    del ones
    if scale != 1.0:
        name += f"_x{scale:g}"
    if d != 128:
        name += f"_d{d}"
    return Workload(name=name, seed=seed, batch=B, num_q_heads=Hq, num_kv_heads=Hkv, head_dim=d,
                    page_size=page, ctx_lens=ctx, new_tokens=new, prefix_len=prefix,
                    block_tables=bt, num_pages=npg, k_chan_scale=ks, v_chan_scale=vs,
                    peaked_frac=(0.01 if peaked_frac is None else peaked_frac))


def make_custom(name: str, seed: int, ctx_lens, num_q_heads: int, num_kv_heads: int,
                prefix_len: int = 0, new_tokens: int = 0, outlier_channels: int = 0,
                outlier_gain: float = 1.0, peaked_frac: float = 0.0, permute: bool = True,
                extra_tokens: int = 0, head_dim: int = 128) -> Workload:
    """Free-form workload for edge cases (empty / ragged sequences, odd lengths)."""
    rng = np.random.default_rng(seed)
    d, page = int(head_dim), PAGE
    ctx = np.asarray(ctx_lens, np.int32)
    ks = np.ones((num_kv_heads, d), np.float32)
    if outlier_channels:
        ks[:, rng.choice(d, outlier_channels, replace=False)] = outlier_gain
    vs = np.ones((num_kv_heads, d), np.float32)
    bt, npg = _tables(rng, ctx, prefix_len, page, max(extra_tokens, new_tokens), permute=permute)
    return Workload(name=name, seed=seed, batch=len(ctx), num_q_heads=num_q_heads,
                    num_kv_heads=num_kv_heads, head_dim=d, page_size=page, ctx_lens=ctx,
                    new_tokens=new_tokens, prefix_len=prefix_len, block_tables=bt, num_pages=npg,
                    k_chan_scale=ks, v_chan_scale=vs, peaked_frac=peaked_frac)
