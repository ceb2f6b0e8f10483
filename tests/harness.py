"""Shared helpers of the GPU parity tests, smoke() and bench.py's verification leg: drive the
CUDA path through the Python binding on seeded workloads, and compute the oracle's answer for
the same bytes.  The CUDA path and the oracle meet only here (test glue)."""
from __future__ import annotations

import numpy as np
import torch

import oracle
import paper_2606_20474_b200 as uq
from paper_2606_20474_b200 import workloads as W
from tests import uq_layout

ATOL, RTOL = 2e-3, 1e-2          # BASELINE.json north_star: 2e-3 absolute / 1e-2 relative


def cfg_of(wl: W.Workload, **kw) -> uq.UQConfig:
    return uq.UQConfig(num_q_heads=wl.num_q_heads, num_kv_heads=wl.num_kv_heads, head_dim=wl.head_dim,
                       page_size=wl.page_size, **kw)


def bits(t: torch.Tensor) -> np.ndarray:
    """bf16 tensor -> uint16 bit patterns on the host (the bytes both sides consume)."""
    return t.detach().contiguous().view(torch.uint16).cpu().numpy()


def append_tokens(cfg, cache, bt_dev, seq_lens_before: np.ndarray, counts: np.ndarray, k_new, v_new,
                  q=None, q_fp8=None):
    dev = cache.device
    cu = np.zeros(len(counts) + 1, np.int32)
    cu[1:] = np.cumsum(counts)
    uq.rotate_quantize_append(cfg, k_new, v_new, torch.from_numpy(cu).to(dev),
                              torch.from_numpy(seq_lens_before.astype(np.int32)).to(dev), bt_dev, cache,
                              q=q, q_fp8=q_fp8)


def fill_cache(cfg, wl: W.Workload, device="cuda", chunk_tokens: int = 1 << 16, lens=None):
    """Fill a fresh cache with every sequence's context through uq_rotate_quantize_append
    (bulk appends of up to chunk_tokens rows; the shared prefix is written once, through
    sequence 0's block table).  Returns (cache, block_tables_dev)."""
    lens = wl.ctx_lens if lens is None else lens
    cache = uq.alloc_cache(cfg, wl.num_pages, device)
    bt_dev = torch.from_numpy(wl.block_tables).to(device)
    B = wl.batch
    if wl.prefix_len:
        done = 0
        while done < wl.prefix_len:
            n = min(chunk_tokens, wl.prefix_len - done)
            k, v = W.gen_kv(wl, -1, done, done + n, device)
            before = np.zeros(B, np.int32); before[0] = done
            counts = np.zeros(B, np.int32); counts[0] = n
            append_tokens(cfg, cache, bt_dev, before, counts, k, v)
            done += n
    for b in range(B):
        priv = int(lens[b]) - wl.prefix_len
        done = 0
        while done < priv:
            n = min(chunk_tokens, priv - done)
            k, v = W.gen_kv(wl, b, done, done + n, device)
            before = np.zeros(B, np.int32); before[b] = wl.prefix_len + done
            counts = np.zeros(B, np.int32); counts[b] = n
            append_tokens(cfg, cache, bt_dev, before, counts, k, v)
            done += n
    return cache, bt_dev


def oracle_sequence_cache(wl: W.Workload, b: int, length: int, device="cuda", c_k=0.156, c_v=0.156):
    """The oracle's logical cache arrays of sequence b from the same generated bf16 bytes."""
    k, v = W.seq_kv(wl, b, length, device)
    return oracle.encode_kv(bits(k), bits(v), c_k, c_v)


def run_decode(cfg, cache, bt_dev, seq_lens: np.ndarray, q, num_splits: int):
    """q bf16 [B, Hq, d] on device -> (out bf16 [B,Hq,d], q_fp8 uint8) via the three ABI calls
    (append with zero new tokens performs the query rotate + FP8 cast)."""
    dev = cache.device
    B = len(seq_lens)
    bufs = uq.StepBuffers(cfg, B, num_splits, dev)
    sl = torch.from_numpy(seq_lens.astype(np.int32)).to(dev)
    empty = torch.zeros((0, cfg.num_kv_heads, cfg.head_dim), dtype=torch.bfloat16, device=dev)
    cu = torch.zeros(B + 1, dtype=torch.int32, device=dev)
    out = uq.decode_step(cfg, bufs, q, empty, empty, cu, sl, sl, bt_dev, cache)
    torch.cuda.synchronize()
    return out.clone(), bufs.q_fp8.clone(), bufs


def check_out(gpu_row: np.ndarray, ref_row: np.ndarray, what=""):
    err = np.abs(gpu_row - ref_row)
    bound = ATOL + RTOL * np.abs(ref_row)
    worst = float((err / bound).max())
    assert worst <= 1.0, f"{what}: max err/bound {worst:.3f}, max abs err {err.max():.3e}, |ref| max {np.abs(ref_row).max():.3e}"
    return worst


def oracle_out(wl, b, length, q_bits_b: np.ndarray, cache_arrays=None, device="cuda", sm_scale=None):
    """float64 oracle output [Hq, d] for sequence b (and the q8 bytes it used)."""
    kc, ks, vc, vs = cache_arrays if cache_arrays is not None else oracle_sequence_cache(wl, b, length, device)
    q8 = oracle.encode_q(q_bits_b)
    return oracle.attention(q8, kc, ks, vc, vs, wl.num_q_heads, wl.num_kv_heads, sm_scale), q8


def compare_cache(cache: torch.Tensor, wl, b: int, length: int, arrays):
    """Bit-exact comparison of the device cache image with the oracle's logical arrays."""
    n_pages = -(-length // wl.page_size)
    idx = torch.from_numpy(wl.block_tables[b][:n_pages].astype(np.int64)).to(cache.device)
    recs = cache.index_select(0, idx).cpu().numpy()                # only this sequence's pages leave the device
    got = uq_layout.gather_sequence(recs, np.arange(n_pages), length)
    for name, g_, o_ in zip(("k_codes", "k_scales", "v_codes", "v_scales"), got, arrays):
        o_ = o_[:length]
        assert g_.shape == o_.shape, (name, g_.shape, o_.shape)
        bad = int((g_ != o_).sum())
        assert bad == 0, f"seq {b}: {name} differs in {bad} of {g_.size} bytes"
