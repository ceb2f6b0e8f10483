"""Parity of the CUDA path (through the C ABI / Python binding) with the float64 oracle.
Codes, scale bytes and q_fp8: bit-exact.  Attention outputs: |gpu - ref| <= 2e-3 + 1e-2 |ref|
(BASELINE.json north_star).  All inputs are seeded and synthetic (workloads.py)."""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_20474_b200 as uq
from paper_2606_20474_b200 import workloads as W
from tests import harness as H
from tests import uq_layout

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _full_check(wl, splits_list, sample_seqs=None, check_cache=True):
    """Fill the cache through the ABI, decode with every slot count of splits_list, then sequence by sequence (the
    oracle's arrays of one sequence at a time: config 3 holds 2.7 M tokens x 8 kv heads) compare the cache image bit
    for bit and every output row of every head within tolerance.  Returns (worst err/bound, sequences checked)."""
    cfg = H.cfg_of(wl)
    cache, bt = H.fill_cache(cfg, wl, DEV)
    q = W.gen_q(wl, DEV)
    qb = H.bits(q)
    seqs = list(range(wl.batch)) if sample_seqs is None else list(sample_seqs)
    outs = []
    for S in splits_list:
        out, q_fp8, _ = H.run_decode(cfg, cache, bt, wl.ctx_lens, q, S)
        outs.append((S, out.float().cpu().numpy().astype(np.float64), q_fp8.cpu().numpy()))
    worst = 0.0
    for b in seqs:
        L = int(wl.ctx_lens[b])
        arrays = H.oracle_sequence_cache(wl, b, L, DEV)
        if check_cache:
            H.compare_cache(cache, wl, b, L, arrays)
        ref, q8 = H.oracle_out(wl, b, L, qb[b], arrays)
        for S, out, q_fp8 in outs:
            assert np.array_equal(q_fp8[b], q8), f"q_fp8 differs for seq {b}"
            worst = max(worst, H.check_out(out[b], ref, f"{wl.name} seq {b} S={S}"))
        del arrays
    return worst, len(seqs)


def test_cfg1_tiny_whole_cache_bit_exact_and_decode():
    wl = W.make_config(1, peaked_frac=0.25)
    _full_check(wl, [1, 4, 7])


@pytest.mark.parametrize("d", [64, 128, 256])
@pytest.mark.parametrize("hq,hkv", [(8, 8), (12, 2), (16, 2), (32, 2), (5, 1)])
def test_ragged_batch_all_gqa_groups(hq, hkv, d):
    # empty, 1-token, ragged tails, several pages; GQA groups 1, 6, 8, 16, 5; head_dim 64 / 128 / 256
    wl = W.make_custom("ragged", 11, [0, 1, 17, 203, 1000, 16, 31, 32], hq, hkv,
                       outlier_channels=3, outlier_gain=8.0, peaked_frac=0.3, head_dim=d)
    _full_check(wl, [1, 3, 64])


def test_zero_length_rows_are_zero():
    wl = W.make_custom("empty", 12, [0, 0, 5], 8, 2)
    cfg = H.cfg_of(wl)
    cache, bt = H.fill_cache(cfg, wl, DEV)
    out, _, _ = H.run_decode(cfg, cache, bt, wl.ctx_lens, W.gen_q(wl, DEV), 2)
    assert torch.all(out[:2] == 0)


def test_incremental_appends_match_bulk_and_oracle():
    """Tokens arriving one at a time / in odd-sized pieces (V-code bytes shared by token pairs,
    page boundaries) give the same cache image as the oracle's encoding."""
    wl = W.make_custom("incr", 13, [75, 40, 1], 8, 2, extra_tokens=0)
    cfg = H.cfg_of(wl)
    cache = uq.alloc_cache(cfg, wl.num_pages, DEV)
    cache.fill_(0xA5)                                   # stale garbage must be overwritten
    bt = torch.from_numpy(wl.block_tables).to(DEV)
    full = [W.gen_kv(wl, b, 0, int(wl.ctx_lens[b]), DEV) for b in range(wl.batch)]
    pos = np.zeros(wl.batch, np.int32)
    pieces = [3, 1, 1, 14, 2, 1, 33, 1, 100]
    for n in pieces:
        counts = np.minimum(n, wl.ctx_lens - pos).astype(np.int32)
        if counts.sum() == 0:
            break
        k = torch.cat([full[b][0][pos[b]:pos[b] + counts[b]] for b in range(wl.batch)])
        v = torch.cat([full[b][1][pos[b]:pos[b] + counts[b]] for b in range(wl.batch)])
        H.append_tokens(cfg, cache, bt, pos, counts, k, v)
        pos = pos + counts
    torch.cuda.synchronize()
    assert np.array_equal(pos, wl.ctx_lens)
    for b in range(wl.batch):
        arrays = H.oracle_sequence_cache(wl, b, int(wl.ctx_lens[b]), DEV)
        H.compare_cache(cache, wl, b, int(wl.ctx_lens[b]), arrays)
    # and decode over the (partly garbage-filled last) pages stays in tolerance
    q = W.gen_q(wl, DEV)
    out, _, _ = H.run_decode(cfg, cache, bt, wl.ctx_lens, q, 2)
    for b in range(wl.batch):
        ref, _ = H.oracle_out(wl, b, int(wl.ctx_lens[b]), H.bits(q)[b])
        H.check_out(out[b].float().cpu().numpy().astype(np.float64), ref, f"incr seq {b}")


@pytest.mark.parametrize("flags", [0, uq.FLAG_SMALL_APPEND_AHEAD])
def test_shared_prefix_steps_cfg4_scaled(flags):
    """Config 4 shape at 1/64 scale: shared prefix pages named by every block table, then three
    timed-style steps (append 1 token per sequence, decode, merge) — also with UQ_FLAG_SMALL_APPEND_AHEAD, under which
    the decode kernel streams every page but a sequence's last two before the append ahead of it has finished."""
    wl = W.make_config(4, scale=1 / 64, peaked_frac=0.05)
    cfg = H.cfg_of(wl, flags=flags)
    cache, bt = H.fill_cache(cfg, wl, DEV)
    S = 3
    bufs = uq.StepBuffers(cfg, wl.batch, S, DEV)
    lens = wl.ctx_lens.copy()
    cu = torch.arange(wl.batch + 1, dtype=torch.int32, device=DEV)
    appended_k, appended_v = [], []
    for step in range(3):
        q = W.gen_q(wl, DEV, step)
        k_new, v_new = W.gen_new_kv(wl, step, DEV)
        appended_k.append(k_new); appended_v.append(v_new)
        before = torch.from_numpy(lens).to(DEV)
        after = torch.from_numpy(lens + 1).to(DEV)
        out = uq.decode_step(cfg, bufs, q, k_new, v_new, cu, before, after, bt, cache)
        torch.cuda.synchronize()
        lens = lens + 1
        out = out.float().cpu().numpy().astype(np.float64)
        for b in (0, wl.batch // 2, wl.batch - 1):
            L0 = int(wl.ctx_lens[b])
            k0, v0 = W.seq_kv(wl, b, L0, DEV)
            k = torch.cat([k0] + [a[b:b + 1] for a in appended_k])
            v = torch.cat([v0] + [a[b:b + 1] for a in appended_v])
            arrays = oracle.encode_kv(H.bits(k), H.bits(v))
            H.compare_cache(cache, wl, b, int(lens[b]), arrays)
            ref, q8 = H.oracle_out(wl, b, int(lens[b]), H.bits(q)[b], arrays)
            assert np.array_equal(bufs.q_fp8[b].cpu().numpy(), q8)
            H.check_out(out[b], ref, f"cfg4 step {step} seq {b}")


@pytest.mark.parametrize("idx,scale,d", [(2, 1 / 16, 128), (3, 1 / 16, 128), (5, 1 / 32, 128), (3, 1 / 16, 64), (3, 1 / 16, 256),
                                         (2, 1 / 16, 256), (5, 1 / 64, 64)])
def test_scaled_configs(idx, scale, d):
    wl = W.make_config(idx, scale=scale, peaked_frac=0.05, head_dim=d)
    S = uq.suggest_num_splits(H.cfg_of(wl), wl.batch, int(wl.ctx_lens.mean()))
    _full_check(wl, sorted({1, S}), sample_seqs=list(range(min(wl.batch, 3))))


@pytest.mark.parametrize("d", [128, 64, 256])
def test_merge_on_hand_made_partials(d):
    rng = np.random.default_rng(21)
    B, Hq, S = 3, 8, 5
    cfg = uq.UQConfig(Hq, 2, head_dim=d)
    acc = rng.standard_normal((B, Hq, S, d)).astype(np.float32)
    m = (rng.standard_normal((B, Hq, S)) * 20).astype(np.float32)
    l = rng.uniform(0.5, 50, (B, Hq, S)).astype(np.float32)
    m[0, 0, 1] = -np.inf; l[0, 0, 1] = 0                 # an empty split
    m[1, :, :] = -np.inf; l[1, :, :] = 0                 # a sequence of length 0
    ml = np.stack([m, l], axis=-1)
    out = torch.empty((B, Hq, d), dtype=torch.bfloat16, device=DEV)
    uq.merge_splits(cfg, torch.from_numpy(acc).to(DEV), torch.from_numpy(ml).to(DEV), out)
    torch.cuda.synchronize()
    out = out.float().cpu().numpy().astype(np.float64)
    a64, m64, l64 = acc.astype(np.float64), m.astype(np.float64), l.astype(np.float64)
    with np.errstate(invalid="ignore"):
        M = m64.max(axis=-1, keepdims=True)
        w = np.where(l64 > 0, np.exp(m64 - M), 0.0)
        den = (w * l64).sum(-1)
        ref = (w[..., None] * a64).sum(-2) / np.where(den > 0, den, 1)[..., None]
    ref[1] = 0
    assert np.all(out[1] == 0)
    assert np.allclose(out, ref, atol=1e-3 + 8e-3 * np.abs(ref).max(), rtol=8e-3)
    assert np.abs(out - ref).max() <= 2 ** -8 * np.abs(ref).max() + 1e-6   # bf16 rounding only


def test_plain_bound_holds_at_the_edge_of_the_guaranteed_domain():
    """include/uq.h "Accuracy domain": the north-star bound |gpu - ref| <= 2e-3 + 1e-2 |ref| — no extra term — is
    guaranteed for inputs whose absolute attention mass A[h, d] = sum_t p_t |vhat[t, d]| stays <= 2 (P enters the PV
    product as fp16: 2^-11 relative per term, so the cancellation error is <= 2^-10 A <= 2e-3).  Here V is scaled so
    that max A sits just below 2 and the attention is diffuse over 700 tokens (outputs are sums of ~700 cancelling
    terms, |out| ~ 0.1): the plain bound must hold for every element, for 1 and 3 slots."""
    L = 700
    wl = W.make_custom("edge", 16, [L, L - 127], 16, 2)
    cfg = H.cfg_of(wl)
    cache = uq.alloc_cache(cfg, wl.num_pages, DEV)
    bt = torch.from_numpy(wl.block_tables).to(DEV)
    kv = [W.gen_kv(wl, b, 0, int(wl.ctx_lens[b]), DEV) for b in range(2)]
    kv = [(k, (v.float() * 2.2).to(torch.bfloat16)) for k, v in kv]
    H.append_tokens(cfg, cache, bt, np.zeros(2, np.int32), wl.ctx_lens.astype(np.int32),
                    torch.cat([k for k, _ in kv]), torch.cat([v for _, v in kv]))
    q = (W.gen_q(wl, DEV).float() * 0.05).to(torch.bfloat16)          # diffuse attention: every token counts
    worst_mass = 0.0
    for S in (1, 3):
        out, _, _ = H.run_decode(cfg, cache, bt, wl.ctx_lens, q, S)
        for b in range(2):
            arrays = oracle.encode_kv(H.bits(kv[b][0]), H.bits(kv[b][1]))
            q8 = oracle.encode_q(H.bits(q)[b])
            ref, probs = oracle.attention(q8, *arrays, wl.num_q_heads, wl.num_kv_heads, None, return_probs=True)
            vhat = np.abs(oracle.dequantize(arrays[2], arrays[3]))                 # [L, Hkv, d]
            G = wl.num_q_heads // wl.num_kv_heads
            mass = np.stack([probs[h] @ vhat[:, h // G] for h in range(wl.num_q_heads)])
            worst_mass = max(worst_mass, float(mass.max()))
            H.check_out(out[b].float().cpu().numpy().astype(np.float64), ref, f"edge of domain seq {b} S={S}")
    assert 1.6 <= worst_mass <= 2.0, worst_mass                        # the input really sits at the edge


def test_wide_scale_spread_and_zero_vectors():
    """OUTSIDE the guaranteed accuracy domain of include/uq.h (absolute attention mass ~ 280 >> 2): V group scales
    spread over > 15 binades inside one page, all-zero K/V tokens, and huge K.  The cache image is still bit-exact; the
    output is checked against the kernel's documented error model (the only test whose bound carries that term)."""
    wl = W.make_custom("spread", 14, [64], 16, 1)
    cfg = H.cfg_of(wl)
    k, v = W.gen_kv(wl, 0, 0, 64, DEV)
    v = v.float()
    v[0:4] *= 2.0 ** 12
    v[4:8, :, 32:64] *= 2.0 ** -20
    v[8] = 0
    k = k.float(); k[8] = 0; k[9] *= 300.0
    k, v = k.to(torch.bfloat16), v.to(torch.bfloat16)
    cache = uq.alloc_cache(cfg, wl.num_pages, DEV)
    bt = torch.from_numpy(wl.block_tables).to(DEV)
    H.append_tokens(cfg, cache, bt, np.zeros(1, np.int32), np.array([64], np.int32), k, v)
    arrays = oracle.encode_kv(H.bits(k), H.bits(v))
    H.compare_cache(cache, wl, 0, 64, arrays)
    q = W.gen_q(wl, DEV) * 0.05                            # diffuse attention: every token counts
    out, _, _ = H.run_decode(cfg, cache, bt, wl.ctx_lens, q.to(torch.bfloat16), 1)
    qb16 = q.to(torch.bfloat16)
    q8 = oracle.encode_q(H.bits(qb16)[0])
    ref, probs = oracle.attention(q8, *arrays, wl.num_q_heads, wl.num_kv_heads, None, return_probs=True)
    got = out[0].float().cpu().numpy().astype(np.float64)
    # V is scaled by 2^12 here, so terms of magnitude ~300 cancel in some outputs.  P enters the PV
    # product as fp16 (relative rounding 2^-11 per term), hence the bound
    # carries 2^-10 * sum_t p_t |vhat_t| next to the north-star terms.
    vhat = np.abs(oracle.dequantize(arrays[2], arrays[3])[:, 0, :])          # [L, d]
    mass = probs @ vhat                                                       # [Hq, d]
    err = np.abs(got - ref)
    bound = 2e-3 + 1e-2 * np.abs(ref) + 2.0 ** -10 * mass
    assert np.all(err <= bound), float((err / bound).max())


def test_permuting_physical_pages_leaves_output_unchanged():
    wl_a = W.make_custom("perm", 15, [300, 77], 8, 1, permute=False)
    wl_b = W.make_custom("perm", 15, [300, 77], 8, 1, permute=True)
    outs = []
    for wl in (wl_a, wl_b):
        cfg = H.cfg_of(wl)
        cache, bt = H.fill_cache(cfg, wl, DEV)
        out, _, _ = H.run_decode(cfg, cache, bt, wl.ctx_lens, W.gen_q(wl, DEV), 2)
        outs.append(out)
    assert not np.array_equal(wl_a.block_tables, wl_b.block_tables)
    assert torch.equal(outs[0], outs[1])


def test_full_size_cfg2_all_32_sequences_in_bench_launch_configuration():
    """BASELINE.json config 2 at FULL size (32 x 32,768 tokens, 64/4 heads) decoded with the num_splits bench.py uses:
    ALL 32 sequences x 64 heads — every code / scale byte of the 1,048,576-token cache bit for bit, every output row
    against the oracle ("attention outputs for all (b, h) on configs 1, 2, 3, 5")."""
    wl = W.make_config(2)
    cfg = H.cfg_of(wl)
    S = uq.suggest_num_splits(cfg, wl.batch, int(wl.ctx_lens.mean()))
    _, n = _full_check(wl, [S], check_cache=True)
    assert n == 32


def test_full_size_cfg3_all_64_sequences():
    """BASELINE.json config 3 at FULL size (64 ragged sequences of 16k-64k tokens, 48/8 heads, GQA 6; 2,720,570 tokens)
    with the split count bench.py uses: ALL 64 sequences x 48 heads, cache image bit for bit and outputs."""
    wl = W.make_config(3)
    cfg = H.cfg_of(wl)
    S = uq.suggest_num_splits(cfg, wl.batch, int(wl.ctx_lens.mean()))
    _, n = _full_check(wl, [S], check_cache=True)
    assert n == 64


def test_full_size_cfg5_all_8_sequences():
    """BASELINE.json config 5 at FULL size (8 x 262,144 tokens, 64/4 heads) with the split count bench.py uses: ALL 8
    sequences x 64 heads, cache image bit for bit and outputs."""
    wl = W.make_config(5)
    cfg = H.cfg_of(wl)
    S = uq.suggest_num_splits(cfg, wl.batch, int(wl.ctx_lens.mean()))
    _, n = _full_check(wl, [S], check_cache=True)
    assert n == 8


def _cfg4_sample(wl, n=32):
    """>= 32 sequences of config 4 chosen by the seed, always including the shortest, the median, the longest and every
    capped (98,000-token) suffix."""
    order = np.argsort(wl.ctx_lens, kind="stable")
    capped = [int(b) for b in np.nonzero(wl.ctx_lens - wl.prefix_len >= 98000)[0]]
    must = [int(order[0]), int(order[len(order) // 2]), int(order[-1])] + capped
    rng = np.random.default_rng(wl.seed + 4444)
    rest = [int(b) for b in rng.permutation(wl.batch) if int(b) not in must]
    return sorted(set(must + rest[:max(0, n - len(set(must)))])), capped


def test_full_size_cfg4_shared_prefix_step_32_sequences_both_decode_paths():
    """BASELINE.json config 4 at FULL size: 256 sequences share a 30,000-token prefix (the same physical pages in every
    block table) and have log-normal private suffixes capped at 98,000; one timed-style step (append 1 token per
    sequence, decode, merge) through BOTH decode paths in bench.py's launch configurations — the plain split-K decode
    and the shared-prefix path (uq_decode_prefix_attention + suffix decode + uq_merge_splits2).  32 seeded sequences
    including the shortest, the median, the longest and all four capped suffixes: cache image (incl. the appended
    token) bit for bit, outputs of both paths against the oracle; all 256 sequences: the two paths against each other."""
    wl = W.make_config(4)
    cfg = H.cfg_of(wl)
    cache, bt = H.fill_cache(cfg, wl, DEV)
    S = uq.suggest_num_splits(cfg, wl.batch, int(wl.ctx_lens.mean()))
    bufs = uq.StepBuffers(cfg, wl.batch, S, DEV)
    q = W.gen_q(wl, DEV, 0)
    k_new, v_new = W.gen_new_kv(wl, 0, DEV)
    cu = torch.arange(wl.batch + 1, dtype=torch.int32, device=DEV)
    before = torch.from_numpy(wl.ctx_lens).to(DEV)
    after = torch.from_numpy(wl.ctx_lens + 1).to(DEV)
    out = uq.decode_step(cfg, bufs, q, k_new, v_new, cu, before, after, bt, cache)
    torch.cuda.synchronize()
    out = out.float().cpu().numpy().astype(np.float64)
    pfx = (int(wl.prefix_len) // 128) * 128
    suf = (wl.ctx_lens + 1 - pfx).astype(np.int64)
    bufs_sp = uq.StepBuffers(cfg, wl.batch, uq.suggest_num_splits_max(cfg, wl.batch, int(suf.mean()), int(suf.max())), DEV)
    bufs_sp.q_fp8.copy_(bufs.q_fp8)
    pb = uq.PrefixBuffers(cfg, wl.batch, uq.suggest_prefix_splits(cfg, wl.batch, pfx), DEV)
    pb.suffix_lens.copy_(torch.from_numpy((wl.ctx_lens + 1 - pfx).astype(np.int32)))
    out_sp = uq.decode_attention_shared_prefix(cfg, bufs_sp, pb, cache, bt, pfx)
    torch.cuda.synchronize()
    out_sp = out_sp.float().cpu().numpy().astype(np.float64)
    assert np.all(np.abs(out_sp - out) <= 2 * (H.ATOL + H.RTOL * np.abs(out)))      # every sequence, against the plain path
    sample, capped = _cfg4_sample(wl)
    assert len(sample) >= 32 and len(capped) >= 1 and set(capped) <= set(sample)
    assert int(np.argmax(wl.ctx_lens)) in sample and int(np.argmin(wl.ctx_lens)) in sample
    q_bits, q_fp8 = H.bits(q), bufs.q_fp8.cpu().numpy()
    kp, vp = W.gen_kv(wl, -1, 0, wl.prefix_len, DEV)                   # the shared prefix rows, generated once
    for b in sample:
        L0 = int(wl.ctx_lens[b])
        ks, vs = W.gen_kv(wl, b, 0, L0 - wl.prefix_len, DEV)
        k = torch.cat([kp, ks, k_new[b:b + 1]])
        v = torch.cat([vp, vs, v_new[b:b + 1]])
        arrays = oracle.encode_kv(H.bits(k), H.bits(v))
        H.compare_cache(cache, wl, b, L0 + 1, arrays)
        ref, q8 = H.oracle_out(wl, b, L0 + 1, q_bits[b], arrays)
        assert np.array_equal(q_fp8[b], q8)
        H.check_out(out[b], ref, f"cfg4 full seq {b} ({L0 + 1} tokens)")
        H.check_out(out_sp[b], ref, f"cfg4 full seq {b} ({L0 + 1} tokens), shared-prefix path")
        del arrays


def test_host_staged_step_equals_device_step_and_oracle():
    """decode_step_host (one staged H2D copy, programmatic launch chain append -> decode -> merge, D2H of O) gives
    bit-for-bit the output of decode_step on device-resident inputs, over several consecutive steps that cross
    a page boundary, and that output is within tolerance of the oracle on the grown context."""
    steps = 3
    wl = W.make_custom("staged", 21, [47, 200, 16], 16, 2, extra_tokens=steps)
    cfg = H.cfg_of(wl)
    B = wl.batch
    lens0 = (wl.ctx_lens - steps).astype(np.int32)
    caches = []
    for _ in range(3):
        cache, bt = H.fill_cache(cfg, wl, DEV, lens=lens0)
        caches.append(cache)
    bufs = [uq.StepBuffers(cfg, B, 3, DEV) for _ in range(3)]
    cu = torch.arange(B + 1, dtype=torch.int32, device=DEV)
    stage = uq.HostStage(cfg, B, B, int(bt.shape[1]), DEV)
    out_host = torch.empty((B, wl.num_q_heads, 128), dtype=torch.bfloat16).pin_memory()
    # the same step as a CUDA graph (HostStepGraph) on a third cache: its own staging block and output
    stage_g = uq.HostStage(cfg, B, B, int(bt.shape[1]), DEV)
    out_host_g = torch.empty((B, wl.num_q_heads, 128), dtype=torch.bfloat16).pin_memory()
    graph = None
    for s in range(steps):
        before = lens0 + s
        q = W.gen_q(wl, DEV, step=s)
        k = torch.cat([W.gen_kv(wl, b, int(before[b]), int(before[b]) + 1, DEV)[0] for b in range(B)])
        v = torch.cat([W.gen_kv(wl, b, int(before[b]), int(before[b]) + 1, DEV)[1] for b in range(B)])
        before_d = torch.from_numpy(before).to(DEV)
        after_d = torch.from_numpy(before + 1).to(DEV)
        ref_out = uq.decode_step(cfg, bufs[0], q, k, v, cu, before_d, after_d, bt, caches[0]).clone()
        stage.h["q"].copy_(q.cpu()); stage.h["k_new"].copy_(k.cpu()); stage.h["v_new"].copy_(v.cpu())
        stage.h["cu_new"].copy_(cu.cpu()); stage.h["seq_lens_before"].copy_(before_d.cpu())
        stage.h["seq_lens_after"].copy_(after_d.cpu()); stage.h["block_tables"].copy_(bt.cpu())
        uq.decode_step_host(cfg, bufs[1], stage, caches[1], out_host)
        torch.cuda.synchronize()
        assert torch.equal(out_host.view(torch.int16), ref_out.cpu().view(torch.int16)), f"step {s}"
        for name in uq.HostStage.FIELDS:
            stage_g.h[name].copy_(stage.h[name])
        if graph is None:                                   # captured with the first step's inputs in the block
            graph = uq.HostStepGraph(cfg, bufs[2], stage_g, caches[2], out_host_g, tables=False)   # tables sent once
        out_host_g.zero_()
        graph.launch()
        torch.cuda.synchronize()
        assert torch.equal(out_host_g.view(torch.int16), ref_out.cpu().view(torch.int16)), f"graph step {s}"
    assert torch.equal(caches[0], caches[1])
    assert torch.equal(caches[0], caches[2])
    for b in range(B):
        ref, _ = H.oracle_out(wl, b, int(wl.ctx_lens[b]), H.bits(q)[b])
        H.check_out(out_host[b].float().numpy().astype(np.float64), ref, f"staged seq {b}")


@pytest.mark.parametrize("flags", [0, uq.FLAG_SMALL_APPEND_AHEAD])
def test_step_graph_equals_direct_calls(flags):
    """uq.StepGraph (decode_step captured as a CUDA graph, inputs rewritten in place between launches) gives the
    direct calls' output bit for bit over consecutive steps, and the same cache image."""
    steps = 3
    wl = W.make_custom("sgraph", 23, [130, 31, 64, 1000], 16, 2, extra_tokens=steps)
    cfg = H.cfg_of(wl, flags=flags)
    B = wl.batch
    lens0 = (wl.ctx_lens - steps).astype(np.int32)
    (cache_a, bt), (cache_b, _) = H.fill_cache(cfg, wl, DEV, lens=lens0), H.fill_cache(cfg, wl, DEV, lens=lens0)
    bufs_a, bufs_b = uq.StepBuffers(cfg, B, 3, DEV), uq.StepBuffers(cfg, B, 3, DEV)
    cu = torch.arange(B + 1, dtype=torch.int32, device=DEV)
    q_g = torch.empty((B, wl.num_q_heads, 128), dtype=torch.bfloat16, device=DEV)
    k_g = torch.empty((B, wl.num_kv_heads, 128), dtype=torch.bfloat16, device=DEV)
    v_g = torch.empty_like(k_g)
    before_g = torch.empty(B, dtype=torch.int32, device=DEV)
    after_g = torch.empty(B, dtype=torch.int32, device=DEV)
    graph = None
    for s_ in range(steps):
        before = lens0 + s_
        q = W.gen_q(wl, DEV, step=s_)
        k = torch.cat([W.gen_kv(wl, b, int(before[b]), int(before[b]) + 1, DEV)[0] for b in range(B)])
        v = torch.cat([W.gen_kv(wl, b, int(before[b]), int(before[b]) + 1, DEV)[1] for b in range(B)])
        before_d, after_d = torch.from_numpy(before).to(DEV), torch.from_numpy(before + 1).to(DEV)
        ref = uq.decode_step(cfg, bufs_a, q, k, v, cu, before_d, after_d, bt, cache_a).clone()
        q_g.copy_(q); k_g.copy_(k); v_g.copy_(v); before_g.copy_(before_d); after_g.copy_(after_d)
        if graph is None:
            graph = uq.StepGraph(cfg, bufs_b, q_g, k_g, v_g, cu, before_g, after_g, bt, cache_b)
        bufs_b.out.zero_()
        out = graph.launch()
        torch.cuda.synchronize()
        assert torch.equal(out.view(torch.int16), ref.view(torch.int16)), f"step {s_}"
    assert torch.equal(cache_a, cache_b)


@pytest.mark.parametrize("d", [64, 256])
def test_append_on_rounding_boundaries_other_head_dims(d):
    """The boundary rows of the test below (E2M1 ties, scale thresholds +- one bf16 step, constant / one-hot / huge /
    tiny / zero rows) at head_dim 64 and 256 — the float64 kernel of those head sizes — bit for bit the oracle's image,
    appended in one call and token by token; and the query bytes."""
    L = 160
    wl = W.make_custom("bound_d", 33 + d, [L], 8, 2, head_dim=d)
    cfg = H.cfg_of(wl)
    g = torch.Generator(device="cpu"); g.manual_seed(99 + d)
    k, v = _boundary_rows(L, g, d)
    k, v = k.to(torch.bfloat16).to(DEV), v.to(torch.bfloat16).to(DEV)
    bt = torch.from_numpy(wl.block_tables).to(DEV)
    ref = oracle.encode_kv(H.bits(k), H.bits(v))
    cache = uq.alloc_cache(cfg, wl.num_pages, DEV); cache.fill_(0x5C)
    H.append_tokens(cfg, cache, bt, np.zeros(1, np.int32), np.array([L], np.int32), k, v)
    torch.cuda.synchronize()
    H.compare_cache(cache, wl, 0, L, ref)
    cache2 = uq.alloc_cache(cfg, wl.num_pages, DEV); cache2.fill_(0xC5)
    pos = 0
    for n in [1, 1, 3, 7, 1, 12, 30, 5, 100]:
        n = min(n, L - pos)
        H.append_tokens(cfg, cache2, bt, np.array([pos], np.int32), np.array([n], np.int32), k[pos:pos + n], v[pos:pos + n])
        pos += n
    torch.cuda.synchronize()
    assert pos == L
    H.compare_cache(cache2, wl, 0, L, ref)
    q = torch.randn((1, 8, d), generator=g)
    q[0, 0] = 0.75; q[0, 1] = 0; q[0, 1, 17] = -2.0; q[0, 2] *= 1e20; q[0, 3] *= 1e-20; q[0, 4] = 0
    q[0, 5] = 448.0 / d ** 0.5
    q = q.to(torch.bfloat16).to(DEV)
    _, q_fp8, _ = H.run_decode(cfg, cache, bt, wl.ctx_lens, q, 1)
    assert np.array_equal(q_fp8[0].cpu().numpy(), oracle.encode_q(H.bits(q)[0]))


def test_append_on_rounding_boundaries_is_bit_exact():
    """The append kernel's float32 fast path must hand every close call to float64: V elements exactly on the
    E2M1 ties (0.25, 0.75, 1.25, 1.75, 2.5, 3.5, 5 times the group scale), group maxima on both sides of the
    scale-exponent thresholds 2^(k-1/2)/c (nextafter in bf16), constant and one-hot K rows (rotated vectors with
    127 exact zeros / 128 equal magnitudes), huge and tiny magnitudes — all compared bit for bit with the oracle."""
    L = 192
    wl = W.make_custom("bound", 31, [L], 8, 2)
    cfg = H.cfg_of(wl)
    g = torch.Generator(device="cpu"); g.manual_seed(1234)
    k = torch.randn((L, 2, 128), generator=g)
    v = torch.randn((L, 2, 128), generator=g)
    ties = torch.tensor([0.25, 0.75, 1.25, 1.75, 2.5, 3.5, 5.0, 6.0, 0.5, 1.0, 1.5, 2.0, 3.0, 4.0, 0.0, -0.25])
    for t in range(0, 64):                                  # V: group max 6 * 2^e -> E = e; the rest sits on ties
        e = (t % 23) - 11
        row = ties[torch.randint(0, 16, (2, 128), generator=g)] * (1.0 if t % 2 else -1.0)
        row[:, ::32] = 6.0                                 # one maximum per 32-group
        v[t] = row * 2.0 ** e
    thr = [2.0 ** (kk - 0.5) / 0.15600000321865082 for kk in range(-6, 7)]
    for t in range(64, 96):                                 # V: group maxima right below / above a scale threshold
        x = torch.tensor(thr[t % len(thr)], dtype=torch.float32).to(torch.bfloat16)
        nb = (x.view(torch.int16) + (1 if t % 2 else -1)).view(torch.bfloat16)
        row = torch.rand((2, 128), generator=g) * float(x) * 0.9
        row[:, ::32] = float(nb) if t % 3 else float(x)
        v[t] = row
    k[96] = 0.75                                            # constant rows: one nonzero rotated value, 127 zeros
    k[97] = -3.0
    k[98] = 0; k[98, :, 5] = 2.0                            # one-hot rows: 128 equal magnitudes
    k[99] = 0; k[99, :, 127] = -1.0 / 3.0
    k[100] *= 1e20; k[101] *= 1e-20; v[100] *= 1e25; v[101] *= 1e-25
    k[102] = 0; v[102] = 0
    k, v = k.to(torch.bfloat16).to(DEV), v.to(torch.bfloat16).to(DEV)
    cache = uq.alloc_cache(cfg, wl.num_pages, DEV)
    bt = torch.from_numpy(wl.block_tables).to(DEV)
    H.append_tokens(cfg, cache, bt, np.zeros(1, np.int32), np.array([L], np.int32), k, v)
    torch.cuda.synchronize()
    arrays = oracle.encode_kv(H.bits(k), H.bits(v))
    H.compare_cache(cache, wl, 0, L, arrays)
    # query rows: constant, one-hot, huge, tiny, zero, and random ones -> q_fp8 bytes against the oracle
    q = torch.randn((1, 8, 128), generator=g)
    q[0, 0] = 0.75; q[0, 1] = 0; q[0, 1, 17] = -2.0; q[0, 2] *= 1e20; q[0, 3] *= 1e-20; q[0, 4] = 0
    q[0, 5] = 448.0 / 11.313708498984761                    # rotated value 448-ish: the saturation boundary
    q = q.to(torch.bfloat16).to(DEV)
    _, q_fp8, _ = H.run_decode(cfg, cache, bt, wl.ctx_lens, q, 1)
    assert np.array_equal(q_fp8[0].cpu().numpy(), oracle.encode_q(H.bits(q)[0]))


def _boundary_rows(L, g, d=128):
    """K / V rows of test_append_on_rounding_boundaries_is_bit_exact (first 103 rows special, the rest N(0,1))."""
    k = torch.randn((L, 2, d), generator=g)
    v = torch.randn((L, 2, d), generator=g)
    ties = torch.tensor([0.25, 0.75, 1.25, 1.75, 2.5, 3.5, 5.0, 6.0, 0.5, 1.0, 1.5, 2.0, 3.0, 4.0, 0.0, -0.25])
    for t in range(0, 64):
        e = (t % 23) - 11
        row = ties[torch.randint(0, 16, (2, d), generator=g)] * (1.0 if t % 2 else -1.0)
        row[:, ::32] = 6.0
        v[t] = row * 2.0 ** e
    thr = [2.0 ** (kk - 0.5) / 0.15600000321865082 for kk in range(-6, 7)]
    for t in range(64, 96):
        x = torch.tensor(thr[t % len(thr)], dtype=torch.float32).to(torch.bfloat16)
        nb = (x.view(torch.int16) + (1 if t % 2 else -1)).view(torch.bfloat16)
        row = torch.rand((2, d), generator=g) * float(x) * 0.9
        row[:, ::32] = float(nb) if t % 3 else float(x)
        v[t] = row
    k[96] = 0.75
    k[97] = -3.0
    k[98] = 0; k[98, :, 5] = 2.0
    k[99] = 0; k[99, :, d - 1] = -1.0 / 3.0
    k[100] *= 1e20; k[101] *= 1e-20; v[100] *= 1e25; v[101] *= 1e-25
    k[102] = 0; v[102] = 0
    return k, v


@pytest.mark.parametrize("start", [0, 5, 37])
def test_bulk_append_kernel_on_rounding_boundaries_and_ragged_ends(start):
    """The bulk append kernel (one warp per aligned block of 32 positions, prefill-sized calls): the same boundary
    rows as above, spread over whole blocks and the partly covered head / tail blocks of the range (the sequence
    starts at position `start`, so rows land in different lanes, octets and pages) — bit for bit the oracle's
    image, and byte-identical to the per-octet kernel (UQ_FLAG_NO_BULK_APPEND) on the same input."""
    L = 1500
    wl = W.make_custom("bulkbound", 77 + start, [start + L], 8, 2)
    g = torch.Generator(device="cpu"); g.manual_seed(4321 + start)
    k, v = _boundary_rows(L, g)
    perm = torch.randperm(L, generator=g)                   # the special rows anywhere in the range
    k, v = k[perm], v[perm]
    k0, v0 = torch.randn((start, 2, 128), generator=g), torch.randn((start, 2, 128), generator=g)
    k, v = torch.cat([k0, k]).to(torch.bfloat16).to(DEV), torch.cat([v0, v]).to(torch.bfloat16).to(DEV)
    bt = torch.from_numpy(wl.block_tables).to(DEV)
    images = []
    for flags in (0, 1):
        cfg = H.cfg_of(wl, flags=flags)
        cache = uq.alloc_cache(cfg, wl.num_pages, DEV)
        cache.fill_(0x3C)
        if start:
            H.append_tokens(cfg, cache, bt, np.zeros(1, np.int32), np.array([start], np.int32), k[:start], v[:start])
        H.append_tokens(cfg, cache, bt, np.array([start], np.int32), np.array([L], np.int32), k[start:], v[start:])
        torch.cuda.synchronize()
        H.compare_cache(cache, wl, 0, start + L, oracle.encode_kv(H.bits(k), H.bits(v)))
        images.append(cache.clone())
    n_rec = -(-(start + L) // 16)
    idx = torch.from_numpy(wl.block_tables[0][:n_rec - 1].astype(np.int64)).to(DEV)   # whole pages: every byte defined
    assert torch.equal(images[0].index_select(0, idx), images[1].index_select(0, idx))


def test_bulk_append_many_sequences_irregular_counts():
    """A prefill-sized call over 24 sequences with irregular starts and counts (zero counts, counts below one
    block, ranges that start and end inside a block): every token of sampled sequences in its slot, bit-exact."""
    B = 24
    rng = np.random.default_rng(99)
    starts = rng.integers(0, 70, B).astype(np.int32)
    counts = rng.integers(0, 400, B).astype(np.int32)
    counts[[3, 11]] = 0
    counts[[5, 17]] = [7, 33]
    wl = W.make_custom("bulkmulti", 4242, [int(x) for x in starts + counts], 8, 2)
    cfg = H.cfg_of(wl)
    assert counts.sum() >= max(1024, 64 * B)                # the call takes the bulk kernel
    cache = uq.alloc_cache(cfg, wl.num_pages, DEV)
    cache.fill_(0xC3)
    bt = torch.from_numpy(wl.block_tables).to(DEV)
    full = [W.gen_kv(wl, b, 0, int(wl.ctx_lens[b]), DEV) for b in range(B)]
    if starts.sum():
        H.append_tokens(cfg, cache, bt, np.zeros(B, np.int32), starts,
                        torch.cat([full[b][0][:starts[b]] for b in range(B)]),
                        torch.cat([full[b][1][:starts[b]] for b in range(B)]))
    H.append_tokens(cfg, cache, bt, starts, counts,
                    torch.cat([full[b][0][starts[b]:] for b in range(B)]),
                    torch.cat([full[b][1][starts[b]:] for b in range(B)]))
    torch.cuda.synchronize()
    for b in range(B):
        L = int(wl.ctx_lens[b])
        if L:
            H.compare_cache(cache, wl, b, L, H.oracle_sequence_cache(wl, b, L, DEV))


@pytest.mark.parametrize("d", [128, 64, 256])
def test_random_small_configs(d):
    """Seeded sweep over head geometries, batch sizes (up to more items than resident CTAs), length mixes (empty,
    one token, tile multiples +-1, ragged) and slot counts 1..6: cache image bit-exact, outputs in tolerance.
    head_dim 128 (24 cases) and 64 / 256 (16 cases each, other seeds)."""
    rng = np.random.default_rng(7 if d == 128 else 7000 + d)
    heads = [(8, 8), (8, 1), (16, 1), (12, 2), (32, 2), (6, 1), (10, 2), (64, 4), (48, 8)]
    for case in range(24 if d == 128 else 16):
        hq, hkv = heads[rng.integers(len(heads))]
        kind = int(rng.integers(6))
        B = int(rng.integers(1, 7)) if kind < 4 else int(rng.integers(40, 130))
        if kind == 0: lens = rng.integers(0, 40, B)
        elif kind == 1: lens = rng.integers(100, 700, B)
        elif kind == 2: lens = rng.integers(0, 3000, B)
        elif kind == 3: lens = np.array([int(rng.integers(1, 5)) * 128 + int(rng.integers(-1, 2)) for _ in range(B)])
        else: lens = rng.integers(0, 260, B)
        if lens.sum() == 0: lens[0] = 1
        S = int(rng.integers(1, 7))
        wl = W.make_custom(f"rnd{case}", 1000 + case, [int(x) for x in lens], hq, hkv,
                           peaked_frac=float(rng.choice([0.0, 0.3])), head_dim=d)
        cfg = H.cfg_of(wl)
        cache, bt = H.fill_cache(cfg, wl, DEV)
        q = W.gen_q(wl, DEV)
        out, q_fp8, _ = H.run_decode(cfg, cache, bt, wl.ctx_lens, q, S)
        out = out.float().cpu().numpy().astype(np.float64)
        for b in rng.choice(B, min(B, 6), replace=False):
            L = int(wl.ctx_lens[b])
            if L == 0:
                assert np.all(out[b] == 0), f"case {case} seq {b}: an empty sequence gives zeros"
                continue
            arrays = H.oracle_sequence_cache(wl, int(b), L, DEV)
            H.compare_cache(cache, wl, int(b), L, arrays)
            ref, q8 = H.oracle_out(wl, int(b), L, H.bits(q)[b], arrays)
            assert np.array_equal(q_fp8[b].cpu().numpy(), q8)
            H.check_out(out[b], ref, f"case {case} {hq}/{hkv} B={B} S={S} seq {b} len {L}")


@pytest.mark.parametrize("B", [33, 700, 1025, 1500])
def test_random_multi_sequence_appends(B):
    """Several sequences per append call with irregular counts (zeros included) over consecutive calls: the guess,
    the two-level warp search (batch <= 1024) and the binary search (beyond) of cu_new all land every token in its
    slot — cache image of sampled sequences bit-exact against the oracle."""
    rng = np.random.default_rng(B)
    lens = rng.integers(0, 50, B)
    lens[rng.integers(0, B, B // 3)] = 0
    wl = W.make_custom(f"ma{B}", 2000 + B, [int(x) for x in lens], 8, 2)
    cfg = H.cfg_of(wl)
    cache = uq.alloc_cache(cfg, wl.num_pages, DEV)
    cache.fill_(0x5A)
    bt = torch.from_numpy(wl.block_tables).to(DEV)
    full, pos = {}, np.zeros(B, np.int32)
    while (pos < wl.ctx_lens).any():
        counts = np.minimum(rng.integers(0, 20, B), wl.ctx_lens - pos).astype(np.int32)
        if counts.sum() == 0:
            continue
        ks, vs = [], []
        for b in np.nonzero(counts)[0]:
            if b not in full:
                full[b] = W.gen_kv(wl, int(b), 0, int(wl.ctx_lens[b]), DEV)
            ks.append(full[b][0][pos[b]:pos[b] + counts[b]])
            vs.append(full[b][1][pos[b]:pos[b] + counts[b]])
        H.append_tokens(cfg, cache, bt, pos, counts, torch.cat(ks), torch.cat(vs))
        pos = pos + counts
    torch.cuda.synchronize()
    for b in rng.choice(B, 10, replace=False):
        L = int(wl.ctx_lens[b])
        if L:
            H.compare_cache(cache, wl, int(b), L, H.oracle_sequence_cache(wl, int(b), L, DEV))


def test_custom_constants_sm_scale_and_c():
    """Non-default uq_config values reach the kernels: softmax scale 0.05 (instead of 1/sqrt(d)) and the paper's
    power-of-two-rule constant c = 0.195 for K and V — cache bit-exact, outputs in tolerance."""
    wl = W.make_custom("consts", 41, [333, 40], 16, 2, peaked_frac=0.3)
    cfg = H.cfg_of(wl, sm_scale=0.05, c_k=0.195, c_v=0.195)
    cache, bt = H.fill_cache(cfg, wl, DEV)
    q = W.gen_q(wl, DEV)
    out, q_fp8, _ = H.run_decode(cfg, cache, bt, wl.ctx_lens, q, 3)
    for b in range(wl.batch):
        L = int(wl.ctx_lens[b])
        arrays = H.oracle_sequence_cache(wl, b, L, DEV, c_k=0.195, c_v=0.195)
        H.compare_cache(cache, wl, b, L, arrays)
        ref, q8 = H.oracle_out(wl, b, L, H.bits(q)[b], arrays, sm_scale=0.05)
        assert np.array_equal(q_fp8[b].cpu().numpy(), q8)
        H.check_out(out[b].float().cpu().numpy().astype(np.float64), ref, f"consts seq {b}")


def test_decode_refuses_more_than_2048_sequences():
    """include/uq.h: at most 2048 sequences per uq_decode_attention call (the tile prefix sums live in shared
    memory); a larger batch is refused on the host with UQ_ERR_INVALID_ARG / UQ_ERR_UNSUPPORTED and nothing is launched."""
    cfg = uq.UQConfig(num_q_heads=8, num_kv_heads=1)
    B = 2049
    cache = uq.alloc_cache(cfg, 4, DEV)
    bt = torch.zeros((B, 1), dtype=torch.int32, device=DEV)
    lens = torch.ones(B, dtype=torch.int32, device=DEV)
    q8 = torch.zeros((B, 8, 128), dtype=torch.uint8, device=DEV)
    acc = torch.zeros((B, 8, 2, 128), dtype=torch.float32, device=DEV)
    ml = torch.zeros((B, 8, 2, 2), dtype=torch.float32, device=DEV)
    with pytest.raises(uq.UQError, match="2048"):
        uq.decode_attention(cfg, q8, cache, bt, lens, 2, acc, ml)
    torch.cuda.synchronize()


@pytest.mark.parametrize("rotate,pow2", [(True, True), (True, False), (False, True), (False, False)])
def test_calibrate_c_matches_the_oracle_objective(rotate, pow2):
    """uq_calibrate_c (Eq.(2)) against oracle.calib_sq_err on keys with outlier
    channels, scale spread over vectors, all-zero vectors and groups: every sum within 1e-11 relative (the float64
    additions are ordered differently), the same argmin, and — on the rotated keys — the paper's constants."""
    g = torch.Generator(device="cpu"); g.manual_seed(77)
    n = 3001                                               # not a multiple of the warps of a CTA
    x = torch.randn((n, 128), generator=g) * torch.exp(0.7 * torch.randn((n, 1), generator=g))
    x[:, [3, 40, 97]] *= 9.0
    x[5] = 0; x[6, 32:64] = 0; x[7] = 2.0 ** -120; x[8] = 3.0e30
    x = x.to(torch.bfloat16)
    cs = np.concatenate([np.arange(0.10, 0.30, 0.0125), [0.156, 0.195, 1.0, 0.5]]).astype(np.float32)   # 20: 8 + 8 + 4
    cfg = uq.UQConfig(num_q_heads=8, num_kv_heads=1)
    sq, nrm = uq.calibrate_c(cfg, x.to(DEV), torch.from_numpy(cs).to(DEV), rotate=rotate, pow2_scale=pow2)
    torch.cuda.synchronize()
    sq, nrm = sq.cpu().numpy(), float(nrm.cpu()[0])
    ref, ref_nrm = oracle.calib_sq_err(H.bits(x), cs, rotate=rotate, pow2=pow2)
    assert nrm == pytest.approx(ref_nrm, rel=1e-11)
    np.testing.assert_allclose(sq, ref, rtol=1e-11, atol=0)
    assert int(np.argmin(sq)) == int(np.argmin(ref))
    if rotate:
        # without the rows of extreme magnitude (they dominate the sums) the rotated keys behave like the paper's:
        # continuous optimum near 0.156 (:128), power-of-two optimum near 0.195 (:333)
        sq2, _ = uq.calibrate_c(cfg, x[9:].contiguous().to(DEV), torch.from_numpy(cs).to(DEV), rotate=True, pow2_scale=pow2)
        best = float(cs[int(torch.argmin(sq2[:16]).item())])
        assert abs(best - (0.195 if pow2 else 0.156)) < 0.03


def test_calibrate_c_other_codebooks_and_fixed_scale():
    """uq_calibrate_c with a codebook other than E2M1 (uniform INT4 magnitudes 0..7 on the absmax scale; 8 Lloyd-Max-
    like magnitudes on a fixed scale, scale_mode 2) against the oracle, on coordinates of random unit vectors
    (the distribution of Fig. 2)."""
    g = torch.Generator(device="cpu"); g.manual_seed(5)
    u = torch.randn((2048, 128), generator=g)
    u = (u / u.norm(dim=1, keepdim=True)).to(torch.bfloat16)
    cfg = uq.UQConfig(num_q_heads=8, num_kv_heads=1)
    lm = np.array([0.1284, 0.3881, 0.6568, 0.9424, 1.2562, 1.6181, 2.0690, 2.7326], np.float32)
    cases = [(0, np.arange(8, dtype=np.float32), np.array([1 / 7, 0.12, 0.2], np.float32)),
             (2, lm, np.array([128 ** -0.5, 0.07, 0.1], np.float32)),
             (2, None, np.array([0.02, 0.05], np.float32))]
    for mode, lev, cs in cases:
        sq, nrm = uq.calibrate_c(cfg, u.to(DEV), torch.from_numpy(cs).to(DEV), rotate=False, scale_mode=mode,
                                 levels=None if lev is None else torch.from_numpy(lev).to(DEV))
        ref, ref_nrm = oracle.calib_sq_err(H.bits(u), cs, rotate=False, scale_mode=mode, levels=lev)
        np.testing.assert_allclose(sq.cpu().numpy(), ref, rtol=1e-11, atol=0)
        assert float(nrm.cpu()[0]) == pytest.approx(ref_nrm, rel=1e-11)


@pytest.mark.parametrize("hq,hkv,lens,prefix,pfx_call,splits", [
    (16, 2, [700, 512, 1300, 497, 900], 496, 384, (2, 3)),          # G = 8, odd batch: the last group has one sequence
    (32, 2, [1500, 1500, 2100, 1281], 1280, 1280, (3, 2)),          # G = 16, a sequence with a 1-token suffix
    (16, 1, [640, 640], 640, 640, (2, 2)),                           # no suffix at all: every suffix slot empty
    (2, 2, [129], 128, 128, (2, 1)),                                 # one sequence, G = 1, a single prefix tile
    (8, 2, [300 + 7 * i for i in range(37)], 256, 256, (4, 2)),      # 37 sequences (10 groups of 4, the last with 1), G = 4
])
def test_shared_prefix_decode_matches_the_oracle_and_the_plain_decode(hq, hkv, lens, prefix, pfx_call, splits):
    """uq_decode_prefix_attention + suffix decode + uq_merge_splits2 on sequences whose block
    tables name the same prefix pages: outputs within tolerance of the float64 oracle for every sequence, and within
    twice that of the plain decode of the same cache (two roundings of the same quantities)."""
    wl = W.make_custom("pfx", 300 + hq + len(lens), lens, hq, hkv, prefix_len=prefix, peaked_frac=0.05)
    cfg = H.cfg_of(wl)
    cache, bt = H.fill_cache(cfg, wl, DEV)
    q = W.gen_q(wl, DEV)
    plain, q_fp8, bufs = H.run_decode(cfg, cache, bt, wl.ctx_lens, q, 3)
    B = wl.batch
    sp, ss = splits
    bufs2 = uq.StepBuffers(cfg, B, ss, DEV)
    bufs2.q_fp8.copy_(q_fp8)
    pb = uq.PrefixBuffers(cfg, B, sp, DEV)
    pb.suffix_lens.copy_(torch.from_numpy((wl.ctx_lens - pfx_call).astype(np.int32)))
    bufs2.partial_acc.fill_(float("nan")); pb.partial_acc.fill_(float("nan"))   # every slot has to be written
    bufs2.partial_ml.fill_(float("nan")); pb.partial_ml.fill_(float("nan"))
    out = uq.decode_attention_shared_prefix(cfg, bufs2, pb, cache, bt, pfx_call)
    torch.cuda.synchronize()
    out = out.float().cpu().numpy().astype(np.float64)
    assert np.isfinite(out).all()
    for b in range(B):
        ref, _ = H.oracle_out(wl, b, int(wl.ctx_lens[b]), H.bits(q)[b])
        H.check_out(out[b], ref, f"shared prefix seq {b}")
    pl = plain.float().cpu().numpy().astype(np.float64)
    assert np.all(np.abs(out - pl) <= 2 * (H.ATOL + H.RTOL * np.abs(pl)))


def test_debug_checks_name_the_first_bad_table_entry_and_leave_good_calls_alone():
    """UQ_FLAG_DEBUG_CHECKS (include/uq.h): with the flag a call whose block table names a page outside the
    cache, whose length exceeds the table, whose cu_new is inconsistent or whose "shared" prefix is not shared is
    refused with UQ_ERR_INVALID_ARG naming the offender — nothing is written; a valid call gives bit for bit the
    result of the same call without the flag."""
    wl = W.make_custom("dbg", 51, [300, 277, 512], 16, 2, prefix_len=256, extra_tokens=4)
    cfg = H.cfg_of(wl)
    dbg = H.cfg_of(wl, flags=uq.FLAG_DEBUG_CHECKS)
    cache, bt = H.fill_cache(dbg, wl, DEV)                  # the fill itself runs under the checks
    cache_ref, _ = H.fill_cache(cfg, wl, DEV)
    assert torch.equal(cache, cache_ref)
    q = W.gen_q(wl, DEV)
    out_ref, q_fp8, bufs = H.run_decode(cfg, cache, bt, wl.ctx_lens, q, 3)
    out_dbg, _, _ = H.run_decode(dbg, cache, bt, wl.ctx_lens, q, 3)
    assert torch.equal(out_ref, out_dbg)
    lens = torch.from_numpy(wl.ctx_lens.astype(np.int32)).to(DEV)
    # (1) an entry outside the cache, inside the used range of sequence 1
    bad = bt.clone(); bad[1, 17] = wl.num_pages
    with pytest.raises(uq.UQError, match=r"block_tables\[1\]\[17\]"):
        uq.decode_attention(dbg, q_fp8, cache, bad, lens, 3, bufs.partial_acc, bufs.partial_ml)
    bad = bt.clone(); bad[0, 0] = -1
    with pytest.raises(uq.UQError, match=r"block_tables\[0\]\[0\] = -1"):
        uq.decode_attention(dbg, q_fp8, cache, bad, lens, 3, bufs.partial_acc, bufs.partial_ml)
    # ... but not one beyond the sequence's last page (never read)
    ok = bt.clone(); ok[1, 20] = 10 ** 6          # seq 1: 277 tokens = pages 0..17
    uq.decode_attention(dbg, q_fp8, cache, ok, lens, 3, bufs.partial_acc, bufs.partial_ml)
    # (2) a length the table cannot hold
    long_lens = lens.clone(); long_lens[2] = bt.shape[1] * 16 + 1
    with pytest.raises(uq.UQError, match="sequence 2"):
        uq.decode_attention(dbg, q_fp8, cache, bt, long_lens, 3, bufs.partial_acc, bufs.partial_ml)
    # (3) append: decreasing cu_new, a write past the table, a bad entry on the page written
    k1, v1 = W.gen_kv(wl, 0, 0, 3, DEV)
    before = cache.clone()
    cu = torch.tensor([0, 2, 1, 3], dtype=torch.int32, device=DEV)
    with pytest.raises(uq.UQError, match="cu_new"):
        uq.rotate_quantize_append(dbg, k1, v1, cu, lens, bt, cache)
    cu = torch.tensor([0, 1, 2, 3], dtype=torch.int32, device=DEV)
    with pytest.raises(uq.UQError, match="sequence 2"):
        uq.rotate_quantize_append(dbg, k1, v1, cu, long_lens, bt, cache)
    bad = bt.clone(); bad[1, 277 // 16] = -5
    with pytest.raises(uq.UQError, match=r"block_tables\[1\]\[17\] = -5"):
        uq.rotate_quantize_append(dbg, k1, v1, cu, lens, bad, cache)
    torch.cuda.synchronize()
    assert torch.equal(cache, before)                       # nothing was written by the refused calls
    uq.rotate_quantize_append(dbg, k1, v1, cu, lens, bt, cache)       # the valid append passes
    # (4) shared prefix that is not shared
    pb = uq.PrefixBuffers(cfg, wl.batch, 2, DEV)
    pb.suffix_lens.copy_(lens - 256)
    bufs2 = uq.StepBuffers(dbg, wl.batch, 2, DEV); bufs2.q_fp8.copy_(q_fp8)
    bad = bt.clone(); bad[2, 7] = bt[2, 20]
    with pytest.raises(uq.UQError, match="not shared"):
        uq.decode_attention_shared_prefix(dbg, bufs2, pb, cache, bad, 256)
    uq.decode_attention_shared_prefix(dbg, bufs2, pb, cache, bt, 256)
    torch.cuda.synchronize()


def test_second_device_of_one_process_if_there_is_one():
    """The library keeps its per-device state (SM count, shared-memory opt-in, TMA descriptors) per device: a decode
    on device 1 after one on device 0 in the same process gives the same output.  Skipped on one-GPU boxes."""
    if torch.cuda.device_count() < 2:
        pytest.skip("one visible device")
    wl = W.make_custom("dev1", 52, [700, 130], 16, 2)
    outs = []
    for dev in ("cuda:0", "cuda:1"):
        with torch.cuda.device(dev):
            cfg = H.cfg_of(wl)
            cache, bt = H.fill_cache(cfg, wl, dev)
            out, _, _ = H.run_decode(cfg, cache, bt, wl.ctx_lens, W.gen_q(wl, dev), 3)
            outs.append(out.cpu())
    assert torch.equal(outs[0], outs[1])


def _fill_baseline_cache(cfg, kv, wl):
    cache = uq.alloc_baseline_cache(cfg, kv, wl.num_pages, DEV)
    cache.fill_(0xFF)                                       # NaN patterns of E4M3 / bf16: stale bytes must never reach an output
    bt = torch.from_numpy(wl.block_tables).to(DEV)
    B = wl.batch
    for b in range(B):
        L = int(wl.ctx_lens[b])
        done = 0
        for n in ([L] if b % 2 == 0 else [min(L, 5), min(max(L - 5, 0), 40), max(L - 45, 0)]):   # one call, or in pieces
            if n == 0:
                continue
            k, v = W.gen_kv(wl, b, done, done + n, DEV)
            before = np.zeros(B, np.int32); before[b] = done
            cu = np.zeros(B + 1, np.int32); cu[b + 1:] = n
            uq.baseline_append(cfg, kv, k, v, torch.from_numpy(cu).to(DEV), torch.from_numpy(before).to(DEV), bt, cache)
            done += n
    torch.cuda.synchronize()
    return cache, bt


@pytest.mark.parametrize("kv", ["fp8", "bf16"])
@pytest.mark.parametrize("hq,hkv", [(16, 1), (12, 2), (8, 8)])
def test_comparison_caches_fp8_and_bf16_kv(kv, hq, hkv):
    """The comparison kernels ("hardware FP8 KV" / BF16 baseline): cache image bit for
    bit (E4M3 bytes of the bf16 values = oracle.cast_e4m3; the bf16 bits themselves), the FP8 query bytes, and the
    decode output within 2e-3 + 1e-2 |ref| of oracle.attention_fp8kv / attention_bf16kv — ragged batch with empty,
    one-token and multi-tile sequences, GQA 16 / 6 / 1, slot counts 1, 3 and 64, peaked queries."""
    fmt = uq.KV_FP8_E4M3 if kv == "fp8" else uq.KV_BF16
    wl = W.make_custom("cmp", 61, [0, 1, 17, 203, 1000, 16, 31, 129], hq, hkv, outlier_channels=3, outlier_gain=8.0,
                       peaked_frac=0.3)
    cfg = H.cfg_of(wl)
    cache, bt = _fill_baseline_cache(cfg, fmt, wl)
    q = W.gen_q(wl, DEV)
    qb = H.bits(q)
    host = cache.cpu().numpy()
    kpage = 2048 if kv == "fp8" else 4096
    lens = torch.from_numpy(wl.ctx_lens.astype(np.int32)).to(DEV)
    empty = torch.zeros((0, hkv, 128), dtype=torch.bfloat16, device=DEV)
    cu0 = torch.zeros(wl.batch + 1, dtype=torch.int32, device=DEV)
    refs = {}
    for b in range(wl.batch):
        L = int(wl.ctx_lens[b])
        if L == 0:
            continue
        k, v = W.seq_kv(wl, b, L, DEV)
        kbits, vbits = H.bits(k), H.bits(v)
        recs = host[wl.block_tables[b][:-(-L // 16)]]                          # [pages, Hkv, rec]
        if kv == "fp8":
            gk = recs[..., :kpage].reshape(-1, hkv, 16, 128).transpose(0, 2, 1, 3).reshape(-1, hkv, 128)[:L]
            gv = recs[..., kpage:].reshape(-1, hkv, 128, 16).transpose(0, 3, 1, 2).reshape(-1, hkv, 128)[:L]
            ref, q8, k8, v8 = oracle.attention_fp8kv(qb[b], kbits, vbits)
            assert np.array_equal(gk, k8) and np.array_equal(gv, v8), f"seq {b}: FP8 cache image differs"
            refs[b] = (ref, q8)
        else:
            r16 = recs.view(np.uint16)
            gk = r16[..., :kpage // 2].reshape(-1, hkv, 16, 128).transpose(0, 2, 1, 3).reshape(-1, hkv, 128)[:L]
            gv = r16[..., kpage // 2:].reshape(-1, hkv, 128, 16).transpose(0, 3, 1, 2).reshape(-1, hkv, 128)[:L]
            assert np.array_equal(gk, kbits) and np.array_equal(gv, vbits), f"seq {b}: BF16 cache image differs"
            refs[b] = (oracle.attention_bf16kv(qb[b], kbits, vbits), None)
    for S in (1, 3, 64):
        bufs = uq.StepBuffers(cfg, wl.batch, S, DEV)
        bufs.partial_acc.fill_(float("nan")); bufs.partial_ml.fill_(float("nan"))
        out = uq.baseline_decode_step(cfg, fmt, bufs, q, empty, empty, cu0, lens, lens, bt, cache)
        torch.cuda.synchronize()
        out = out.float().cpu().numpy().astype(np.float64)
        assert np.all(out[0] == 0)                                              # the empty sequence
        for b, (ref, q8) in refs.items():
            if q8 is not None:
                assert np.array_equal(bufs.q_fp8[b].cpu().numpy(), q8), f"seq {b}: FP8 query bytes differ"
            H.check_out(out[b], ref, f"{kv} kv seq {b} S={S}")


def test_ultra_tq_cache_and_decode_against_the_oracle_of_algorithm_2():
    """Ultra-TQ comparison path (Alg. 2, last item): uq_tq_append's cache image —
    codebook indices, bf16 block norms, uniform V codes, bf16 (scale, zero) — and the rotated bf16 query bit for bit against
    oracle/ultra_tq.py, read back through the independent unpacker of tests/uq_layout.py; uq_tq_decode_attention + merge
    within 2e-3 + 1e-2 |ref| of its float64 attention, for a ragged batch (empty, one token, page and tile boundaries,
    multi-tile), GQA 16 and 6, slot counts 1, 3 and 64, tokens appended one sequence at a time AND several per call."""
    from oracle import ultra_tq as T
    from . import uq_layout as UL
    cb = np.asarray(W.TQ_CODEBOOK, np.float32)
    for hq, hkv in ((16, 1), (12, 2)):
        wl = W.make_custom("tq", 71, [0, 1, 17, 203, 1000, 16, 31, 129], hq, hkv, outlier_channels=3, outlier_gain=8.0,
                           peaked_frac=0.3)
        cfg = H.cfg_of(wl)
        assert uq.baseline_record_bytes(cfg, uq.KV_ULTRA_TQ) == UL.TQ_RECORD
        cache = uq.alloc_baseline_cache(cfg, uq.KV_ULTRA_TQ, wl.num_pages, DEV)
        bt = torch.from_numpy(wl.block_tables).to(DEV)
        B = wl.batch
        # first half of every sequence in one call for all sequences, the rest sequence by sequence
        half = (wl.ctx_lens // 2).astype(np.int32)
        ks, vs = [], []
        for b in range(B):
            k, v = W.seq_kv(wl, b, int(wl.ctx_lens[b]), DEV) if wl.ctx_lens[b] else (None, None)
            ks.append(k); vs.append(v)
        cu = np.concatenate([[0], np.cumsum(half)]).astype(np.int32)
        if cu[-1]:
            k1 = torch.cat([ks[b][:half[b]] for b in range(B) if half[b]]); v1 = torch.cat([vs[b][:half[b]] for b in range(B) if half[b]])
            uq.tq_append(cfg, cb, k1.contiguous(), v1.contiguous(), torch.from_numpy(cu).to(DEV),
                         torch.zeros(B, dtype=torch.int32, device=DEV), bt, cache)
        for b in range(B):
            n = int(wl.ctx_lens[b] - half[b])
            if n == 0:
                continue
            before = np.zeros(B, np.int32); before[b] = half[b]
            cu = np.zeros(B + 1, np.int32); cu[b + 1:] = n
            uq.tq_append(cfg, cb, ks[b][half[b]:].contiguous(), vs[b][half[b]:].contiguous(), torch.from_numpy(cu).to(DEV),
                         torch.from_numpy(before).to(DEV), bt, cache)
        q = W.gen_q(wl, DEV)
        q_rot = torch.empty_like(q)
        lens = torch.from_numpy(wl.ctx_lens.astype(np.int32)).to(DEV)
        empty = torch.zeros((0, hkv, 128), dtype=torch.bfloat16, device=DEV)
        uq.tq_append(cfg, cb, empty, empty, torch.zeros(B + 1, dtype=torch.int32, device=DEV), lens, bt, cache, q=q, q_rot=q_rot)
        torch.cuda.synchronize()
        host = cache.cpu().numpy()
        qb = H.bits(q)
        assert np.array_equal(H.bits(q_rot).reshape(-1, 128), T.bf16_bits(T.encode_q(qb.reshape(-1, 128)))), "rotated bf16 query differs"
        refs = {}
        for b in range(B):
            L = int(wl.ctx_lens[b])
            if L == 0:
                continue
            kbits, vbits = H.bits(ks[b]).reshape(L * hkv, 128), H.bits(vs[b]).reshape(L * hkv, 128)
            ki, kn = T.encode_k(kbits, cb)
            vc, vsc, vz = T.encode_v(vbits)
            gi, gn, gc, gs, gz = UL.gather_tq_sequence(host, wl.block_tables[b], L)
            sh = lambda a: a.reshape(L, hkv, -1)
            assert np.array_equal(gi, sh(ki)), f"seq {b}: codebook indices differ"
            assert np.array_equal(gn, sh(T.bf16_bits(kn))), f"seq {b}: block norms differ"
            assert np.array_equal(gc, sh(vc)), f"seq {b}: V codes differ"
            assert np.array_equal(gs, sh(T.bf16_bits(vsc))) and np.array_equal(gz, sh(T.bf16_bits(vz))), f"seq {b}: V scale / zero differ"
            refs[b] = T.attention(qb[b], sh(ki), sh(kn), sh(vc), sh(vsc), sh(vz), cb, hkv)
        for S in (1, 3, 64):
            bufs = uq.StepBuffers(cfg, B, S, DEV)
            bufs.partial_acc.fill_(float("nan")); bufs.partial_ml.fill_(float("nan"))
            uq.tq_decode_attention(cfg, cb, q_rot, cache, bt, lens, S, bufs.partial_acc, bufs.partial_ml)
            uq.merge_splits(cfg, bufs.partial_acc, bufs.partial_ml, bufs.out)
            torch.cuda.synchronize()
            out = bufs.out.float().cpu().numpy().astype(np.float64)
            assert np.all(out[0] == 0)                                          # the empty sequence
            for b, ref in refs.items():
                H.check_out(out[b], ref, f"ultra-tq seq {b} S={S} heads {hq}/{hkv}")


def test_ultra_tq_scaled_config3_sampled_sequences():
    """Ultra-TQ on config 3's shape at 0.2 x (13 ragged sequences of 4,180-13,037 tokens, 48/8 heads = GQA 6: several
    units per CTA, slots from uq_suggest_num_splits): three sequences — the longest, the shortest, one in between — cache
    image bit for bit and outputs within 2e-3 + 1e-2 |ref| of the oracle of Algorithm 2; the rest must be finite."""
    from oracle import ultra_tq as T
    from . import uq_layout as UL
    cb = np.asarray(W.TQ_CODEBOOK, np.float32)
    wl = W.make_config(3, scale=0.2)
    cfg = H.cfg_of(wl)
    B, hkv = wl.batch, wl.num_kv_heads
    cache = uq.alloc_baseline_cache(cfg, uq.KV_ULTRA_TQ, wl.num_pages, DEV)
    cache.fill_(0xFF)                                                        # stale bytes: NaN patterns in norms / scales
    bt = torch.from_numpy(wl.block_tables).to(DEV)
    for b in range(B):
        L = int(wl.ctx_lens[b])
        k, v = W.seq_kv(wl, b, L, DEV)
        before = np.zeros(B, np.int32)
        cu = np.zeros(B + 1, np.int32); cu[b + 1:] = L
        uq.tq_append(cfg, cb, k.contiguous(), v.contiguous(), torch.from_numpy(cu).to(DEV), torch.from_numpy(before).to(DEV), bt, cache)
    q = W.gen_q(wl, DEV)
    q_rot = torch.empty_like(q)
    lens = torch.from_numpy(wl.ctx_lens.astype(np.int32)).to(DEV)
    empty = torch.zeros((0, hkv, 128), dtype=torch.bfloat16, device=DEV)
    uq.tq_append(cfg, cb, empty, empty, torch.zeros(B + 1, dtype=torch.int32, device=DEV), lens, bt, cache, q=q, q_rot=q_rot)
    S = uq.suggest_num_splits(cfg, B, int(wl.ctx_lens.mean()))
    bufs = uq.StepBuffers(cfg, B, S, DEV)
    bufs.partial_acc.fill_(float("nan")); bufs.partial_ml.fill_(float("nan"))
    uq.tq_decode_attention(cfg, cb, q_rot, cache, bt, lens, S, bufs.partial_acc, bufs.partial_ml)
    uq.merge_splits(cfg, bufs.partial_acc, bufs.partial_ml, bufs.out)
    torch.cuda.synchronize()
    out = bufs.out.float().cpu().numpy().astype(np.float64)
    assert np.isfinite(out).all()
    host = cache.cpu().numpy()
    qb = H.bits(q)
    order = np.argsort(wl.ctx_lens)
    for b in (int(order[-1]), int(order[0]), int(order[len(order) // 2])):
        L = int(wl.ctx_lens[b])
        k, v = W.seq_kv(wl, b, L, DEV)
        ki, kn = T.encode_k(H.bits(k).reshape(L * hkv, 128), cb)
        vc, vsc, vz = T.encode_v(H.bits(v).reshape(L * hkv, 128))
        gi, gn, gc, gs, gz = UL.gather_tq_sequence(host, wl.block_tables[b], L)
        sh = lambda a: a.reshape(L, hkv, -1)
        assert np.array_equal(gi, sh(ki)) and np.array_equal(gn, sh(T.bf16_bits(kn))), f"seq {b}: K image differs"
        assert np.array_equal(gc, sh(vc)) and np.array_equal(gs, sh(T.bf16_bits(vsc))) and np.array_equal(gz, sh(T.bf16_bits(vz))), \
            f"seq {b}: V image differs"
        ref = T.attention(qb[b], sh(ki), sh(kn), sh(vc), sh(vsc), sh(vz), cb, hkv)
        H.check_out(out[b], ref, f"ultra-tq config 3 x 0.2, seq {b} ({L} tokens), S={S}")


def test_distortion_study_has_the_shape_of_fig_2b():
    """paper_2606_20474_b200.distortion (the shape of Fig. 2b) on 4,096
    vectors per head size: raw-absmax FP4 is an order of magnitude off; the constant closes most of the gap to the
    Lloyd-Max codebook; 0.156 beats the MX rule with the continuous scale and 0.195 beats 0.156 with the power-of-two
    scale (the paper's "power-of-two-optimal value"); the figures do not depend on d."""
    from paper_2606_20474_b200 import distortion
    rows = distortion.study(n_vectors=4096, seed=3, device=DEV)
    assert set(rows) == {64, 128, 256}
    for d, r in rows.items():
        assert 0.0085 < r["lloyd-max"] < 0.0100, (d, r)
        assert r["fp4 c=1.0"] > 8 * r["fp4 0.156"], (d, r)
        assert r["lloyd-max"] < r["fp4 0.156"] < r["fp4 mx"], (d, r)
        assert r["fp4 0.195p"] < r["fp4 0.156p"], (d, r)
        assert r["fp4 0.156"] < r["fp4 0.195p"], (d, r)
        assert abs(r["fp4 0.156"] - rows[128]["fp4 0.156"]) < 0.1 * rows[128]["fp4 0.156"], (d, r)


@pytest.mark.parametrize("d", [256, 64])
def test_full_size_cfg3_shape_at_other_head_dims_sampled_sequences(d):
    """The shapes `bench.py --config 3 --head-dim 256 | 64` time (config 3: 64 ragged sequences of 16k-64k tokens, 48/8
    heads), at FULL size and with the slot count bench.py uses: the longest, the shortest and a middle sequence — cache
    image bit for bit, FP8 query bytes, every output row of every head within 2e-3 + 1e-2 |ref| (full-size
    parity in the launch configuration that is timed; head sizes of PAPER.md:322)."""
    wl = W.make_config(3, head_dim=d)
    cfg = H.cfg_of(wl)
    S = uq.suggest_num_splits(cfg, wl.batch, int(wl.ctx_lens.mean()))
    order = np.argsort(wl.ctx_lens, kind="stable")
    _, n = _full_check(wl, [S], sample_seqs=[int(order[-1]), int(order[0]), int(order[len(order) // 2])], check_cache=True)
    assert n == 3


@pytest.mark.parametrize("kv", ["fp8", "bf16", "tq"])
def test_full_size_cfg2_comparison_caches_sampled_sequences(kv):
    """The comparison kernels on the shape `bench.py --config 2 --kv fp8 | bf16 | tq` times (32 x 32,768 tokens, 64/4 heads)
    at FULL size with bench.py's slot count: sequences 0, 13 and 31, all 64 heads, within 2e-3 + 1e-2 |ref| of the float64
    attention over that cache's own contents (oracle.attention_fp8kv / attention_bf16kv / ultra_tq.attention)."""
    from oracle import ultra_tq as T
    wl = W.make_config(2)
    cfg = H.cfg_of(wl)
    B, hkv = wl.batch, wl.num_kv_heads
    S = uq.suggest_num_splits(cfg, B, int(wl.ctx_lens.mean()))
    bt = torch.from_numpy(wl.block_tables).to(DEV)
    lens = torch.from_numpy(wl.ctx_lens.astype(np.int32)).to(DEV)
    empty = torch.zeros((0, hkv, 128), dtype=torch.bfloat16, device=DEV)
    cu0 = torch.zeros(B + 1, dtype=torch.int32, device=DEV)
    q = W.gen_q(wl, DEV)
    qb = H.bits(q)
    bufs = uq.StepBuffers(cfg, B, S, DEV)
    cb = np.asarray(W.TQ_CODEBOOK, np.float32)
    if kv == "tq":
        cache = uq.alloc_baseline_cache(cfg, uq.KV_ULTRA_TQ, wl.num_pages, DEV)
        for b in range(B):
            L = int(wl.ctx_lens[b])
            k, v = W.seq_kv(wl, b, L, DEV)
            cu = np.zeros(B + 1, np.int32); cu[b + 1:] = L
            uq.tq_append(cfg, cb, k.contiguous(), v.contiguous(), torch.from_numpy(cu).to(DEV),
                         torch.zeros(B, dtype=torch.int32, device=DEV), bt, cache)
        q_rot = torch.empty_like(q)
        uq.tq_append(cfg, cb, empty, empty, cu0, lens, bt, cache, q=q, q_rot=q_rot)
        uq.tq_decode_attention(cfg, cb, q_rot, cache, bt, lens, S, bufs.partial_acc, bufs.partial_ml)
        uq.merge_splits(cfg, bufs.partial_acc, bufs.partial_ml, bufs.out)
        out = bufs.out
    else:
        fmt = uq.KV_FP8_E4M3 if kv == "fp8" else uq.KV_BF16
        cache, _ = _fill_baseline_cache(cfg, fmt, wl)
        out = uq.baseline_decode_step(cfg, fmt, bufs, q, empty, empty, cu0, lens, lens, bt, cache)
    torch.cuda.synchronize()
    out = out.float().cpu().numpy().astype(np.float64)
    assert np.isfinite(out).all()
    for b in (0, 13, 31):
        L = int(wl.ctx_lens[b])
        k, v = W.seq_kv(wl, b, L, DEV)
        kbits, vbits = H.bits(k), H.bits(v)
        if kv == "fp8":
            ref = oracle.attention_fp8kv(qb[b], kbits, vbits)[0]
        elif kv == "bf16":
            ref = oracle.attention_bf16kv(qb[b], kbits, vbits)
        else:
            ki, kn = T.encode_k(kbits.reshape(L * hkv, 128), cb)
            vc, vsc, vz = T.encode_v(vbits.reshape(L * hkv, 128))
            sh = lambda a: a.reshape(L, hkv, -1)
            ref = T.attention(qb[b], sh(ki), sh(kn), sh(vc), sh(vsc), sh(vz), cb, hkv)
        H.check_out(out[b], ref, f"{kv} kv, config 2 full size, seq {b}, S={S}")
