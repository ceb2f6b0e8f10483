"""The seeded workload generators reproduce the shapes SURVEY.md §8 computed for BASELINE.json's
configs, and are position-addressed (any caller regenerates the same bytes)."""
import numpy as np
import torch

from paper_2606_20474_b200 import workloads as W


def test_config_shapes_match_baseline():
    w2 = W.make_config(2)
    assert (w2.batch, w2.num_q_heads, w2.num_kv_heads) == (32, 64, 4)
    assert w2.total_tokens == 1_048_576 and w2.num_pages == 65_536
    assert w2.kv_bytes_per_step() == 570_425_344            # 570.4 MB
    assert sorted(w2.block_tables.ravel().tolist()) == list(range(65_536))   # a permutation
    assert int((w2.k_chan_scale[0] == 8).sum()) == 3
    w3 = W.make_config(3)
    assert (w3.batch, w3.num_q_heads, w3.num_kv_heads) == (64, 48, 8)
    assert w3.ctx_lens.min() >= 16384 and w3.ctx_lens.max() <= 65536
    w5 = W.make_config(5)
    assert w5.total_tokens == 8 * 262_144 and w5.kv_bytes_per_step() == 1_140_850_688
    w1 = W.make_config(1)
    assert np.array_equal(w1.block_tables[0], np.arange(64)) and int((w1.k_chan_scale == 10).sum()) == 4


def test_cfg4_prefix_pages_are_shared():
    w4 = W.make_config(4)
    assert w4.batch == 256 and w4.prefix_len == 30_000 and w4.new_tokens == 1
    n_prefix = 30_000 // 16
    assert np.all(w4.block_tables[:, :n_prefix] == np.arange(n_prefix))
    assert (w4.ctx_lens - 30_000).max() <= 98_000
    med = np.median(w4.ctx_lens - 30_000)
    assert 7_000 < med < 14_000
    # private pages are disjoint between sequences
    priv = []
    for b in range(w4.batch):
        n = -(-(int(w4.ctx_lens[b]) + 64 - 30_000) // 16)
        priv.append(w4.block_tables[b, n_prefix:n_prefix + n])
    allp = np.concatenate(priv)
    assert len(np.unique(allp)) == len(allp) and allp.min() >= n_prefix


def test_generators_are_position_addressed():
    wl = W.make_config(2, scale=1 / 64)
    k1, v1 = W.gen_kv(wl, 3, 100, 5000)
    k2, v2 = W.gen_kv(wl, 3, 4000, 4500)
    assert torch.equal(k1[3900:4400], k2) and torch.equal(v1[3900:4400], v2)
    ka, _ = W.seq_kv(wl, 1, 50)
    kb, _ = W.seq_kv(wl, 1, 80)
    assert torch.equal(ka, kb[:50])
    q = W.gen_q(W.make_config(1, peaked_frac=0.5))
    assert q.shape == (1, 8, 128) and q.dtype == torch.bfloat16
