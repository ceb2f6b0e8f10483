"""uq_decode_attention_static (include/uq.h "Decode without allocation"): decode + merge with the split partials in the
library's static device array.  Collected LAST on purpose (the suite runs with pytest -x): a failure here hides nothing.
The entry point runs the same kernels as uq_decode_attention + uq_merge_splits, so its output is compared with that
path's bit for bit AND, like every other parity test, with the float64 oracle within the north-star bound — on two
calls in a row of different shapes, so that the second call runs over what the first left in the array."""
import numpy as np
import pytest
import torch

import paper_2606_20474_b200 as uq
from paper_2606_20474_b200 import workloads as W

from . import harness as H

pytestmark = pytest.mark.gpu


def _static_vs_existing(wl, num_splits, sample):
    cfg = H.cfg_of(wl)
    cache, bt = H.fill_cache(cfg, wl, "cuda")
    q = W.gen_q(wl, "cuda")
    out_ref, q_fp8, _ = H.run_decode(cfg, cache, bt, wl.ctx_lens, q, num_splits)      # existing path, caller buffers
    sl = torch.from_numpy(wl.ctx_lens.astype(np.int32)).cuda()
    out = torch.full((wl.batch, wl.num_q_heads, wl.head_dim), float("nan"), dtype=torch.bfloat16, device="cuda")
    before = torch.cuda.memory_allocated()
    uq.decode_attention_static(cfg, q_fp8, cache, bt, sl, num_splits, out)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before
    a, b = out.float().cpu().numpy().astype(np.float64), out_ref.float().cpu().numpy().astype(np.float64)
    live = wl.ctx_lens > 0
    assert np.array_equal(a[live], b[live]), "static-scratch path differs from uq_decode_attention + uq_merge_splits"
    assert np.all(a[~live] == 0.0)
    for s in sample:                                                                     # and against the oracle
        L = int(wl.ctx_lens[s])
        ref, _ = H.oracle_out(wl, s, L, H.bits(q)[s])
        H.check_out(a[s], ref, f"{wl.name} seq {s} (static scratch)")


def test_static_scratch_two_calls_in_a_row():
    assert uq.static_scratch_bytes() == 32 << 20
    # call 1: ragged lengths over several tiles, an empty sequence, 5 slots
    wl1 = W.make_custom("noalloc_a", 4101, [1500, 0, 129, 2048, 777, 16], 16, 2, peaked_frac=0.25)
    _static_vs_existing(wl1, 5, [0, 2, 4])
    # call 2: another shape and slot count over the array as call 1 left it
    wl2 = W.make_custom("noalloc_b", 4102, [300, 4096, 1], 32, 4, peaked_frac=0.25)
    _static_vs_existing(wl2, 3, [0, 2])
    # and the first shape again (slots that call 2 overwrote with other rows)
    _static_vs_existing(wl1, 2, [3])


def test_static_scratch_limit_is_an_error():
    wl = W.make_custom("noalloc_big", 4103, [64] * 256, 64, 4)
    cfg = H.cfg_of(wl)
    need = uq.decode_static_scratch_needed(cfg, wl.batch, 8)
    assert need == 256 * 64 * 8 * 128 * 4 + 256 * 64 * 8 * 8 and need > uq.static_scratch_bytes()
    cache, bt = H.fill_cache(cfg, wl, "cuda")
    sl = torch.from_numpy(wl.ctx_lens.astype(np.int32)).cuda()
    q8 = torch.zeros((wl.batch, wl.num_q_heads, wl.head_dim), dtype=torch.uint8, device="cuda")
    out = torch.zeros((wl.batch, wl.num_q_heads, wl.head_dim), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(uq.UQError, match="static scratch"):
        uq.decode_attention_static(cfg, q8, cache, bt, sl, 8, out)
    uq.decode_attention_static(cfg, q8, cache, bt, sl, 3, out)                          # 3 slots fit (24.2 MiB)
    torch.cuda.synchronize()
