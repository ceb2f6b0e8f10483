"""CPU-side checks of the boundary: libuq.so builds for sm_100a, loads without a GPU, exports
every symbol include/uq.h declares, and validates arguments on the host (no compute calls)."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_2606_20474_b200 as uq
from paper_2606_20474_b200 import binding, build
from tests import uq_layout

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding._load()


def test_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "uq.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(uq_[a-z_0-9]+)\s*\(", hdr))
    assert {"uq_rotate_quantize_append", "uq_decode_attention", "uq_merge_splits"} <= declared
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in uq.h but not exported"


def test_record_bytes_is_4_25_bits_per_element(lib):
    cfg = uq.UQConfig(64, 4)
    assert uq.cache_record_bytes(cfg) == uq.RECORD_BYTES == 2176
    assert 2176 * 8 / (16 * 128 * 2) == 4.25
    count = uq_layout.used_byte_mask()
    assert np.all(count[:1024] == 1) and np.all(count[1024:2048] == 2) and np.all(count[2048:] == 1)
    for d in (64, 256):                                    # the other supported head sizes: 17 d bytes, no padding
        assert uq.cache_record_bytes(uq.UQConfig(64, 4, head_dim=d)) == uq.record_bytes(d) == 17 * d
        assert 17 * d * 8 / (16 * d * 2) == 4.25
        count = uq_layout.used_byte_mask(d)
        assert np.all(count[:8 * d] == 1) and np.all(count[8 * d:16 * d] == 2) and np.all(count[16 * d:] == 1)


def test_host_side_validation(lib):
    c = uq.UQConfig(64, 4).c()
    f = lib.uq_merge_splits
    assert f(None, None, None, 1, 1, None, None) == 1      # UQ_ERR_INVALID_ARG: NULL config
    assert b"NULL" in lib.uq_last_error_string()
    bad = uq.UQConfig(64, 5).c()
    assert f(ctypes.byref(bad), None, None, 1, 1, None, None) == 1
    bad = uq.UQConfig(64, 4, head_dim=96).c()
    assert f(ctypes.byref(bad), None, None, 1, 1, None, None) == 2   # UQ_ERR_UNSUPPORTED
    bad = uq.UQConfig(64, 2).c()                           # GQA group 32
    assert f(ctypes.byref(bad), None, None, 1, 1, None, None) == 2
    assert f(ctypes.byref(c), None, None, 1, 1, None, None) == 1     # NULL buffers
    assert lib.uq_decode_attention(ctypes.byref(c), None, None, 1, None, 1, None, 1, 1, None, None, None) == 1
    assert lib.uq_rotate_quantize_append(ctypes.byref(c), None, None, None, None, None, 1, 1, 4, None, 1,
                                         None, None, None) == 1
    assert uq.cache_record_bytes(uq.UQConfig(64, 4, page_size=32)) == 0


def test_prefix_decode_and_calibrate_validate_on_the_host(lib):
    c = uq.UQConfig(64, 4).c()
    fake = ctypes.c_void_p(0x1000)                          # aligned, never dereferenced: validation comes first
    f = lib.uq_decode_prefix_attention
    assert f(ctypes.byref(c), None, None, 1, None, 1, 1, 128, 2, None, None, None) == 1
    assert f(ctypes.byref(c), fake, fake, 64, fake, 64, 4, 100, 2, fake, fake, None) == 1    # prefix_len % 128
    assert b"128" in lib.uq_last_error_string()
    assert f(ctypes.byref(c), fake, fake, 64, fake, 4, 4, 128, 2, fake, fake, None) == 1     # prefix beyond max_pages
    assert f(ctypes.byref(c), fake, fake, 64, fake, 64, 4, 128, 1, fake, fake, None) == 1    # num_splits < 2
    g = lib.uq_calibrate_c
    assert g(ctypes.byref(c), fake, 8, 1, fake, 4, 3, None, fake, fake, None) == 1           # scale_mode out of range
    assert g(ctypes.byref(c), fake, 8, 1, fake, 4, 1, fake, fake, fake, None) == 1           # power-of-two scale + levels
    assert lib.uq_merge_splits2(ctypes.byref(c), None, None, 2, None, None, 2, 1, None, None) == 1
    assert uq.suggest_num_splits_max(uq.UQConfig(64, 4), 256, 16500, 98000) > uq.suggest_num_splits(uq.UQConfig(64, 4), 256, 16500)
    for d in (64, 256):                                     # the shared-prefix decode and the calibration exist for head_dim 128
        cd = uq.UQConfig(64, 4, head_dim=d).c()
        assert f(ctypes.byref(cd), fake, fake, 64, fake, 64, 4, 128, 2, fake, fake, None) == 2
        assert g(ctypes.byref(cd), fake, 8, 1, fake, 4, 1, None, fake, fake, None) == 2


def test_workspace_query_and_debug_flag_on_the_host(lib):
    """uq_decode_workspace_bytes: 0 bytes for any supported geometry, argument errors reported; the
    debug flag is a known bit of uq_config.flags, other bits are refused."""
    assert uq.decode_workspace_bytes(uq.UQConfig(64, 4), 32, 6) == 0
    assert uq.decode_workspace_bytes(uq.UQConfig(48, 8), 2048, 64) == 0
    c = uq.UQConfig(64, 4).c()
    n = ctypes.c_size_t(7)
    assert lib.uq_decode_workspace_bytes(ctypes.byref(c), 0, 1, ctypes.byref(n)) == 1
    assert lib.uq_decode_workspace_bytes(ctypes.byref(c), 1, 1, None) == 1
    bad = uq.UQConfig(64, 4, page_size=32).c()
    assert lib.uq_decode_workspace_bytes(ctypes.byref(bad), 1, 1, ctypes.byref(n)) == 2
    ok = uq.UQConfig(64, 4, flags=uq.FLAG_DEBUG_CHECKS | uq.FLAG_NO_BULK_APPEND)
    assert uq.cache_record_bytes(ok) == 2176
    assert uq.cache_record_bytes(uq.UQConfig(64, 4, flags=uq.FLAG_SMALL_APPEND_AHEAD)) == 2176
    assert uq.cache_record_bytes(uq.UQConfig(64, 4, flags=8)) == 0
    assert b"flags" in lib.uq_last_error_string()


def test_binding_refuses_cpu_tensors(lib):
    import torch
    cfg = uq.UQConfig(8, 1)
    out = torch.zeros((1, 8, 128), dtype=torch.bfloat16)
    with pytest.raises(uq.UQError):
        uq.merge_splits(cfg, torch.zeros((1, 8, 1, 128)), torch.zeros((1, 8, 1, 2)), out)


def test_argument_checks_of_the_round_2_entry_points_need_no_gpu(lib):
    """Host-side validation of uq_decode_attention_static, uq_tq_append and uq_tq_decode_attention returns before any
    CUDA call: sizes beyond the static scratch, a missing / unsorted codebook, the wrong entry point for a format."""
    cfg = uq.UQConfig(64, 4).c()
    n = ctypes.c_size_t(0)
    assert lib.uq_decode_static_scratch_needed(ctypes.byref(cfg), 32, 6, ctypes.byref(n)) == 0
    assert n.value == 32 * 64 * 6 * 128 * 4 + 32 * 64 * 6 * 8
    assert lib.uq_static_scratch_bytes() == 32 << 20
    one = ctypes.c_void_p(256)                          # never dereferenced: the size check comes first
    assert lib.uq_decode_attention_static(ctypes.byref(cfg), one, one, 10, one, 4, one, 256, 8, one, None) == 2
    assert b"static scratch" in lib.uq_last_error_string()
    assert lib.uq_decode_static_scratch_needed(ctypes.byref(cfg), 0, 6, ctypes.byref(n)) == 1
    assert lib.uq_baseline_record_bytes(ctypes.byref(cfg), 3) == 2432
    good = (ctypes.c_float * 16)(*[float(i) - 7.5 for i in range(16)])
    bad = (ctypes.c_float * 16)(*([0.0] * 16))
    cb = lambda a: ctypes.cast(a, ctypes.c_void_p)
    assert lib.uq_tq_append(ctypes.byref(cfg), None, one, one, one, one, one, 4, 1, 1, one, 10, None, None, None) == 1
    assert lib.uq_tq_append(ctypes.byref(cfg), cb(bad), one, one, one, one, one, 4, 1, 1, one, 10, None, None, None) == 1
    assert b"ascending" in lib.uq_last_error_string()
    assert lib.uq_tq_append(ctypes.byref(cfg), cb(good), one, one, one, one, one, 4, 1, 1, one, 10, one, None, None) == 1
    assert lib.uq_tq_decode_attention(ctypes.byref(cfg), cb(bad), one, one, 10, one, 4, one, 1, 1, one, one, None) == 1
    assert lib.uq_baseline_append(ctypes.byref(cfg), 3, one, one, one, one, one, 4, 1, 1, one, 10, None, None, None) == 1
    assert b"uq_tq_append" in lib.uq_last_error_string()
    d64 = uq.UQConfig(64, 4, head_dim=64).c()
    assert lib.uq_tq_append(ctypes.byref(d64), cb(good), one, one, one, one, one, 4, 1, 1, one, 10, None, None, None) == 2


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_20474_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in src and "from oracle" not in src and "uq_oracle" not in src, fn


def test_host_stage_layout_one_block():
    """HostStage: the seven step inputs are disjoint, 256-byte aligned views of one host block and of
    one device block with the same layout (here the 'device' block is a CPU tensor: layout only)."""
    import torch
    cfg = uq.UQConfig(8, 2)
    st = uq.HostStage(cfg, batch=3, total_new=5, max_pages=7, device="cpu")
    assert tuple(st.h["q"].shape) == (3, 8, 128) and st.h["q"].dtype == torch.bfloat16
    assert tuple(st.h["k_new"].shape) == (5, 2, 128) and tuple(st.h["block_tables"].shape) == (3, 7)
    base_h, base_d = st.host.data_ptr(), st.dev.data_ptr()
    spans = []
    for name in uq.HostStage.FIELDS:
        h, d = st.h[name], st.d[name]
        off = h.data_ptr() - base_h
        assert off == d.data_ptr() - base_d and off % 256 == 0
        assert h.shape == d.shape and h.dtype == d.dtype
        spans.append((off, off + h.numel() * h.element_size()))
    spans.sort()
    assert all(a1 <= b0 for (_, a1), (b0, _) in zip(spans, spans[1:])) and spans[-1][1] <= st.nbytes
    for i, name in enumerate(uq.HostStage.FIELDS):
        st.h[name].view(torch.uint8).fill_(i + 1)
    st.upload()
    for i, name in enumerate(uq.HostStage.FIELDS):
        assert bool((st.d[name].view(torch.uint8) == i + 1).all())
