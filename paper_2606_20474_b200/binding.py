"""ctypes binding of libuq.so.  Same names and argument order as include/uq.h; torch tensors
are passed as raw device pointers, the current torch CUDA stream as the stream argument."""
from __future__ import annotations

import ctypes
import dataclasses
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libuq.so")
_lib = None

RECORD_BYTES = 2176          # head_dim 128; in general 17 * head_dim (record_bytes())


def record_bytes(head_dim: int = 128) -> int:
    """Bytes of one (page, kv head) record: 16 tokens x (d/2 + d/32) x 2 = 17 d (include/uq.h)."""
    return 17 * int(head_dim)


class UQError(RuntimeError):
    pass


class _CConfig(ctypes.Structure):
    _fields_ = [("num_q_heads", ctypes.c_int32), ("num_kv_heads", ctypes.c_int32),
                ("head_dim", ctypes.c_int32), ("page_size", ctypes.c_int32),
                ("group_size", ctypes.c_int32), ("c_k", ctypes.c_float), ("c_v", ctypes.c_float),
                ("sm_scale", ctypes.c_float), ("flags", ctypes.c_uint32)]


@dataclasses.dataclass
class UQConfig:
    num_q_heads: int
    num_kv_heads: int
    head_dim: int = 128
    page_size: int = 16
    group_size: int = 32
    c_k: float = 0.156
    c_v: float = 0.156
    sm_scale: float = 0.0       # 0 => 1/sqrt(head_dim)
    flags: int = 0

    def c(self) -> _CConfig:
        return _CConfig(self.num_q_heads, self.num_kv_heads, self.head_dim, self.page_size,
                        self.group_size, self.c_k, self.c_v, self.sm_scale, self.flags)


def library_path() -> str:
    return _LIB_PATH


def _load():
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise UQError(f"{_LIB_PATH} is missing: build it with `python -m paper_2606_20474_b200.build` "
                      "(there is no CPU fallback)")
    lib = ctypes.CDLL(_LIB_PATH)
    vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
    cfgp = ctypes.POINTER(_CConfig)
    lib.uq_last_error_string.restype = ctypes.c_char_p
    lib.uq_last_error_string.argtypes = []
    lib.uq_cache_record_bytes.restype = ctypes.c_size_t
    lib.uq_cache_record_bytes.argtypes = [cfgp]
    lib.uq_rotate_quantize_append.restype = i32
    lib.uq_rotate_quantize_append.argtypes = [cfgp, vp, vp, vp, vp, vp, i32, i32, i32, vp, i64, vp, vp, vp]
    lib.uq_decode_attention.restype = i32
    lib.uq_decode_attention.argtypes = [cfgp, vp, vp, i64, vp, i32, vp, i32, i32, vp, vp, vp]
    lib.uq_merge_splits.restype = i32
    lib.uq_merge_splits.argtypes = [cfgp, vp, vp, i32, i32, vp, vp]
    lib.uq_decode_prefix_attention.restype = i32
    lib.uq_decode_prefix_attention.argtypes = [cfgp, vp, vp, i64, vp, i32, i32, i32, i32, vp, vp, vp]
    lib.uq_merge_splits2.restype = i32
    lib.uq_merge_splits2.argtypes = [cfgp, vp, vp, i32, vp, vp, i32, i32, vp, vp]
    lib.uq_calibrate_c.restype = i32
    lib.uq_calibrate_c.argtypes = [cfgp, vp, i64, i32, vp, i32, i32, vp, vp, vp, vp]
    lib.uq_decode_workspace_bytes.restype = i32
    lib.uq_decode_workspace_bytes.argtypes = [cfgp, i32, i32, ctypes.POINTER(ctypes.c_size_t)]
    lib.uq_baseline_record_bytes.restype = ctypes.c_size_t
    lib.uq_baseline_record_bytes.argtypes = [cfgp, i32]
    lib.uq_baseline_append.restype = i32
    lib.uq_baseline_append.argtypes = [cfgp, i32, vp, vp, vp, vp, vp, i32, i32, i32, vp, i64, vp, vp, vp]
    lib.uq_baseline_decode_attention.restype = i32
    lib.uq_baseline_decode_attention.argtypes = [cfgp, i32, vp, vp, i64, vp, i32, vp, i32, i32, vp, vp, vp]
    lib.uq_tq_append.restype = i32
    lib.uq_tq_append.argtypes = [cfgp, vp, vp, vp, vp, vp, vp, i32, i32, i32, vp, i64, vp, vp, vp]
    lib.uq_tq_decode_attention.restype = i32
    lib.uq_tq_decode_attention.argtypes = [cfgp, vp, vp, vp, i64, vp, i32, vp, i32, i32, vp, vp, vp]
    lib.uq_static_scratch_bytes.restype = ctypes.c_size_t
    lib.uq_static_scratch_bytes.argtypes = []
    lib.uq_decode_static_scratch_needed.restype = i32
    lib.uq_decode_static_scratch_needed.argtypes = [cfgp, i32, i32, ctypes.POINTER(ctypes.c_size_t)]
    lib.uq_decode_attention_static.restype = i32
    lib.uq_decode_attention_static.argtypes = [cfgp, vp, vp, i64, vp, i32, vp, i32, i32, vp, vp]
    lib.uq_suggest_num_splits.restype = i32
    lib.uq_suggest_num_splits.argtypes = [cfgp, i32, i32]
    lib.uq_suggest_prefix_splits.restype = i32
    lib.uq_suggest_prefix_splits.argtypes = [cfgp, i32, i32]
    lib.uq_suggest_num_splits_max.restype = i32
    lib.uq_suggest_num_splits_max.argtypes = [cfgp, i32, i32, i32]
    _lib = lib
    return lib


def last_error() -> str:
    return _load().uq_last_error_string().decode()


def _check(status: int, what: str) -> None:
    if status != 0:
        raise UQError(f"{what} failed with status {status}: {last_error()}")


def _p(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _stream(stream) -> ctypes.c_void_p:
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def _dev(t: torch.Tensor, dtype, name: str) -> torch.Tensor:
    if not t.is_cuda:
        raise UQError(f"{name} must be a CUDA tensor (no CPU path exists)")
    if t.dtype != dtype or not t.is_contiguous():
        raise UQError(f"{name} must be contiguous {dtype}, got {t.dtype} contiguous={t.is_contiguous()}")
    return t


def cache_record_bytes(cfg: UQConfig) -> int:
    c = cfg.c()
    return int(_load().uq_cache_record_bytes(ctypes.byref(c)))


FLAG_NO_BULK_APPEND = 1
FLAG_DEBUG_CHECKS = 2
FLAG_SMALL_APPEND_AHEAD = 4


def decode_workspace_bytes(cfg: UQConfig, batch: int, num_splits: int) -> int:
    """uq_decode_workspace_bytes: device scratch the decode calls need beyond the partial buffers (0 in this version)."""
    c = cfg.c()
    n = ctypes.c_size_t(0)
    _check(_load().uq_decode_workspace_bytes(ctypes.byref(c), int(batch), int(num_splits), ctypes.byref(n)),
           "uq_decode_workspace_bytes")
    return int(n.value)


def suggest_num_splits(cfg: UQConfig, batch: int, avg_seq_len: int) -> int:
    c = cfg.c()
    return int(_load().uq_suggest_num_splits(ctypes.byref(c), int(batch), int(avg_seq_len)))


def suggest_num_splits_max(cfg: UQConfig, batch: int, avg_seq_len: int, max_seq_len: int) -> int:
    c = cfg.c()
    return int(_load().uq_suggest_num_splits_max(ctypes.byref(c), int(batch), int(avg_seq_len), int(max_seq_len)))


def suggest_prefix_splits(cfg: UQConfig, batch: int, prefix_len: int) -> int:
    c = cfg.c()
    return int(_load().uq_suggest_prefix_splits(ctypes.byref(c), int(batch), int(prefix_len)))


def alloc_cache(cfg: UQConfig, num_pages: int, device="cuda") -> torch.Tensor:
    """uint8 [num_pages, num_kv_heads, 17 * head_dim] (2176 at head_dim 128; layout: include/uq.h)."""
    return torch.zeros((num_pages, cfg.num_kv_heads, record_bytes(cfg.head_dim)), dtype=torch.uint8, device=device)


def rotate_quantize_append(cfg: UQConfig, k_new, v_new, cu_new, seq_lens, block_tables, cache,
                           q=None, q_fp8=None, stream=None) -> None:
    """uq_rotate_quantize_append (Alg. 1 l.1-6).  k_new/v_new bf16 [total_new, Hkv, d]."""
    lib = _load()
    _dev(k_new, torch.bfloat16, "k_new"); _dev(v_new, torch.bfloat16, "v_new")
    _dev(cu_new, torch.int32, "cu_new"); _dev(seq_lens, torch.int32, "seq_lens")
    _dev(block_tables, torch.int32, "block_tables"); _dev(cache, torch.uint8, "cache")
    if q is not None:
        _dev(q, torch.bfloat16, "q"); _dev(q_fp8, torch.uint8, "q_fp8")
    c = cfg.c()
    batch = seq_lens.shape[0]
    st = lib.uq_rotate_quantize_append(ctypes.byref(c), _p(k_new), _p(v_new), _p(cu_new), _p(seq_lens),
                                       _p(block_tables), block_tables.shape[1], batch, k_new.shape[0],
                                       _p(cache), cache.shape[0], _p(q), _p(q_fp8), _stream(stream))
    _check(st, "uq_rotate_quantize_append")


def calibrate_c(cfg: UQConfig, x, c_grid, rotate: bool = True, pow2_scale: bool = True, scale_mode=None, levels=None,
                stream=None):
    """uq_calibrate_c (Eq.(2)).  x bf16 [n, head_dim], c_grid float32 [n_c] (CUDA tensors); scale_mode
    0 (s = c m), 1 (the deployed power of two) or 2 (s = c), default 1 if pow2_scale else 0; levels None (E2M1) or
    float32 [8] on the device.  Returns (sq_err float64 [n_c], sq_norm float64 [1]) on the device; the calibrated
    constant is c_grid[sq_err.argmin()]."""
    lib = _load()
    _dev(x, torch.bfloat16, "x"); _dev(c_grid, torch.float32, "c_grid")
    if levels is not None:
        _dev(levels, torch.float32, "levels")
        if levels.numel() != 8:
            raise UQError("levels must hold 8 magnitudes")
    if x.dim() != 2 or x.shape[1] != cfg.head_dim:
        raise UQError(f"x must be [n, {cfg.head_dim}], got {tuple(x.shape)}")
    mode = (1 if pow2_scale else 0) if scale_mode is None else int(scale_mode)
    sq_err = torch.empty(c_grid.shape[0], dtype=torch.float64, device=x.device)
    sq_norm = torch.empty(1, dtype=torch.float64, device=x.device)
    c = cfg.c()
    st = lib.uq_calibrate_c(ctypes.byref(c), _p(x), x.shape[0], int(bool(rotate)), _p(c_grid), c_grid.shape[0],
                            mode, _p(levels), _p(sq_err), _p(sq_norm), _stream(stream))
    _check(st, "uq_calibrate_c")
    return sq_err, sq_norm


def decode_attention(cfg: UQConfig, q_fp8, cache, block_tables, seq_lens, num_splits: int,
                     partial_acc, partial_ml, stream=None) -> None:
    """uq_decode_attention (Alg. 1 l.7-8, split-K partials)."""
    lib = _load()
    _dev(q_fp8, torch.uint8, "q_fp8"); _dev(cache, torch.uint8, "cache")
    _dev(block_tables, torch.int32, "block_tables"); _dev(seq_lens, torch.int32, "seq_lens")
    _dev(partial_acc, torch.float32, "partial_acc"); _dev(partial_ml, torch.float32, "partial_ml")
    c = cfg.c()
    st = lib.uq_decode_attention(ctypes.byref(c), _p(q_fp8), _p(cache), cache.shape[0], _p(block_tables),
                                 block_tables.shape[1], _p(seq_lens), seq_lens.shape[0], int(num_splits),
                                 _p(partial_acc), _p(partial_ml), _stream(stream))
    _check(st, "uq_decode_attention")


def merge_splits(cfg: UQConfig, partial_acc, partial_ml, out, stream=None) -> None:
    """uq_merge_splits: out bf16 [batch, Hq, d]."""
    lib = _load()
    _dev(partial_acc, torch.float32, "partial_acc"); _dev(partial_ml, torch.float32, "partial_ml")
    _dev(out, torch.bfloat16, "out")
    c = cfg.c()
    st = lib.uq_merge_splits(ctypes.byref(c), _p(partial_acc), _p(partial_ml), out.shape[0],
                             partial_ml.shape[2], _p(out), _stream(stream))
    _check(st, "uq_merge_splits")


def static_scratch_bytes() -> int:
    """uq_static_scratch_bytes: size of the library's static split-partial array (UQ_STATIC_SCRATCH_BYTES)."""
    return int(_load().uq_static_scratch_bytes())


def decode_static_scratch_needed(cfg: UQConfig, batch: int, num_splits: int) -> int:
    """uq_decode_static_scratch_needed: bytes of that array a uq_decode_attention_static call of this shape uses."""
    lib = _load()
    n = ctypes.c_size_t(0)
    c = cfg.c()
    _check(lib.uq_decode_static_scratch_needed(ctypes.byref(c), int(batch), int(num_splits), ctypes.byref(n)),
           "uq_decode_static_scratch_needed")
    return int(n.value)


def decode_attention_static(cfg: UQConfig, q_fp8, cache, block_tables, seq_lens, num_splits: int, out, stream=None) -> None:
    """uq_decode_attention_static: decode + merge with the split partials in the library's static device array — the
    call allocates nothing.  out bf16 [batch, Hq, d].  Calls that overlap on the GPU race on that array."""
    lib = _load()
    _dev(q_fp8, torch.uint8, "q_fp8"); _dev(cache, torch.uint8, "cache")
    _dev(block_tables, torch.int32, "block_tables"); _dev(seq_lens, torch.int32, "seq_lens")
    _dev(out, torch.bfloat16, "out")
    c = cfg.c()
    st = lib.uq_decode_attention_static(ctypes.byref(c), _p(q_fp8), _p(cache), cache.shape[0], _p(block_tables),
                                        block_tables.shape[1], _p(seq_lens), seq_lens.shape[0], int(num_splits),
                                        _p(out), _stream(stream))
    _check(st, "uq_decode_attention_static")


class PrefixBuffers:
    """Device scratch of the shared-prefix decode: the prefix partials (a second set next to StepBuffers') and the
    suffix lengths / block-table view the suffix call reads.  `suffix_lens` (int32 [batch], = seq_lens - prefix_len)
    is the caller's to fill."""

    def __init__(self, cfg: UQConfig, batch: int, prefix_splits: int, device="cuda"):
        self.prefix_splits = prefix_splits
        self.partial_acc = torch.empty((batch, cfg.num_q_heads, prefix_splits, cfg.head_dim), dtype=torch.float32, device=device)
        self.partial_ml = torch.empty((batch, cfg.num_q_heads, prefix_splits, 2), dtype=torch.float32, device=device)
        self.suffix_lens = torch.empty((batch,), dtype=torch.int32, device=device)


def decode_attention_shared_prefix(cfg: UQConfig, bufs: "StepBuffers", pbufs: PrefixBuffers, cache, block_tables,
                                   prefix_len: int, stream=None, mark=None) -> torch.Tensor:
    """Decode + merge for sequences that share their first prefix_len tokens (a multiple of 128; same pages in every
    block table): uq_decode_prefix_attention over the prefix, uq_decode_attention over the private suffixes
    (pbufs.suffix_lens, the block tables from page prefix_len / page_size on), uq_merge_splits2.  bufs.q_fp8 holds
    the encoded queries.  Returns bufs.out.  mark (timing only): called with 0, 1, 2 before the prefix call, between
    the two decode calls and after the suffix call (bench.py records an event each time)."""
    lib = _load()
    _dev(cache, torch.uint8, "cache"); _dev(block_tables, torch.int32, "block_tables")
    c = cfg.c()
    batch, max_pages = block_tables.shape
    pp = prefix_len // cfg.page_size
    if mark is not None:
        mark(0)
    st = lib.uq_decode_prefix_attention(ctypes.byref(c), _p(bufs.q_fp8), _p(cache), cache.shape[0], _p(block_tables),
                                        max_pages, batch, int(prefix_len), pbufs.prefix_splits, _p(pbufs.partial_acc),
                                        _p(pbufs.partial_ml), _stream(stream))
    _check(st, "uq_decode_prefix_attention")
    if mark is not None:
        mark(1)
    bt_suffix = ctypes.c_void_p(block_tables.data_ptr() + 4 * pp)      # row stride stays max_pages
    st = lib.uq_decode_attention(ctypes.byref(c), _p(bufs.q_fp8), _p(cache), cache.shape[0], bt_suffix, max_pages,
                                 _p(pbufs.suffix_lens), batch, bufs.num_splits, _p(bufs.partial_acc),
                                 _p(bufs.partial_ml), _stream(stream))
    _check(st, "uq_decode_attention (suffix)")
    if mark is not None:
        mark(2)
    st = lib.uq_merge_splits2(ctypes.byref(c), _p(pbufs.partial_acc), _p(pbufs.partial_ml), pbufs.prefix_splits,
                              _p(bufs.partial_acc), _p(bufs.partial_ml), bufs.num_splits, batch, _p(bufs.out),
                              _stream(stream))
    _check(st, "uq_merge_splits2")
    return bufs.out


class StepBuffers:
    """Device scratch for one decode step (caller-owned memory, allocated once)."""

    def __init__(self, cfg: UQConfig, batch: int, num_splits: int, device="cuda"):
        self.num_splits = num_splits
        self.q_fp8 = torch.empty((batch, cfg.num_q_heads, cfg.head_dim), dtype=torch.uint8, device=device)
        self.partial_acc = torch.empty((batch, cfg.num_q_heads, num_splits, cfg.head_dim),
                                       dtype=torch.float32, device=device)
        self.partial_ml = torch.empty((batch, cfg.num_q_heads, num_splits, 2), dtype=torch.float32, device=device)
        self.out = torch.empty((batch, cfg.num_q_heads, cfg.head_dim), dtype=torch.bfloat16, device=device)
        self.seq_lens_after = torch.empty((batch,), dtype=torch.int32, device=device)
        self.cu_new = torch.empty((batch + 1,), dtype=torch.int32, device=device)


def decode_step(cfg: UQConfig, bufs: StepBuffers, q, k_new, v_new, cu_new, seq_lens_before,
                seq_lens_after, block_tables, cache, stream=None) -> torch.Tensor:
    """One whole hot-path step on device-resident inputs: quantize-on-append of the step's new
    tokens (k_new may have 0 rows) with the query rotate+cast, split-K decode, merge."""
    rotate_quantize_append(cfg, k_new, v_new, cu_new, seq_lens_before, block_tables, cache,
                           q=q, q_fp8=bufs.q_fp8, stream=stream)
    decode_attention(cfg, bufs.q_fp8, cache, block_tables, seq_lens_after, bufs.num_splits,
                     bufs.partial_acc, bufs.partial_ml, stream=stream)
    merge_splits(cfg, bufs.partial_acc, bufs.partial_ml, bufs.out, stream=stream)
    return bufs.out


class HostStage:
    """A step's inputs laid back to back in ONE pinned host block with a device block of the same layout, so
    that they cross PCIe in a single copy: q bf16 [batch, Hq, d], k_new / v_new bf16 [total_new, Hkv, d],
    cu_new i32 [batch + 1], seq_lens_before / seq_lens_after i32 [batch], block_tables i32 [batch, max_pages].
    The caller writes the host views (`.h[name]`), `upload()` enqueues the copy, the kernels read `.d[name]`.
    The block tables come last in the block: they change only when a sequence crosses a page boundary (every 16th
    token), so `upload(tables=False)` leaves them out and the caller sends them with `upload_tables()` when they did."""

    FIELDS = ("q", "k_new", "v_new", "cu_new", "seq_lens_before", "seq_lens_after", "block_tables")

    def __init__(self, cfg: UQConfig, batch: int, total_new: int, max_pages: int, device="cuda"):
        d = cfg.head_dim
        spec = {
            "q": ((batch, cfg.num_q_heads, d), torch.bfloat16),
            "k_new": ((total_new, cfg.num_kv_heads, d), torch.bfloat16),
            "v_new": ((total_new, cfg.num_kv_heads, d), torch.bfloat16),
            "cu_new": ((batch + 1,), torch.int32),
            "seq_lens_before": ((batch,), torch.int32),
            "seq_lens_after": ((batch,), torch.int32),
            "block_tables": ((batch, max_pages), torch.int32),
        }
        offs, total = {}, 0
        for name in self.FIELDS:
            shape, dtype = spec[name]
            n = int(torch.tensor(shape).prod().item()) * torch.empty((), dtype=dtype).element_size()
            offs[name] = (total, n)
            total = (total + n + 255) // 256 * 256          # every field 256-byte aligned (the kernels ask for 16)
        self.nbytes = total
        self.step_nbytes = offs["block_tables"][0]          # everything before the block tables: a step's own inputs
        self.host = torch.empty(total, dtype=torch.uint8)
        if torch.device(device).type == "cuda":
            self.host = self.host.pin_memory()
        self.dev = torch.empty(total, dtype=torch.uint8, device=device)

        def views(block):
            return {name: block[o:o + n].view(spec[name][1]).view(spec[name][0]) for name, (o, n) in offs.items()}
        self.h, self.d = views(self.host), views(self.dev)

    def upload(self, tables: bool = True):
        n = self.nbytes if tables else self.step_nbytes
        self.dev[:n].copy_(self.host[:n], non_blocking=True)    # on the current stream

    def upload_tables(self):
        self.dev[self.step_nbytes:].copy_(self.host[self.step_nbytes:], non_blocking=True)


def decode_step_host(cfg: UQConfig, bufs: StepBuffers, stage: HostStage, cache, out_host, stream=None,
                     tables: bool = True) -> torch.Tensor:
    """The step with HOST (pinned) inputs and output: the step's query, new K/V rows, lengths and block tables
    (stage.h, filled by the caller) are copied host->device in one copy, the attention output device->host.
    The KV cache itself is the resident state and stays in HBM."""
    stage.upload(tables)
    dv = stage.d
    out = decode_step(cfg, bufs, dv["q"], dv["k_new"], dv["v_new"], dv["cu_new"], dv["seq_lens_before"],
                      dv["seq_lens_after"], dv["block_tables"], cache, stream=stream)
    out_host.copy_(out, non_blocking=True)
    return out_host


class StepGraph:
    """decode_step on device-resident inputs captured once as a CUDA graph (the three kernels with their
    programmatic-launch edges): a step costs the host one graph launch — what matters when the step is short
    (config 1: three launches from Python take longer than the kernels).  All addresses are those of the tensors
    given here: the caller rewrites them in place between launches.  The constructor runs the step once."""

    def __init__(self, cfg: UQConfig, bufs: StepBuffers, q, k_new, v_new, cu_new, seq_lens_before, seq_lens_after,
                 block_tables, cache):
        args = (cfg, bufs, q, k_new, v_new, cu_new, seq_lens_before, seq_lens_after, block_tables, cache)
        decode_step(*args)                                           # first-call set-up happens outside the capture
        torch.cuda.current_stream().synchronize()
        self.graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(self.graph):
            decode_step(*args)
        self.out = bufs.out

    def launch(self) -> torch.Tensor:
        self.graph.replay()
        return self.out


class HostStepGraph:
    """decode_step_host captured once as a CUDA graph — the host->device copy of the staged inputs, the three kernels
    (their programmatic-launch edges are kept by the capture) and the device->host copy of O — so that a step costs
    the host one graph launch.  All addresses are those of `stage`, `bufs`, `cache` and `out_host`: the caller
    rewrites `stage.h[...]` between launches.  `launch()` enqueues on the current stream."""

    def __init__(self, cfg: UQConfig, bufs: StepBuffers, stage: HostStage, cache, out_host, tables: bool = True):
        """tables=False: the captured step uploads the step's own inputs only; the caller sends the block tables with
        stage.upload_tables() whenever they change (the constructor sends them once)."""
        decode_step_host(cfg, bufs, stage, cache, out_host)          # first-call set-up happens outside the capture
        torch.cuda.current_stream().synchronize()
        self.graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(self.graph):                           # torch's capture stream becomes the current one
            decode_step_host(cfg, bufs, stage, cache, out_host, tables=tables)
        self.out_host = out_host

    def launch(self) -> torch.Tensor:
        self.graph.replay()
        return self.out_host


# ----------------------------------------------------------------------------- comparison caches (include/uq.h)
KV_FP8_E4M3 = 1
KV_BF16 = 2
KV_ULTRA_TQ = 3


def _codebook(codebook):
    cb = (ctypes.c_float * 16)(*[float(v) for v in codebook])
    return cb


def tq_append(cfg: UQConfig, codebook, k_new, v_new, cu_new, seq_lens, block_tables, cache, q=None, q_rot=None, stream=None) -> None:
    """uq_tq_append (Alg. 2 l.1-5): new rows into the Ultra-TQ cache (alloc_baseline_cache(cfg, KV_ULTRA_TQ, ...)); q bf16
    -> q_rot bf16 = bf16(R q).  codebook: 16 ascending floats (host)."""
    lib = _load()
    _dev(k_new, torch.bfloat16, "k_new"); _dev(v_new, torch.bfloat16, "v_new")
    _dev(cu_new, torch.int32, "cu_new"); _dev(seq_lens, torch.int32, "seq_lens")
    _dev(block_tables, torch.int32, "block_tables"); _dev(cache, torch.uint8, "cache")
    if q is not None:
        _dev(q, torch.bfloat16, "q"); _dev(q_rot, torch.bfloat16, "q_rot")
    c = cfg.c()
    cb = _codebook(codebook)
    st = lib.uq_tq_append(ctypes.byref(c), ctypes.cast(cb, ctypes.c_void_p), _p(k_new), _p(v_new), _p(cu_new), _p(seq_lens),
                          _p(block_tables), block_tables.shape[1], seq_lens.shape[0], k_new.shape[0], _p(cache),
                          cache.shape[0], _p(q), _p(q_rot), _stream(stream))
    _check(st, "uq_tq_append")


def tq_decode_attention(cfg: UQConfig, codebook, q_rot, cache, block_tables, seq_lens, num_splits: int, partial_acc,
                        partial_ml, stream=None) -> None:
    """uq_tq_decode_attention (Alg. 2 l.6-8): split-K partials over the Ultra-TQ cache; merge_splits finishes."""
    lib = _load()
    _dev(q_rot, torch.bfloat16, "q_rot"); _dev(cache, torch.uint8, "cache")
    _dev(block_tables, torch.int32, "block_tables"); _dev(seq_lens, torch.int32, "seq_lens")
    _dev(partial_acc, torch.float32, "partial_acc"); _dev(partial_ml, torch.float32, "partial_ml")
    c = cfg.c()
    cb = _codebook(codebook)
    st = lib.uq_tq_decode_attention(ctypes.byref(c), ctypes.cast(cb, ctypes.c_void_p), _p(q_rot), _p(cache), cache.shape[0],
                                    _p(block_tables), block_tables.shape[1], _p(seq_lens), seq_lens.shape[0], int(num_splits),
                                    _p(partial_acc), _p(partial_ml), _stream(stream))
    _check(st, "uq_tq_decode_attention")


def baseline_record_bytes(cfg: UQConfig, kv_format: int) -> int:
    c = cfg.c()
    return int(_load().uq_baseline_record_bytes(ctypes.byref(c), int(kv_format)))


def alloc_baseline_cache(cfg: UQConfig, kv_format: int, num_pages: int, device="cuda") -> torch.Tensor:
    """uint8 [num_pages, num_kv_heads, 4096 (FP8) | 8192 (BF16)]: K rows [16 tok][128] then V [128 ch][16 tok]."""
    n = baseline_record_bytes(cfg, kv_format)
    if n == 0:
        raise UQError(f"uq_baseline_record_bytes: {last_error()}")
    return torch.zeros((num_pages, cfg.num_kv_heads, n), dtype=torch.uint8, device=device)


def baseline_append(cfg: UQConfig, kv_format: int, k_new, v_new, cu_new, seq_lens, block_tables, cache, q=None, q_out=None,
                    stream=None) -> None:
    """uq_baseline_append: store new K/V rows in the FP8-E4M3 / BF16 comparison cache (FP8: also q -> q_out E4M3)."""
    lib = _load()
    _dev(k_new, torch.bfloat16, "k_new"); _dev(v_new, torch.bfloat16, "v_new")
    _dev(cu_new, torch.int32, "cu_new"); _dev(seq_lens, torch.int32, "seq_lens")
    _dev(block_tables, torch.int32, "block_tables"); _dev(cache, torch.uint8, "cache")
    if q is not None and q_out is not None:
        _dev(q, torch.bfloat16, "q"); _dev(q_out, torch.uint8, "q_out")
    c = cfg.c()
    st = lib.uq_baseline_append(ctypes.byref(c), int(kv_format), _p(k_new), _p(v_new), _p(cu_new), _p(seq_lens),
                                _p(block_tables), block_tables.shape[1], seq_lens.shape[0], k_new.shape[0], _p(cache),
                                cache.shape[0], _p(q) if q_out is not None else None, _p(q_out), _stream(stream))
    _check(st, "uq_baseline_append")


def baseline_decode_attention(cfg: UQConfig, kv_format: int, q_enc, cache, block_tables, seq_lens, num_splits: int,
                              partial_acc, partial_ml, stream=None) -> None:
    """uq_baseline_decode_attention: split-K partials over the comparison cache (q_enc: uint8 E4M3 or bf16)."""
    lib = _load()
    _dev(q_enc, torch.uint8 if kv_format == KV_FP8_E4M3 else torch.bfloat16, "q_enc"); _dev(cache, torch.uint8, "cache")
    _dev(block_tables, torch.int32, "block_tables"); _dev(seq_lens, torch.int32, "seq_lens")
    _dev(partial_acc, torch.float32, "partial_acc"); _dev(partial_ml, torch.float32, "partial_ml")
    c = cfg.c()
    st = lib.uq_baseline_decode_attention(ctypes.byref(c), int(kv_format), _p(q_enc), _p(cache), cache.shape[0],
                                          _p(block_tables), block_tables.shape[1], _p(seq_lens), seq_lens.shape[0],
                                          int(num_splits), _p(partial_acc), _p(partial_ml), _stream(stream))
    _check(st, "uq_baseline_decode_attention")


def baseline_decode_step(cfg: UQConfig, kv_format: int, bufs: "StepBuffers", q, k_new, v_new, cu_new, seq_lens_before,
                         seq_lens_after, block_tables, cache, stream=None) -> torch.Tensor:
    """One step over a comparison cache: append (+ query cast for FP8), split-K decode, merge.  Returns bufs.out."""
    fp8 = kv_format == KV_FP8_E4M3
    baseline_append(cfg, kv_format, k_new, v_new, cu_new, seq_lens_before, block_tables, cache,
                    q=q if fp8 else None, q_out=bufs.q_fp8 if fp8 else None, stream=stream)
    baseline_decode_attention(cfg, kv_format, bufs.q_fp8 if fp8 else q, cache, block_tables, seq_lens_after,
                              bufs.num_splits, bufs.partial_acc, bufs.partial_ml, stream=stream)
    merge_splits(cfg, bufs.partial_acc, bufs.partial_ml, bufs.out, stream=stream)
    return bufs.out
