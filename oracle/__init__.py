"""ctypes front end of the float64 CPU oracle (oracle/uq_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  The product package never imports this module,
and this module never imports the product package.

All arrays are numpy; "logical" cache arrays are
    codes  uint8 [n_vec, d/2]   (element 2j in bits 0-3 of byte j, 2j+1 in bits 4-7)
    scales uint8 [n_vec, d/32]  (UE8M0 byte = E + 127)
following Algorithm 1 of the paper.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "uq_oracle.c")
_LIB = os.path.join(_HERE, "libuq_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile uq_oracle.c with gcc -O2 (no fast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = ctypes.CDLL(build())
    u8p = ctypes.POINTER(ctypes.c_uint8)
    u16p = ctypes.POINTER(ctypes.c_uint16)
    f64p = ctypes.POINTER(ctypes.c_double)
    lib.uqo_bf16_to_double.restype = ctypes.c_double
    lib.uqo_bf16_to_double.argtypes = [ctypes.c_uint16]
    lib.uqo_kappa.restype = ctypes.c_double
    lib.uqo_kappa.argtypes = [ctypes.c_int]
    lib.uqo_hadamard.restype = None
    lib.uqo_hadamard.argtypes = [f64p, ctypes.c_int, f64p]
    lib.uqo_scale_exponent.restype = ctypes.c_int
    lib.uqo_scale_exponent.argtypes = [ctypes.c_double, ctypes.c_double]
    lib.uqo_e2m1_encode.restype = ctypes.c_uint8
    lib.uqo_e2m1_encode.argtypes = [ctypes.c_double, ctypes.c_int]
    lib.uqo_e2m1_level.restype = ctypes.c_double
    lib.uqo_e2m1_level.argtypes = [ctypes.c_uint8]
    lib.uqo_dequant.restype = ctypes.c_double
    lib.uqo_dequant.argtypes = [ctypes.c_uint8, ctypes.c_uint8]
    lib.uqo_quantize_vector.restype = None
    lib.uqo_quantize_vector.argtypes = [f64p, ctypes.c_int, ctypes.c_double, u8p, u8p]
    lib.uqo_encode_kv.restype = None
    lib.uqo_encode_kv.argtypes = [u16p, u16p, ctypes.c_int64, ctypes.c_int, ctypes.c_float,
                                  ctypes.c_float, u8p, u8p, u8p, u8p]
    lib.uqo_e4m3_encode.restype = ctypes.c_uint8
    lib.uqo_e4m3_encode.argtypes = [ctypes.c_double]
    lib.uqo_e4m3_decode.restype = ctypes.c_double
    lib.uqo_e4m3_decode.argtypes = [ctypes.c_uint8]
    lib.uqo_encode_q.restype = None
    lib.uqo_encode_q.argtypes = [u16p, ctypes.c_int64, ctypes.c_int, u8p]
    lib.uqo_attention.restype = None
    lib.uqo_attention.argtypes = [u8p, u8p, u8p, u8p, u8p, ctypes.c_int64, ctypes.c_int,
                                  ctypes.c_int, ctypes.c_int, ctypes.c_double, f64p, f64p]
    lib.uqo_attention_dense.restype = None
    lib.uqo_attention_dense.argtypes = [f64p, f64p, f64p, ctypes.c_int64, ctypes.c_int,
                                        ctypes.c_int, ctypes.c_int, ctypes.c_double, f64p]
    lib.uqo_calib_sq_err.restype = None
    lib.uqo_calib_sq_err.argtypes = [u16p, ctypes.c_int64, ctypes.c_int, ctypes.c_int,
                                     ctypes.POINTER(ctypes.c_float), ctypes.c_int, ctypes.c_int,
                                     ctypes.POINTER(ctypes.c_float), f64p, f64p]
    lib.uqo_cast_e4m3.restype = None
    lib.uqo_cast_e4m3.argtypes = [u16p, ctypes.c_int64, u8p]
    lib.uqo_e4m3_to_double.restype = None
    lib.uqo_e4m3_to_double.argtypes = [u8p, ctypes.c_int64, f64p]
    lib.uqo_num_threads.restype = ctypes.c_int
    lib.uqo_set_num_threads.argtypes = [ctypes.c_int]
    _lib = lib
    return lib


def _ptr(a: np.ndarray, ctype):
    return a.ctypes.data_as(ctypes.POINTER(ctype))


def _c(a, dtype) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=dtype)


# ------------------------------------------------------------------ scalar helpers
def kappa(d: int) -> float:
    return _load().uqo_kappa(d)


def bf16_to_double(bits) -> np.ndarray:
    """Exact float64 value of bf16 bit patterns (uint16 array)."""
    bits = np.asarray(bits, dtype=np.uint16)
    return (bits.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def hadamard(x) -> np.ndarray:
    """y = H_d x / sqrt(d) for one vector (dense product, Sylvester order)."""
    x = _c(x, np.float64)
    y = np.empty_like(x)
    _load().uqo_hadamard(_ptr(x, ctypes.c_double), x.shape[0], _ptr(y, ctypes.c_double))
    return y


def scale_exponent(c: float, m: float) -> int:
    return _load().uqo_scale_exponent(float(c), float(m))


def e2m1_encode(y: float, E: int) -> int:
    return _load().uqo_e2m1_encode(float(y), int(E))


def e2m1_level(code: int) -> float:
    return _load().uqo_e2m1_level(int(code))


def dequant(code: int, scale_byte: int) -> float:
    return _load().uqo_dequant(int(code), int(scale_byte))


def e4m3_encode(y: float) -> int:
    return _load().uqo_e4m3_encode(float(y))


def e4m3_decode(b: int) -> float:
    return _load().uqo_e4m3_decode(int(b))


def num_threads() -> int:
    return _load().uqo_num_threads()


def set_num_threads(n: int) -> None:
    _load().uqo_set_num_threads(int(n))


# ------------------------------------------------------------------ vector / bulk
def quantize_vector(y, c: float):
    """Alg. 1 l.2-5 on one (already rotated or unrotated) vector of doubles."""
    y = _c(y, np.float64)
    d = y.shape[0]
    packed = np.empty(d // 2, np.uint8)
    scales = np.empty(d // 32, np.uint8)
    _load().uqo_quantize_vector(_ptr(y, ctypes.c_double), d, float(c),
                                _ptr(packed, ctypes.c_uint8), _ptr(scales, ctypes.c_uint8))
    return packed, scales


def encode_kv(k_bits, v_bits, c_k: float = 0.156, c_v: float = 0.156):
    """Alg. 1 "Write".  k_bits, v_bits: uint16 bf16 patterns [..., d].  Returns the logical
    arrays (k_codes, k_scales, v_codes, v_scales) with the leading dims of the input."""
    k_bits = _c(k_bits, np.uint16)
    v_bits = _c(v_bits, np.uint16)
    d = k_bits.shape[-1]
    lead = k_bits.shape[:-1]
    n = int(np.prod(lead)) if lead else 1
    kc = np.empty((n, d // 2), np.uint8)
    ks = np.empty((n, d // 32), np.uint8)
    vc = np.empty((n, d // 2), np.uint8)
    vs = np.empty((n, d // 32), np.uint8)
    _load().uqo_encode_kv(_ptr(k_bits, ctypes.c_uint16), _ptr(v_bits, ctypes.c_uint16), n, d,
                          ctypes.c_float(c_k), ctypes.c_float(c_v),
                          _ptr(kc, ctypes.c_uint8), _ptr(ks, ctypes.c_uint8),
                          _ptr(vc, ctypes.c_uint8), _ptr(vs, ctypes.c_uint8))
    return (kc.reshape(lead + (d // 2,)), ks.reshape(lead + (d // 32,)),
            vc.reshape(lead + (d // 2,)), vs.reshape(lead + (d // 32,)))


def calib_sq_err(x_bits, c_grid, rotate: bool = True, pow2: bool = True, scale_mode: int | None = None, levels=None):
    """Objective of Eq.(2) on a grid of constants: x_bits uint16 bf16 patterns [n, d], c_grid
    float32 [n_c].  Returns (sq_err float64 [n_c], sq_norm float): sums over all elements of (z - zhat)^2 and
    z^2, z rotated if `rotate`.  scale_mode 0: s = c*m; 1: the deployed power-of-two scale (Alg. 1 l.3); 2: s = c
    (no absmax); default 1 if pow2 else 0.  levels: None (E2M1) or 8 ascending magnitudes of another codebook."""
    x_bits = _c(x_bits, np.uint16)
    c_grid = _c(c_grid, np.float32)
    n, d = x_bits.shape
    mode = (1 if pow2 else 0) if scale_mode is None else int(scale_mode)
    lev = None if levels is None else _c(levels, np.float32)
    sq_err = np.zeros(c_grid.shape[0], np.float64)
    sq_norm = np.zeros(1, np.float64)
    _load().uqo_calib_sq_err(_ptr(x_bits, ctypes.c_uint16), n, d, int(bool(rotate)), _ptr(c_grid, ctypes.c_float),
                             c_grid.shape[0], mode, None if lev is None else _ptr(lev, ctypes.c_float),
                             _ptr(sq_err, ctypes.c_double), _ptr(sq_norm, ctypes.c_double))
    return sq_err, float(sq_norm[0])


def encode_q(q_bits) -> np.ndarray:
    """Alg. 1 l.6: rotate, cast to E4M3 bytes.  q_bits uint16 [..., d] -> uint8 [..., d]."""
    q_bits = _c(q_bits, np.uint16)
    d = q_bits.shape[-1]
    n = q_bits.size // d
    out = np.empty(q_bits.shape, np.uint8)
    _load().uqo_encode_q(_ptr(q_bits, ctypes.c_uint16), n, d, _ptr(out, ctypes.c_uint8))
    return out


def unpack_codes(packed) -> np.ndarray:
    """uint8 [..., d/2] -> uint8 codes [..., d] (one 4-bit code per byte)."""
    packed = np.asarray(packed, np.uint8)
    out = np.empty(packed.shape[:-1] + (packed.shape[-1] * 2,), np.uint8)
    out[..., 0::2] = packed & 0xF
    out[..., 1::2] = packed >> 4
    return out


def dequantize(packed, scales) -> np.ndarray:
    """Eq.(1) on logical arrays: float64 [..., d]."""
    codes = unpack_codes(packed)
    levels = np.array([e2m1_level(c) for c in range(16)], np.float64)
    scales = np.asarray(scales, np.uint8)
    exp = np.repeat(scales.astype(np.int64) - 127, 32, axis=-1)
    return np.ldexp(levels[codes], exp)


def attention(q8, k_codes, k_scales, v_codes, v_scales, num_q_heads: int, num_kv_heads: int,
              sm_scale: float | None = None, return_probs: bool = False):
    """Alg. 1 "Decode" l.7-8 for ONE sequence: q8 uint8 [Hq, d]; logical cache arrays
    [L, Hkv, d/2] / [L, Hkv, d/32].  Returns float64 out [Hq, d] (and p [Hq, L])."""
    q8 = _c(q8, np.uint8)
    k_codes = _c(k_codes, np.uint8)
    k_scales = _c(k_scales, np.uint8)
    v_codes = _c(v_codes, np.uint8)
    v_scales = _c(v_scales, np.uint8)
    d = q8.shape[-1]
    L = k_codes.shape[0]
    if sm_scale is None or sm_scale == 0:
        sm_scale = 1.0 / np.sqrt(float(d))
    out = np.zeros((num_q_heads, d), np.float64)
    probs = np.zeros((num_q_heads, max(L, 1)), np.float64) if return_probs else None
    _load().uqo_attention(_ptr(q8, ctypes.c_uint8), _ptr(k_codes, ctypes.c_uint8),
                          _ptr(k_scales, ctypes.c_uint8), _ptr(v_codes, ctypes.c_uint8),
                          _ptr(v_scales, ctypes.c_uint8), L, num_q_heads, num_kv_heads, d,
                          float(sm_scale), _ptr(out, ctypes.c_double),
                          _ptr(probs, ctypes.c_double) if return_probs else None)
    if return_probs:
        return out, probs[:, :L]
    return out


def attention_dense(q, k, v, sm_scale: float | None = None) -> np.ndarray:
    """Unquantised softmax attention in float64 (context only): q [Hq,d], k,v [L,Hkv,d]."""
    q = _c(q, np.float64)
    k = _c(k, np.float64)
    v = _c(v, np.float64)
    Hq, d = q.shape
    L, Hkv = k.shape[0], k.shape[1]
    if sm_scale is None or sm_scale == 0:
        sm_scale = 1.0 / np.sqrt(float(d))
    out = np.zeros((Hq, d), np.float64)
    _load().uqo_attention_dense(_ptr(q, ctypes.c_double), _ptr(k, ctypes.c_double),
                                _ptr(v, ctypes.c_double), L, Hq, Hkv, d, float(sm_scale),
                                _ptr(out, ctypes.c_double))
    return out


# ------------------------------------------------------------------ comparison caches (DESIGN reading G19)
def cast_e4m3(x_bits) -> np.ndarray:
    """bf16 bit patterns -> OCP E4M3 bytes of the values themselves (no rotation, scale 1): the FP8-KV cache entry."""
    x_bits = _c(x_bits, np.uint16)
    out = np.empty(x_bits.shape, np.uint8)
    _load().uqo_cast_e4m3(_ptr(x_bits, ctypes.c_uint16), x_bits.size, _ptr(out, ctypes.c_uint8))
    return out


def e4m3_to_double(b) -> np.ndarray:
    b = _c(b, np.uint8)
    out = np.empty(b.shape, np.float64)
    _load().uqo_e4m3_to_double(_ptr(b, ctypes.c_uint8), b.size, _ptr(out, ctypes.c_double))
    return out


def attention_fp8kv(q_bits, k_bits, v_bits, sm_scale: float | None = None):
    """FP8-E4M3 KV attention for ONE sequence: q bf16 bits [Hq, d], k / v bf16 bits [L, Hkv, d]; every tensor is cast to
    E4M3 (cast_e4m3), then plain float64 softmax attention over the decoded values.  Returns (out [Hq, d], q8, k8, v8)."""
    q8, k8, v8 = cast_e4m3(q_bits), cast_e4m3(k_bits), cast_e4m3(v_bits)
    out = attention_dense(e4m3_to_double(q8), e4m3_to_double(k8), e4m3_to_double(v8), sm_scale)
    return out, q8, k8, v8


def attention_bf16kv(q_bits, k_bits, v_bits, sm_scale: float | None = None) -> np.ndarray:
    """BF16 KV attention for ONE sequence: float64 softmax attention over the exact values of the bf16 inputs."""
    return attention_dense(bf16_to_double(q_bits), bf16_to_double(k_bits), bf16_to_double(v_bits), sm_scale)
