"""Float64 oracle of the paper's Algorithm 2, "Calibrated LUT int4 KV encoding (Ultra-TQ)" — the
codebook path that UltraQuant replaces; built here only as the last comparison kernel of SURVEY 8(f) rank 4.

TEST INFRASTRUCTURE ONLY (as oracle/__init__.py): plain numpy, one step per line of the algorithm, in its order.

Algorithm 2 leaves open what a "block norm", the metadata types and the decode arithmetic are; the readings (DESIGN.md
G20) are:
  * rotation R and group size g = 32 as in Algorithm 1 ("rotation R; group size g");
  * l.3 "K: store block norm": the l2 norm of the 32 rotated coordinates of the block (TurboQuant's unit-sphere scaling,
    PAPER.md:39), accumulated in coordinate order, stored as bf16 (round to nearest even); the coordinate is divided by
    the STORED norm before the codebook search;
  * l.3 "nearest C_K index": argmin_i |u - C_K[i]|, ties to the lower index; C_K (16 float32 values) is an INPUT
    ("codebook C_K": calibrated offline, out of scope here);
  * l.4 "V: store block (scale, zero); 4-bit uniform": zero = min, scale = (max - min) / 15 over the block, both stored
    as bf16 (RNE); code = clamp(rint((v - zero) / scale), 0, 15), scale 0 -> code 0;
  * l.7 "K: dequant via C_K . norm": bf16(bf16(C_K[idx]) * norm);  "V: scale . code + zero": bf16(scale * code + zero);
  * l.5 / l.8: Q <- R Q rounded to bf16; QK and PV "on dequantized K, V": plain softmax attention (scale 1/sqrt(d)).
parity unpinned: the conventions above (the paper prints no worked example of Algorithm 2); the arithmetic itself is
pinned by tests/test_oracle_pins.py P15-P17.
"""
from __future__ import annotations

import numpy as np

from . import attention_dense, bf16_to_double, hadamard

GROUP = 32


def rotate_rows(x) -> np.ndarray:
    """R applied to every row of x [n, d] (oracle.hadamard takes one vector)."""
    x = np.asarray(x, np.float64)
    return np.stack([hadamard(row) for row in x]) if len(x) else x.copy()


def bf16_rne(x) -> np.ndarray:
    """float64 -> the nearest bf16 value (8 significant bits, ties to even), returned as float64.  Written out: the
    quantum of a value in [2^e, 2^(e+1)) is 2^(e-7); values below the bf16 normal range do not occur in this path."""
    x = np.asarray(x, np.float64)
    out = np.zeros_like(x)
    nz = x != 0
    _, e = np.frexp(x[nz])                       # |x| = m 2^e, m in [0.5, 1)
    quantum = np.ldexp(1.0, e - 8)               # 2^((e-1)-7)
    out[nz] = np.rint(x[nz] / quantum) * quantum
    return out


def bf16_bits(x) -> np.ndarray:
    """bf16-representable float64 values -> their 16-bit patterns."""
    f = np.ascontiguousarray(np.asarray(x, np.float64).astype(np.float32))
    assert np.array_equal(f.astype(np.float64), np.asarray(x, np.float64)), "value is not a float32"
    b = f.view(np.uint32)
    assert not np.any(b & 0xFFFF), "value is not a bf16"
    return (b >> 16).astype(np.uint16)


def encode_k(k_bits, codebook):
    """Alg. 2 l.1-3.  k_bits uint16 bf16 patterns [n, d]; codebook 16 float32 values, ascending.
    Returns (idx uint8 [n, d] in 0..15, norm float64 [n, d/32] = the stored bf16 norms)."""
    c = np.asarray(codebook, np.float32).astype(np.float64)
    assert c.shape == (16,)
    x = rotate_rows(bf16_to_double(k_bits))                               # l.1: K <- R K
    n, d = x.shape
    xb = x.reshape(n, d // GROUP, GROUP)                                  # l.2: g-channel blocks
    acc = np.zeros((n, d // GROUP), np.float64)
    for j in range(GROUP):                                                # l.3: block norm, coordinate order
        acc = acc + xb[:, :, j] * xb[:, :, j]
    norm = bf16_rne(np.sqrt(acc))
    with np.errstate(divide="ignore", invalid="ignore"):
        u = np.where(norm[:, :, None] > 0, xb / norm[:, :, None], 0.0)
    dist = np.abs(u[..., None] - c)                                       # l.3: nearest C_K index (argmin: first minimum)
    idx = np.argmin(dist, axis=-1).astype(np.uint8)
    return idx.reshape(n, d), norm


def encode_v(v_bits):
    """Alg. 2 l.2, l.4.  v_bits uint16 bf16 patterns [n, d] (V is not rotated).
    Returns (code uint8 [n, d] in 0..15, scale float64 [n, d/32], zero float64 [n, d/32]) — scale, zero bf16 values."""
    v = bf16_to_double(v_bits)
    n, d = v.shape
    vb = v.reshape(n, d // GROUP, GROUP)
    mn, mx = vb.min(axis=-1), vb.max(axis=-1)
    scale = bf16_rne((mx - mn) / 15.0)
    zero = bf16_rne(mn)
    with np.errstate(divide="ignore", invalid="ignore"):
        t = np.where(scale[:, :, None] > 0, (vb - zero[:, :, None]) / scale[:, :, None], 0.0)
    code = np.clip(np.rint(t), 0, 15).astype(np.uint8)
    return code.reshape(n, d), scale, zero


def dequant_k(idx, norm, codebook) -> np.ndarray:
    """Alg. 2 l.7: C_K[idx] . norm, both factors bf16, the product rounded to bf16."""
    c = bf16_rne(np.asarray(codebook, np.float32).astype(np.float64))
    n, d = idx.shape
    return bf16_rne(c[idx].reshape(n, d // GROUP, GROUP) * norm[:, :, None]).reshape(n, d)


def dequant_v(code, scale, zero) -> np.ndarray:
    """Alg. 2 l.7: scale . code + zero, rounded to bf16 once."""
    n, d = code.shape
    c = code.reshape(n, d // GROUP, GROUP).astype(np.float64)
    return bf16_rne(scale[:, :, None] * c + zero[:, :, None]).reshape(n, d)


def encode_q(q_bits) -> np.ndarray:
    """Alg. 2 l.5: Q <- R Q, rounded to bf16 (float64 values)."""
    return bf16_rne(rotate_rows(bf16_to_double(q_bits)))


def attention(q_bits, k_idx, k_norm, v_code, v_scale, v_zero, codebook, num_kv_heads: int, sm_scale=None) -> np.ndarray:
    """Alg. 2 l.5-8 for ONE sequence: q_bits [Hq, d]; k_idx / v_code [L, Hkv, d]; k_norm / v_scale / v_zero
    [L, Hkv, d/32].  Returns the float64 output [Hq, d]."""
    L, Hkv, d = k_idx.shape
    assert Hkv == num_kv_heads
    q = encode_q(q_bits)
    k = dequant_k(k_idx.reshape(L * Hkv, d), k_norm.reshape(L * Hkv, -1), codebook).reshape(L, Hkv, d)
    v = dequant_v(v_code.reshape(L * Hkv, d), v_scale.reshape(L * Hkv, -1), v_zero.reshape(L * Hkv, -1)).reshape(L, Hkv, d)
    return attention_dense(q, k, v, sm_scale)
