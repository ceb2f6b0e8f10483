"""Independent unpacker of the physical cache record documented in include/uq.h ("PHYSICAL
CACHE LAYOUT"), written from that description only.  Test glue: it maps a device cache image
back to the LOGICAL arrays the oracle produces (packed codes [.., d/2], scale bytes [.., d/32]).
Pure index arithmetic — none of the method's arithmetic lives here.  head_dim d in {64, 128, 256}:
record = 17 d bytes = K codes [0, 8d) | V codes [8d, 16d) | K scales [16d, 16d + d/2) | V scales."""
import functools

import numpy as np

RECORD = 2176          # head_dim 128
PAGE = 16


def record_bytes(d: int = 128) -> int:
    return 17 * d


@functools.lru_cache(maxsize=None)
def _indices(d: int):
    ng = d // 32
    # K codes, logical order: token slot t at (d/2) t, byte j = channels 2j, 2j+1
    kc = np.zeros((PAGE, d // 2), np.int64)
    for t in range(PAGE):
        for j in range(d // 2):
            kc[t, j] = (d // 2) * t + j
    # V codes, token-major nibbles: the 32-bit word at 8d + 4d (t>>3) + 128 (c>>5) + 4 (c&31) holds channel c of
    # the eight tokens of the octet; token t in bits 4(t&7)..4(t&7)+3
    vc = np.zeros((PAGE, d), np.int64)
    sh = np.zeros((PAGE, d), np.int64)
    for t in range(PAGE):
        for c in range(d):
            word = 8 * d + 4 * d * (t >> 3) + 128 * (c >> 5) + 4 * (c & 31)
            bit = 4 * (t & 7)
            vc[t, c] = word + bit // 8            # little-endian byte of the word
            sh[t, c] = bit % 8
    # K scales: token t's d/32 group bytes (group 0 first) at 16d + (d/32) t
    ks = np.zeros((PAGE, ng), np.int64)
    for t in range(PAGE):
        for gr in range(ng):
            ks[t, gr] = 16 * d + ng * t + gr
    # V scales: token t, group g at 16d + d/2 + (d/4)(t>>3) + 8 g + (t&7)
    vs = np.zeros((PAGE, ng), np.int64)
    for t in range(PAGE):
        for gr in range(ng):
            vs[t, gr] = 16 * d + d // 2 + (d // 4) * (t >> 3) + 8 * gr + (t & 7)
    return kc, vc, sh, ks, vs


def unpack_records(rec: np.ndarray):
    """rec uint8 [..., 17 d] -> logical (k_codes [...,16,d/2], k_scales [...,16,d/32],
    v_codes [...,16,d/2], v_scales [...,16,d/32])."""
    rec = np.asarray(rec, np.uint8)
    d = rec.shape[-1] // 17
    assert rec.shape[-1] == 17 * d and d in (64, 128, 256), rec.shape
    KC, VC, VSH, KS, VS = _indices(d)
    kc = rec[..., KC]
    ks = rec[..., KS]
    vs = rec[..., VS]
    vn = (rec[..., VC] >> VSH.astype(np.uint8)) & 0xF          # one 4-bit code per channel
    vc = (vn[..., 0::2] | (vn[..., 1::2] << 4)).astype(np.uint8)
    return kc, ks, vc, vs


def gather_sequence(cache: np.ndarray, block_table: np.ndarray, length: int):
    """Logical arrays of one sequence: codes [L, Hkv, d/2], scales [L, Hkv, d/32] (K then V)."""
    n_pages = -(-length // PAGE)
    recs = cache[block_table[:n_pages]]                           # [n_pages, Hkv, 17 d]
    kc, ks, vc, vs = unpack_records(recs)                         # [n_pages, Hkv, 16, .]
    def fix(a):
        a = np.moveaxis(a, 2, 1)                                  # [n_pages, 16, Hkv, .]
        return a.reshape(n_pages * PAGE, a.shape[2], a.shape[3])[:length]
    return fix(kc), fix(ks), fix(vc), fix(vs)


def used_byte_mask(d: int = 128):
    """Every one of the 17 d record bytes is addressed exactly once per full page (no padding)."""
    KC, VC, _, KS, VS = _indices(d)
    count = np.zeros(record_bytes(d), np.int64)
    np.add.at(count, KC.ravel(), 1)
    np.add.at(count, KS.ravel(), 1)
    np.add.at(count, VS.ravel(), 1)
    np.add.at(count, VC.ravel(), 1)                               # two tokens (nibbles) per V byte
    return count


# ----------------------------------------------------------------------------- Ultra-TQ comparison cache (include/uq.h)
TQ_RECORD = 2432


def unpack_tq_records(rec: np.ndarray):
    """rec uint8 [..., 2432] -> logical (k_idx [...,16,128] in 0..15, k_norm uint16 bf16 bits [...,16,4],
    v_code [...,16,128], v_scale bits [...,16,4], v_zero bits [...,16,4]), from the layout table of include/uq.h."""
    rec = np.asarray(rec, np.uint8)
    assert rec.shape[-1] == TQ_RECORD
    lead = rec.shape[:-1]
    kb = rec[..., 0:1024].reshape(*lead, 16, 64)                      # token t at 64 t, byte j = channels 2j, 2j + 1
    k_idx = np.stack([kb & 0xF, kb >> 4], axis=-1).reshape(*lead, 16, 128)
    k_norm = np.ascontiguousarray(rec[..., 1024:1152]).view(np.uint16).reshape(*lead, 16, 4)   # 1024 + 8 t + 2 g
    vw = np.ascontiguousarray(rec[..., 1152:2176]).view(np.uint32).reshape(*lead, 128, 2)      # channel c, word t >> 3
    v_code = np.zeros((*lead, 16, 128), np.uint8)
    for t in range(16):
        tt = t & 7
        nib = (tt >> 1) + 4 * (tt & 1)                                # token 2n in nibble n, token 2n + 1 in nibble n + 4
        v_code[..., t, :] = (vw[..., :, t >> 3] >> np.uint32(4 * nib)) & 0xF
    meta = np.ascontiguousarray(rec[..., 2176:2432]).view(np.uint16).reshape(*lead, 4, 2, 16)  # block g: scales, zeros
    v_scale = np.moveaxis(meta[..., :, 0, :], -1, -2)                 # [..., 16 tokens, 4 blocks]
    v_zero = np.moveaxis(meta[..., :, 1, :], -1, -2)
    return k_idx, k_norm, v_code, v_scale, v_zero


def gather_tq_sequence(cache: np.ndarray, block_table: np.ndarray, length: int):
    """Logical arrays of one sequence, each [L, Hkv, .]."""
    n_pages = -(-length // PAGE)
    parts = unpack_tq_records(cache[block_table[:n_pages]])            # [n_pages, Hkv, 16, .]
    def fix(a):
        a = np.moveaxis(a, 2, 1)
        return a.reshape(n_pages * PAGE, a.shape[2], a.shape[3])[:length]
    return tuple(fix(a) for a in parts)
