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
