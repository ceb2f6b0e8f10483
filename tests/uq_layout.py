"""Independent unpacker of the physical cache record documented in include/uq.h ("PHYSICAL
CACHE LAYOUT"), written from that description only.  Test glue: it maps a device cache image
back to the LOGICAL arrays the oracle produces (packed codes [.., 64], scale bytes [.., 4]).
Pure index arithmetic — none of the method's arithmetic lives here."""
import numpy as np

RECORD = 2176
PAGE = 16


def _k_code_index():
    """idx[t, j] = record byte holding logical K byte j (channels 2j, 2j+1) of token slot t."""
    idx = np.zeros((PAGE, 64), np.int64)
    for t in range(PAGE):
        for j in range(64):
            idx[t, j] = 64 * t + j                # logical order
    return idx


def _v_code_index():
    """(byte index, nibble shift) of V code of (token slot t, channel d)."""
    idx = np.zeros((PAGE, 128), np.int64)
    sh = np.zeros((PAGE, 128), np.int64)
    for t in range(PAGE):
        for d in range(128):
            word = 1024 + 512 * (t >> 3) + 128 * (d >> 5) + 4 * (d & 31)
            bit = 4 * (t & 7)                      # token t in bits 4(t&7)..4(t&7)+3 of the word
            idx[t, d] = word + bit // 8            # little-endian byte of the word
            sh[t, d] = bit % 8
    return idx, sh


def _k_scale_index():
    idx = np.zeros((PAGE, 4), np.int64)
    for t in range(PAGE):
        for gr in range(4):
            idx[t, gr] = 2048 + 4 * t + gr
    return idx


def _v_scale_index():
    idx = np.zeros((PAGE, 4), np.int64)
    for t in range(PAGE):
        for gr in range(4):
            idx[t, gr] = 2112 + 32 * (t >> 3) + 8 * gr + (t & 7)
    return idx


_KC = _k_code_index()
_VC, _VSH = _v_code_index()
_KS = _k_scale_index()
_VS = _v_scale_index()


def unpack_records(rec: np.ndarray):
    """rec uint8 [..., 2176] -> logical (k_codes [...,16,64], k_scales [...,16,4],
    v_codes [...,16,64], v_scales [...,16,4])."""
    rec = np.asarray(rec, np.uint8)
    kc = rec[..., _KC]
    ks = rec[..., _KS]
    vs = rec[..., _VS]
    vn = (rec[..., _VC] >> _VSH.astype(np.uint8)) & 0xF          # one 4-bit code per channel
    vc = (vn[..., 0::2] | (vn[..., 1::2] << 4)).astype(np.uint8)
    return kc, ks, vc, vs


def gather_sequence(cache: np.ndarray, block_table: np.ndarray, length: int):
    """Logical arrays of one sequence: codes [L, Hkv, 64], scales [L, Hkv, 4] (K then V)."""
    n_pages = -(-length // PAGE)
    recs = cache[block_table[:n_pages]]                           # [n_pages, Hkv, 2176]
    kc, ks, vc, vs = unpack_records(recs)                         # [n_pages, Hkv, 16, .]
    def fix(a):
        a = np.moveaxis(a, 2, 1)                                  # [n_pages, 16, Hkv, .]
        return a.reshape(n_pages * PAGE, a.shape[2], a.shape[3])[:length]
    return fix(kc), fix(ks), fix(vc), fix(vs)


def used_byte_mask():
    """Every one of the 2176 record bytes is addressed exactly once per full page (no padding)."""
    count = np.zeros(RECORD, np.int64)
    np.add.at(count, _KC.ravel(), 1)
    np.add.at(count, _KS.ravel(), 1)
    np.add.at(count, _VS.ravel(), 1)
    np.add.at(count, _VC.ravel(), 1)                              # two tokens (nibbles) per V byte
    return count
