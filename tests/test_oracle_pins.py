"""Pins P1-P9: the oracle checked against what the paper and the mathematics fix — never
against itself and never against the CUDA path.  (DESIGN.md "Pins".)"""
import ctypes
import math
import os
import subprocess

import numpy as np
import pytest
import torch

import oracle

HERE = os.path.dirname(os.path.abspath(__file__))
LEVELS = [0.0, 0.5, 1.0, 1.5, 2.0, 3.0, 4.0, 6.0]          # PAPER.md:124 (also in golden/)


def _golden():
    out = {}
    with open(os.path.join(HERE, "golden", "paper_constants.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if "=" in line:
                k, v = line.split("=")
                out[k.strip()] = v.strip()
    return out


# ----------------------------------------------------------------------------- P1 Hadamard
@pytest.mark.parametrize("d", [32, 64, 128, 256])
def test_p1_hadamard_structure(d):
    kap = oracle.kappa(d)
    assert kap == pytest.approx(d ** -0.5, rel=1e-15)
    # kappa is the CORRECTLY ROUNDED 2^(-log2(d)/2): its square brackets 1/d within 1 ulp
    assert abs(kap * kap * d - 1.0) < 4e-16
    H = np.stack([oracle.hadamard(np.eye(d)[j]) for j in range(d)], axis=1) / kap
    # entries are exactly +-1 with the Sylvester sign pattern (-1)^popcount(i&j)
    i, j = np.meshgrid(np.arange(d), np.arange(d), indexing="ij")
    sign = 1 - 2 * (np.vectorize(lambda a: bin(a).count("1"))(i & j) & 1)
    assert np.array_equal(H, sign.astype(np.float64))
    # H H^T = d I exactly (integers)
    assert np.array_equal(H @ H.T, d * np.eye(d))
    # Kronecker recursion H_{2n} = [[H_n, H_n], [H_n, -H_n]]
    h = d // 2
    assert np.array_equal(H[:h, :h], H[:h, h:]) and np.array_equal(H[:h, :h], -H[h:, h:])
    assert np.array_equal(H[:2, :2], np.array([[1.0, 1.0], [1.0, -1.0]]))


def test_p1_rotation_is_orthonormal_involution():
    rng = np.random.default_rng(0)
    for d in (64, 128, 256):
        x = rng.standard_normal(d)
        y = oracle.hadamard(x)
        assert np.linalg.norm(y) == pytest.approx(np.linalg.norm(x), rel=1e-14)
        assert np.allclose(oracle.hadamard(y), x, atol=1e-14)
        e0 = np.zeros(d)
        e0[0] = 1.0
        assert np.array_equal(oracle.hadamard(e0), np.full(d, oracle.kappa(d)))
        # (Rq).(Rk) = q.k : the identity the decode step relies on
        q = rng.standard_normal(d)
        assert np.dot(oracle.hadamard(q), y) == pytest.approx(np.dot(q, x), abs=1e-12)


# ----------------------------------------------------------------------------- P2 decode table
def test_p2_decode_table_matches_eq1():
    g = _golden()
    assert [float(v) for v in g["e2m1_levels"].split()] == LEVELS
    bias = int(g["scale_bias"])
    for byte in (0, 1, 126, 127, 128, 254):
        for code in range(16):
            mag = LEVELS[code & 7]
            want = (-mag if code & 8 else mag) * 2.0 ** (byte - bias)      # Eq.(1)
            assert oracle.dequant(code, byte) == want
    assert oracle.dequant(8, 127) == 0.0                                   # -0 decodes to 0
    assert oracle.dequant(7, 127) == 6.0 and oracle.dequant(15, 128) == -12.0


def test_p2_exact_round_trip_of_representable_values():
    # a group holding levels of F times 2^k, max level 6: m = 6*2^k, c*m = 0.936*2^k -> E = k
    rng = np.random.default_rng(1)
    for k in (-20, -3, 0, 1, 9):
        idx = rng.integers(0, 8, size=128)
        idx[::32] = 7                                    # every group contains the level 6
        sgn = rng.choice([-1.0, 1.0], size=128)
        y = sgn * np.array(LEVELS)[idx] * 2.0 ** k
        packed, scales = oracle.quantize_vector(y, 0.156)
        assert np.all(scales == 127 + k)
        assert np.array_equal(oracle.dequantize(packed, scales), y)
        codes = oracle.unpack_codes(packed)
        assert np.array_equal(codes & 7, idx)
        assert np.all((codes[idx == 0] & 8) == 0)        # zero never carries a sign (G7)


# ----------------------------------------------------------------------------- P3 brute force
def test_p3_nearest_level_brute_force():
    """For every r on a grid holding all midpoints, the encoder's code is the argmin of
    |r - level| over the 8 magnitudes, ties to the even code, clamp above 6."""
    lev = np.array(LEVELS)
    for E in (-5, -1, 0, 3):
        for n in range(0, 10 * 1024 + 1):
            r = n / 1024.0
            dist = np.abs(r - lev)
            best = np.flatnonzero(dist == dist.min())
            want = int(best[0]) if len(best) == 1 else int([b for b in best if b % 2 == 0][0])
            y = math.ldexp(r, E)
            assert oracle.e2m1_encode(y, E) == want, (r, E)
            got_neg = oracle.e2m1_encode(-y, E)
            assert got_neg == (want | 8 if want else 0)
    # all 16 codes x several scales: encode(decode(code)) is the identity (except -0 -> +0)
    for byte in (100, 127, 140):
        for code in range(16):
            v = oracle.dequant(code, byte)
            assert oracle.e2m1_encode(v, byte - 127) == (0 if code == 8 else code)


# ----------------------------------------------------------------------------- P4 thresholds
def test_p4_scale_thresholds():
    c = float(np.float32(0.156))                       # the constant reaches the rule as a float
    assert c == 0.15600000321865082
    for k in range(-6, 7):
        thr = 2.0 ** (k - 0.5) / c                     # E switches from k-1 to k here
        lo, hi = np.nextafter(thr, 0), np.nextafter(thr, np.inf)
        # thr itself is irrational-adjacent; step a few ulps each side to be independent of
        # how 2^(k-0.5) rounded
        for _ in range(4):
            lo, hi = np.nextafter(lo, 0), np.nextafter(hi, np.inf)
        assert oracle.scale_exponent(c, lo) == k - 1
        assert oracle.scale_exponent(c, hi) == k
        assert oracle.scale_exponent(c, thr * 1.3) == k
    assert oracle.scale_exponent(c, 0.0) == -127
    assert oracle.scale_exponent(c, 1e-300) == -127 and oracle.scale_exponent(c, 1e300) == 127
    # equals round(log2(c*m)) evaluated in extended precision for random m
    rng = np.random.default_rng(2)
    for m in np.exp(rng.uniform(-40, 40, 2000)):
        want = int(np.rint(np.log2(np.longdouble(c) * np.longdouble(m))))
        assert oracle.scale_exponent(c, m) == want
    # invariant: the group max lands in [4.5327, 9.0655) grid units (so it encodes to 4 or 6)
    for m in np.exp(rng.uniform(-10, 10, 500)):
        E = oracle.scale_exponent(c, m)
        r = m / 2.0 ** E
        assert 2.0 ** -0.5 / c * 0.999999 <= r < 2.0 ** 0.5 / c * 1.000001
        assert oracle.e2m1_encode(m, E) in (6, 7)


# ----------------------------------------------------------------------------- P5 fingerprints
def test_p5_statistical_fingerprints():
    """i.i.d. N(0,1) groups, c = 0.156 (values from the survey's Monte-Carlo, SURVEY.md §8c P5,
    an independent numpy prototype): E histogram, clamp rate, code histogram, relative MSE."""
    rng = np.random.default_rng(3)
    n = 20000
    y = rng.standard_normal((n, 128))
    packs = [oracle.quantize_vector(v, float(np.float32(0.156))) for v in y]
    packed = np.stack([p[0] for p in packs])
    scales = np.stack([p[1] for p in packs])
    frac125 = np.mean(scales == 125)
    frac126 = np.mean(scales == 126)
    assert frac125 == pytest.approx(0.468, abs=0.01) and frac126 == pytest.approx(0.532, abs=0.01)
    assert np.mean((scales < 125) | (scales > 126)) < 2e-3
    E = np.repeat(scales.astype(np.int64) - 127, 32, axis=1)
    r = np.abs(y) / 2.0 ** E
    assert np.mean(r > 6) == pytest.approx(0.0554, abs=0.003)
    codes = oracle.unpack_codes(packed)
    hist = np.bincount((codes & 7).ravel(), minlength=8) / codes.size
    want = [0.0757, 0.1479, 0.1377, 0.1229, 0.1509, 0.1403, 0.1222, 0.1024]
    assert np.allclose(hist, want, atol=0.004)
    deq = oracle.dequantize(packed, scales)
    rel_mse = np.mean((deq - y) ** 2) / np.mean(y ** 2)
    assert rel_mse == pytest.approx(0.0178, abs=0.001)


# ----------------------------------------------------------------------------- P6 sizes
def test_p6_sizes():
    g = _golden()
    packed, scales = oracle.quantize_vector(np.ones(128), 0.156)
    assert packed.nbytes + scales.nbytes == 68
    per_group = (packed.nbytes + scales.nbytes) // (128 // int(g["group_size"]))
    assert per_group == int(g["bytes_per_group"])
    assert per_group * 8 / int(g["group_size"]) == float(g["bits_per_element"])


# ----------------------------------------------------------------------------- P7 the two constants
def _mse_for_c(y, c, power_of_two):
    """Eq.(2) objective E[(z - s q(z/s))^2] with s = c*m (continuous) or 2^round(log2(c*m)),
    evaluated with an INDEPENDENT numpy nearest-level quantiser (argmin over the level set)."""
    lev = np.array([-6, -4, -3, -2, -1.5, -1, -0.5, 0, 0.5, 1, 1.5, 2, 3, 4, 6], np.float64)
    m = np.abs(y).max(axis=1, keepdims=True)
    s = c * m
    if power_of_two:
        s = 2.0 ** np.rint(np.log2(s))
    z = y / s
    q = lev[np.abs(z[..., None] - lev).argmin(axis=-1)]
    return np.mean((y - s * q) ** 2)


def test_p7_paper_constants_fix_the_reading_of_round():
    """PAPER.md:128 gives c = 0.156 as the MSE optimum of Eq.(2); PAPER.md:333 calls 0.195 "the
    power-of-two-optimal value".  With round-to-nearest in E = round(log2(c m)) the power-of-two
    optimum on Gaussian groups sits at ~0.196 (floor would give ~0.28, ceil ~0.14) and the
    continuous-scale optimum at ~0.16 — so "round" is round-to-nearest (reading G4)."""
    g = _golden()
    rng = np.random.default_rng(4)
    y = rng.standard_normal((12000, 32))
    cs = np.arange(0.10, 0.32, 0.004)
    cont = [_mse_for_c(y, c, False) for c in cs]
    p2 = [_mse_for_c(y, c, True) for c in cs]
    c_cont = cs[int(np.argmin(cont))]
    c_p2 = cs[int(np.argmin(p2))]
    assert abs(c_cont - float(g["c_default"])) < 0.02
    assert abs(c_p2 - float(g["c_power_of_two_optimal"])) < 0.02
    # and the ORACLE's rule reproduces the power-of-two objective at the paper's two constants
    for c in (0.156, 0.195):
        deq = np.stack([oracle.dequantize(*oracle.quantize_vector(np.tile(v, 4), c))[:32] for v in y[:3000]])
        mse_oracle = np.mean((deq - y[:3000]) ** 2)
        assert mse_oracle == pytest.approx(_mse_for_c(y[:3000], c, True), rel=1e-9)


def test_p7_c_equal_one_uses_no_shrinkage():
    # c = 1.0 is "raw absmax with no shrinkage": the group max maps near 1.0
    rng = np.random.default_rng(5)
    y = rng.standard_normal(128)
    packed, scales = oracle.quantize_vector(y, 1.0)
    codes = oracle.unpack_codes(packed) & 7
    assert codes.max() <= 3                              # nothing above 1.5 grid units is used


# ----------------------------------------------------------------------------- P11 the Eq.(2) objective (O11)
def _bf16_bits(a):
    return (torch.from_numpy(np.asarray(a, np.float32)).to(torch.bfloat16).view(torch.uint16).numpy())


@pytest.mark.parametrize("pow2", [False, True])
def test_p11_objective_equals_an_independent_numpy_quantiser(pow2):
    """oracle.calib_sq_err without rotation against _mse_for_c above (argmin over the level set, numpy log2 /
    rint for the exponent): the same mean squared error for every c of a grid (a tie between two levels costs
    the same whichever is taken)."""
    rng = np.random.default_rng(21)
    bits = _bf16_bits(rng.standard_normal((400, 128)) * np.exp(rng.standard_normal((400, 1))))
    y = oracle.bf16_to_double(bits)
    cs = np.array([0.1, 0.14, 0.156, 0.17, 0.195, 0.25, 0.4, 1.0], np.float32)
    sq, nrm = oracle.calib_sq_err(bits, cs, rotate=False, pow2=pow2)
    assert nrm == pytest.approx(float((y ** 2).sum()), rel=1e-13)
    for j, c in enumerate(cs):
        ref = _mse_for_c(y.reshape(-1, 32), float(c), pow2) * y.size
        assert sq[j] == pytest.approx(ref, rel=1e-10), (pow2, c)


def test_p11_exactly_representable_inputs_have_zero_error_and_rotation_keeps_the_norm():
    rng = np.random.default_rng(22)
    lev = np.array(LEVELS + [-v for v in LEVELS[1:]])
    e = rng.integers(-6, 7, (64, 4))
    x = lev[rng.integers(0, 15, (64, 4, 32))] * 2.0 ** e[..., None]
    x[:, :, 0] = 6.0 * 2.0 ** e                              # group max 6 * 2^e: E = e at c = 0.156 (0.936 * 2^e)
    bits = _bf16_bits(x.reshape(64, 128))
    sq, nrm = oracle.calib_sq_err(bits, np.array([0.156], np.float32), rotate=False, pow2=True)
    assert sq[0] == 0.0 and nrm == float((x ** 2).sum())
    # rotation: H/sqrt(d) is orthogonal, so sum z^2 is the same with and without it
    g = _bf16_bits(rng.standard_normal((50, 128)))
    _, n0 = oracle.calib_sq_err(g, np.array([0.156], np.float32), rotate=False)
    _, n1 = oracle.calib_sq_err(g, np.array([0.156], np.float32), rotate=True)
    assert n1 == pytest.approx(n0, rel=1e-13)


def test_p11_paper_ordering_of_the_constants_on_rotated_vectors():
    """PAPER.md:128, :333 and Table 5: on rotated keys the MSE optimum of Eq.(2) is 0.156, the power-of-two
    optimum 0.195, and c = 1.0 is far worse than either — here on rotated unit-sphere-like vectors (Fig. 2)."""
    g = _golden()
    rng = np.random.default_rng(23)
    x = rng.standard_normal((3000, 128))
    x[:, rng.choice(128, 3, replace=False)] *= 8.0           # outlier channels: the rotation spreads them
    bits = _bf16_bits(x)
    cs = np.arange(0.10, 0.32, 0.004).astype(np.float32)
    cont, _ = oracle.calib_sq_err(bits, cs, rotate=True, pow2=False)
    p2, _ = oracle.calib_sq_err(bits, cs, rotate=True, pow2=True)
    assert abs(float(cs[int(np.argmin(cont))]) - float(g["c_default"])) < 0.02
    assert abs(float(cs[int(np.argmin(p2))]) - float(g["c_power_of_two_optimal"])) < 0.02
    three, _ = oracle.calib_sq_err(bits, np.array([0.156, 0.195, 1.0], np.float32), rotate=True, pow2=False)
    assert three[0] < three[1] < three[2] and three[2] > 5 * three[0]


def _lloyd_max_gaussian_magnitudes():
    """Lloyd's algorithm for a 16-level quantiser of N(0,1) (the published fixed-point iteration: thresholds =
    midpoints, centroids = conditional means), run here on the closed-form Gaussian integrals; returns the 8
    positive centroids."""
    from scipy.stats import norm
    c = np.linspace(0.1, 2.5, 8)
    for _ in range(500):
        t = np.concatenate([[0.0], 0.5 * (c[:-1] + c[1:]), [np.inf]])
        c = (norm.pdf(t[:-1]) - norm.pdf(t[1:])) / (norm.cdf(t[1:]) - norm.cdf(t[:-1]))
    return c


def test_p11_other_codebooks_and_the_fixed_scale():
    """scale_mode 2 (s = c, no absmax) and `levels` against numpy restatements, on the distribution of Fig. 2
    (PAPER.md:118-120): coordinates of random unit vectors, d = 64, 128, 256.  The analytical Lloyd-Max codebook at
    the fixed scale 1/sqrt(d) has a lower MSE than absmax-scaled FP4 at any of the paper's constants (Fig. 2b: "FP4
    has higher MSE than analytical Lloyd-Max"), and c = 0.156 beats c = 1.0 by a wide margin (Table 5)."""
    lm = _lloyd_max_gaussian_magnitudes()
    assert lm[0] == pytest.approx(0.1284, abs=2e-3) and lm[-1] == pytest.approx(2.7326, abs=2e-3)   # textbook table
    rng = np.random.default_rng(31)
    for d in (64, 128, 256):
        u = rng.standard_normal((512 * 128 // d, d))
        u /= np.linalg.norm(u, axis=1, keepdims=True)
        bits = _bf16_bits(u.reshape(-1, 128))
        y = oracle.bf16_to_double(bits)
        one = lambda c, mode, lev=None: oracle.calib_sq_err(bits, np.array([c], np.float32), rotate=False,
                                                            scale_mode=mode, levels=lev)[0][0] / y.size
        mse_lm = one(d ** -0.5, 2, lm)
        mse_opt, mse_195, mse_one = one(0.156, 0), one(0.195, 0), one(1.0, 0)
        mse_int4 = one(1.0 / 7.0, 0, np.arange(8.0))
        assert mse_lm < min(mse_opt, mse_195, mse_one)
        assert mse_opt < mse_195 < mse_one and mse_one > 5 * mse_opt
        # numpy restatements: the fixed-scale Lloyd-Max quantiser, and absmax INT4 (grid m/7 * {-7..7})
        s = np.float64(np.float32(d ** -0.5))
        lev = np.concatenate([-lm[::-1], lm]).astype(np.float32).astype(np.float64)
        q = lev[np.abs(y[..., None] / s - lev).argmin(axis=-1)]
        assert mse_lm == pytest.approx(np.mean((y - s * q) ** 2), rel=1e-10)
        yg = y.reshape(-1, 32)
        sg = np.float64(np.float32(1.0 / 7.0)) * np.abs(yg).max(axis=1, keepdims=True)
        qi = np.clip(np.floor(np.abs(yg) / sg + 0.5), 0, 7) * np.sign(yg)
        assert mse_int4 == pytest.approx(np.mean((yg - sg * qi) ** 2), rel=1e-9)


# ----------------------------------------------------------------------------- P8 library casts
@pytest.fixture(scope="module")
def libcasts():
    inc = "/usr/local/cuda/include"
    if not os.path.exists(os.path.join(inc, "cuda_fp4.h")):
        pytest.skip("CUDA toolkit headers not present")
    src = os.path.join(HERE, "helpers", "cuda_host_casts.cpp")
    so = os.path.join(HERE, "helpers", "cuda_host_casts.so")
    if not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
        subprocess.run(["g++", "-O1", "-shared", "-fPIC", f"-I{inc}", "-o", so, src], check=True)
    lib = ctypes.CDLL(so)
    for f in (lib.lib_e2m1, lib.lib_e4m3):
        f.argtypes = [ctypes.c_double]
        f.restype = ctypes.c_ubyte
    return lib


def test_p8_e2m1_matches_cuda_host_routine(libcasts):
    rng = np.random.default_rng(6)
    xs = np.concatenate([np.arange(-8, 8, 1 / 64.0), rng.standard_normal(4000) * 3,
                         [0.25, 0.75, 1.25, 1.75, 2.5, 3.5, 5.0, 6.0, 1e9, -1e9]])
    for x in xs:
        got = oracle.e2m1_encode(float(x), 0)
        ref = libcasts.lib_e2m1(float(x))
        if (ref & 7) == 0:
            ref = 0                                      # G7: we store canonical +0, CUDA keeps the sign
        assert got == ref, x


def test_p8_e4m3_matches_torch_and_cuda_host_routine(libcasts):
    rng = np.random.default_rng(7)
    xs = np.concatenate([rng.standard_normal(5000) * 4, rng.standard_normal(2000) * 0.01,
                         np.arange(0, 2 ** -5, 2 ** -12), [2 ** -10, 1.5 * 2 ** -9, 447.9, 448.0,
                                                         449.0, 463.9, 1e4, -1e4, 0.0, 2 ** -6]])
    t = torch.tensor(xs, dtype=torch.float64).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    for x, tb in zip(xs, t):
        got = oracle.e4m3_encode(float(x))
        ref = libcasts.lib_e4m3(float(x))
        if (ref & 0x7F) == 0:
            ref = 0
        assert got == ref, x
        if abs(x) < 464 and (tb & 0x7F) != 0:
            assert got == tb, x                          # torch saturates to NaN beyond 464; we clamp
    # all 256 bytes decode per the closed form, and encode(decode(b)) == b
    for b in range(256):
        if (b & 0x7F) == 0x7F:
            continue                                     # NaN pattern: never produced
        v = oracle.e4m3_decode(b)
        ef, mf = (b >> 3) & 15, b & 7
        want = (mf / 8.0) * 2.0 ** -6 if ef == 0 else (1 + mf / 8.0) * 2.0 ** (ef - 7)
        assert abs(v) == want
        assert oracle.e4m3_encode(v) == (0 if (b & 0x7F) == 0 else b)
    assert oracle.e4m3_decode(0x7E) == 448.0


# ----------------------------------------------------------------------------- P9 attention
def _random_cache(rng, L, Hkv, d=128):
    k = rng.standard_normal((L, Hkv, d)).astype(np.float32)
    v = rng.standard_normal((L, Hkv, d)).astype(np.float32)
    kb = torch.from_numpy(k).to(torch.bfloat16).view(torch.uint16).numpy()
    vb = torch.from_numpy(v).to(torch.bfloat16).view(torch.uint16).numpy()
    return kb, vb


def test_p9_attention_closed_forms():
    rng = np.random.default_rng(8)
    Hq, Hkv, d = 8, 2, 128
    kb, vb = _random_cache(rng, 37, Hkv)
    kc, ks, vc, vs = oracle.encode_kv(kb, vb)
    qb = torch.from_numpy(rng.standard_normal((Hq, d)).astype(np.float32)).to(torch.bfloat16)
    q8 = oracle.encode_q(qb.view(torch.uint16).numpy())
    out, p = oracle.attention(q8, kc, ks, vc, vs, Hq, Hkv, return_probs=True)
    assert np.allclose(p.sum(axis=1), 1.0, atol=1e-14)               # rows of P sum to 1
    # L = 1: out = vhat_0
    out1 = oracle.attention(q8, kc[:1], ks[:1], vc[:1], vs[:1], Hq, Hkv)
    vhat = oracle.dequantize(vc, vs)
    for h in range(Hq):
        assert np.array_equal(out1[h], vhat[0, h // (Hq // Hkv)])
    # all keys equal: out = mean of vhat
    kc_eq = np.repeat(kc[:1], 37, axis=0)
    ks_eq = np.repeat(ks[:1], 37, axis=0)
    out_eq = oracle.attention(q8, kc_eq, ks_eq, vc, vs, Hq, Hkv)
    for h in range(Hq):
        assert np.allclose(out_eq[h], vhat[:, h // (Hq // Hkv)].mean(axis=0), atol=1e-13)
    # L = 0: zeros
    assert np.array_equal(oracle.attention(q8, kc[:0], ks[:0], vc[:0], vs[:0], Hq, Hkv), np.zeros((Hq, d)))
    # equals torch SDPA in float64 on the dequantised tensors (library routine)
    khat = oracle.dequantize(kc, ks)
    qd = np.array([[oracle.e4m3_decode(int(b)) for b in row] for row in q8])
    G = Hq // Hkv
    tq = torch.from_numpy(qd)[None, :, None, :]
    tk = torch.from_numpy(khat).permute(1, 0, 2).repeat_interleave(G, dim=0)[None]
    tv = torch.from_numpy(vhat).permute(1, 0, 2).repeat_interleave(G, dim=0)[None]
    ref = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv)[0, :, 0].numpy()
    assert np.allclose(out, ref, atol=1e-12)
    # the GQA map is contiguous groups: head h <-> kv head h // G (a swapped map would differ)
    assert not np.allclose(out[0], ref[G], atol=1e-6)


def test_p9_split_merge_identity_and_page_permutation():
    """A split-K evaluation with the merge formula of include/uq.h equals the unsplit oracle."""
    rng = np.random.default_rng(9)
    Hq, Hkv, d, L = 4, 1, 128, 203
    kb, vb = _random_cache(rng, L, Hkv)
    kc, ks, vc, vs = oracle.encode_kv(kb, vb)
    q8 = oracle.encode_q(torch.from_numpy(rng.standard_normal((Hq, d)).astype(np.float32))
                         .to(torch.bfloat16).view(torch.uint16).numpy())
    full = oracle.attention(q8, kc, ks, vc, vs, Hq, Hkv)
    khat, vhat = oracle.dequantize(kc, ks)[:, 0], oracle.dequantize(vc, vs)[:, 0]
    qd = np.array([[oracle.e4m3_decode(int(b)) for b in row] for row in q8])
    z = (qd @ khat.T) / math.sqrt(d)
    bounds = [0, 16, 64, 64, 160, L]                    # includes an empty split
    ms, ls, accs = [], [], []
    for a, b in zip(bounds[:-1], bounds[1:]):
        if a == b:
            ms.append(np.full(Hq, -np.inf)); ls.append(np.zeros(Hq)); accs.append(np.zeros((Hq, d)))
            continue
        m = z[:, a:b].max(axis=1)
        e = np.exp(z[:, a:b] - m[:, None])
        ms.append(m); ls.append(e.sum(axis=1)); accs.append(e @ vhat[a:b])
    M = np.max(np.stack(ms), axis=0)
    w = [np.exp(m - M) for m in ms]
    num = sum(wi[:, None] * ai for wi, ai in zip(w, accs))
    den = sum(wi * li for wi, li in zip(w, ls))
    assert np.allclose(num / den[:, None], full, atol=1e-12)
    # without quantisation (Rq).(Rk) = q.k: dense attention is rotation invariant
    qf = rng.standard_normal((Hq, d)); kf = rng.standard_normal((L, 1, d)); vf = rng.standard_normal((L, 1, d))
    a = oracle.attention_dense(qf, kf, vf)
    qr = np.stack([oracle.hadamard(x) for x in qf])
    kr = np.stack([oracle.hadamard(x) for x in kf[:, 0]])[:, None]
    assert np.allclose(oracle.attention_dense(qr, kr, vf), a, atol=1e-12)


def test_k_is_rotated_and_v_is_not():
    """Alg. 1 l.1: "rotate keys; V unrotated" — V codes equal direct quantisation of V, K codes
    equal quantisation of R*K, and nothing per-token is stored besides codes + group scales."""
    rng = np.random.default_rng(10)
    kb, vb = _random_cache(rng, 5, 2)
    kc, ks, vc, vs = oracle.encode_kv(kb, vb)
    for t in range(5):
        for h in range(2):
            x = oracle.bf16_to_double(vb[t, h])
            p, s = oracle.quantize_vector(x, float(np.float32(0.156)))
            assert np.array_equal(p, vc[t, h]) and np.array_equal(s, vs[t, h])
            y = oracle.hadamard(oracle.bf16_to_double(kb[t, h]))
            p, s = oracle.quantize_vector(y, float(np.float32(0.156)))
            assert np.array_equal(p, kc[t, h]) and np.array_equal(s, ks[t, h])
    assert kc.shape[-1] + ks.shape[-1] == 68 and vc.shape[-1] + vs.shape[-1] == 68


# ----------------------------------------------------------------------------- P12 query encoder (Alg. 1 l.6)
@pytest.mark.parametrize("d", [64, 128, 256])
def test_p12_encode_q_is_e4m3_of_the_rotated_query_element_for_element(d):
    """`encode_q` (Alg. 1 l.6: "Q <- R*Q; Q <- cast_fp8_e4m3(Q)") against its parts, each pinned on its own
    (P1 the rotation, P8 the cast): byte i of row n == e4m3_encode(hadamard(bf16_to_double(row n))[i]), on random rows,
    one-hot rows (every rotated element +-kappa*x: a missing rotation or a wrong kappa changes every byte), rows that
    saturate (|Rq| > 448), rows with a single non-zero in the LAST channel (element order / transposed index), huge,
    tiny and zero rows.  Then against the library cast (torch float8_e4m3fn, P8) of an independently rotated query
    (numpy float64 matmul with the Sylvester matrix built here) wherever that cast is defined (|y| < 464)."""
    rng = np.random.default_rng(120 + d)
    rows = [rng.standard_normal(d) for _ in range(6)]
    e = np.zeros(d); e[0] = 3.0; rows.append(e)                       # one-hot, first channel: all +3*kappa
    e = np.zeros(d); e[d - 1] = -2.5; rows.append(e)                  # one-hot, last channel: signs follow popcount(i & (d-1))
    e = np.zeros(d); e[5] = 1.0; e[d // 2 + 1] = -7.0; rows.append(e)
    rows.append(np.full(d, 448.0 / math.sqrt(d) * 1.5))               # rotated element 0 = 672 > 448: saturates, the rest 0
    rows.append(rng.standard_normal(d) * 300.0)                       # many elements beyond 448
    rows.append(rng.standard_normal(d) * 1e-3)                        # subnormal E4M3 range
    rows.append(rng.standard_normal(d) * 1e20)
    rows.append(rng.standard_normal(d) * 1e-20)
    rows.append(np.zeros(d))
    x = torch.from_numpy(np.stack(rows).astype(np.float32)).to(torch.bfloat16)
    bits = x.view(torch.uint16).numpy()
    got = oracle.encode_q(bits)
    assert got.shape == bits.shape and got.dtype == np.uint8
    # (a) element for element against the pinned parts
    for n in range(bits.shape[0]):
        y = oracle.hadamard(oracle.bf16_to_double(bits[n]))
        want = np.array([oracle.e4m3_encode(float(v)) for v in y], np.uint8)
        assert np.array_equal(got[n], want), f"row {n}"
    # (b) against an independent rotation + the library cast
    i, j = np.meshgrid(np.arange(d), np.arange(d), indexing="ij")
    H = 1.0 - 2.0 * (np.vectorize(lambda a: bin(a).count("1"))(i & j) & 1)
    y_ind = (H @ x.double().numpy().T).T * (2.0 ** (-0.5 * math.log2(d)))
    ok = np.abs(y_ind) < 448.0
    lib = torch.from_numpy(y_ind).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    lib = np.where((lib & 0x7F) == 0, 0, lib)                          # -0 is never stored (reading G7)
    # y_ind carries float64 rounding of the kappa product only when d is an odd power of two; a value within 1e-12
    # relative of an E4M3 rounding boundary could flip there, everything else must agree exactly
    mism = (got != lib) & ok
    assert mism.sum() == 0, f"{int(mism.sum())} bytes differ from the library cast"
    sat = np.abs(y_ind) >= 448.0
    assert np.all((got[sat] & 0x7F) == 0x7E)                           # saturation to +-448 (reading G9)
    assert sat.sum() >= d // 4                                         # the saturating rows really saturate
    # one-hot rows: every byte is the same magnitude, signs follow the Sylvester pattern of that column
    mag = got[6] & 0x7F
    assert len(set(mag.tolist())) == 1 and np.all(got[6] < 0x80)
    pop = np.array([bin(a & (d - 1)).count("1") & 1 for a in range(d)])
    assert np.array_equal(got[7] >> 7, 1 - pop)                        # x = -2.5 e_{d-1}: y_i = -2.5 kappa (-1)^popcount(i)


# ----------------------------------------------------------------------------- P13 unquantised attention (context figure)
def test_p13_attention_dense_against_sdpa_and_closed_forms():
    """`attention_dense` (textbook softmax attention over unquantised doubles; feeds only the context figure
    quant_error_vs_bf16) against torch float64 SDPA (library routine) with GQA, a non-default scale, and the closed
    forms: L = 1 -> out = v_0; all keys equal -> the mean of v; one dominant key -> its value; L = 0 -> zeros."""
    rng = np.random.default_rng(13)
    Hq, Hkv, d, L = 12, 3, 64, 91
    G = Hq // Hkv
    q = rng.standard_normal((Hq, d)); k = rng.standard_normal((L, Hkv, d)); v = rng.standard_normal((L, Hkv, d))
    for scale in (None, 0.3):
        out = oracle.attention_dense(q, k, v, scale)
        tq = torch.from_numpy(q)[None, :, None, :]
        tk = torch.from_numpy(k).permute(1, 0, 2).repeat_interleave(G, dim=0)[None]
        tv = torch.from_numpy(v).permute(1, 0, 2).repeat_interleave(G, dim=0)[None]
        ref = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv, scale=scale)[0, :, 0].numpy()
        assert np.allclose(out, ref, atol=1e-13)
        assert not np.allclose(out[0], ref[G], atol=1e-6)              # contiguous GQA groups, not interleaved
    out1 = oracle.attention_dense(q, k[:1], v[:1])
    for h in range(Hq):
        assert np.array_equal(out1[h], v[0, h // G])
    keq = np.repeat(k[:1], L, axis=0)
    oeq = oracle.attention_dense(q, keq, v)
    for h in range(Hq):
        assert np.allclose(oeq[h], v[:, h // G].mean(axis=0), atol=1e-13)
    kd = k.copy(); kd[17] = 0.0
    qd = np.zeros((Hq, d)); qd[:, 3] = 1.0
    kd[:, :, 3] = 0.0; kd[17, :, 3] = 4000.0                           # logit 4000/8 = 500 above all others
    od = oracle.attention_dense(qd, kd, v)
    for h in range(Hq):
        assert np.allclose(od[h], v[17, h // G], atol=1e-13)
    assert np.array_equal(oracle.attention_dense(q, k[:0], v[:0]), np.zeros((Hq, d)))


# ----------------------------------------------------------------------------- P14 comparison caches (FP8 KV / BF16 KV)
def test_p14_fp8_kv_cast_and_attention_are_the_pinned_parts():
    """The FP8-KV comparison cache ("hardware FP8 KV"; DESIGN reading G19): `cast_e4m3` == e4m3_encode of the
    bf16 value element for element (P8 pins that scalar) == the library cast (torch float8_e4m3fn) below 448, saturating
    above, no -0; `e4m3_to_double` == the closed form for all 256 bytes; `attention_fp8kv` == float64 SDPA over the
    library-decoded tensors; `attention_bf16kv` == float64 SDPA over the bf16 values."""
    rng = np.random.default_rng(14)
    x = np.concatenate([rng.standard_normal(4000) * 3, rng.standard_normal(300) * 300, [0.0, -0.0, 448.0, -448.0, 464.0, 1e30,
                        -1e30, 2.0 ** -9, 2.0 ** -10, -(2.0 ** -10), 1.5 * 2.0 ** -9, 2.0 ** -6, 0.0175]])
    xb = torch.from_numpy(x.astype(np.float32)).to(torch.bfloat16)
    bits = xb.view(torch.uint16).numpy()
    got = oracle.cast_e4m3(bits)
    want = np.array([oracle.e4m3_encode(float(v)) for v in oracle.bf16_to_double(bits)], np.uint8)
    assert np.array_equal(got, want)
    xv = xb.double().numpy()
    ok = np.abs(xv) < 448.0
    lib = xb.to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    lib = np.where((lib & 0x7F) == 0, 0, lib)
    assert np.array_equal(got[ok], lib[ok])
    assert np.all((got[~ok] & 0x7F) == 0x7E) and (~ok).sum() > 20
    assert not np.any(got == 0x80)
    allb = np.arange(256, dtype=np.uint8)
    dec = oracle.e4m3_to_double(allb)
    ef, mf = (allb >> 3) & 0xF, allb & 7
    closed = np.where(ef == 0, mf * 2.0 ** -9, (1 + mf / 8.0) * 2.0 ** (ef.astype(np.float64) - 7)) * np.where(allb & 0x80, -1.0, 1.0)
    assert np.array_equal(dec, closed)
    # attention over the two comparison caches
    Hq, Hkv, d, L = 8, 2, 128, 77
    G = Hq // Hkv
    q = torch.from_numpy(rng.standard_normal((Hq, d)).astype(np.float32)).to(torch.bfloat16)
    k = torch.from_numpy(rng.standard_normal((L, Hkv, d)).astype(np.float32) * 2).to(torch.bfloat16)
    v = torch.from_numpy(rng.standard_normal((L, Hkv, d)).astype(np.float32)).to(torch.bfloat16)
    qb, kb, vb = (t.view(torch.uint16).numpy() for t in (q, k, v))
    def sdpa(tq, tk, tv):
        tq = tq[None, :, None, :]
        tk = tk.permute(1, 0, 2).repeat_interleave(G, dim=0)[None]
        tv = tv.permute(1, 0, 2).repeat_interleave(G, dim=0)[None]
        return torch.nn.functional.scaled_dot_product_attention(tq, tk, tv)[0, :, 0].numpy()
    out8, q8, k8, v8 = oracle.attention_fp8kv(qb, kb, vb)
    f8 = lambda t: t.to(torch.float8_e4m3fn).double()
    assert np.allclose(out8, sdpa(f8(q), f8(k), f8(v)), atol=1e-12)
    assert np.array_equal(k8, k.to(torch.float8_e4m3fn).view(torch.uint8).numpy() * (np.abs(k.double().numpy()) >= 2.0 ** -10))
    out16 = oracle.attention_bf16kv(qb, kb, vb)
    assert np.allclose(out16, sdpa(q.double(), k.double(), v.double()), atol=1e-12)
    assert not np.allclose(out8, out16, atol=1e-3)                  # the two caches really differ


# ----------------------------------------------------------------------------- P15-P17 Ultra-TQ (Alg. 2)
def _bf16_bits_of(x):
    return torch.from_numpy(np.asarray(x, np.float32)).to(torch.bfloat16).view(torch.uint16).numpy()


def test_p15_bf16_rne_is_the_library_rounding():
    """`ultra_tq.bf16_rne` (written from the definition: quantum 2^(e-7), ties to even) == the library cast float32 ->
    bfloat16 on random magnitudes, on exact ties (odd / even neighbours) and at binade boundaries."""
    from oracle import ultra_tq as T
    rng = np.random.default_rng(15)
    x = (rng.standard_normal(200000) * np.exp(rng.uniform(-30, 30, 200000))).astype(np.float32)
    ties = np.array([1.0 + 2.0 ** -8, 1.0 + 3 * 2.0 ** -8, 1.0 + 2.0 ** -8 + 2.0 ** -20, 2.0 - 2.0 ** -8, 255.5, 256.5, -1.00390625,
                     0.0, 3.0e-5, 65504.0], np.float32)
    x = np.concatenate([x, ties, -ties])
    want = torch.from_numpy(x).to(torch.bfloat16).double().numpy()
    assert np.array_equal(T.bf16_rne(x.astype(np.float64)), want)
    assert T.bf16_rne(np.array([1.0 + 2.0 ** -8]))[0] == 1.0 and T.bf16_rne(np.array([1.0 + 3 * 2.0 ** -8]))[0] == 1.0 + 2.0 ** -6
    assert np.array_equal(T.bf16_bits(want), torch.from_numpy(x).to(torch.bfloat16).view(torch.uint16).numpy())


def test_p16_ultra_tq_encoders_closed_forms_and_brute_force():
    """Alg. 2 l.1-4.  K: a one-hot key a e_0 rotates to a/sqrt(d) (+-1 pattern of Hadamard row 0 = all +): every block has
    norm a sqrt(32/d) and every coordinate u = 1/sqrt(32) -> the codebook entry nearest to 0.17678 (index 11 of the
    input table), a e_1 alternates signs (indices 11, 4); the index is the brute-force nearest entry (python floats) and
    the stored norm the bf16 of the plain l2 norm; reconstruction error of Gaussian keys is that of a 16-level
    Lloyd-Max quantiser (relative MSE 0.0095 +- 15 %).  V: a block zero + scale * (codes) with bf16 scale / zero comes back
    exactly; a constant block has scale 0, codes 0 and decodes exactly; |v - vhat| <= scale/2 + one bf16 rounding."""
    from oracle import ultra_tq as T
    from paper_2606_20474_b200 import workloads as W
    cb = np.asarray(W.TQ_CODEBOOK, np.float32)
    assert np.all(np.diff(cb) > 0) and np.allclose(cb, -cb[::-1])
    d = 128
    for j, want in ((0, [11] * 4), (1, [11, 4] * 2)):
        k = np.zeros((1, d), np.float32); k[0, j] = 3.0
        idx, norm = T.encode_k(_bf16_bits_of(k), cb)
        assert np.array_equal(norm[0], T.bf16_rne(np.full(4, 3.0 * np.sqrt(32.0 / d))))
        assert list(idx[0, :4]) == want and set(idx[0]) <= {4, 11}
    rng = np.random.default_rng(16)
    kb = _bf16_bits_of(rng.standard_normal((64, d)) * np.exp(rng.uniform(-3, 3, (64, 1))))
    idx, norm = T.encode_k(kb, cb)
    x = np.stack([oracle.hadamard(r) for r in oracle.bf16_to_double(kb)])
    for r in range(0, 64, 7):                                  # brute force, scalar python arithmetic
        for g in range(4):
            blk = [float(v) for v in x[r, 32 * g:32 * g + 32]]
            n2 = 0.0
            for v in blk:
                n2 = n2 + v * v
            ns = float(T.bf16_rne(np.array([n2 ** 0.5]))[0])
            assert ns == norm[r, g]
            for c in range(32):
                u = blk[c] / ns
                best = min(range(16), key=lambda i: (abs(u - float(cb[i])), i))
                assert best == idx[r, 32 * g + c]
    kh = T.dequant_k(idx, norm, cb)
    rel = float(((kh - x) ** 2).sum() / (x ** 2).sum())
    assert 0.0080 < rel < 0.0110, rel                          # 16-level Lloyd-Max of a Gaussian: 0.0095
    # V
    scale, zero = 0.375, -2.5                                  # bf16 values
    codes = rng.integers(0, 16, (5, d)); codes[:, ::32] = 0; codes[:, 1::32] = 15
    v = zero + scale * codes                                   # exact in bf16 (<= 8 significant bits)
    code, sc, ze = T.encode_v(_bf16_bits_of(v))
    assert np.array_equal(code, codes) and np.all(sc == scale) and np.all(ze == zero)
    assert np.array_equal(T.dequant_v(code, sc, ze), v)
    const = np.full((2, d), 1.75)
    code, sc, ze = T.encode_v(_bf16_bits_of(const))
    assert not code.any() and not sc.any() and np.array_equal(T.dequant_v(code, sc, ze), const)
    vb = _bf16_bits_of(rng.standard_normal((64, d)) * 3)
    code, sc, ze = T.encode_v(vb)
    v = oracle.bf16_to_double(vb)
    vh = T.dequant_v(code, sc, ze)
    bound = np.repeat(sc, 32, axis=1) * 0.5 * (1 + 2.0 ** -6) + np.abs(v) * 2.0 ** -8 + 16 * np.repeat(sc, 32, axis=1) * 2.0 ** -8
    assert np.all(np.abs(v - vh) <= bound)
    assert code.min() == 0 and code.max() == 15


def test_p17_ultra_tq_attention_special_cases_and_sdpa():
    """Alg. 2 l.5-8: one token -> the output is the dequantised value row of the head's kv head; every key equal -> the mean
    of the value rows; in general == float64 torch SDPA over (bf16(R q), dequant_k, dequant_v)."""
    from oracle import ultra_tq as T
    from paper_2606_20474_b200 import workloads as W
    cb = np.asarray(W.TQ_CODEBOOK, np.float32)
    rng = np.random.default_rng(17)
    Hq, Hkv, d, L = 8, 2, 128, 45
    G = Hq // Hkv
    qb = _bf16_bits_of(rng.standard_normal((Hq, d)))
    kb = _bf16_bits_of(rng.standard_normal((L, Hkv, d)) * 2)
    vb = _bf16_bits_of(rng.standard_normal((L, Hkv, d)))
    ki, kn = T.encode_k(kb.reshape(L * Hkv, d), cb)
    vc, vs, vz = T.encode_v(vb.reshape(L * Hkv, d))
    sh = lambda a: a.reshape(L, Hkv, -1)
    out = T.attention(qb, sh(ki), sh(kn), sh(vc), sh(vs), sh(vz), cb, Hkv)
    q = torch.from_numpy(T.encode_q(qb))
    k = torch.from_numpy(T.dequant_k(ki, kn, cb).reshape(L, Hkv, d))
    v = torch.from_numpy(T.dequant_v(vc, vs, vz).reshape(L, Hkv, d))
    ref = torch.nn.functional.scaled_dot_product_attention(
        q.view(Hkv, G, d), k.permute(1, 0, 2), v.permute(1, 0, 2)).reshape(Hq, d).numpy()
    assert np.abs(out - ref).max() < 1e-12
    one = T.attention(qb, sh(ki)[:1], sh(kn)[:1], sh(vc)[:1], sh(vs)[:1], sh(vz)[:1], cb, Hkv)
    assert np.array_equal(one, np.repeat(v[0].numpy(), G, axis=0))
    same = lambda a: np.repeat(sh(a)[:1], L, axis=0)
    eq = T.attention(qb, same(ki), same(kn), sh(vc), sh(vs), sh(vz), cb, Hkv)
    assert np.abs(eq - np.repeat(v.numpy().mean(axis=0), G, axis=0)).max() < 1e-12
    # the rotation is the pinned one (P1 / P12) and the query is rounded to bf16 once
    assert np.array_equal(T.encode_q(qb)[3], T.bf16_rne(oracle.hadamard(oracle.bf16_to_double(qb[3]))))
