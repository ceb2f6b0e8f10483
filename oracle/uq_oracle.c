/*
 * uq_oracle.c — plain, slow, float64 CPU oracle for UltraQuant's hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing in the product path (the CUDA library, its
 * Python binding) may include, link, import or call this file.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs use it.
 * It shares no code, header, table or constant generator with the CUDA path.
 *
 * Written from /root/reference/PAPER.md (arxiv/paper_2606_20474):
 *   Algorithm 1 "FP4-ConstOpt KV encoding (Ultra-Quant)"
 *   Section 5.1 cache layout (32-channel groups, 17 B/group)
 *   Section 5.2 dequantisation rule Eq.(1)
 *   Section 5.3 level set F and scale s = c*m
 * Readings of what the paper leaves open are listed in DESIGN.md ("Readings").
 *
 * Every function follows the paper's steps in the paper's order, in double
 * precision, with no tiling, paging, online softmax or split-K.
 *
 * Pins (tests/test_oracle_pins.py): Hadamard orthogonality and Kronecker
 * structure, decode table vs Eq.(1), exact round trip, brute-force nearest
 * level, scale thresholds, statistical fingerprints, the paper's two constants
 * (0.156 / 0.195), library E2M1/E4M3 casts, softmax closed forms, torch SDPA; the Eq.(2)
 * objective (O11) against an independent numpy quantiser, exactly representable inputs
 * (zero error), the rotation's norm invariance and the paper's ordering of c (P11);
 * uqo_encode_q element for element against hadamard + e4m3_encode and against the library
 * cast of an independently rotated query, on random / one-hot / saturating rows (P12);
 * uqo_attention_dense against float64 SDPA and the L = 1 / equal-keys / dominant-key closed
 * forms (P13); the FP8-KV casts uqo_cast_e4m3 / uqo_e4m3_to_double element for element against
 * e4m3_encode / e4m3_decode (P8) and the library cast (P14).
 * Parity unpinned: the attention *output values* for concrete inputs (the paper
 * prints no worked example) — pinned only through the closed forms above.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define UQ_GROUP 32

/* ---- O1: exact double of a bf16 bit pattern (Alg. 1 "Require: K, V (BF16)") */
double uqo_bf16_to_double(uint16_t h) {
  uint32_t u = ((uint32_t)h) << 16;
  float f;
  memcpy(&f, &u, 4);
  return (double)f;
}

/* ---- O2: rotation R = H_d / sqrt(d), Sylvester order (Alg. 1 l.1/l.6)
 * H[i][j] = (-1)^popcount(i & j).  Dense product, no butterfly.
 * kappa_d is the correctly rounded double of 2^(-log2(d)/2), written as a hex literal. */
static int popcount_u32(uint32_t v) {
  int c = 0;
  while (v) { c += (int)(v & 1u); v >>= 1; }
  return c;
}

double uqo_kappa(int d) {
  switch (d) {
    case 32:  return 0x1.6a09e667f3bcdp-3;   /* 2^-2.5 */
    case 64:  return 0x1p-3;                 /* 2^-3   */
    case 128: return 0x1.6a09e667f3bcdp-4;   /* 2^-3.5 */
    case 256: return 0x1p-4;                 /* 2^-4   */
    default:  return 0.0;
  }
}

/* The matrix is written out once per d (entries exactly +1.0 / -1.0 from the popcount rule) and then
 * used as a plain dense matrix: y_i = kappa * sum_j H[i][j] * x[j], j ascending.  A product by +-1.0 is
 * exact, so this is the same sum, term for term, as adding +x[j] or -x[j]. */
#define UQ_MAX_D 256
static double uqo_H[4][UQ_MAX_D * UQ_MAX_D];   /* d = 32, 64, 128, 256 */
static int uqo_H_ready[4];

static const double* uqo_hadamard_matrix(int d) {
  const int slot = d == 32 ? 0 : d == 64 ? 1 : d == 128 ? 2 : d == 256 ? 3 : -1;
  if (slot < 0) return NULL;
  double* H = uqo_H[slot];
  int ready;
#pragma omp atomic read
  ready = uqo_H_ready[slot];
  if (!ready) {
#pragma omp critical(uqo_hadamard_table)
    {
      if (!uqo_H_ready[slot]) {
        for (int i = 0; i < d; ++i)
          for (int j = 0; j < d; ++j)
            H[i * d + j] = (popcount_u32((uint32_t)i & (uint32_t)j) & 1) ? -1.0 : 1.0;
#pragma omp flush
#pragma omp atomic write
        uqo_H_ready[slot] = 1;
      }
    }
  }
  return H;
}

void uqo_hadamard(const double* x, int d, double* y) {
  const double kappa = uqo_kappa(d);
  const double* H = uqo_hadamard_matrix(d);
  if (!H) { for (int i = 0; i < d; ++i) y[i] = 0.0; return; }
  for (int i = 0; i < d; ++i) {
    double acc = 0.0;
    for (int j = 0; j < d; ++j) acc += H[i * d + j] * x[j];
    y[i] = acc * kappa;
  }
}

/* ---- O4: per-group scale exponent E = round(log2(c*m)) (Alg. 1 l.3)
 * "round" = round to nearest integer (reading G4).  Evaluated without a log2
 * call: t = f * 2^e with f in [0.5,1); round(log2 t) = e if f > 1/sqrt(2) else e-1.  The
 * double 0x1.6a09e667f3bcdp-1 is the smallest double above 1/sqrt(2); f is a double, so
 * f >= that constant  <=>  f > 1/sqrt(2).  Clamp to the UE8M0 range; byte = E + 127. */
int uqo_scale_exponent(double c, double m) {
  double t = c * m;
  if (!(t > 0.0)) return -127;
  int e;
  double f = frexp(t, &e);
  int E = (f >= 0x1.6a09e667f3bcdp-1) ? e : e - 1;
  if (E < -127) E = -127;
  if (E > 127) E = 127;
  return E;
}

/* ---- O5: nearest level in F = {0,.5,1,1.5,2,3,4,6} (Alg. 1 l.4; F at :124)
 * r = |y| / 2^E.  Ties go to the code with even mantissa bit; r > 6 clamps to 6; a zero
 * magnitude never carries a sign (readings G6, G7).  Code = sign<<3 | magnitude. */
uint8_t uqo_e2m1_encode(double y, int E) {
  double r = ldexp(fabs(y), -E);
  int mag = (r > 0.25) + (r >= 0.75) + (r > 1.25) + (r >= 1.75) + (r > 2.5) + (r >= 3.5) + (r > 5.0);
  uint8_t code = (uint8_t)mag;
  if (mag != 0 && y < 0.0) code |= 8u;
  return code;
}

/* ---- O8: Eq.(1) value = code * 2^(byte-127) (Alg. 1 l.7 :260) */
double uqo_e2m1_level(uint8_t code) {
  static const double F[8] = {0.0, 0.5, 1.0, 1.5, 2.0, 3.0, 4.0, 6.0};
  double v = F[code & 7u];
  return (code & 8u) ? -v : v;
}

double uqo_dequant(uint8_t code, uint8_t scale_byte) {
  return ldexp(uqo_e2m1_level(code), (int)scale_byte - 127);
}

/* ---- O3-O6: quantise one d-vector (already rotated or not) into packed codes + scale bytes.
 * Groups are contiguous 32-channel slices (Alg. 1 l.2).  Packing: byte j holds
 * element 2j in bits 0-3 and element 2j+1 in bits 4-7; scale bytes in group order (G8). */
void uqo_quantize_vector(const double* y, int d, double c, uint8_t* packed /*d/2*/, uint8_t* scales /*d/32*/) {
  for (int g = 0; g < d / UQ_GROUP; ++g) {
    const double* yg = y + g * UQ_GROUP;
    double m = 0.0;
    for (int i = 0; i < UQ_GROUP; ++i) {
      double a = fabs(yg[i]);
      if (a > m) m = a;
    }
    int E = uqo_scale_exponent(c, m);
    scales[g] = (uint8_t)(E + 127);
    for (int i = 0; i < UQ_GROUP; i += 2) {
      uint8_t lo = uqo_e2m1_encode(yg[i], E);
      uint8_t hi = uqo_e2m1_encode(yg[i + 1], E);
      packed[(g * UQ_GROUP + i) / 2] = (uint8_t)(lo | (hi << 4));
    }
  }
}

/* ---- Alg. 1 "Write" over n_vec vectors of d channels (one vector per
 * (token, kv_head)).  K is rotated, V is not ("rotate keys; V unrotated", :251).
 * Outputs are LOGICAL arrays: codes [n_vec][d/2], scales [n_vec][d/32].  The only
 * parallelism is an outer loop over independent vectors (for timing on many cores). */
void uqo_encode_kv(const uint16_t* k_bf16, const uint16_t* v_bf16, int64_t n_vec, int d,
                   float c_k, float c_v,
                   uint8_t* k_codes, uint8_t* k_scales, uint8_t* v_codes, uint8_t* v_scales) {
  const int ng = d / UQ_GROUP;
#pragma omp parallel
  {
    double* x = (double*)malloc(sizeof(double) * (size_t)d);
    double* y = (double*)malloc(sizeof(double) * (size_t)d);
#pragma omp for schedule(static)
    for (int64_t n = 0; n < n_vec; ++n) {
      if (k_bf16) {
        for (int i = 0; i < d; ++i) x[i] = uqo_bf16_to_double(k_bf16[n * d + i]);
        uqo_hadamard(x, d, y);                                   /* l.1 */
        uqo_quantize_vector(y, d, (double)c_k, k_codes + n * (d / 2), k_scales + n * ng); /* l.2-5 */
      }
      if (v_bf16) {
        for (int i = 0; i < d; ++i) x[i] = uqo_bf16_to_double(v_bf16[n * d + i]);
        uqo_quantize_vector(x, d, (double)c_v, v_codes + n * (d / 2), v_scales + n * ng);
      }
    }
    free(x);
    free(y);
  }
}

/* ---- O11: the objective of Eq.(2) on a grid of constants: for every c_j,
 *     sq_err[j] = sum over all elements z of (z - zhat_j(z))^2,   sq_norm = sum z^2,
 * with z the rotated vector (rotate != 0: Alg. 1 l.1) or the vector itself, m the absmax of
 * z's 32-channel group and
 *   scale_mode 0: s = c_j*m, the scale of Eq.(2) as printed; zhat = s * q(z/s), q = nearest level;
 *   scale_mode 1: s = 2^E, E = round(log2(c_j*m)) (O4): the quantiser Alg. 1 deploys
 *                 (l.3-5, :253-255) followed by Eq.(1); zhat = dequant(encode(z, E), E);
 *   scale_mode 2: s = c_j, no absmax: a fixed grid for vectors of known norm (the per-token
 *                 l2-norm schemes the paper compares with, :116-120 and Fig. 2).
 * Levels: levels == NULL -> F = {0,.5,1,1.5,2,3,4,6} with the tie rule of O5 (the only choice
 * for scale_mode 1); else 8 ascending magnitudes L_0..L_7 of a symmetric 15/16-level codebook
 * (uniform INT4: 0..7; Lloyd-Max centroids: Fig. 2a), q(r) = the L_i nearest to r, a tie going
 * to the smaller one (the squared error of a tie does not depend on the choice).
 * c_j is a float (as uq_config.c_k) used as (double)c_j.  A group with s = 0 contributes 0.
 * E[.] of Eq.(2) is sq_err / (n_vec*d); its argmin over j is the calibrated constant (:128).
 * Plain loops, vector after vector, one double accumulator per c_j. */
static int uqo_mag_of_ratio(double r) {
  return (r > 0.25) + (r >= 0.75) + (r > 1.25) + (r >= 1.75) + (r > 2.5) + (r >= 3.5) + (r > 5.0);
}

void uqo_calib_sq_err(const uint16_t* x_bf16, int64_t n_vec, int d, int rotate, const float* c_grid,
                      int n_c, int scale_mode, const float* levels /*[8] or NULL*/,
                      double* sq_err /*[n_c]*/, double* sq_norm /*[1]*/) {
  double F[8] = {0.0, 0.5, 1.0, 1.5, 2.0, 3.0, 4.0, 6.0};
  if (levels) for (int i = 0; i < 8; ++i) F[i] = (double)levels[i];
  double* x = (double*)malloc(sizeof(double) * (size_t)d);
  double* y = (double*)malloc(sizeof(double) * (size_t)d);
  for (int j = 0; j < n_c; ++j) sq_err[j] = 0.0;
  *sq_norm = 0.0;
  for (int64_t n = 0; n < n_vec; ++n) {
    for (int i = 0; i < d; ++i) x[i] = uqo_bf16_to_double(x_bf16[n * d + i]);
    if (rotate) uqo_hadamard(x, d, y);
    else memcpy(y, x, sizeof(double) * (size_t)d);
    for (int i = 0; i < d; ++i) *sq_norm += y[i] * y[i];
    for (int g = 0; g < d / UQ_GROUP; ++g) {
      const double* yg = y + g * UQ_GROUP;
      double m = 0.0;
      for (int i = 0; i < UQ_GROUP; ++i) {
        double a = fabs(yg[i]);
        if (a > m) m = a;
      }
      for (int j = 0; j < n_c; ++j) {
        const double c = (double)c_grid[j];
        if (scale_mode == 1) {
          int E = uqo_scale_exponent(c, m);
          for (int i = 0; i < UQ_GROUP; ++i) {
            double zh = uqo_dequant(uqo_e2m1_encode(yg[i], E), (uint8_t)(E + 127));
            double e = yg[i] - zh;
            sq_err[j] += e * e;
          }
        } else {
          double s = (scale_mode == 2) ? c : c * m;
          if (!(s > 0.0)) continue;
          for (int i = 0; i < UQ_GROUP; ++i) {
            double r = fabs(yg[i]) / s;
            int mag;
            if (levels) {
              mag = 0;
              for (int k = 0; k < 7; ++k) mag += (r > 0.5 * (F[k] + F[k + 1]));
            } else {
              mag = uqo_mag_of_ratio(r);
            }
            double zh = (yg[i] < 0.0 ? -F[mag] : F[mag]) * s;
            double e = yg[i] - zh;
            sq_err[j] += e * e;
          }
        }
      }
    }
  }
  free(x);
  free(y);
}

/* ---- O7: cast_fp8_e4m3 (Alg. 1 l.6).  OCP E4M3 "FN": bias 7, normals
 * 2^-6..448, subnormal step 2^-9, no infinities; round to nearest even, saturate to 448,
 * no -0 stored (readings G7, G9).  Directly from the double, one rounding. */
uint8_t uqo_e4m3_encode(double y) {
  double a = fabs(y);
  uint8_t mag;
  if (!(a > 0.0)) {
    mag = 0;
  } else if (a >= 448.0) {
    mag = 0x7E;                                  /* 448 = 1.75 * 2^8 */
  } else if (a < 0x1p-6) {
    int n = (int)rint(ldexp(a, 9));              /* subnormal quantum 2^-9; n==8 is the min normal */
    mag = (uint8_t)n;                            /* n in 0..8: 8 -> exponent field 1, mantissa 0 */
  } else {
    int e;
    (void)frexp(a, &e);
    e -= 1;                                      /* a = 1.xxx * 2^e */
    int n = (int)rint(ldexp(a, 3 - e));          /* n in [8,16] */
    if (n == 16) { n = 8; e += 1; }
    if (e > 8 || (e == 8 && n > 14)) {
      mag = 0x7E;
    } else {
      mag = (uint8_t)(((e + 7) << 3) | (n - 8));
    }
  }
  if (mag != 0 && y < 0.0) mag |= 0x80u;
  return mag;
}

double uqo_e4m3_decode(uint8_t b) {
  int ef = (b >> 3) & 0xF;
  int mf = b & 7;
  double v = (ef == 0) ? ldexp((double)mf, -9) : ldexp(1.0 + (double)mf / 8.0, ef - 7);
  return (b & 0x80u) ? -v : v;
}

/* Q <- R*Q ; Q <- cast_fp8_e4m3(Q)  (Alg. 1 l.6).  q_bf16 [n_vec][d] -> q8 [n_vec][d]. */
void uqo_encode_q(const uint16_t* q_bf16, int64_t n_vec, int d, uint8_t* q8) {
#pragma omp parallel
  {
    double* x = (double*)malloc(sizeof(double) * (size_t)d);
    double* y = (double*)malloc(sizeof(double) * (size_t)d);
#pragma omp for schedule(static)
    for (int64_t n = 0; n < n_vec; ++n) {
      for (int i = 0; i < d; ++i) x[i] = uqo_bf16_to_double(q_bf16[n * d + i]);
      uqo_hadamard(x, d, y);
      for (int i = 0; i < d; ++i) q8[n * d + i] = uqo_e4m3_encode(y[i]);
    }
    free(x);
    free(y);
  }
}

/* ---- O8-O10: Alg. 1 "Decode" l.7-8 as the textbook definition.
 * One sequence of L tokens.  Logical cache arrays: codes [L][Hkv][d/2], scales [L][Hkv][d/32].
 * q8 [Hq][d] E4M3 bytes.  q head h uses kv head h / (Hq/Hkv) (reading G11).
 *   z_t   = sm_scale * sum_i q8[h,i] * khat[t,i]
 *   p_t   = exp(z_t - max z) / sum_t exp(z_t - max z)
 *   out[h] = sum_t p_t * vhat[t,:]          (no inverse rotation: V was never rotated)
 * L == 0 gives a row of zeros.  If probs != NULL it receives p [Hq][L]. */
void uqo_attention(const uint8_t* q8, const uint8_t* k_codes, const uint8_t* k_scales,
                   const uint8_t* v_codes, const uint8_t* v_scales,
                   int64_t L, int Hq, int Hkv, int d, double sm_scale,
                   double* out /*[Hq][d]*/, double* probs /*[Hq][L] or NULL*/) {
  const int G = Hq / Hkv;
  const int ng = d / UQ_GROUP;
#pragma omp parallel for schedule(dynamic, 1)
  for (int h = 0; h < Hq; ++h) {
    const int kvh = h / G;
    double* o = out + (size_t)h * d;
    for (int i = 0; i < d; ++i) o[i] = 0.0;
    if (L <= 0) continue;
    double* z = (double*)malloc(sizeof(double) * (size_t)L);
    double* qd = (double*)malloc(sizeof(double) * (size_t)d);
    for (int i = 0; i < d; ++i) qd[i] = uqo_e4m3_decode(q8[(size_t)h * d + i]);
    double zmax = -INFINITY;
    for (int64_t t = 0; t < L; ++t) {
      const uint8_t* kc = k_codes + ((size_t)t * Hkv + kvh) * (d / 2);
      const uint8_t* ks = k_scales + ((size_t)t * Hkv + kvh) * ng;
      double acc = 0.0;
      for (int i = 0; i < d; ++i) {
        uint8_t code = (i & 1) ? (uint8_t)(kc[i / 2] >> 4) : (uint8_t)(kc[i / 2] & 0xF);
        acc += qd[i] * uqo_dequant(code, ks[i / UQ_GROUP]);      /* l.7 then l.8 (QK) */
      }
      z[t] = sm_scale * acc;
      if (z[t] > zmax) zmax = z[t];
    }
    double denom = 0.0;
    for (int64_t t = 0; t < L; ++t) { z[t] = exp(z[t] - zmax); denom += z[t]; }
    for (int64_t t = 0; t < L; ++t) {
      double p = z[t] / denom;
      if (probs) probs[(size_t)h * L + t] = p;
      const uint8_t* vc = v_codes + ((size_t)t * Hkv + kvh) * (d / 2);
      const uint8_t* vs = v_scales + ((size_t)t * Hkv + kvh) * ng;
      for (int i = 0; i < d; ++i) {
        uint8_t code = (i & 1) ? (uint8_t)(vc[i / 2] >> 4) : (uint8_t)(vc[i / 2] & 0xF);
        o[i] += p * uqo_dequant(code, vs[i / UQ_GROUP]);         /* l.8 (PV) */
      }
    }
    free(z);
    free(qd);
  }
}

/* Same result for a query/key/value set given as doubles (no quantisation): used only to
 * report the error against unquantised BF16-input attention "as context" (BASELINE.json). */
void uqo_attention_dense(const double* q /*[Hq][d]*/, const double* k /*[L][Hkv][d]*/,
                         const double* v /*[L][Hkv][d]*/, int64_t L, int Hq, int Hkv, int d,
                         double sm_scale, double* out) {
  const int G = Hq / Hkv;
#pragma omp parallel for schedule(dynamic, 1)
  for (int h = 0; h < Hq; ++h) {
    const int kvh = h / G;
    double* o = out + (size_t)h * d;
    for (int i = 0; i < d; ++i) o[i] = 0.0;
    if (L <= 0) continue;
    double* z = (double*)malloc(sizeof(double) * (size_t)L);
    double zmax = -INFINITY;
    for (int64_t t = 0; t < L; ++t) {
      const double* kt = k + ((size_t)t * Hkv + kvh) * d;
      double acc = 0.0;
      for (int i = 0; i < d; ++i) acc += q[(size_t)h * d + i] * kt[i];
      z[t] = sm_scale * acc;
      if (z[t] > zmax) zmax = z[t];
    }
    double denom = 0.0;
    for (int64_t t = 0; t < L; ++t) { z[t] = exp(z[t] - zmax); denom += z[t]; }
    for (int64_t t = 0; t < L; ++t) {
      double p = z[t] / denom;
      const double* vt = v + ((size_t)t * Hkv + kvh) * d;
      for (int i = 0; i < d; ++i) o[i] += p * vt[i];
    }
    free(z);
  }
}

/* ---- Comparison systems of the paper's Section 7 (PAPER.md:163-171; Table 3, :293-301): "hardware FP8 KV" and the
 * BF16 baseline, as CACHES for the same attention.  The paper names them and nothing more;
 * DESIGN.md reading G19: FP8 KV = K and V stored as OCP E4M3 bytes of the bf16 values themselves (no rotation, scale 1
 * — the engine default without calibrated scales), round to nearest even, saturating, +0 only, i.e. uqo_e4m3_encode
 * per element; the query is cast the same way; BF16 KV = the bf16 values as they are.  Attention over either is
 * uqo_attention_dense on the decoded doubles (uqo_e4m3_decode / uqo_bf16_to_double): the textbook definition. */
void uqo_cast_e4m3(const uint16_t* x_bf16, int64_t n, uint8_t* out) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) out[i] = uqo_e4m3_encode(uqo_bf16_to_double(x_bf16[i]));
}

void uqo_e4m3_to_double(const uint8_t* b, int64_t n, double* out) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) out[i] = uqo_e4m3_decode(b[i]);
}

/* Number of OpenMP threads the loops above will use (reported as cpu_baseline.cores). */
#ifdef _OPENMP
#include <omp.h>
int uqo_num_threads(void) { return omp_get_max_threads(); }
void uqo_set_num_threads(int n) { omp_set_num_threads(n); }
#else
int uqo_num_threads(void) { return 1; }
void uqo_set_num_threads(int n) { (void)n; }
#endif
