// uq_append.cu — quantize-on-append: Alg. 1 "Write" l.1-5 and "Decode" l.6 of
// arxiv/paper_2606_20474.
//
// Record layout: include/uq.h.  One warp per (aligned octet of token positions, kv head) or per (sequence, q head).  A lane owns 4 consecutive
// channels of the 128-channel vector.  The Walsh-Hadamard rotation is an in-register butterfly:
// index bits 0-1 inside the lane, bits 2-6 through warp shuffles.  All of it runs in float64:
// sums of 128 bf16 values are exact in double, so every rounding decision (scale exponent,
// E2M1 level, E4M3 byte) is taken on the same real numbers the float64 oracle sees
// (reading G1).  __dadd_rn/__dmul_rn keep the compiler from contracting into FMAs.
#include <cuda.h>

#include "uq_common.cuh"
#include "uq_quant.cuh"

namespace uq {
namespace {

// ---------------------------------------------------------------- float32 fast path
// The float64 path above takes every rounding decision on exact sums.  The fast path computes the same vector in
// float32 with a proven error bound and accepts a decision only if the whole error interval falls on one side of
// every rounding boundary (the decision functions are monotone, so equal results at both ends of the interval
// mean the exact value gives that result too); otherwise the warp redoes the vector in float64.  Results are
// therefore identical to the float64 path bit for bit — only the time differs.
//
// Error bound of the rotated value z_i (float32) against the oracle's y_i (float64, exact sums): seven levels of
// float32 additions give |sum - exact| <= ((1+u)^7 - 1) S with u = 2^-24 and S = sum_i |x_i|; the float32 constant
// 2^-3.5 and the final product add 2u|y| <= 2u S: |z_i - y_i| <= 9.0001 u kappa S < 4.75e-8 S.  kBound leaves 5 %
// for the float32 evaluation of S and of the bound itself.
constexpr float kBound = 5.0e-8f;

__device__ __forceinline__ void load4f(const uint16_t* row, int lane, float (&x)[4]) {
  const uint2 raw = *reinterpret_cast<const uint2*>(row + 4 * lane);
  x[0] = __uint_as_float(raw.x << 16);
  x[1] = __uint_as_float(raw.x & 0xFFFF0000u);
  x[2] = __uint_as_float(raw.y << 16);
  x[3] = __uint_as_float(raw.y & 0xFFFF0000u);
}

// four values -> four E2M1 codes (hardware conversion: round to nearest, ties to the even code, saturating),
// code i in bits 4i..4i+3; "-0" (only the sign bit set) is mapped to +0 as in the float64 path
__device__ __forceinline__ uint32_t e2m1x4(float r0, float r1, float r2, float r3) {
  uint32_t n;
  asm("{\n.reg .b8 t0, t1;\n.reg .b16 h;\n"
      "cvt.rn.satfinite.e2m1x2.f32 t0, %2, %1;\n"
      "cvt.rn.satfinite.e2m1x2.f32 t1, %4, %3;\n"
      "mov.b16 h, {t0, t1};\ncvt.u32.u16 %0, h;\n}\n" : "=r"(n) : "f"(r0), "f"(r1), "f"(r2), "f"(r3));
  const uint32_t t = n & 0x7777u;
  const uint32_t nz = ((t + 0x7777u) | t) & 0x8888u;       // bit 3 of a nibble set iff its magnitude is not 0
  return n & (0x7777u | nz);
}

// round(log2 t) for a positive normal float t by integer arithmetic on its bits: the exponent, plus one if the
// significand is at least sqrt(2) (0x3504F3 = float32 significand bits of sqrt(2), rounded down).  Monotone in t.
__device__ __forceinline__ int round_log2_f32(float t) {
  return (int)((__float_as_uint(t) + (0x800000u - 0x3504F3u)) >> 23) - 127;
}
// E = round(log2(c m)) for m known to +-radius: both ends of the error interval of t = c m — widened by 3.4 u t
// for the float32 product and the float32 sqrt(2) — must give the same exponent; false otherwise.
__device__ __forceinline__ bool scale_exponent_f32(float c, float m, float radius, int& E) {
  const float t = __fmul_rn(c, m);
  const float d = __fmaf_rn(t, 2.0e-7f, __fmul_rn(__fmul_rn(c, radius), 1.0001f));
  const float lo = t - d, hi = t + d;
  E = round_log2_f32(hi);
  return (lo > 1e-30f) && (hi < 1e30f) && (round_log2_f32(lo) == E);
}

// 2^-E as a float (|E| <= 100 is checked by the callers)
__device__ __forceinline__ float pow2_neg(int E) { return __uint_as_float((uint32_t)(127 - E) << 23); }

// y = H_128 x * 2^-3.5 in float32 for the lane's 4 channels; eps = bound of |x[i] - exact|; false if the vector is
// outside the range the bound was derived for (underflow / overflow / NaN: float64 takes those).
__device__ __forceinline__ bool wht128_f32(const uint16_t* row, int lane, float (&x)[4], float& eps) {
  load4f(row, lane, x);
  float S = (fabsf(x[0]) + fabsf(x[1])) + (fabsf(x[2]) + fabsf(x[3]));
#pragma unroll
  for (int k = 1; k < 32; k <<= 1) S += __shfl_xor_sync(kFull, S, k);
  // butterflies: index bits 0-1 inside the lane, bits 2-6 through shuffles
  const float a0 = x[0] + x[1], a1 = x[0] - x[1], a2 = x[2] + x[3], a3 = x[2] - x[3];
  x[0] = a0 + a2; x[2] = a0 - a2; x[1] = a1 + a3; x[3] = a1 - a3;
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    const float sgn = ((lane >> k) & 1) ? -1.0f : 1.0f;
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const float other = __shfl_xor_sync(kFull, x[r], 1 << k);
      x[r] = __fmaf_rn(x[r], sgn, other);               // exact product: one rounding, as an addition
    }
  }
  const float kappa = 0x1.6a09e6p-4f;                     // float32 nearest to 2^-3.5
#pragma unroll
  for (int r = 0; r < 4; ++r) x[r] = __fmul_rn(x[r], kappa);
  eps = __fmul_rn(S, kBound);
  return (S > 1e-30f) && (S < 1e30f);                     // no underflow / overflow / NaN games on the fast path
}

// four values -> four OCP E4M3 bytes (hardware conversion: round to nearest even, saturating to +-448), value i in
// byte i; "-0" is mapped to +0 as in the float64 path
__device__ __forceinline__ uint32_t e4m3x4(float r0, float r1, float r2, float r3) {
  uint32_t n;
  asm("{\n.reg .b16 h0, h1;\n"
      "cvt.rn.satfinite.e4m3x2.f32 h0, %2, %1;\n"
      "cvt.rn.satfinite.e4m3x2.f32 h1, %4, %3;\n"
      "mov.b32 %0, {h0, h1};\n}\n" : "=r"(n) : "f"(r0), "f"(r1), "f"(r2), "f"(r3));
  const uint32_t t = n & 0x7F7F7F7Fu;
  const uint32_t nz = ((t + 0x7F7F7F7Fu) | t) & 0x80808080u;   // bit 7 of a byte set iff its magnitude is not 0
  return n & (0x7F7F7F7Fu | nz);
}

// Query row, float32: the four E4M3 bytes of the lane; false if any element's error interval straddles a rounding
// boundary of E4M3 (the conversion is monotone).
__device__ __forceinline__ bool encode_q_fast(const uint16_t* qrow, int lane, uint32_t& w) {
  float x[4], eps;
  const bool ok = wht128_f32(qrow, lane, x, eps);
  const float er = __fmaf_rn(eps, 1.0001f, 1e-37f);       // the two additions below round: widen by their ulp as well
  float lo[4], hi[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const float slack = __fmaf_rn(fabsf(x[i]), 1.2e-7f, er);
    lo[i] = x[i] - slack;
    hi[i] = x[i] + slack;
  }
  w = e4m3x4(lo[0], lo[1], lo[2], lo[3]);
  return ok && (w == e4m3x4(hi[0], hi[1], hi[2], hi[3]));
}

// K of one token, float32: codes (as store_k packs them) and scale exponent; false if any decision is unsafe.
__device__ __forceinline__ bool encode_k_fast(const uint16_t* krow, int lane, double c_k, uint32_t& h16, int& E) {
  float x[4], eps;
  bool ok = wht128_f32(krow, lane, x, eps);
  // ---- scale exponent of the group (8 lanes x 4 channels)
  float m = fmaxf(fmaxf(fabsf(x[0]), fabsf(x[1])), fmaxf(fabsf(x[2]), fabsf(x[3])));
#pragma unroll
  for (int s = 1; s <= 4; s <<= 1) m = fmaxf(m, __shfl_xor_sync(kFull, m, s));
  ok = scale_exponent_f32((float)c_k, m, eps, E) && ok && (E >= -100) && (E <= 100);
  // ---- codes: the error interval of every element must round to one code
  const float sc = pow2_neg(ok ? E : 0);
  const float er = __fmaf_rn(__fmul_rn(eps, sc), 1.0001f, 1.2e-6f);   // + the rounding of the two additions below
  float r[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) r[i] = __fmul_rn(x[i], sc);  // exact (power of two)
  const uint32_t lo = e2m1x4(r[0] - er, r[1] - er, r[2] - er, r[3] - er);
  const uint32_t hi = e2m1x4(r[0] + er, r[1] + er, r[2] + er, r[3] + er);
  h16 = lo;
  return ok && (lo == hi);
}

// V of one token, float32: exact (no rotation: the bf16 values themselves are scaled by a power of two); only the
// scale exponent needs the float64 product c * m.  Returns the codes as encode_v does; false -> use encode_v.
__device__ __forceinline__ bool encode_v_fast(const uint16_t* vrow, int lane, double c_v, uint32_t& codes, int& E) {
  float x[4];
  load4f(vrow, lane, x);
  float m = fmaxf(fmaxf(fabsf(x[0]), fabsf(x[1])), fmaxf(fabsf(x[2]), fabsf(x[3])));
#pragma unroll
  for (int s = 1; s <= 4; s <<= 1) m = fmaxf(m, __shfl_xor_sync(kFull, m, s));
  const bool zero = (m == 0.0f);                           // an all-zero group: E = -127, codes 0 (as scale_exponent)
  const bool ok = zero || (scale_exponent_f32((float)c_v, m, 0.0f, E) && (E >= -100) && (E <= 100));
  const float sc = pow2_neg((ok && !zero) ? E : 0);
  const uint32_t h = e2m1x4(__fmul_rn(x[0], sc), __fmul_rn(x[1], sc), __fmul_rn(x[2], sc), __fmul_rn(x[3], sc));
  codes = zero ? 0u : ((h & 0xFu) | ((h & 0xF0u) << 4) | ((h & 0xF00u) << 8) | ((h & 0xF000u) << 12));
  if (zero) E = -127;
  return ok;
}

// Encode + store K of one token: codes into the word-permuted K block, scale word.
__device__ __forceinline__ void store_k(const uint16_t* krow, uint8_t* rec, int t, int lane, double c_k) {
  uint32_t h16;
  int E;
  if (!__all_sync(kFull, encode_k_fast(krow, lane, c_k, h16, E))) {   // float64 when any decision was too close
    double x[4];
    load4(krow, lane, x);
    wht128(x, lane);
    E = group_exponent(x, c_k);
    h16 = e2m1_code(x[0], E) | (e2m1_code(x[1], E) << 4) | (e2m1_code(x[2], E) << 8) | (e2m1_code(x[3], E) << 12);
  }
  const uint32_t other = __shfl_down_sync(kFull, h16, 1);
  if ((lane & 1) == 0) {                      // logical order: word j = channels 8j..8j+7
    *reinterpret_cast<uint32_t*>(rec + kOffKCodes + 64 * t + 4 * (lane >> 1)) = h16 | (other << 16);
  }
  const uint32_t b = (uint32_t)(E + 127);
  const uint32_t w = __shfl_sync(kFull, b, 0) | (__shfl_sync(kFull, b, 8) << 8) |
                     (__shfl_sync(kFull, b, 16) << 16) | (__shfl_sync(kFull, b, 24) << 24);
  if (lane == 0) *reinterpret_cast<uint32_t*>(rec + kOffKScales + 4 * t) = w;
}

// Encode V of one token: returns the lane's four 4-bit codes (one per byte of the result) and
// stores the token's scale bytes.
__device__ __forceinline__ uint32_t encode_v(const uint16_t* vrow, uint8_t* rec, int t, int lane, double c_v) {
  uint32_t codes;
  int E;
  if (!__all_sync(kFull, encode_v_fast(vrow, lane, c_v, codes, E))) {
    double x[4];
    load4(vrow, lane, x);
    E = group_exponent(x, c_v);
    codes = e2m1_code(x[0], E) | (e2m1_code(x[1], E) << 8) | (e2m1_code(x[2], E) << 16) | (e2m1_code(x[3], E) << 24);
  }
  if ((lane & 7) == 0) rec[kOffVScales + 32 * (t >> 3) + 8 * (lane >> 3) + (t & 7)] = (uint8_t)(E + 127);
  return codes;
}

// Sequence b owns the work units off(b) .. off(b+1)-1 with off(b) = (cu_new[b] >> SHIFT) + 2 b (its new tokens touch
// at most (count >> SHIFT) + 2 aligned blocks of 2^SHIFT positions).  Returns the largest b < batch with off(b) <= u:
// a guess for evenly spread tokens checked with two independent loads; else a two-level search by the whole warp
// (32 entries per level, one load per lane and a ballot), or a binary search beyond 1024 sequences.
template <int SHIFT>
__device__ __forceinline__ int find_sequence(const int32_t* __restrict__ cu_new, int batch, int u, int n_units, int lane) {
  auto off = [&](int i) { return (cu_new[i] >> SHIFT) + 2 * i; };
  int b = max(0, min((int)((float)u * (float)batch / (float)n_units), batch - 1));   // only a guess: verified next
  if (!(off(b) <= u && u < off(b + 1))) {
    if (batch <= 1024) {
      const int step = (batch + 31) >> 5;             // entries per first-level block
      const int i1 = min((lane + 1) * step, batch);
      const int blk = __popc(__ballot_sync(kFull, off(i1) <= u && i1 < batch));   // blocks wholly <= u
      const int base = min(blk * step, batch - 1);
      const int i2 = min(base + lane, batch - 1);
      const unsigned le = __ballot_sync(kFull, lane < step && base + lane < batch && off(i2) <= u);
      b = base + (31 - __clz((int)(le | 1u)));        // off(base) <= u always holds
    } else {
      int lo = 0, hi = batch;
      while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (off(mid) <= u) lo = mid; else hi = mid;
      }
      b = lo;
    }
  }
  return b;
}

// One warp: K and V of the call's positions t_lo .. t_hi-1 inside the aligned octet q0 .. q0+7 of a sequence whose
// first new token (row c0 of k_new / v_new) lands at position p0.  An octet's V codes are 128 whole 32-bit words (one
// per channel, a nibble per token) = 512 contiguous bytes of the record, written with one 16-byte store per lane; the
// tokens of the octet that are not part of the range keep their nibbles (masked merge).
__device__ __forceinline__ void append_octet(const uint16_t* __restrict__ k_new, const uint16_t* __restrict__ v_new,
                                             uint8_t* rec, int c0, int p0, int q0, int t_lo, int t_hi, int h, int Hkv,
                                             int lane, double c_k, double c_v) {
  // token-major nibbles: channel d lives in word 512*(t>>3) + 4 d of the V codes, token t in nibble t & 7
  uint4* dst = reinterpret_cast<uint4*>(rec + kOffVCodes + 512 * ((q0 >> 3) & 1) + 16 * lane);
  const bool whole = (t_hi - t_lo == 8);
  uint4 old = make_uint4(0u, 0u, 0u, 0u);
  if (!whole) old = *dst;                             // the other tokens' nibbles: loaded under the encoding below
  uint32_t vw[4] = {0u, 0u, 0u, 0u};                  // V code words of channels 4 lane .. 4 lane + 3
  for (int pos = t_lo; pos < t_hi; ++pos) {
    const long long row = ((long long)(c0 + (pos - p0)) * Hkv + h) * kHeadDim;
    store_k(k_new + row, rec, pos & 15, lane, c_k);
    const uint32_t c = encode_v(v_new + row, rec, pos & 15, lane, c_v);
#pragma unroll
    for (int r = 0; r < 4; ++r) vw[r] |= ((c >> (8 * r)) & 0xFu) << (4 * (pos & 7));
  }
  if (whole) {
    *dst = make_uint4(vw[0], vw[1], vw[2], vw[3]);
  } else {                                            // keep the nibbles of the other tokens of the octet
    const uint32_t below_hi = (t_hi - q0 == 8) ? 0xFFFFFFFFu : ((1u << (4 * (t_hi - q0))) - 1u);
    const uint32_t m = below_hi & ~((1u << (4 * (t_lo - q0))) - 1u);
    *dst = make_uint4((old.x & ~m) | (vw[0] & m), (old.y & ~m) | (vw[1] & m), (old.z & ~m) | (vw[2] & m),
                      (old.w & ~m) | (vw[3] & m));
  }
}

// V of the single position pos (octet q0) redone in float64 by the warp: the token's nibbles are merged into the
// words the octet already holds.
__device__ __forceinline__ void append_octet_v(const uint16_t* __restrict__ v_new, uint8_t* rec, int c0, int p0, int q0,
                                               int pos, int h, int Hkv, int lane, double c_v) {
  uint4* dst = reinterpret_cast<uint4*>(rec + kOffVCodes + 512 * ((q0 >> 3) & 1) + 16 * lane);
  const uint4 old = *dst;
  const long long row = ((long long)(c0 + (pos - p0)) * Hkv + h) * kHeadDim;
  const uint32_t c = encode_v(v_new + row, rec, pos & 15, lane, c_v);
  const uint32_t m = 0xFu << (4 * (pos & 7));
  uint32_t vw[4];
#pragma unroll
  for (int r = 0; r < 4; ++r) vw[r] = ((c >> (8 * r)) & 0xFu) << (4 * (pos & 7));
  *dst = make_uint4((old.x & ~m) | vw[0], (old.y & ~m) | vw[1], (old.z & ~m) | vw[2], (old.w & ~m) | vw[3]);
}

__global__ void __launch_bounds__(128)
append_kernel(const uint16_t* __restrict__ k_new, const uint16_t* __restrict__ v_new,
              const int32_t* __restrict__ cu_new, const int32_t* __restrict__ seq_lens,
              const int32_t* __restrict__ block_tables, int max_pages, int batch, int total_new,
              int Hq, int Hkv, uint8_t* __restrict__ cache, const uint16_t* __restrict__ q,
              uint8_t* __restrict__ q_fp8, double c_k, double c_v) {
  pdl_launch_dependents();
  pdl_wait();                                          // inputs and cache may come from the kernel before this one
  const int lane = threadIdx.x & 31;
  // grid: y < Hkv -> K/V of kv head y, unit 4 x + warp;  y >= Hkv -> query rows.
  // A K/V unit is one aligned octet of token positions (8 k .. 8 k + 7) of one sequence: its V codes are 128
  // whole 32-bit words (one per channel, a nibble per token) = 512 contiguous bytes of the record, written with one
  // 16-byte store per lane; the tokens of the octet that are not part of this call keep their nibbles.  The
  // position of a sequence's first new token is device data, so units are dealt out by an upper bound that needs
  // cu_new only: sequence b owns units off(b) .. off(b+1)-1 with off(b) = (cu_new[b] >> 3) + 2 b (its tokens touch at
  // most (count >> 3) + 2 octets); surplus units exit.
  if ((int)blockIdx.y < Hkv) {
    const int u = (int)blockIdx.x * 4 + (int)(threadIdx.x >> 5), h = (int)blockIdx.y;
    const int n_units = (total_new >> 3) + 2 * batch;
    if (total_new == 0 || u >= n_units) return;
    const int b = find_sequence<3>(cu_new, batch, u, n_units, lane);
    const int c0 = cu_new[b], cnt = cu_new[b + 1] - c0, p0 = seq_lens[b];
    const int q0 = ((p0 >> 3) + (u - ((c0 >> 3) + 2 * b))) << 3;     // first position of this unit's octet
    const int t_lo = max(p0, q0), t_hi = min(p0 + cnt, q0 + 8);   // the call's positions inside the octet
    if (t_lo >= t_hi) return;
    {   // the first token's rows on their way while the page is looked up (a decode step is a chain of latencies)
      const long long row0 = ((long long)(c0 + (t_lo - p0)) * Hkv + h) * kHeadDim + 4 * lane;
      asm volatile("prefetch.global.L1 [%0];" ::"l"(k_new + row0));
      asm volatile("prefetch.global.L1 [%0];" ::"l"(v_new + row0));
    }
    const int page = block_tables[(long long)b * max_pages + (q0 >> 4)];
    uint8_t* rec = cache + ((long long)page * Hkv + h) * kRecordBytes;
    append_octet(k_new, v_new, rec, c0, p0, q0, t_lo, t_hi, h, Hkv, lane, c_k, c_v);
    return;
  }
  const long long qu = ((long long)((int)blockIdx.y - Hkv) * gridDim.x + blockIdx.x) * 4 + (threadIdx.x >> 5);
  if (q != nullptr && qu < (long long)batch * Hq) {
    uint32_t w;
    if (!__all_sync(kFull, encode_q_fast(q + qu * kHeadDim, lane, w))) {   // float64 when any byte was too close
      double x[4];
      load4(q + qu * kHeadDim, lane, x);
      wht128(x, lane);
      w = e4m3_byte(x[0]) | (e4m3_byte(x[1]) << 8) | (e4m3_byte(x[2]) << 16) | (e4m3_byte(x[3]) << 24);
    }
    *reinterpret_cast<uint32_t*>(q_fp8 + qu * kHeadDim + 4 * lane) = w;
  }
}

// ---------------------------------------------------------------- bulk (prefill-sized) append
// SURVEY 8(f) rank 1.  The kernel above spends a warp on every vector: 326 warp instructions per (token, kv head),
// a third of them shuffles and lane bookkeeping.  Here a warp takes one page (16 aligned positions) of one kv head,
// stages its K and V rows in shared memory with four TMA tensor copies (k_new / v_new seen as
// [rows][kv heads x 128] bf16, box 16 rows x 64 channels, completion on an mbarrier) and works in two thread mappings:
//   K      lanes t and t + 16 = token t, 64 channels (two whole scale groups) each: six butterfly levels are
//          in-register add/sub pairs (five of them on packed float32 pairs), the level between the two halves is a
//          shuffle of those pairs; the same float32 error-interval test as the fast path above decides every scale exponent
//          and code; 32 B of codes and two scale bytes are stored per lane;
//   V      pass 1, lane = (token, channel half): group maxima by packed 16-bit integer maxima of the bf16
//          magnitudes -> scale exponent, scale bytes, and the power-of-two multipliers left in shared memory;
//          pass 2, lane = 4 channels: eight tokens of a channel make one 32-bit word of the token-major layout
//          (four cvt.e2m1x2 per word), one 16-byte store per lane and octet.
// A vector whose interval test fails (0.45 % of N(0,1) keys) is redone by the whole warp with store_k /
// append_octet_v (float64), after the fast lanes have stored; a page that the call covers only partly goes through
// append_octet octet by octet.  The bytes written are those of the kernel above in every case.
// (First version: a block of 32 positions per warp, lane = token with all 128 channels in registers — 78 instead
// of 90 instructions per vector but 168 registers, 11 warps per SM; this one runs 20 warps per SM and is 6-10 %
// faster, profiles/r01_append_bulk_cfg2.md.)
constexpr int kBulkWarps = 4;
#ifndef UQ_BULK_CTAS
#define UQ_BULK_CTAS 5
#endif
// Shared memory per warp: the K and the V rows of its 16 tokens (one page) as two channel halves each — a TMA tensor
// tile of [16 tokens][64 channels] bf16 = 16 rows of 128 B with the 128-byte swizzle (16-byte chunk c of row r sits
// at chunk c ^ (r & 7)), so a lane reading its own row with 16-byte loads is bank-conflict free — and 16 x 4 V
// multipliers.
constexpr int kBulkHalf = 16 * 128;                    // 2048
constexpr int kBulkTiles = 4 * kBulkHalf;              // K lo, K hi, V lo, V hi: 8192 per warp
constexpr int kBulkSmem = kBulkWarps * (kBulkTiles + 256) + 1024;   // + alignment slack (the swizzle atom is 1024 B)

// eight values -> eight E2M1 codes, value i in bits 4i..4i+3 (raw hardware result: may hold "-0")
__device__ __forceinline__ uint32_t e2m1x8(float r0, float r1, float r2, float r3, float r4, float r5, float r6, float r7) {
  uint32_t n;
  asm("{\n.reg .b8 t0, t1, t2, t3;\n"
      "cvt.rn.satfinite.e2m1x2.f32 t0, %2, %1;\n"
      "cvt.rn.satfinite.e2m1x2.f32 t1, %4, %3;\n"
      "cvt.rn.satfinite.e2m1x2.f32 t2, %6, %5;\n"
      "cvt.rn.satfinite.e2m1x2.f32 t3, %8, %7;\n"
      "mov.b32 %0, {t0, t1, t2, t3};\n}\n"
      : "=r"(n) : "f"(r0), "f"(r1), "f"(r2), "f"(r3), "f"(r4), "f"(r5), "f"(r6), "f"(r7));
  return n;
}
__device__ __forceinline__ uint32_t canon_e2m1x8(uint32_t n) {   // "-0" (only the sign bit of a nibble set) -> +0
  const uint32_t t = n & 0x77777777u;
  const uint32_t nz = ((t + 0x77777777u) | t) & 0x88888888u;   // bit 3 of a nibble set iff its magnitude is not 0
  return n & (0x77777777u | nz);
}

// Packed float32 pairs (one instruction, two IEEE results: each half rounds exactly as the scalar operation does).
__device__ __forceinline__ uint64_t pack2(float a, float b) {
  uint64_t v;
  asm("mov.b64 %0, {%1, %2};" : "=l"(v) : "f"(a), "f"(b));
  return v;
}
__device__ __forceinline__ void unpack2(uint64_t v, float& a, float& b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b) {
  uint64_t d;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}
__device__ __forceinline__ uint64_t mul2(uint64_t a, uint64_t b) {
  uint64_t d;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c) {
  uint64_t d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}

// one butterfly level over the 32 pairs {x[2i], x[2i+1]} of a lane (64 channels): element index bit log2(2 HP).
// a - b is fma(b, -1, a): the product is exact, so it rounds once, like the subtraction.
template <int HP>
__device__ __forceinline__ void wht_level2(uint64_t (&p)[32], uint64_t minus1) {
#pragma unroll
  for (int k = 0; k < 16; ++k) {
    const int j = ((k / HP) * 2 * HP) + (k % HP);
    const uint64_t a = p[j], b = p[j + HP];
    p[j] = add2(a, b);
    p[j + HP] = fma2(b, minus1, a);
  }
}

__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// K of one token by the two lanes t and t + 16: lane t + 16 hf holds channels 64 hf .. 64 hf + 63 (row t of channel
// half hf of the tile, two whole scale groups).  Returns the lane's 8 code words and 2 scale bytes; false if any of
// ITS decisions is unsafe.
__device__ __forceinline__ bool bulk_encode_k(uint32_t tile, int lane, float c_k, uint32_t (&codes)[8], uint32_t& scale_half) {
  const int t = lane & 15, hf = lane >> 4;
  const uint32_t row = tile + kBulkHalf * hf + 128 * t, sw = (uint32_t)(t & 7);
  uint32_t mine[32];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(mine[4 * j]), "=r"(mine[4 * j + 1]), "=r"(mine[4 * j + 2]),
                 "=r"(mine[4 * j + 3]) : "r"(row + ((((uint32_t)j) ^ sw) << 4)));
  }
  // index bit 0 while unpacking, bits 1-5 on packed pairs in the lane, bit 6 (the other channel half lives in lane ^ 16)
  // last: x = lower + upper in lanes 0-15, lower - upper in lanes 16-31.  One rounding per output and level in any
  // order of the levels (the bound kBound is for exactly this: seven levels).
  uint64_t p[32];                                        // p[i] = {x[2i], x[2i+1]} of this lane's 64 channels
  float s0 = 0.f, s1 = 0.f;                              // sum |x_i| over this lane's inputs: two chains
#pragma unroll
  for (int i = 0; i < 32; ++i) {
    const float a = __uint_as_float(mine[i] << 16), b = __uint_as_float(mine[i] & 0xFFFF0000u);
    s0 += fabsf(a); s1 += fabsf(b);
    p[i] = pack2(__fadd_rn(a, b), __fsub_rn(a, b));
  }
  float S = s0 + s1;
  S += __shfl_xor_sync(kFull, S, 16);                    // the token's 128 inputs
  const uint64_t minus1 = pack2(-1.0f, -1.0f);
  wht_level2<1>(p, minus1); wht_level2<2>(p, minus1); wht_level2<4>(p, minus1); wht_level2<8>(p, minus1);
  wht_level2<16>(p, minus1);
  {
    const float sgn = hf ? -1.0f : 1.0f;
    const uint64_t sgn2 = pack2(sgn, sgn);
#pragma unroll
    for (int i = 0; i < 32; ++i) {
      const uint32_t lo = (uint32_t)p[i], hi = (uint32_t)(p[i] >> 32);
      const uint64_t oth = (uint64_t)__shfl_xor_sync(kFull, lo, 16) | ((uint64_t)__shfl_xor_sync(kFull, hi, 16) << 32);
      p[i] = fma2(p[i], sgn2, oth);                      // exact product: one rounding
    }
  }
  const float kappa = 0x1.6a09e6p-4f;                    // float32 nearest to 2^-3.5
  const float eps = __fmul_rn(S, kBound);
  bool ok = (S > 1e-30f) && (S < 1e30f);
  scale_half = 0u;
#pragma unroll
  for (int g = 0; g < 2; ++g) {
    float m = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) {
      float a, b;
      unpack2(p[16 * g + i], a, b);
      m = fmaxf(m, fmaxf(fabsf(a), fabsf(b)));
    }
    m = __fmul_rn(m, kappa);                             // = max |fl(kappa x_i)|: rounding is monotone
    int E;
    const bool okg = scale_exponent_f32(c_k, m, eps, E) && (E >= -100) && (E <= 100);
    ok = ok && okg;
    if (!okg) E = 0;
    scale_half |= (uint32_t)(E + 127) << (8 * g);
    const float sc = pow2_neg(E);
    const float ksc = __fmul_rn(kappa, sc);              // exact: fl(x kappa) 2^-E = fl(x (kappa 2^-E))
    const float er = __fmaf_rn(__fmul_rn(eps, sc), 1.0001f, 1.2e-6f);   // + the rounding of the two additions below
    const uint64_t ksc2 = pack2(ksc, ksc), per = pack2(er, er), mer = pack2(-er, -er);
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      float lo[8], hi[8];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const uint64_t r = mul2(p[16 * g + 4 * w + i], ksc2);
        unpack2(add2(r, mer), lo[2 * i], lo[2 * i + 1]);
        unpack2(add2(r, per), hi[2 * i], hi[2 * i + 1]);
      }
      const uint32_t cl = e2m1x8(lo[0], lo[1], lo[2], lo[3], lo[4], lo[5], lo[6], lo[7]);
      const uint32_t ch = e2m1x8(hi[0], hi[1], hi[2], hi[3], hi[4], hi[5], hi[6], hi[7]);
      ok = ok && (cl == ch);                           // raw codes: an interval over 0 counts as undecided too
      codes[4 * g + w] = canon_e2m1x8(cl);
    }
  }
  return ok;
}

__global__ void __launch_bounds__(32 * kBulkWarps, UQ_BULK_CTAS)
append_bulk_kernel(const __grid_constant__ CUtensorMap tmap_k, const __grid_constant__ CUtensorMap tmap_v,
                   const uint16_t* __restrict__ k_new, const uint16_t* __restrict__ v_new,
                   const int32_t* __restrict__ cu_new, const int32_t* __restrict__ seq_lens,
                   const int32_t* __restrict__ block_tables, int max_pages, int batch, int total_new, int Hkv,
                   uint8_t* __restrict__ cache, double c_k, double c_v) {
  extern __shared__ __align__(16) uint8_t bulk_smem[];
  __shared__ __align__(8) uint64_t bars[kBulkWarps][2];
  pdl_launch_dependents();
  pdl_wait();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int u = (int)blockIdx.x * kBulkWarps + warp, h = (int)blockIdx.y;
  const int n_units = (total_new >> 4) + 2 * batch;
  if (u >= n_units) return;                            // warps are independent: no CTA-wide barrier below
  const int b = find_sequence<4>(cu_new, batch, u, n_units, lane);
  const int c0 = cu_new[b], cnt = cu_new[b + 1] - c0, p0 = seq_lens[b];
  const int q0 = ((p0 >> 4) + (u - ((c0 >> 4) + 2 * b))) << 4;      // first position of this unit's page
  const int t_lo = max(p0, q0), t_hi = min(p0 + cnt, q0 + 16);      // the call's positions inside the page
  if (t_lo >= t_hi) return;
  const bool whole = (t_hi - t_lo == 16);

  // ---------------- whole page: rows -> shared memory (issued before the page lookup)
  const uint32_t sbase = (smem_addr(bulk_smem) + 1023u) & ~1023u;
  const uint32_t sK = sbase + warp * kBulkTiles, sV = sK + 2 * kBulkHalf, sM = sbase + kBulkWarps * kBulkTiles + 256 * warp;
  const uint32_t barK = smem_addr(&bars[warp][0]), barV = barK + 8;
  if (whole && lane == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(barK));
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(barV));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(barK), "r"(2 * kBulkHalf) : "memory");
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(barV), "r"(2 * kBulkHalf) : "memory");
    const int row0 = c0 + (q0 - p0);                   // k_new / v_new row of the page's first token
#pragma unroll
    for (int hf = 0; hf < 2; ++hf) {
      asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                   ::"r"(sK + kBulkHalf * hf), "l"(&tmap_k), "r"(h * kHeadDim + 64 * hf), "r"(row0), "r"(barK) : "memory");
    }
#pragma unroll
    for (int hf = 0; hf < 2; ++hf) {
      asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                   ::"r"(sV + kBulkHalf * hf), "l"(&tmap_v), "r"(h * kHeadDim + 64 * hf), "r"(row0), "r"(barV) : "memory");
    }
  }
  __syncwarp();
  const int page = block_tables[(long long)b * max_pages + (q0 >> 4)];
  uint8_t* const rec = cache + ((long long)page * Hkv + h) * kRecordBytes;

  if (!whole) {                                        // head / tail of a sequence's range: octet by octet
    for (int o = 0; o < 2; ++o) {
      const int qo = q0 + 8 * o, lo = max(t_lo, qo), hi = min(t_hi, qo + 8);
      if (lo >= hi) continue;
      append_octet(k_new, v_new, rec, c0, p0, qo, lo, hi, h, Hkv, lane, c_k, c_v);
      __syncwarp();
    }
    return;
  }

  const int t = lane & 15, hf = lane >> 4;             // this lane's token slot and channel half
  auto wait = [](uint32_t bar) {
    asm volatile("{\n.reg .pred p;\nW_%=:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], 0;\n@p bra D_%=;\nbra W_%=;\nD_%=:\n}\n"
                 ::"r"(bar) : "memory");
  };

  // ---------------- K: lanes t and t + 16 = token t
  wait(barK);
  unsigned bad_k;
  {
    uint32_t codes[8], scale_half;
    const bool ok = bulk_encode_k(sK, lane, (float)c_k, codes, scale_half);
    bad_k = __ballot_sync(kFull, !ok);
    bad_k = (bad_k | (bad_k >> 16)) & 0xFFFFu;         // tokens with an undecided half
    if (!((bad_k >> t) & 1u)) {
      uint4* dst = reinterpret_cast<uint4*>(rec + kOffKCodes + 64 * t + 32 * hf);
      dst[0] = make_uint4(codes[0], codes[1], codes[2], codes[3]);
      dst[1] = make_uint4(codes[4], codes[5], codes[6], codes[7]);
      *reinterpret_cast<uint16_t*>(rec + kOffKScales + 4 * t + 2 * hf) = (uint16_t)scale_half;
    }
  }

  // ---------------- V pass 1: lane = (token, channel half): two groups
  wait(barV);
  unsigned bad_v;
  {
    const uint32_t vrow = sV + kBulkHalf * hf + 128 * t, sw = (uint32_t)(t & 7);
    bool ok = true;
    float mult[2];
    uint32_t bytes = 0u;
#pragma unroll
    for (int gg = 0; gg < 2; ++gg) {
      uint32_t mx = 0u;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        uint4 w;
        asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(w.x), "=r"(w.y), "=r"(w.z), "=r"(w.w)
                     : "r"(vrow + ((((uint32_t)(4 * gg + j)) ^ sw) << 4)));
        mx = __vmaxu2(mx, __vmaxu2(__vmaxu2(w.x & 0x7FFF7FFFu, w.y & 0x7FFF7FFFu), __vmaxu2(w.z & 0x7FFF7FFFu, w.w & 0x7FFF7FFFu)));
      }
      const float m = __uint_as_float(max(mx >> 16, mx & 0xFFFFu) << 16);   // bf16 magnitudes order like their bits
      int E = -127;
      const bool zero = (m == 0.0f);
      const bool okg = zero || (scale_exponent_f32((float)c_v, m, 0.0f, E) && (E >= -100) && (E <= 100));
      ok = ok && okg;
      mult[gg] = (okg && !zero) ? pow2_neg(E) : 1.0f;
      if (zero || !okg) E = -127;
      bytes |= (uint32_t)(E + 127) << (8 * gg);
    }
    asm volatile("st.shared.v2.f32 [%0], {%1,%2};" ::"r"(sM + 16 * t + 8 * hf), "f"(mult[0]), "f"(mult[1]) : "memory");
    bad_v = __ballot_sync(kFull, !ok);
    bad_v = (bad_v | (bad_v >> 16)) & 0xFFFFu;
    if (!((bad_v >> t) & 1u)) {                          // group g = 2 hf + gg of token t: byte 32 (t >> 3) + 8 g + (t & 7)
      uint8_t* sb = rec + kOffVScales + 32 * (t >> 3) + 16 * hf + (t & 7);
      sb[0] = (uint8_t)(bytes & 0xFFu);
      sb[8] = (uint8_t)(bytes >> 8);
    }
  }
  __syncwarp();

  // ---------------- V pass 2: lane = channels 4 lane .. 4 lane + 3 (group lane >> 3), an octet of tokens per word
  const uint32_t vsrc = sV + kBulkHalf * (lane >> 4) + 8 * (lane & 1), vchunk = (uint32_t)((lane & 15) >> 1);
#pragma unroll
  for (int o = 0; o < 2; ++o) {
    float r[4][8];
#pragma unroll
    for (int tt = 0; tt < 8; ++tt) {
      uint32_t w0, w1;
      float mu;
      asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(w0), "=r"(w1)
                   : "r"(vsrc + 128 * (8 * o + tt) + ((vchunk ^ (uint32_t)tt) << 4)));   // row & 7 = tt
      asm volatile("ld.shared.f32 %0, [%1];" : "=f"(mu) : "r"(sM + 16 * (8 * o + tt) + 4 * (lane >> 3)));
      r[0][tt] = __fmul_rn(__uint_as_float(w0 << 16), mu);
      r[1][tt] = __fmul_rn(__uint_as_float(w0 & 0xFFFF0000u), mu);
      r[2][tt] = __fmul_rn(__uint_as_float(w1 << 16), mu);
      r[3][tt] = __fmul_rn(__uint_as_float(w1 & 0xFFFF0000u), mu);
    }
    uint32_t vw[4];
#pragma unroll
    for (int c = 0; c < 4; ++c)
      vw[c] = canon_e2m1x8(e2m1x8(r[c][0], r[c][1], r[c][2], r[c][3], r[c][4], r[c][5], r[c][6], r[c][7]));
    *reinterpret_cast<uint4*>(rec + kOffVCodes + 512 * o + 16 * lane) = make_uint4(vw[0], vw[1], vw[2], vw[3]);
  }

  // ---------------- vectors the float32 intervals could not decide: the whole warp, float64
  if (bad_k | bad_v) {
    __syncwarp();
    while (bad_k) {
      const int tk = __ffs(bad_k) - 1;
      bad_k &= bad_k - 1;
      const long long rw = ((long long)(c0 + (q0 - p0) + tk) * Hkv + h) * kHeadDim;
      store_k(k_new + rw, rec, tk, lane, c_k);
    }
    while (bad_v) {
      const int tv = __ffs(bad_v) - 1;
      bad_v &= bad_v - 1;
      const int pos = q0 + tv;
      append_octet_v(v_new, rec, c0, p0, pos & ~7, pos, h, Hkv, lane, c_v);
      __syncwarp();
    }
  }
}

// 2-D TMA view of k_new / v_new: [rows][kv heads x 128] bf16; box = 16 rows x 64 channels (128 B: the widest row the
// 128-byte swizzle takes), so a page's K (or V) rows of one kv head are two tensor copies.
int32_t rows_map(const void* rows, long long n_rows, int Hkv, CUtensorMap* out) {
  const EncodeTiledFn encode = encode_tiled_fn();
  if (!encode) return UQ_ERR_CUDA;
  const cuuint64_t gdim[2] = {(cuuint64_t)Hkv * kHeadDim, (cuuint64_t)n_rows};
  const cuuint64_t gstr[1] = {(cuuint64_t)Hkv * kHeadDim * 2};
  const cuuint32_t box[2] = {64, 16};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult cr = encode(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(rows), gdim, gstr, box, estr,
                             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (cr != CUDA_SUCCESS) {
    set_error("append: cuTensorMapEncodeTiled failed with CUresult %d", (int)cr);
    return UQ_ERR_CUDA;
  }
  return UQ_OK;
}


// ---------------------------------------------------------------- head_dim 64 / 256: the float64 path, any D
// One warp per (aligned octet of positions, kv head) or per query row, dealt out exactly as in append_kernel; a lane
// owns N = D/32 consecutive channels (2 or 8), a 32-channel scale group is 32/N lanes.  Everything is float64 on exact
// sums (uq_quant.cuh's rules: the decisions are the oracle's); no float32 fast path and no bulk kernel for these head
// sizes — the tuned kernels above are written for head_dim 128, the geometry of every BASELINE.json config.
template <int D>
__device__ __forceinline__ void load_row(const uint16_t* row, int lane, double (&x)[D / 32]) {
  if constexpr (D == 64) {
    const uint32_t raw = *reinterpret_cast<const uint32_t*>(row + 2 * lane);
    x[0] = bf16_bits_to_double(raw & 0xFFFFu);
    x[1] = bf16_bits_to_double(raw >> 16);
  } else if constexpr (D == 128) {
    load4(row, lane, x);
  } else {
    const uint4 raw = *reinterpret_cast<const uint4*>(row + 8 * lane);
    const uint32_t w[4] = {raw.x, raw.y, raw.z, raw.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      x[2 * i] = bf16_bits_to_double(w[i] & 0xFFFFu);
      x[2 * i + 1] = bf16_bits_to_double(w[i] >> 16);
    }
  }
}

// y = H_D x / sqrt(D) (Sylvester order): index bits 0..log2(N)-1 inside the lane, the other five through shuffles
template <int D>
__device__ __forceinline__ void wht_any(double (&x)[D / 32], int lane) {
  constexpr int N = D / 32;
#pragma unroll
  for (int h = 1; h < N; h <<= 1) {
#pragma unroll
    for (int i = 0; i < N; ++i) {
      if ((i & h) == 0) {
        const double a = x[i], b = x[i | h];
        x[i] = __dadd_rn(a, b);
        x[i | h] = __dadd_rn(a, -b);
      }
    }
  }
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    const bool upper = (lane >> k) & 1;
#pragma unroll
    for (int r = 0; r < N; ++r) {
      const double other = __shfl_xor_sync(kFull, x[r], 1 << k);
      x[r] = upper ? __dadd_rn(other, -x[r]) : __dadd_rn(x[r], other);
    }
  }
  // correctly rounded 2^(-log2(D)/2): exact powers of two for D = 64 and 256
  const double kappa = D == 64 ? 0x1p-3 : D == 256 ? 0x1p-4 : 0x1.6a09e667f3bcdp-4;
#pragma unroll
  for (int r = 0; r < N; ++r) x[r] = __dmul_rn(x[r], kappa);
}

// scale exponent of the lane's 32-channel group (32/N lanes)
template <int D>
__device__ __forceinline__ int group_exponent_any(const double (&y)[D / 32], double c) {
  constexpr int N = D / 32;
  double m = fabs(y[0]);
#pragma unroll
  for (int r = 1; r < N; ++r) m = fmax(m, fabs(y[r]));
#pragma unroll
  for (int s = 1; s < 32 / N; s <<= 1) m = fmax(m, __shfl_xor_sync(kFull, m, s));
  return scale_exponent(c, m);
}

template <int D>
__device__ __forceinline__ void append_octet_any(const uint16_t* __restrict__ k_new, const uint16_t* __restrict__ v_new,
                                                 uint8_t* rec, int c0, int p0, int q0, int t_lo, int t_hi, int h, int Hkv,
                                                 int lane, double c_k, double c_v) {
  using R = RecordGeo<D>;
  constexpr int N = D / 32, LPG = 32 / N;               // channels per lane, lanes per scale group
  uint32_t* dst = reinterpret_cast<uint32_t*>(rec + R::kVCodes + 4 * D * ((q0 >> 3) & 1) + 4 * N * lane);
  uint32_t vw[N];
#pragma unroll
  for (int r = 0; r < N; ++r) vw[r] = 0u;
  for (int pos = t_lo; pos < t_hi; ++pos) {
    const long long row = ((long long)(c0 + (pos - p0)) * Hkv + h) * D;
    const int t = pos & 15;
    double x[N];
    // ---- K: rotate, group exponent, codes in logical order, scale bytes
    load_row<D>(k_new + row, lane, x);
    wht_any<D>(x, lane);
    int E = group_exponent_any<D>(x, c_k);
    uint32_t kc = 0u;
#pragma unroll
    for (int r = 0; r < N; ++r) kc |= e2m1_code(x[r], E) << (4 * r);
    if constexpr (N == 2) rec[R::kKCodes + (D / 2) * t + lane] = (uint8_t)kc;
    else *reinterpret_cast<uint32_t*>(rec + R::kKCodes + (D / 2) * t + 4 * lane) = kc;
    if ((lane % LPG) == 0) rec[R::kKScales + (D / 32) * t + lane / LPG] = (uint8_t)(E + 127);
    // ---- V: no rotation; the token's nibble of every channel word, scale bytes
    load_row<D>(v_new + row, lane, x);
    E = group_exponent_any<D>(x, c_v);
#pragma unroll
    for (int r = 0; r < N; ++r) vw[r] |= e2m1_code(x[r], E) << (4 * (pos & 7));
    if ((lane % LPG) == 0) rec[R::kVScales + (D / 4) * (t >> 3) + 8 * (lane / LPG) + (t & 7)] = (uint8_t)(E + 127);
  }
  // the tokens of the octet that are not part of the call keep their nibbles
  const uint32_t below_hi = (t_hi - q0 == 8) ? 0xFFFFFFFFu : ((1u << (4 * (t_hi - q0))) - 1u);
  const uint32_t m = below_hi & ~((1u << (4 * (t_lo - q0))) - 1u);
#pragma unroll
  for (int r = 0; r < N; ++r) dst[r] = (m == 0xFFFFFFFFu) ? vw[r] : ((dst[r] & ~m) | (vw[r] & m));
}

template <int D>
__global__ void __launch_bounds__(128)
append_any_kernel(const uint16_t* __restrict__ k_new, const uint16_t* __restrict__ v_new,
                  const int32_t* __restrict__ cu_new, const int32_t* __restrict__ seq_lens,
                  const int32_t* __restrict__ block_tables, int max_pages, int batch, int total_new,
                  int Hq, int Hkv, uint8_t* __restrict__ cache, const uint16_t* __restrict__ q,
                  uint8_t* __restrict__ q_fp8, double c_k, double c_v) {
  pdl_launch_dependents();
  pdl_wait();
  constexpr int N = D / 32;
  const int lane = threadIdx.x & 31;
  if ((int)blockIdx.y < Hkv) {                         // K/V units: see append_kernel
    const int u = (int)blockIdx.x * 4 + (int)(threadIdx.x >> 5), h = (int)blockIdx.y;
    const int n_units = (total_new >> 3) + 2 * batch;
    if (total_new == 0 || u >= n_units) return;
    const int b = find_sequence<3>(cu_new, batch, u, n_units, lane);
    const int c0 = cu_new[b], cnt = cu_new[b + 1] - c0, p0 = seq_lens[b];
    const int q0 = ((p0 >> 3) + (u - ((c0 >> 3) + 2 * b))) << 3;
    const int t_lo = max(p0, q0), t_hi = min(p0 + cnt, q0 + 8);
    if (t_lo >= t_hi) return;
    const int page = block_tables[(long long)b * max_pages + (q0 >> 4)];
    uint8_t* rec = cache + ((long long)page * Hkv + h) * RecordGeo<D>::kBytes;
    append_octet_any<D>(k_new, v_new, rec, c0, p0, q0, t_lo, t_hi, h, Hkv, lane, c_k, c_v);
    return;
  }
  const long long qu = ((long long)((int)blockIdx.y - Hkv) * gridDim.x + blockIdx.x) * 4 + (threadIdx.x >> 5);
  if (q != nullptr && qu < (long long)batch * Hq) {    // query rows: rotate, E4M3 bytes
    double x[N];
    load_row<D>(q + qu * D, lane, x);
    wht_any<D>(x, lane);
    if constexpr (N == 2) {
      *reinterpret_cast<uint16_t*>(q_fp8 + qu * D + 2 * lane) = (uint16_t)(e4m3_byte(x[0]) | (e4m3_byte(x[1]) << 8));
    } else {
#pragma unroll
      for (int w = 0; w < N / 4; ++w)
        *reinterpret_cast<uint32_t*>(q_fp8 + qu * D + N * lane + 4 * w) =
            e4m3_byte(x[4 * w]) | (e4m3_byte(x[4 * w + 1]) << 8) | (e4m3_byte(x[4 * w + 2]) << 16) | (e4m3_byte(x[4 * w + 3]) << 24);
    }
  }
}

}  // namespace
}  // namespace uq

extern "C" int32_t uq_rotate_quantize_append(const uq_config* cfg, const void* k_new, const void* v_new,
                                             const int32_t* cu_new, const int32_t* seq_lens,
                                             const int32_t* block_tables, int32_t max_pages,
                                             int32_t batch, int32_t total_new, void* cache,
                                             int64_t num_pages, const void* q, void* q_fp8,
                                             void* stream) {
  using namespace uq;
  NvtxRange nvtx_range("uq_rotate_quantize_append");
  int32_t st = check_config(cfg);
  if (st != UQ_OK) return st;
  if (batch <= 0 || total_new < 0 || max_pages <= 0 || num_pages <= 0) {
    set_error("append: batch/max_pages/num_pages must be positive, total_new >= 0");
    return UQ_ERR_INVALID_ARG;
  }
  if (total_new > 0 && (!k_new || !v_new || !cu_new || !seq_lens || !block_tables || !cache)) {
    set_error("append: NULL pointer");
    return UQ_ERR_INVALID_ARG;
  }
  if ((q == nullptr) != (q_fp8 == nullptr)) {
    set_error("append: q and q_fp8 must both be given or both be NULL");
    return UQ_ERR_INVALID_ARG;
  }
  if (((uintptr_t)k_new | (uintptr_t)v_new | (uintptr_t)q) & 7u || ((uintptr_t)cache & 15u) ||
      ((uintptr_t)q_fp8 & 3u)) {
    set_error("append: misaligned pointer (k/v/q 8 B, cache 16 B, q_fp8 4 B)");
    return UQ_ERR_INVALID_ARG;
  }
  const long long q_rows = q ? (long long)batch * cfg->num_q_heads : 0;
  if (total_new == 0 && q_rows == 0) return UQ_OK;
  if ((cfg->flags & UQ_FLAG_DEBUG_CHECKS) && total_new > 0) {
    st = debug_check_tables("uq_rotate_quantize_append", block_tables, max_pages, batch, num_pages, seq_lens, cu_new,
                            total_new, 0, cfg->page_size, 1, (cudaStream_t)stream);
    if (st != UQ_OK) return st;
  }
  if (cfg->head_dim == 256 && (((uintptr_t)k_new | (uintptr_t)v_new | (uintptr_t)q) & 15u)) {
    set_error("append: head_dim 256 needs k_new / v_new / q 16-byte aligned");
    return UQ_ERR_INVALID_ARG;
  }
  if (cfg->head_dim != kHeadDim) {                     // head_dim 64 / 256: the generic float64 kernel, same grid shape
    long long gx = total_new > 0 ? (((long long)(total_new >> 3) + 2LL * batch) + 3) / 4 : 0;
    gx = gx > (q_rows + 4 * 60000LL - 1) / (4 * 60000LL) ? gx : (q_rows + 4 * 60000LL - 1) / (4 * 60000LL);
    if (gx < 1) gx = 1;
    const long long gy = cfg->num_kv_heads + (q_rows + 4 * gx - 1) / (4 * gx);
    if (gx > 0x7fffffffLL || gy > 65535) {
      set_error("append: too many work units");
      return UQ_ERR_INVALID_ARG;
    }
    auto kern = cfg->head_dim == 64 ? append_any_kernel<64> : append_any_kernel<256>;
    return check_cuda(launch_pdl(kern, dim3((unsigned)gx, (unsigned)gy), dim3(128), 0, (cudaStream_t)stream,
                                 (const uint16_t*)k_new, (const uint16_t*)v_new, cu_new, seq_lens, block_tables,
                                 (int)max_pages, (int)batch, (int)total_new, (int)cfg->num_q_heads,
                                 (int)cfg->num_kv_heads, (uint8_t*)cache, (const uint16_t*)q, (uint8_t*)q_fp8,
                                 (double)cfg->c_k, (double)cfg->c_v),
                      "uq_rotate_quantize_append (head_dim 64/256) launch");
  }
  // Prefill-sized calls (on average 64 or more new tokens per sequence): K/V through append_bulk_kernel, one warp per
  // page; the kernel below then only encodes the query rows.  Same bytes either way.
  if (total_new >= 1024 && (long long)total_new >= 64LL * batch && !(((uintptr_t)k_new | (uintptr_t)v_new) & 15u) &&
      !(cfg->flags & UQ_FLAG_NO_BULK_APPEND)) {
    st = opt_in_dynamic_smem((const void*)append_bulk_kernel, kBulkSmem, "append: cudaFuncSetAttribute");
    if (st != UQ_OK) return st;
    CUtensorMap tmap_k, tmap_v;
    st = rows_map(k_new, total_new, cfg->num_kv_heads, &tmap_k);
    if (st == UQ_OK) st = rows_map(v_new, total_new, cfg->num_kv_heads, &tmap_v);
    if (st != UQ_OK) return st;
    const long long n_units = (long long)(total_new >> 4) + 2LL * batch;
    const long long bx = (n_units + kBulkWarps - 1) / kBulkWarps;
    if (bx > 0x7fffffffLL) {
      set_error("append: too many work units");
      return UQ_ERR_INVALID_ARG;
    }
    st = check_cuda(launch_pdl(append_bulk_kernel, dim3((unsigned)bx, (unsigned)cfg->num_kv_heads), dim3(32 * kBulkWarps),
                               (size_t)kBulkSmem, (cudaStream_t)stream, tmap_k, tmap_v, (const uint16_t*)k_new,
                               (const uint16_t*)v_new, cu_new, seq_lens, block_tables, (int)max_pages, (int)batch, (int)total_new,
                               (int)cfg->num_kv_heads, (uint8_t*)cache, (double)cfg->c_k, (double)cfg->c_v),
                    "uq_rotate_quantize_append (bulk) launch");
    if (st != UQ_OK || q_rows == 0) return st;
    total_new = 0;                                     // the query rows are left
  }
  // grid.x: blocks of 4 K/V units (one aligned octet of positions each; grid.y = kv head) — widened if the query
  // rows would need more than 60000 further grid rows; grid.y beyond the kv heads: query rows, 4 * grid.x per row
  long long gx = total_new > 0 ? (((long long)(total_new >> 3) + 2LL * batch) + 3) / 4 : 0;
  gx = gx > (q_rows + 4 * 60000LL - 1) / (4 * 60000LL) ? gx : (q_rows + 4 * 60000LL - 1) / (4 * 60000LL);
  if (gx < 1) gx = 1;
  const long long gy = cfg->num_kv_heads + (q_rows + 4 * gx - 1) / (4 * gx);
  if (gx > 0x7fffffffLL || gy > 65535) {
    set_error("append: too many work units");
    return UQ_ERR_INVALID_ARG;
  }
  return check_cuda(launch_pdl(append_kernel, dim3((unsigned)gx, (unsigned)gy), dim3(128), 0, (cudaStream_t)stream,
                               (const uint16_t*)k_new, (const uint16_t*)v_new, cu_new, seq_lens, block_tables,
                               (int)max_pages, (int)batch, (int)total_new, (int)cfg->num_q_heads,
                               (int)cfg->num_kv_heads, (uint8_t*)cache, (const uint16_t*)q, (uint8_t*)q_fp8,
                               (double)cfg->c_k, (double)cfg->c_v),
                    "uq_rotate_quantize_append launch");
}
