// uq_append.cu — quantize-on-append: Alg. 1 "Write" l.1-5 and "Decode" l.6 of
// arxiv/paper_2606_20474.
//
// Record layout: include/uq.h.  One warp per (new token pair, kv head) or per (sequence, q head).  A lane owns 4 consecutive
// channels of the 128-channel vector.  The Walsh-Hadamard rotation is an in-register butterfly:
// index bits 0-1 inside the lane, bits 2-6 through warp shuffles.  All of it runs in float64:
// sums of 128 bf16 values are exact in double, so every rounding decision (scale exponent,
// E2M1 level, E4M3 byte) is taken on the same real numbers the float64 oracle sees
// (reading G1).  __dadd_rn/__dmul_rn keep the compiler from contracting into FMAs.
#include "uq_common.cuh"

namespace uq {
namespace {

constexpr unsigned kFull = 0xffffffffu;

__device__ __forceinline__ double bf16_bits_to_double(uint32_t bits16) {
  return (double)__uint_as_float(bits16 << 16);
}

// y = H_128 x * 2^-3.5 for the 4 channels {4*lane .. 4*lane+3} held in x[0..3].
__device__ __forceinline__ void wht128(double (&x)[4], int lane) {
  // index bit 0
  double a0 = __dadd_rn(x[0], x[1]), a1 = __dadd_rn(x[0], -x[1]);
  double a2 = __dadd_rn(x[2], x[3]), a3 = __dadd_rn(x[2], -x[3]);
  // index bit 1
  x[0] = __dadd_rn(a0, a2);
  x[2] = __dadd_rn(a0, -a2);
  x[1] = __dadd_rn(a1, a3);
  x[3] = __dadd_rn(a1, -a3);
  // index bits 2..6 = lane bits 0..4
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    const bool upper = (lane >> k) & 1;
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const double other = __shfl_xor_sync(kFull, x[r], 1 << k);
      x[r] = upper ? __dadd_rn(other, -x[r]) : __dadd_rn(x[r], other);
    }
  }
  const double kappa = 0x1.6a09e667f3bcdp-4;  // correctly rounded 2^-3.5
#pragma unroll
  for (int r = 0; r < 4; ++r) x[r] = __dmul_rn(x[r], kappa);
}

// E = round(log2(c*m)) by exponent extraction and one compare against the double just above
// 1/sqrt(2) (no log2 evaluation); clamped to the UE8M0 range.  PAPER.md:253.
__device__ __forceinline__ int scale_exponent(double c, double m) {
  const double t = __dmul_rn(c, m);
  if (!(t > 0.0)) return -127;
  const long long bits = __double_as_longlong(t);
  const int ef = (int)((bits >> 52) & 0x7FF);
  if (ef == 0) return -127;
  const double f = __longlong_as_double((bits & 0x000FFFFFFFFFFFFFLL) | (1022LL << 52));
  int E = (f >= 0x1.6a09e667f3bcdp-1) ? ef - 1022 : ef - 1023;
  return max(-127, min(127, E));
}

// Nearest level of |y|/2^E in {0,.5,1,1.5,2,3,4,6}, ties to the even code, clamp at 6, +0 only.
__device__ __forceinline__ uint32_t e2m1_code(double y, int E) {
  const double inv = __longlong_as_double((long long)(1023 - E) << 52);
  const double r = __dmul_rn(fabs(y), inv);
  const uint32_t mag = (r > 0.25) + (r >= 0.75) + (r > 1.25) + (r >= 1.75) + (r > 2.5) +
                       (r >= 3.5) + (r > 5.0);
  return (mag != 0 && y < 0.0) ? (mag | 8u) : mag;
}

// OCP E4M3, round-to-nearest-even from the double, saturating, +0 only.  PAPER.md:259.
__device__ __forceinline__ uint32_t e4m3_byte(double y) {
  const double a = fabs(y);
  uint32_t mag;
  if (!(a > 0.0)) {
    mag = 0;
  } else if (a >= 448.0) {
    mag = 0x7E;
  } else if (a < 0x1p-6) {
    mag = (uint32_t)__double2int_rn(__dmul_rn(a, 512.0));
  } else {
    const long long bits = __double_as_longlong(a);
    int e = (int)((bits >> 52) & 0x7FF) - 1023;
    const double sc = __longlong_as_double((long long)(1023 + 3 - e) << 52);
    int n = __double2int_rn(__dmul_rn(a, sc));
    if (n == 16) { n = 8; e += 1; }
    mag = (e > 8 || (e == 8 && n > 14)) ? 0x7Eu : (uint32_t)(((e + 7) << 3) | (n - 8));
  }
  return (mag != 0 && y < 0.0) ? (mag | 0x80u) : mag;
}

// Group (8 lanes x 4 channels) absmax -> exponent; returns E, identical in all 8 lanes.
__device__ __forceinline__ int group_exponent(const double (&y)[4], double c) {
  double m = fmax(fmax(fabs(y[0]), fabs(y[1])), fmax(fabs(y[2]), fabs(y[3])));
#pragma unroll
  for (int s = 1; s <= 4; s <<= 1) m = fmax(m, __shfl_xor_sync(kFull, m, s));
  return scale_exponent(c, m);
}

__device__ __forceinline__ void load4(const uint16_t* row, int lane, double (&x)[4]) {
  const uint2 raw = *reinterpret_cast<const uint2*>(row + 4 * lane);
  x[0] = bf16_bits_to_double(raw.x & 0xFFFFu);
  x[1] = bf16_bits_to_double(raw.x >> 16);
  x[2] = bf16_bits_to_double(raw.y & 0xFFFFu);
  x[3] = bf16_bits_to_double(raw.y >> 16);
}

// Encode + store K of one token: codes into the word-permuted K block, scale word.
__device__ __forceinline__ void store_k(const uint16_t* krow, uint8_t* rec, int t, int lane, double c_k) {
  double x[4];
  load4(krow, lane, x);
  wht128(x, lane);
  const int E = group_exponent(x, c_k);
  uint32_t h16 = e2m1_code(x[0], E) | (e2m1_code(x[1], E) << 4) | (e2m1_code(x[2], E) << 8) |
                 (e2m1_code(x[3], E) << 12);
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
  double x[4];
  load4(vrow, lane, x);
  const int E = group_exponent(x, c_v);
  if ((lane & 7) == 0) rec[kOffVScales + 32 * (t >> 3) + 8 * (lane >> 3) + (t & 7)] = (uint8_t)(E + 127);
  return e2m1_code(x[0], E) | (e2m1_code(x[1], E) << 8) | (e2m1_code(x[2], E) << 16) |
         (e2m1_code(x[3], E) << 24);
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
  const long long unit = (long long)blockIdx.x * 4 + (threadIdx.x >> 5);
  const long long kv_units = (long long)total_new * Hkv;
  if (unit < kv_units) {
    const int n = (int)(unit / Hkv), h = (int)(unit % Hkv);
    // largest b with cu_new[b] <= n: first the guess for evenly spread tokens (the decode step appends one
    // token per sequence) checked with two independent loads, else a binary search (log2(batch) dependent loads)
    int b = (int)(((long long)n * batch) / total_new);
    if (!(cu_new[b] <= n && n < cu_new[b + 1])) {
      int lo = 0, hi = batch;
      while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (cu_new[mid] <= n) lo = mid; else hi = mid;
      }
      b = lo;
    }
    const int j = n - cu_new[b];
    const int pos = seq_lens[b] + j;
    const bool odd = pos & 1;
    if (odd && j > 0) return;                 // handled by the warp of the even partner
    const bool has_b = !odd && (n + 1 < cu_new[b + 1]);
    const int page = block_tables[(long long)b * max_pages + (pos >> 4)];
    const int t = pos & 15;
    uint8_t* rec = cache + ((long long)page * Hkv + h) * kRecordBytes;
    const uint16_t* krow = k_new + ((long long)n * Hkv + h) * kHeadDim;
    const uint16_t* vrow = v_new + ((long long)n * Hkv + h) * kHeadDim;
    store_k(krow, rec, t, lane, c_k);
    const uint32_t ca = encode_v(vrow, rec, t, lane, c_v);
    uint32_t cb = 0;
    if (has_b) {
      store_k(krow + (long long)Hkv * kHeadDim, rec, t + 1, lane, c_k);
      cb = encode_v(vrow + (long long)Hkv * kHeadDim, rec, t + 1, lane, c_v);
    }
    // token-major nibbles: channel d = 4*lane + r lives in word 512*(t>>3) + 128*(d>>5) + 4*(d&31),
    // tokens (t, t+1) share byte (t&7)>>1 of that word
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const int d = 4 * lane + r;
      uint8_t* dst = rec + kOffVCodes + 512 * (t >> 3) + 128 * (d >> 5) + 4 * (d & 31) + ((t & 7) >> 1);
      const uint32_t a4 = (ca >> (8 * r)) & 0xF, b4 = (cb >> (8 * r)) & 0xF;
      *dst = odd ? (uint8_t)((*dst & 0x0F) | (a4 << 4)) : (uint8_t)(a4 | (b4 << 4));
    }
    return;
  }
  const long long qu = unit - kv_units;
  if (q != nullptr && qu < (long long)batch * Hq) {
    double x[4];
    load4(q + qu * kHeadDim, lane, x);
    wht128(x, lane);
    const uint32_t w = e4m3_byte(x[0]) | (e4m3_byte(x[1]) << 8) | (e4m3_byte(x[2]) << 16) |
                       (e4m3_byte(x[3]) << 24);
    *reinterpret_cast<uint32_t*>(q_fp8 + qu * kHeadDim + 4 * lane) = w;
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
  const long long units = (long long)total_new * cfg->num_kv_heads +
                          (q ? (long long)batch * cfg->num_q_heads : 0);
  if (units == 0) return UQ_OK;
  const long long blocks = (units + 3) / 4;
  if (blocks > 0x7fffffffLL) {
    set_error("append: too many work units");
    return UQ_ERR_INVALID_ARG;
  }
  return check_cuda(launch_pdl(append_kernel, dim3((unsigned)blocks), dim3(128), 0, (cudaStream_t)stream,
                               (const uint16_t*)k_new, (const uint16_t*)v_new, cu_new, seq_lens, block_tables,
                               (int)max_pages, (int)batch, (int)total_new, (int)cfg->num_q_heads,
                               (int)cfg->num_kv_heads, (uint8_t*)cache, (const uint16_t*)q, (uint8_t*)q_fp8,
                               (double)cfg->c_k, (double)cfg->c_v),
                    "uq_rotate_quantize_append launch");
}
