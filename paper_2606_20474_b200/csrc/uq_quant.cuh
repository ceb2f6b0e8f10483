// uq_quant.cuh — the float64 reference arithmetic of the quantiser, shared by the append kernels (uq_append.cu) and
// the calibration kernel (uq_calib.cu): Alg. 1 l.1-4 of arxiv/paper_2606_20474.  One warp per
// 128-channel vector, a lane owns 4 consecutive channels.  All of it in float64: sums of 128 bf16 values are exact
// in double, so every rounding decision is taken on the same real numbers the float64 oracle sees (DESIGN.md
// reading G1).  __dadd_rn / __dmul_rn keep the compiler from contracting into FMAs.  CUDA path only.
#pragma once
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

}  // namespace
}  // namespace uq
