// uq_calib.cu — the objective of Eq.(2) of arxiv/paper_2606_20474 on a grid of constants c:
// "This one-dimensional minimization is solved once, offline, on captured rotated key activations" (:128).
// SURVEY 8(f) rank 3.  Contract: include/uq.h (uq_calibrate_c).
//
// One warp per vector at a time (a lane owns 4 channels; rotation and quantiser are the float64 reference
// arithmetic of uq_quant.cuh, the same decisions the append kernels take), warps stride over the vectors.  The grid
// of constants is walked eight at a time with eight float64 accumulators per lane; a warp reduces them by shuffles
// and adds them to the result with one atomicAdd per constant, so the sums are those of the oracle up to the order
// of the float64 additions.
#include "uq_common.cuh"
#include "uq_quant.cuh"

namespace uq {
namespace {

constexpr int kCalibWarps = 8;
constexpr int kChunk = 8;                              // constants per pass over the vectors

__device__ __forceinline__ double e2m1_level_of(uint32_t mag) {   // {0,.5,1,1.5,2,3,4,6}[mag]
  return mag < 4u ? 0.5 * (double)mag : (mag == 4u ? 2.0 : (mag == 5u ? 3.0 : (mag == 6u ? 4.0 : 6.0)));
}
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o; o >>= 1) v = __dadd_rn(v, __shfl_xor_sync(kFull, v, o));
  return v;
}

__global__ void __launch_bounds__(32 * kCalibWarps)
calib_kernel(const uint16_t* __restrict__ x, long long n_vec, int rotate, const float* __restrict__ c_grid, int n_c,
             int scale_mode, const float* __restrict__ levels, double* __restrict__ sq_err, double* __restrict__ sq_norm) {
  const int lane = threadIdx.x & 31;
  // a codebook other than E2M1: its 8 magnitudes and the 7 midpoints between them (a tie goes to the smaller level)
  double lv[8], th[7];
  if (levels != nullptr) {
#pragma unroll
    for (int i = 0; i < 8; ++i) lv[i] = (double)levels[i];
#pragma unroll
    for (int i = 0; i < 7; ++i) th[i] = __dmul_rn(0.5, __dadd_rn(lv[i], lv[i + 1]));
  }
  const long long w0 = (long long)blockIdx.x * kCalibWarps + (threadIdx.x >> 5), nw = (long long)gridDim.x * kCalibWarps;
  for (int j0 = 0; j0 < n_c; j0 += kChunk) {
    double c[kChunk], acc[kChunk], nrm = 0.0;
#pragma unroll
    for (int j = 0; j < kChunk; ++j) {
      c[j] = (double)c_grid[min(j0 + j, n_c - 1)];     // past the end: a repeat that is not added
      acc[j] = 0.0;
    }
    for (long long v = w0; v < n_vec; v += nw) {
      double y[4];
      load4(x + v * kHeadDim, lane, y);
      if (rotate) wht128(y, lane);                     // Alg. 1 l.1
      if (j0 == 0) {
#pragma unroll
        for (int r = 0; r < 4; ++r) nrm = __dadd_rn(nrm, __dmul_rn(y[r], y[r]));
      }
      double m = fmax(fmax(fabs(y[0]), fabs(y[1])), fmax(fabs(y[2]), fabs(y[3])));   // l.3: the group's absmax
#pragma unroll
      for (int s = 1; s <= 4; s <<= 1) m = fmax(m, __shfl_xor_sync(kFull, m, s));
#pragma unroll
      for (int j = 0; j < kChunk; ++j) {
        if (scale_mode == 1) {                         // Alg. 1 l.3-5 and Eq.(1): the deployed quantiser
          const int E = scale_exponent(c[j], m);
          const double s = __longlong_as_double((long long)(1023 + E) << 52);   // 2^E, |E| <= 127
#pragma unroll
          for (int r = 0; r < 4; ++r) {
            const uint32_t code = e2m1_code(y[r], E);
            const double lev = e2m1_level_of(code & 7u);
            const double e = __dadd_rn(y[r], -__dmul_rn((code & 8u) ? -lev : lev, s));
            acc[j] = __dadd_rn(acc[j], __dmul_rn(e, e));
          }
        } else {                                       // Eq.(2) as printed: s = c m; or the fixed scale s = c
          const double s = (scale_mode == 2) ? c[j] : __dmul_rn(c[j], m);
          if (s > 0.0) {
#pragma unroll
            for (int r = 0; r < 4; ++r) {
              const double q = __ddiv_rn(fabs(y[r]), s);
              double lev;
              if (levels != nullptr) {
                lev = lv[0];
#pragma unroll
                for (int i = 0; i < 7; ++i) lev = (q > th[i]) ? lv[i + 1] : lev;
              } else {
                const uint32_t mag = (q > 0.25) + (q >= 0.75) + (q > 1.25) + (q >= 1.75) + (q > 2.5) + (q >= 3.5) + (q > 5.0);
                lev = e2m1_level_of(mag);
              }
              const double e = __dadd_rn(y[r], -__dmul_rn(y[r] < 0.0 ? -lev : lev, s));
              acc[j] = __dadd_rn(acc[j], __dmul_rn(e, e));
            }
          }
        }
      }
    }
#pragma unroll
    for (int j = 0; j < kChunk; ++j) {
      const double t = warp_sum(acc[j]);
      if (lane == 0 && j0 + j < n_c) atomicAdd(sq_err + j0 + j, t);
    }
    if (j0 == 0) {
      const double t = warp_sum(nrm);
      if (lane == 0) atomicAdd(sq_norm, t);
    }
  }
}

}  // namespace
}  // namespace uq

extern "C" int32_t uq_calibrate_c(const uq_config* cfg, const void* x, int64_t n_vec, int32_t rotate,
                                  const float* c_grid, int32_t n_c, int32_t scale_mode, const float* levels,
                                  double* sq_err, double* sq_norm, void* stream) {
  using namespace uq;
  NvtxRange nvtx_range("uq_calibrate_c");
  int32_t st = check_config(cfg);
  if (st != UQ_OK) return st;
  st = require_head_dim_128(cfg, "uq_calibrate_c");
  if (st != UQ_OK) return st;
  if (!x || !c_grid || !sq_err || !sq_norm || n_vec <= 0 || n_c <= 0) {
    set_error("calibrate: NULL pointer or non-positive size");
    return UQ_ERR_INVALID_ARG;
  }
  if (scale_mode < 0 || scale_mode > 2 || (scale_mode == 1 && levels != nullptr)) {
    set_error("calibrate: scale_mode must be 0, 1 or 2, and the power-of-two scale (1) takes the E2M1 levels only");
    return UQ_ERR_INVALID_ARG;
  }
  if (((uintptr_t)x & 7u) || ((uintptr_t)sq_err & 7u) || ((uintptr_t)sq_norm & 7u) || ((uintptr_t)c_grid & 3u)) {
    set_error("calibrate: misaligned pointer (x 8 B, sq_err / sq_norm 8 B, c_grid 4 B)");
    return UQ_ERR_INVALID_ARG;
  }
  cudaStream_t s = (cudaStream_t)stream;
  cudaError_t e = cudaMemsetAsync(sq_err, 0, sizeof(double) * (size_t)n_c, s);
  if (e == cudaSuccess) e = cudaMemsetAsync(sq_norm, 0, sizeof(double), s);
  if (e != cudaSuccess) return check_cuda(e, "calibrate: cudaMemsetAsync");
  int sm_count = 0;
  st = current_device_sms(&sm_count);
  if (st != UQ_OK) return st;
  long long blocks = (n_vec + kCalibWarps - 1) / kCalibWarps;
  if (blocks > 8LL * sm_count) blocks = 8LL * sm_count;   // a multiple of the SM count; warps stride over the vectors
  calib_kernel<<<(unsigned)blocks, 32 * kCalibWarps, 0, s>>>((const uint16_t*)x, (long long)n_vec, (int)rotate, c_grid,
                                                             (int)n_c, (int)scale_mode, levels, sq_err, sq_norm);
  return check_cuda(cudaGetLastError(), "uq_calibrate_c launch");
}
