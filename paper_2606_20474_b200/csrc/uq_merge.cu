// uq_merge.cu — merge of split-K partials (flash-decoding reduction; not in the paper, exact
// reassociation of the softmax in Alg. 1 l.8; format in include/uq.h).
//
// One warp per (sequence, query head); a lane owns 4 of the 128 output channels (one 16-byte
// load per split, coalesced 512 B per warp).  HBM-bound: reads S*(512+8) B, writes 256 B per row.
#include <cuda_bf16.h>

#include "uq_common.cuh"

namespace uq {
namespace {

__global__ void __launch_bounds__(128)
merge_kernel(const float* __restrict__ acc, const float* __restrict__ ml, int rows, int S,
             __nv_bfloat16* __restrict__ out) {
  pdl_launch_dependents();
  pdl_wait();                                          // the partials come from the kernel before this one
  const int lane = threadIdx.x & 31;
  const int row = blockIdx.x * 4 + (threadIdx.x >> 5);
  if (row >= rows) return;
  const float2* ml2 = reinterpret_cast<const float2*>(ml) + (long long)row * S;
  const float4* a4 = reinterpret_cast<const float4*>(acc) + (long long)row * S * 32 + lane;
  float4 num = make_float4(0.f, 0.f, 0.f, 0.f);
  float den = 0.f;
  if (S <= 8) {
    // the usual case, one round of loads: every lane reads all (m, l) pairs (broadcast) and its 16 bytes of every
    // accumulator before anything is used; the maximum needs no exchange between lanes
    float2 v[8];
    float4 a[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const bool in = k < S;
      v[k] = in ? ml2[k] : make_float2(0.f, 0.f);
      a[k] = in ? a4[(long long)k * 32] : make_float4(0.f, 0.f, 0.f, 0.f);
    }
    float M = -INFINITY;
#pragma unroll
    for (int k = 0; k < 8; ++k)
      if (v[k].y > 0.0f) M = fmaxf(M, v[k].x);
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      if (!(v[k].y > 0.0f)) continue;                  // empty slot (or past the last one)
      const float w = __expf(v[k].x - M);
      num.x = fmaf(w, a[k].x, num.x);
      num.y = fmaf(w, a[k].y, num.y);
      num.z = fmaf(w, a[k].z, num.z);
      num.w = fmaf(w, a[k].w, num.w);
      den = fmaf(w, v[k].y, den);
    }
  } else {
    // pass 1: M = max over non-empty splits (lanes stride over splits, then warp max)
    float M = -INFINITY;
    for (int s = lane; s < S; s += 32) {
      const float2 v = ml2[s];
      if (v.y > 0.0f) M = fmaxf(M, v.x);
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, o));
    if (M > -INFINITY) {
      // eight slots at a time, all loads issued before the first use (the kernel is latency-bound)
      for (int s0 = 0; s0 < S; s0 += 8) {
        float2 v[8];
        float4 a[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const bool in = s0 + k < S;
          v[k] = in ? ml2[s0 + k] : make_float2(0.f, 0.f);
          a[k] = in ? a4[(long long)(s0 + k) * 32] : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          if (!(v[k].y > 0.0f)) continue;              // empty slot (or past the last one)
          const float w = __expf(v[k].x - M);
          num.x = fmaf(w, a[k].x, num.x);
          num.y = fmaf(w, a[k].y, num.y);
          num.z = fmaf(w, a[k].z, num.z);
          num.w = fmaf(w, a[k].w, num.w);
          den = fmaf(w, v[k].y, den);
        }
      }
    }
  }
  const float inv = den > 0.f ? 1.0f / den : 0.f;
  __nv_bfloat162 lo = __floats2bfloat162_rn(num.x * inv, num.y * inv);
  __nv_bfloat162 hi = __floats2bfloat162_rn(num.z * inv, num.w * inv);
  uint2 packed;
  packed.x = *reinterpret_cast<uint32_t*>(&lo);
  packed.y = *reinterpret_cast<uint32_t*>(&hi);
  *reinterpret_cast<uint2*>(out + (long long)row * kHeadDim + 4 * lane) = packed;
}

// Two sets of partials per row (shared-prefix decode: the prefix slots and the suffix slots live in separate
// arrays).  One warp per row, a lane owns 4 channels; first the maximum over both sets, then the weighted sums.
__global__ void __launch_bounds__(128)
merge2_kernel(const float* __restrict__ acc_a, const float* __restrict__ ml_a, int Sa, const float* __restrict__ acc_b,
              const float* __restrict__ ml_b, int Sb, int rows, __nv_bfloat16* __restrict__ out) {
  pdl_launch_dependents();
  pdl_wait();
  const int lane = threadIdx.x & 31;
  const int row = blockIdx.x * 4 + (threadIdx.x >> 5);
  if (row >= rows) return;
  const float2* mla = reinterpret_cast<const float2*>(ml_a) + (long long)row * Sa;
  const float2* mlb = reinterpret_cast<const float2*>(ml_b) + (long long)row * Sb;
  const float4* aa = reinterpret_cast<const float4*>(acc_a) + (long long)row * Sa * 32 + lane;
  const float4* ab = reinterpret_cast<const float4*>(acc_b) + (long long)row * Sb * 32 + lane;
  float M = -INFINITY;
  for (int s = 0; s < Sa + Sb; ++s) {
    const float2 v = s < Sa ? mla[s] : mlb[s - Sa];
    if (v.y > 0.0f) M = fmaxf(M, v.x);
  }
  float4 num = make_float4(0.f, 0.f, 0.f, 0.f);
  float den = 0.f;
  for (int s = 0; s < Sa + Sb; ++s) {
    const float2 v = s < Sa ? mla[s] : mlb[s - Sa];
    if (!(v.y > 0.0f)) continue;                       // empty slot
    const float4 a = s < Sa ? aa[(long long)s * 32] : ab[(long long)(s - Sa) * 32];
    const float w = __expf(v.x - M);
    num.x = fmaf(w, a.x, num.x);
    num.y = fmaf(w, a.y, num.y);
    num.z = fmaf(w, a.z, num.z);
    num.w = fmaf(w, a.w, num.w);
    den = fmaf(w, v.y, den);
  }
  const float inv = den > 0.f ? 1.0f / den : 0.f;
  __nv_bfloat162 lo = __floats2bfloat162_rn(num.x * inv, num.y * inv);
  __nv_bfloat162 hi = __floats2bfloat162_rn(num.z * inv, num.w * inv);
  uint2 packed;
  packed.x = *reinterpret_cast<uint32_t*>(&lo);
  packed.y = *reinterpret_cast<uint32_t*>(&hi);
  *reinterpret_cast<uint2*>(out + (long long)row * kHeadDim + 4 * lane) = packed;
}

// head_dim 64 / 256 (and a cross-check of the kernels above at 128): one warp per row, a lane takes channels
// lane, lane + 32, ... (coalesced 128-byte reads); one or two sets of partials.
__global__ void __launch_bounds__(128)
merge_any_kernel(const float* __restrict__ acc_a, const float* __restrict__ ml_a, int Sa, const float* __restrict__ acc_b,
                 const float* __restrict__ ml_b, int Sb, int rows, int D, __nv_bfloat16* __restrict__ out) {
  pdl_launch_dependents();
  pdl_wait();
  const int lane = threadIdx.x & 31;
  const int row = blockIdx.x * 4 + (threadIdx.x >> 5);
  if (row >= rows) return;
  const float2* mla = reinterpret_cast<const float2*>(ml_a) + (long long)row * Sa;
  const float2* mlb = reinterpret_cast<const float2*>(ml_b) + (long long)row * Sb;
  float M = -INFINITY;
  for (int s = 0; s < Sa + Sb; ++s) {
    const float2 v = s < Sa ? mla[s] : mlb[s - Sa];
    if (v.y > 0.0f) M = fmaxf(M, v.x);
  }
  float num[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  float den = 0.f;
  const int n = D >> 5;                                // channels per lane: 2, 4 or 8
  for (int s = 0; s < Sa + Sb; ++s) {
    const float2 v = s < Sa ? mla[s] : mlb[s - Sa];
    if (!(v.y > 0.0f)) continue;                       // empty slot: its accumulator row is not read
    const float* a = s < Sa ? acc_a + ((long long)row * Sa + s) * D : acc_b + ((long long)row * Sb + (s - Sa)) * D;
    const float w = __expf(v.x - M);
#pragma unroll
    for (int i = 0; i < 8; ++i)
      if (i < n) num[i] = fmaf(w, a[lane + 32 * i], num[i]);
    den = fmaf(w, v.y, den);
  }
  const float inv = den > 0.f ? 1.0f / den : 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i)
    if (i < n) out[(long long)row * D + lane + 32 * i] = __float2bfloat16_rn(num[i] * inv);
}

}  // namespace
}  // namespace uq

extern "C" int32_t uq_merge_splits(const uq_config* cfg, const float* partial_acc, const float* partial_ml,
                                   int32_t batch, int32_t num_splits, void* out_bf16, void* stream) {
  using namespace uq;
  NvtxRange nvtx_range("uq_merge_splits");
  int32_t st = check_config(cfg);
  if (st != UQ_OK) return st;
  if (batch <= 0 || num_splits <= 0 || !partial_acc || !partial_ml || !out_bf16) {
    set_error("merge: NULL pointer or non-positive batch/num_splits");
    return UQ_ERR_INVALID_ARG;
  }
  if (((uintptr_t)partial_acc & 15u) || ((uintptr_t)partial_ml & 7u) || ((uintptr_t)out_bf16 & 7u)) {
    set_error("merge: misaligned pointer (partial_acc 16 B, partial_ml 8 B, out 8 B)");
    return UQ_ERR_INVALID_ARG;
  }
  const int rows = batch * cfg->num_q_heads;
  if (cfg->head_dim != kHeadDim)
    return check_cuda(launch_pdl(merge_any_kernel, dim3((rows + 3) / 4), dim3(128), 0, (cudaStream_t)stream, partial_acc,
                                 partial_ml, (int)num_splits, partial_acc, partial_ml, 0, rows, (int)cfg->head_dim,
                                 (__nv_bfloat16*)out_bf16),
                      "uq_merge_splits (head_dim 64/256) launch");
  return check_cuda(launch_pdl(merge_kernel, dim3((rows + 3) / 4), dim3(128), 0, (cudaStream_t)stream, partial_acc,
                               partial_ml, rows, (int)num_splits, (__nv_bfloat16*)out_bf16),
                    "uq_merge_splits launch");
}

extern "C" int32_t uq_merge_splits2(const uq_config* cfg, const float* acc_a, const float* ml_a, int32_t splits_a,
                                    const float* acc_b, const float* ml_b, int32_t splits_b, int32_t batch,
                                    void* out_bf16, void* stream) {
  using namespace uq;
  NvtxRange nvtx_range("uq_merge_splits2");
  int32_t st = check_config(cfg);
  if (st != UQ_OK) return st;
  if (batch <= 0 || splits_a <= 0 || splits_b <= 0 || !acc_a || !ml_a || !acc_b || !ml_b || !out_bf16) {
    set_error("merge2: NULL pointer or non-positive batch/splits");
    return UQ_ERR_INVALID_ARG;
  }
  if ((((uintptr_t)acc_a | (uintptr_t)acc_b) & 15u) || (((uintptr_t)ml_a | (uintptr_t)ml_b | (uintptr_t)out_bf16) & 7u)) {
    set_error("merge2: misaligned pointer (partial_acc 16 B, partial_ml 8 B, out 8 B)");
    return UQ_ERR_INVALID_ARG;
  }
  const int rows = batch * cfg->num_q_heads;
  if (cfg->head_dim != kHeadDim)
    return check_cuda(launch_pdl(merge_any_kernel, dim3((rows + 3) / 4), dim3(128), 0, (cudaStream_t)stream, acc_a, ml_a,
                                 (int)splits_a, acc_b, ml_b, (int)splits_b, rows, (int)cfg->head_dim,
                                 (__nv_bfloat16*)out_bf16),
                      "uq_merge_splits2 (head_dim 64/256) launch");
  return check_cuda(launch_pdl(merge2_kernel, dim3((rows + 3) / 4), dim3(128), 0, (cudaStream_t)stream, acc_a, ml_a,
                               (int)splits_a, acc_b, ml_b, (int)splits_b, rows, (__nv_bfloat16*)out_bf16),
                    "uq_merge_splits2 launch");
}
