// uq_tq_append.cu — the write path of the paper's Algorithm 2, "Calibrated LUT int4 KV encoding (Ultra-TQ)"
// (PAPER.md:453-473, l.1-4), and the rotated bf16 query of l.5: the codebook cache that uq_tq_decode_attention
// (uq_decode_cmp.cu) reads — the last comparison kernel of SURVEY 8(f) rank 4.  Readings: DESIGN.md G20.
// One warp per new (token, kv head) row and per query row, a lane owns 4 consecutive channels; every decision (norm,
// nearest codebook entry, scale / zero, uniform code) is taken in float64 on the same real numbers as the oracle:
// not a tuned kernel.  CUDA path only; the oracle shares nothing with this file.
#include <cuda_bf16.h>

#include "uq_quant.cuh"

namespace uq {
namespace {

// double -> the nearest bf16 (ties to even) and back
__device__ __forceinline__ double bf16_rne(double x, uint32_t* bits) {
  const __nv_bfloat16 h = __double2bfloat16(x);
  *bits = __bfloat16_as_ushort(h);
  return (double)__bfloat162float(h);
}

__global__ void __launch_bounds__(128)
append_tq_kernel(const uint16_t* __restrict__ k_new, const uint16_t* __restrict__ v_new, const int32_t* __restrict__ cu_new,
                 const int32_t* __restrict__ seq_lens, const int32_t* __restrict__ block_tables, int max_pages, int batch,
                 int total_new, int Hq, int Hkv, uint8_t* __restrict__ cache, const uint16_t* __restrict__ q,
                 uint16_t* __restrict__ q_rot, const TqCodebook cb) {
  pdl_launch_dependents();
  pdl_wait();
  const int lane = threadIdx.x & 31;
  const long long u = (long long)blockIdx.x * 4 + (threadIdx.x >> 5);
  const long long n_kv = (long long)total_new * Hkv;
  if (u >= n_kv) {                                     // l.5: Q <- R Q, rounded to bf16
    const long long qu = u - n_kv;
    if (q != nullptr && qu < (long long)batch * Hq) {
      double x[4];
      load4(q + qu * kHeadDim, lane, x);
      wht128(x, lane);
      uint32_t b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) bf16_rne(x[i], &b[i]);
      *reinterpret_cast<uint2*>(q_rot + qu * kHeadDim + 4 * lane) = make_uint2(b[0] | (b[1] << 16), b[2] | (b[3] << 16));
    }
    return;
  }
  const int row = (int)(u / Hkv), h = (int)(u - (long long)row * Hkv);
  int lo = 0, hi = batch;                              // the sequence of new row `row`: largest b with cu_new[b] <= row
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (cu_new[mid] <= row) lo = mid; else hi = mid;
  }
  const int b = lo, pos = seq_lens[b] + (row - cu_new[b]), t = pos & 15;
  const int page = block_tables[(long long)b * max_pages + (pos >> 4)];
  uint8_t* rec = cache + ((long long)page * Hkv + h) * kTqRecord;
  const long long src = ((long long)row * Hkv + h) * kHeadDim;
  const int g = lane >> 3, l8 = lane & 7;              // 32-channel block, lane within it

  // ---- K (l.1-3): rotate, block norm (coordinate order), nearest codebook entry of x / norm
  {
    double x[4];
    load4(k_new + src, lane, x);
    wht128(x, lane);
    double acc = 0.0;
#pragma unroll
    for (int s = 0; s < 8; ++s) {                      // the block's 32 squares in coordinate order: lane s of the block adds its 4
      double a = acc;
#pragma unroll
      for (int i = 0; i < 4; ++i) a = __dadd_rn(a, __dmul_rn(x[i], x[i]));
      acc = __shfl_sync(kFull, a, 8 * g + s);
    }
    uint32_t nbits;
    const double ns = bf16_rne(sqrt(acc), &nbits);
    uint32_t idx[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const double uu = ns > 0.0 ? __ddiv_rn(x[i], ns) : 0.0;
      int best = 0;
      double bd = fabs(__dadd_rn(uu, -(double)cb.c[0]));
#pragma unroll
      for (int c = 1; c < 16; ++c) {
        const double dd = fabs(__dadd_rn(uu, -(double)cb.c[c]));
        if (dd < bd) { bd = dd; best = c; }            // ties keep the lower index
      }
      idx[i] = (uint32_t)best;
    }
    *reinterpret_cast<uint16_t*>(rec + 64 * t + 2 * lane) = (uint16_t)(idx[0] | (idx[1] << 4) | (idx[2] << 8) | (idx[3] << 12));
    if (l8 == 0) *reinterpret_cast<uint16_t*>(rec + kTqKNorms + 8 * t + 2 * g) = (uint16_t)nbits;
  }
  // ---- V (l.4): block (scale, zero) = ((max - min) / 15, min) as bf16, uniform 4-bit codes
  {
    double v[4];
    load4(v_new + src, lane, v);
    double mn = fmin(fmin(v[0], v[1]), fmin(v[2], v[3])), mx = fmax(fmax(v[0], v[1]), fmax(v[2], v[3]));
#pragma unroll
    for (int s = 1; s <= 4; s <<= 1) {
      mn = fmin(mn, __shfl_xor_sync(kFull, mn, s));
      mx = fmax(mx, __shfl_xor_sync(kFull, mx, s));
    }
    uint32_t sbits, zbits;
    const double scale = bf16_rne(__ddiv_rn(__dadd_rn(mx, -mn), 15.0), &sbits), zero = bf16_rne(mn, &zbits);
    // V codes [channel][8 bytes]: word t >> 3 of the channel, token 2n of the octet in nibble n, token 2n + 1 in nibble
    // n + 4; other tokens of the word may be written by other warps of this call: the nibble goes in atomically
    const int tt = t & 7, sh = 4 * ((tt >> 1) + 4 * (tt & 1));
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      double code = scale > 0.0 ? rint(__ddiv_rn(__dadd_rn(v[i], -zero), scale)) : 0.0;
      code = fmin(fmax(code, 0.0), 15.0);
      uint32_t* w = reinterpret_cast<uint32_t*>(rec + kTqVCodes + 8 * (4 * lane + i) + 4 * (t >> 3));
      atomicAnd(w, ~(0xFu << sh));
      atomicOr(w, (uint32_t)code << sh);
    }
    if (l8 == 0) {                                     // block g: scales of the 16 tokens, then their zeros
      *reinterpret_cast<uint16_t*>(rec + kTqVMeta + 64 * g + 2 * t) = (uint16_t)sbits;
      *reinterpret_cast<uint16_t*>(rec + kTqVMeta + 64 * g + 32 + 2 * t) = (uint16_t)zbits;
    }
  }
}

}  // namespace
}  // namespace uq

extern "C" int32_t uq_tq_append(const uq_config* cfg, const float* codebook_k, const void* k_new, const void* v_new,
                                const int32_t* cu_new, const int32_t* seq_lens, const int32_t* block_tables,
                                int32_t max_pages, int32_t batch, int32_t total_new, void* cache, int64_t num_pages,
                                const void* q, void* q_rot, void* stream) {
  using namespace uq;
  NvtxRange nvtx_range("uq_tq_append");
  int32_t st = check_config(cfg);
  if (st != UQ_OK) return st;
  st = require_head_dim_128(cfg, "uq_tq_append");
  if (st != UQ_OK) return st;
  if (!codebook_k || batch <= 0 || total_new < 0 || max_pages <= 0 || num_pages <= 0) {
    set_error("uq_tq_append: codebook_k is NULL, or batch / max_pages / num_pages not positive, or total_new < 0");
    return UQ_ERR_INVALID_ARG;
  }
  if (total_new > 0 && (!k_new || !v_new || !cu_new || !seq_lens || !block_tables || !cache)) {
    set_error("uq_tq_append: NULL pointer");
    return UQ_ERR_INVALID_ARG;
  }
  if ((q == nullptr) != (q_rot == nullptr)) {
    set_error("uq_tq_append: q and q_rot must both be given or both be NULL");
    return UQ_ERR_INVALID_ARG;
  }
  if ((((uintptr_t)k_new | (uintptr_t)v_new | (uintptr_t)q | (uintptr_t)q_rot) & 7u) || ((uintptr_t)cache & 15u)) {
    set_error("uq_tq_append: misaligned pointer (k / v / q / q_rot 8 B, cache 16 B)");
    return UQ_ERR_INVALID_ARG;
  }
  TqCodebook cb;
  for (int i = 0; i < 16; ++i) {
    cb.c[i] = codebook_k[i];
    if (!(cb.c[i] == cb.c[i]) || (i > 0 && !(cb.c[i] > cb.c[i - 1]))) {
      set_error("uq_tq_append: codebook_k must be 16 finite values in ascending order");
      return UQ_ERR_INVALID_ARG;
    }
  }
  if (cfg->flags & UQ_FLAG_DEBUG_CHECKS) {
    st = debug_check_tables("uq_tq_append", block_tables, max_pages, batch, num_pages, seq_lens, cu_new, total_new, 0,
                            cfg->page_size, 1, (cudaStream_t)stream);
    if (st != UQ_OK) return st;
  }
  const long long units = (long long)total_new * cfg->num_kv_heads + (q ? (long long)batch * cfg->num_q_heads : 0);
  if (units == 0) return UQ_OK;
  const long long blocks = (units + 3) / 4;
  if (blocks > 0x7fffffffLL) {
    set_error("uq_tq_append: too many rows for one call");
    return UQ_ERR_INVALID_ARG;
  }
  return check_cuda(launch_pdl(append_tq_kernel, dim3((unsigned)blocks), dim3(128), 0, (cudaStream_t)stream,
                               (const uint16_t*)k_new, (const uint16_t*)v_new, cu_new, seq_lens, block_tables, (int)max_pages,
                               (int)batch, (int)total_new, (int)cfg->num_q_heads, (int)cfg->num_kv_heads, (uint8_t*)cache,
                               (const uint16_t*)q, (uint16_t*)q_rot, cb),
                    "uq_tq_append launch");
}
