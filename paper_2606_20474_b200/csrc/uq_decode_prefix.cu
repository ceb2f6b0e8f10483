// uq_decode_prefix.cu — entry point of the shared-prefix ("cascade") decode: uq_decode_prefix_attention validates its
// arguments here and launches the kernel of uq_decode_prefix_m.cu (query rows of 8 / 16 sequences on the M side of the
// score tile).  The round-1 kernel that lived in this file — tokens on the TMEM lanes, the heads of four sequences side
// by side on the columns, one group of four softmax warps and one consensus barrier per sequence: 334 us for the
// 30,000-token prefix of config 4 — was replaced in round 2 (the history has it).
#include <cuda.h>

#include "uq_common.cuh"

extern "C" int32_t uq_decode_prefix_attention(const uq_config* cfg, const void* q_fp8, const void* cache,
                                              int64_t num_pages, const int32_t* block_tables, int32_t max_pages,
                                              int32_t batch, int32_t prefix_len, int32_t num_splits,
                                              float* partial_acc, float* partial_ml, void* stream) {
  using namespace uq;
  NvtxRange nvtx_range("uq_decode_prefix_attention");
  int32_t st = check_config(cfg);
  if (st != UQ_OK) return st;
  st = require_head_dim_128(cfg, "uq_decode_prefix_attention");
  if (st != UQ_OK) return st;
  if (!q_fp8 || !cache || !block_tables || !partial_acc || !partial_ml || batch <= 0 || max_pages <= 0 ||
      num_pages <= 0) {
    set_error("decode_prefix: NULL pointer or non-positive size");
    return UQ_ERR_INVALID_ARG;
  }
  if (prefix_len <= 0 || prefix_len % 128 != 0 || prefix_len / kPage > max_pages) {
    set_error("decode_prefix: prefix_len must be a positive multiple of 128 tokens within max_pages");
    return UQ_ERR_INVALID_ARG;
  }
  if (num_splits < 2) {
    set_error("decode_prefix: num_splits must be at least 2");
    return UQ_ERR_INVALID_ARG;
  }
  if (((uintptr_t)cache & 31u) || ((uintptr_t)q_fp8 & 15u) || ((uintptr_t)partial_acc & 15u) ||
      ((uintptr_t)partial_ml & 7u)) {
    set_error("decode_prefix: misaligned pointer (cache 32 B, q_fp8 16 B, partial_acc 16 B, partial_ml 8 B)");
    return UQ_ERR_INVALID_ARG;
  }
  const long long records = (long long)num_pages * cfg->num_kv_heads;
  if (records > 0x7fffffffLL) {
    set_error("decode_prefix: num_pages * num_kv_heads must be < 2^31");
    return UQ_ERR_INVALID_ARG;
  }
  if (cfg->flags & UQ_FLAG_DEBUG_CHECKS) {
    st = debug_check_tables("uq_decode_prefix_attention", block_tables, max_pages, batch, num_pages, nullptr, nullptr, 0,
                            prefix_len / cfg->page_size, cfg->page_size, 2, (cudaStream_t)stream);
    if (st != UQ_OK) return st;
  }
  return launch_prefix_m(cfg, q_fp8, cache, records, block_tables, max_pages, batch, prefix_len, num_splits, partial_acc,
                           partial_ml, (cudaStream_t)stream);
}
