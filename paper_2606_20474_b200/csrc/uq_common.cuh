// uq_common.cuh — shared host-side helpers of libuq.so (error string, config checks) and the
// record-layout constants documented in include/uq.h.  CUDA path only; the oracle shares
// nothing with this file.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/uq.h"

namespace uq {

constexpr int kHeadDim = 128;
constexpr int kGroup = 32;
constexpr int kPage = 16;
constexpr int kRecordBytes = UQ_RECORD_BYTES;  // 2176
constexpr int kOffKCodes = 0;
constexpr int kOffVCodes = 1024;
constexpr int kOffKScales = 2048;
constexpr int kOffVScales = 2112;

void set_error(const char* fmt, ...);
int32_t check_config(const uq_config* cfg);  // UQ_OK / UQ_ERR_*; sets the error string
int32_t check_cuda(cudaError_t e, const char* what);

inline float resolved_sm_scale(const uq_config* cfg) {
  return cfg->sm_scale != 0.0f ? cfg->sm_scale : 0.08838834764831845f;  // 1/sqrt(128)
}

}  // namespace uq
