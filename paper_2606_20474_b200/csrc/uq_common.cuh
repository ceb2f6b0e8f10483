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

// Programmatic dependent launch.  The three kernels of a decode step (append -> decode -> merge) are short and
// run back to back on one stream: each is launched with programmatic stream serialization, announces right
// away that its dependents may be launched (their CTAs become resident and run their own prologue as resources
// allow), and waits for the grid before it in the stream — complete, memory visible — before it touches
// global memory that grid may have written.  Behind a kernel that is not part of the scheme (or a copy) the
// launch is ordered as usual.
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
#endif
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream,
                              Args&&... args) {
  cudaLaunchConfig_t lc = {};
  lc.gridDim = grid;
  lc.blockDim = block;
  lc.dynamicSmemBytes = smem;
  lc.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  lc.attrs = attr;
  lc.numAttrs = 1;
  return cudaLaunchKernelEx(&lc, kernel, KArgs(args)...);
}

// TMA descriptors of the decode kernels (uq_decode.cu): the K codes of the cache as a packed 4-bit tensor (cached
// per cache pointer), and q_fp8 as [rows][128] bytes with a box of 16 rows.
#ifdef CUDA_VERSION
int32_t k_code_map(const void* cache, long long records, CUtensorMap* out);
int32_t q_map(const void* q_fp8, long long rows, CUtensorMap* out);
#endif

inline float resolved_sm_scale(const uq_config* cfg) {
  return cfg->sm_scale != 0.0f ? cfg->sm_scale : 0.08838834764831845f;  // 1/sqrt(128)
}

}  // namespace uq
