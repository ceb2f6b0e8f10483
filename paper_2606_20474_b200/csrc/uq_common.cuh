// uq_common.cuh — shared host-side helpers of libuq.so (error string, config checks) and the
// record-layout constants documented in include/uq.h.  CUDA path only; the oracle shares
// nothing with this file.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/uq.h"

namespace uq {

constexpr int kHeadDim = 128;                  // the head_dim the tuned kernels are written for
constexpr int kGroup = 32;
constexpr int kPage = 16;
constexpr int kRecordBytes = UQ_RECORD_BYTES;  // 2176
constexpr int kOffKCodes = 0;
constexpr int kOffVCodes = 1024;
constexpr int kOffKScales = 2048;
constexpr int kOffVScales = 2112;

// Record geometry for head_dim D in {64, 128, 256} (include/uq.h "PHYSICAL CACHE LAYOUT"): 16 tokens x (D/2 + D/32)
// bytes for K and the same for V = 17 D bytes; K codes | V codes | K scales | V scales.
template <int D>
struct RecordGeo {
  static_assert(D == 64 || D == 128 || D == 256, "head_dim must be 64, 128 or 256");
  static constexpr int kGroups = D / kGroup;           // scale bytes per vector
  static constexpr int kBytes = 17 * D;                // 1088 / 2176 / 4352
  static constexpr int kKCodes = 0;                    // 16 x D/2
  static constexpr int kVCodes = 8 * D;                // 2 octets x D words
  static constexpr int kKScales = 16 * D;              // 16 x D/32
  static constexpr int kVScales = 16 * D + D / 2;      // 2 octets x D/32 groups x 8
  static constexpr int kRest = 9 * D;                  // the record without its K codes
};
static_assert(RecordGeo<128>::kBytes == kRecordBytes && RecordGeo<128>::kVCodes == kOffVCodes &&
              RecordGeo<128>::kKScales == kOffKScales && RecordGeo<128>::kVScales == kOffVScales, "layout");

// NVTX range around an ABI call (tracing).  nvtx3 is header-only and does nothing unless a tool (nsys, ncu
// --nvtx) has injected its library into the process: one predictable branch per call otherwise.
struct NvtxRange {
  explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
  ~NvtxRange() { nvtxRangePop(); }
  NvtxRange(const NvtxRange&) = delete;
  NvtxRange& operator=(const NvtxRange&) = delete;
};

// Ultra-TQ comparison cache (Alg. 2; include/uq.h "ULTRA-TQ"): record regions and the codebook as it
// is handed to the kernels (by value: 16 levels)
constexpr int kTqRecord = 2432;                // K indices 1024 | K block norms 128 | V codes 1024 | V scale / zero 256
constexpr int kTqKNorms = 1024, kTqVCodes = 1152, kTqVMeta = 2176;
struct TqCodebook {
  float c[16];
};

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

// Per-DEVICE host state (uq_api.cu).  The library may be called on several devices of one process (the caller's
// cudaSetDevice decides): the SM count sizes the one-wave grids, and the dynamic-shared-memory opt-in of a kernel is a
// per-device function attribute.  Both are looked up for the current device under a mutex.
int32_t current_device_sms(int* sms);                                   // UQ_OK / UQ_ERR_CUDA
int32_t opt_in_dynamic_smem(const void* kernel, int bytes, const char* what);   // once per (kernel, device)

// UQ_FLAG_DEBUG_CHECKS (uq_debug.cu): validates on the device the table entries / lengths a call is going to use and
// synchronises the stream; mode 0 decode, 1 append, 2 shared prefix (fixed_pages entries equal to sequence 0's).
int32_t debug_check_tables(const char* who, const int32_t* block_tables, int max_pages, int batch, long long num_pages,
                           const int32_t* seq_lens, const int32_t* cu_new, int total_new, int fixed_pages, int page,
                           int mode, cudaStream_t stream);

// TMA descriptors.  cuTensorMapEncodeTiled is fetched once through the runtime (no link-time dependency on
// libcuda); k_code_map: the K codes of the cache as a packed 4-bit tensor (descriptors cached per cache pointer);
// q_map: q_fp8 as [rows][128] bytes with a box of 16 rows.
#ifdef CUDA_VERSION
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn();                                        // nullptr (error string set) if unavailable
int32_t launch_prefix_m(const uq_config* cfg, const void* q_fp8, const void* cache, long long records,
                        const int32_t* block_tables, int32_t max_pages, int32_t batch, int32_t prefix_len,
                        int32_t num_splits, float* partial_acc, float* partial_ml, cudaStream_t stream);
int32_t k_code_map(const void* cache, long long records, int head_dim, CUtensorMap* out, CUtensorMap* out_rest = nullptr);
int32_t q_map(const void* q_fp8, long long rows, int head_dim, CUtensorMap* out);
#endif

inline float resolved_sm_scale(const uq_config* cfg) {
  if (cfg->sm_scale != 0.0f) return cfg->sm_scale;
  return cfg->head_dim == 64 ? 0.125f : cfg->head_dim == 256 ? 0.0625f : 0.08838834764831845f;  // 1/sqrt(head_dim)
}
// entry points whose kernels exist for head_dim 128 only
int32_t require_head_dim_128(const uq_config* cfg, const char* who);

}  // namespace uq
