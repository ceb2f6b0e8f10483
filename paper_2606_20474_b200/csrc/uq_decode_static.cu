// uq_decode_static.cu — uq_decode_attention_static: split-K decode + merge for callers that cannot allocate (code under
// CUDA graph capture, serving loops and harnesses that forbid cudaMalloc).  The split partials (partial_acc / partial_ml of
// include/uq.h, the only scratch the decode path uses) live in a file-scope __device__ array of UQ_STATIC_SCRATCH_BYTES
// that every GPU which loads libuq.so holds until the process exits; the caller passes inputs and the output only.
// The entry point calls no cudaMalloc / cudaFree and no allocating library routine: it resolves the array's device
// address once per device, lays the two partial buffers out in it and calls the existing uq_decode_attention and
// uq_merge_splits on them (same kernels, same arithmetic, same error bound).
// CUDA path only; the oracle shares nothing with this file.
#include <mutex>

#include "uq_common.cuh"

namespace uq {
namespace {

// In host code this name is a host-side stand-in for the array, NOT a device address: only device code may name it
// directly; host code takes its address with cudaGetSymbolAddress (scratch_of below) and passes that to the kernels.
static __device__ __align__(256) unsigned char g_static_scratch[UQ_STATIC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
std::mutex g_mutex;
unsigned char* g_scratch_ptr[kMaxDevices] = {};        // per device: the array's address there (each GPU has its own copy)

// The address of g_static_scratch on the CURRENT device, looked up once per device with that device current.
int32_t scratch_of(unsigned char** ptr) {
  int dev = -1;
  int32_t st = check_cuda(cudaGetDevice(&dev), "uq_decode_attention_static: cudaGetDevice");
  if (st != UQ_OK) return st;
  if (dev < 0 || dev >= kMaxDevices) {
    set_error("uq_decode_attention_static: device ordinal %d outside the supported range [0, %d)", dev, kMaxDevices);
    return UQ_ERR_UNSUPPORTED;
  }
  std::lock_guard<std::mutex> lock(g_mutex);
  if (!g_scratch_ptr[dev]) {
    void* p = nullptr;
    st = check_cuda(cudaGetSymbolAddress(&p, g_static_scratch), "uq_decode_attention_static: cudaGetSymbolAddress");
    if (st != UQ_OK) return st;
    if (!p || ((uintptr_t)p & 255u)) {
      set_error("uq_decode_attention_static: the static scratch resolved to %p (expected a 256-byte aligned device address)", p);
      return UQ_ERR_CUDA;
    }
    g_scratch_ptr[dev] = (unsigned char*)p;
  }
  *ptr = g_scratch_ptr[dev];
  return UQ_OK;
}

}  // namespace
}  // namespace uq

extern "C" size_t uq_static_scratch_bytes(void) { return (size_t)UQ_STATIC_SCRATCH_BYTES; }

extern "C" int32_t uq_decode_static_scratch_needed(const uq_config* cfg, int32_t batch, int32_t num_splits, size_t* bytes) {
  using namespace uq;
  int32_t st = check_config(cfg);
  if (st != UQ_OK) return st;
  if (!bytes || batch <= 0 || num_splits <= 0) {
    set_error("uq_decode_static_scratch_needed: NULL pointer or non-positive batch / num_splits");
    return UQ_ERR_INVALID_ARG;
  }
  const unsigned long long slots = (unsigned long long)batch * (unsigned long long)cfg->num_q_heads * (unsigned long long)num_splits;
  const unsigned long long acc = (slots * (unsigned long long)cfg->head_dim * sizeof(float) + 255ull) & ~255ull;
  *bytes = (size_t)(acc + slots * 2ull * sizeof(float));
  return UQ_OK;
}

extern "C" int32_t uq_decode_attention_static(const uq_config* cfg, const void* q_fp8, const void* cache, int64_t num_pages,
                                              const int32_t* block_tables, int32_t max_pages, const int32_t* seq_lens,
                                              int32_t batch, int32_t num_splits, void* out_bf16, void* stream) {
  using namespace uq;
  NvtxRange nvtx_range("uq_decode_attention_static");
  size_t need = 0;
  int32_t st = uq_decode_static_scratch_needed(cfg, batch, num_splits, &need);
  if (st != UQ_OK) return st;
  if (need > (size_t)UQ_STATIC_SCRATCH_BYTES) {
    set_error("uq_decode_attention_static: batch %d x %d query heads x %d splits x head_dim %d needs %zu bytes of split "
              "partials, more than the %zu-byte static scratch (UQ_STATIC_SCRATCH_BYTES): lower num_splits or use "
              "uq_decode_attention + uq_merge_splits with buffers of your own",
              batch, cfg->num_q_heads, num_splits, cfg->head_dim, need, (size_t)UQ_STATIC_SCRATCH_BYTES);
    return UQ_ERR_UNSUPPORTED;
  }
  if (!out_bf16) {
    set_error("uq_decode_attention_static: out_bf16 is NULL");
    return UQ_ERR_INVALID_ARG;
  }
  unsigned char* scratch = nullptr;
  st = scratch_of(&scratch);
  if (st != UQ_OK) return st;
  const size_t slots = (size_t)batch * cfg->num_q_heads * num_splits;
  float* partial_acc = (float*)scratch;
  float* partial_ml = (float*)(scratch + ((slots * cfg->head_dim * sizeof(float) + 255u) & ~(size_t)255u));
  // Nothing in the scratch has to start at zero: the decode kernel writes (m, l) of EVERY slot on every call (an unused
  // slot as (-inf, 0)) and the merge reads the acc row of a slot only if its l is not 0, so what the last call left
  // behind is never read.
  st = uq_decode_attention(cfg, q_fp8, cache, num_pages, block_tables, max_pages, seq_lens, batch, num_splits, partial_acc,
                           partial_ml, stream);
  if (st != UQ_OK) return st;
  return uq_merge_splits(cfg, partial_acc, partial_ml, batch, num_splits, out_bf16, stream);
}
