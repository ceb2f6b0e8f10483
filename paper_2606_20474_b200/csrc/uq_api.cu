// uq_api.cu — host-side plumbing of libuq.so: error string, config validation, small queries.
#include <stdarg.h>

#include <mutex>

#include "uq_common.cuh"

namespace uq {

static thread_local char g_err[256] = "no error";

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}

int32_t check_config(const uq_config* cfg) {
  if (cfg == nullptr) {
    set_error("uq_config is NULL");
    return UQ_ERR_INVALID_ARG;
  }
  if (cfg->num_q_heads <= 0 || cfg->num_kv_heads <= 0 || cfg->head_dim <= 0 ||
      cfg->page_size <= 0 || cfg->group_size <= 0) {
    set_error("uq_config: non-positive dimension");
    return UQ_ERR_INVALID_ARG;
  }
  if (cfg->num_q_heads % cfg->num_kv_heads != 0) {
    set_error("uq_config: num_q_heads %d not a multiple of num_kv_heads %d", cfg->num_q_heads,
              cfg->num_kv_heads);
    return UQ_ERR_INVALID_ARG;
  }
  if (!(cfg->c_k > 0.0f) || !(cfg->c_v > 0.0f)) {
    set_error("uq_config: c_k and c_v must be positive");
    return UQ_ERR_INVALID_ARG;
  }
  if ((cfg->flags & ~(uint32_t)(UQ_FLAG_NO_BULK_APPEND | UQ_FLAG_DEBUG_CHECKS | UQ_FLAG_SMALL_APPEND_AHEAD)) != 0) {
    set_error("uq_config: unknown bit in flags");
    return UQ_ERR_INVALID_ARG;
  }
  if ((cfg->head_dim != 64 && cfg->head_dim != 128 && cfg->head_dim != 256) || cfg->group_size != kGroup ||
      cfg->page_size != kPage) {
    set_error("unsupported geometry: head_dim %d group %d page %d (supported: 64|128|256 / 32 / 16)",
              cfg->head_dim, cfg->group_size, cfg->page_size);
    return UQ_ERR_UNSUPPORTED;
  }
  if (cfg->num_q_heads / cfg->num_kv_heads > 16) {
    set_error("unsupported GQA group %d (> 16)", cfg->num_q_heads / cfg->num_kv_heads);
    return UQ_ERR_UNSUPPORTED;
  }
  return UQ_OK;
}

int32_t require_head_dim_128(const uq_config* cfg, const char* who) {
  if (cfg->head_dim == kHeadDim) return UQ_OK;
  set_error("%s: head_dim %d is not supported by this entry point (128 only)", who, cfg->head_dim);
  return UQ_ERR_UNSUPPORTED;
}

int32_t check_cuda(cudaError_t e, const char* what) {
  if (e == cudaSuccess) return UQ_OK;
  set_error("%s: %s", what, cudaGetErrorString(e));
  return UQ_ERR_CUDA;
}

// ---------------------------------------------------------------- per-device host state
namespace {
constexpr int kMaxDevices = 64;
std::mutex g_dev_mu;
int g_sms[kMaxDevices];                                // 0 = not looked up yet
struct OptIn { const void* kernel; int device; int bytes; };
OptIn g_optin[256];
int g_optin_n = 0;
}  // namespace

int32_t current_device_sms(int* sms) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return check_cuda(e, "cudaGetDevice");
  std::lock_guard<std::mutex> lock(g_dev_mu);
  if (dev >= 0 && dev < kMaxDevices && g_sms[dev] > 0) { *sms = g_sms[dev]; return UQ_OK; }
  int v = 0;
  e = cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess || v <= 0) return check_cuda(e != cudaSuccess ? e : cudaErrorUnknown, "cudaDeviceGetAttribute(SM count)");
  if (dev >= 0 && dev < kMaxDevices) g_sms[dev] = v;
  *sms = v;
  return UQ_OK;
}

int32_t opt_in_dynamic_smem(const void* kernel, int bytes, const char* what) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return check_cuda(e, "cudaGetDevice");
  std::lock_guard<std::mutex> lock(g_dev_mu);
  for (int i = 0; i < g_optin_n; ++i)
    if (g_optin[i].kernel == kernel && g_optin[i].device == dev && g_optin[i].bytes >= bytes) return UQ_OK;
  e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if (e != cudaSuccess) return check_cuda(e, what);
  if (g_optin_n < 256) g_optin[g_optin_n++] = OptIn{kernel, dev, bytes};   // a full table only costs a repeated call
  return UQ_OK;
}

EncodeTiledFn encode_tiled_fn() {
  static std::mutex mu;
  static EncodeTiledFn encode = nullptr;
  std::lock_guard<std::mutex> lock(mu);
  if (!encode) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess || fn == nullptr) {
      set_error("cuTensorMapEncodeTiled is not available from this driver");
      return nullptr;
    }
    encode = (EncodeTiledFn)fn;
  }
  return encode;
}

}  // namespace uq

extern "C" const char* uq_last_error_string(void) { return uq::g_err; }

extern "C" size_t uq_cache_record_bytes(const uq_config* cfg) {
  if (uq::check_config(cfg) != UQ_OK) return 0;
  return (size_t)cfg->page_size * (size_t)(cfg->head_dim / 2 + cfg->head_dim / cfg->group_size) * 2;
}

extern "C" int32_t uq_decode_workspace_bytes(const uq_config* cfg, int32_t batch, int32_t num_splits, size_t* bytes) {
  const int32_t st = uq::check_config(cfg);
  if (st != UQ_OK) return st;
  if (batch <= 0 || num_splits <= 0 || bytes == nullptr) {
    uq::set_error("uq_decode_workspace_bytes: non-positive size or NULL result pointer");
    return UQ_ERR_INVALID_ARG;
  }
  // The decode kernels keep their schedule (tile prefix sums), their rings and their accumulators in shared memory and
  // TMEM, and the split partials are the caller's buffers: no device scratch beyond them.
  *bytes = 0;
  return UQ_OK;
}

extern "C" int32_t uq_suggest_num_splits(const uq_config* cfg, int32_t batch, int32_t avg_seq_len) {
  if (uq::check_config(cfg) != UQ_OK || batch <= 0) return 1;
  int sms = 148;
  if (uq::current_device_sms(&sms) != UQ_OK) sms = 148;   // no device (a host-only caller sizing buffers): B200's count
  // uq_decode_attention gives every resident CTA (2 per SM) one equal range of 128-token tiles; an item
  // (sequence, kv head) of T tiles then spans about T / range + 1 CTAs = slots.  Leave room for sequences
  // twice the average length.
  const int64_t items = (int64_t)batch * cfg->num_kv_heads;
  const int64_t slots = (int64_t)sms * (cfg->head_dim == 256 ? 1 : 2);   // resident decode CTAs
  const int64_t pages = (avg_seq_len + cfg->page_size - 1) / cfg->page_size;
  const int64_t tiles = (pages + 7) / 8 > 0 ? (pages + 7) / 8 : 1;
  int64_t range = (items * tiles + slots - 1) / slots;
  if (range < 1) range = 1;
  int64_t s = (2 * tiles + range - 1) / range + 1;
  if (s > tiles + 1) s = tiles + 1;
  if (s < 2) s = 2;
  if (s > 64) s = 64;
  return (int32_t)s;
}

extern "C" int32_t uq_suggest_num_splits_max(const uq_config* cfg, int32_t batch, int32_t avg_seq_len,
                                             int32_t max_seq_len) {
  // As above with the longest sequence known: the balanced schedule makes every range long enough for the longest
  // item to fit into num_splits - 1 of them, so a skewed length mix (the private suffixes of a shared-prefix batch:
  // mean 16k, maximum 98k tokens) needs max_tiles / range + 2 slots or every CTA's range is stretched.
  const int32_t base = uq_suggest_num_splits(cfg, batch, avg_seq_len);
  if (uq::check_config(cfg) != UQ_OK || batch <= 0 || max_seq_len <= avg_seq_len) return base;
  int sms = 148;
  if (uq::current_device_sms(&sms) != UQ_OK) sms = 148;   // no device (a host-only caller sizing buffers): B200's count
  const int64_t tiles_avg = ((int64_t)avg_seq_len + 127) / 128 > 0 ? ((int64_t)avg_seq_len + 127) / 128 : 1;
  const int64_t tiles_max = ((int64_t)max_seq_len + 127) / 128;
  const int64_t resident = (int64_t)sms * (cfg->head_dim == 256 ? 1 : 2);
  int64_t range = ((int64_t)batch * cfg->num_kv_heads * tiles_avg + resident - 1) / resident;
  if (range < 1) range = 1;
  int64_t s = tiles_max / range + 2;
  if (s < base) s = base;
  if (s > 64) s = 64;
  return (int32_t)s;
}

extern "C" int32_t uq_suggest_prefix_splits(const uq_config* cfg, int32_t batch, int32_t prefix_len) {
  // uq_decode_prefix_attention: items = (group of 8 or 16 sequences, kv head), prefix_len / 128 tiles each, one equal
  // tile range per SM; an item then spans about tiles / range + 1 ranges = slots.
  if (uq::check_config(cfg) != UQ_OK || batch <= 0 || prefix_len < 128) return 2;
  int sms = 148;
  if (uq::current_device_sms(&sms) != UQ_OK) sms = 148;
  const int nseq = (cfg->num_q_heads / cfg->num_kv_heads) > 8 ? 8 : 16;
  const int64_t tiles = prefix_len / 128;
  const int64_t total = (int64_t)((batch + nseq - 1) / nseq) * cfg->num_kv_heads * tiles;
  int64_t range = (total + sms - 1) / sms;
  if (range < 1) range = 1;
  int64_t s = (tiles + range - 1) / range + 1;
  if (s < 2) s = 2;
  if (s > 64) s = 64;
  return (int32_t)s;
}
