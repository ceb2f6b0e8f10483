// uq_debug.cu — UQ_FLAG_DEBUG_CHECKS (include/uq.h): device-side validation of what the host cannot see — the block
// tables, lengths and cu_new of a call live in device memory, and Alg. 1's "Require" says nothing about
// paging, so an entry outside the cache is silent undefined behaviour in the hot kernels.  With the flag set every
// entry point first runs this kernel over exactly the table entries / lengths the call is going to use, copies a
// 4-word report back and SYNCHRONISES the stream (the one documented exception to "never synchronises"; the call is
// then not capturable into a CUDA graph): the first offender is named in uq_last_error_string() and nothing else is
// launched.  CUDA path only.
#include <mutex>

#include "uq_common.cuh"

namespace uq {
namespace {

// report of the current device: {offenders, kind, sequence, index, value}
__device__ int g_report[5];

enum Kind { kBadLen = 1, kBadCount = 2, kBadEntry = 3, kPrefixDiffers = 4, kBadCu = 5 };

__device__ __forceinline__ void report(int kind, int b, int idx, int val) {
  if (atomicAdd(&g_report[0], 1) == 0) {
    g_report[1] = kind; g_report[2] = b; g_report[3] = idx; g_report[4] = val;
  }
}

// One CTA per sequence.  mode 0 (decode): pages [0, ceil(seq_lens[b] / page)); mode 1 (append): the pages positions
// seq_lens[b] .. seq_lens[b] + count - 1 fall into, count = cu_new[b+1] - cu_new[b]; mode 2 (shared prefix): pages
// [0, fixed_pages), which must also equal sequence 0's.
__global__ void check_tables_kernel(const int32_t* __restrict__ block_tables, int max_pages, int batch, long long num_pages,
                                    const int32_t* __restrict__ seq_lens, const int32_t* __restrict__ cu_new, int total_new,
                                    int fixed_pages, int page, int mode) {
  const int b = blockIdx.x;
  int p0 = 0, p1 = 0;
  if (mode == 0) {
    const int L = seq_lens[b];
    if (L < 0 || (long long)L > (long long)max_pages * page) { if (threadIdx.x == 0) report(kBadLen, b, max_pages * page, L); return; }
    p1 = (L + page - 1) / page;
  } else if (mode == 1) {
    const int c0 = cu_new[b], c1 = cu_new[b + 1], n = c1 - c0;
    if (b == 0 && c0 != 0 && threadIdx.x == 0) report(kBadCu, 0, 0, c0);
    if (b == batch - 1 && c1 != total_new && threadIdx.x == 0) report(kBadCu, batch, total_new, c1);
    if (n < 0) { if (threadIdx.x == 0) report(kBadCount, b, c0, c1); return; }
    if (n == 0) return;
    const int L = seq_lens[b];
    if (L < 0 || (long long)L + n > (long long)max_pages * page) { if (threadIdx.x == 0) report(kBadLen, b, max_pages * page, L + n); return; }
    p0 = L / page;
    p1 = (L + n + page - 1) / page;
  } else {
    p1 = fixed_pages;
  }
  const int32_t* row = block_tables + (long long)b * max_pages;
  for (int p = p0 + (int)threadIdx.x; p < p1; p += (int)blockDim.x) {
    const int e = row[p];
    if (e < 0 || (long long)e >= num_pages) report(kBadEntry, b, p, e);
    else if (mode == 2 && e != block_tables[p]) report(kPrefixDiffers, b, p, e);
  }
}

std::mutex g_dbg_mu;

}  // namespace

int32_t debug_check_tables(const char* who, const int32_t* block_tables, int max_pages, int batch, long long num_pages,
                           const int32_t* seq_lens, const int32_t* cu_new, int total_new, int fixed_pages, int page,
                           int mode, cudaStream_t stream) {
  std::lock_guard<std::mutex> lock(g_dbg_mu);          // one report buffer per device
  void* rep = nullptr;
  cudaError_t e = cudaGetSymbolAddress(&rep, g_report);
  if (e == cudaSuccess) e = cudaMemsetAsync(rep, 0, sizeof(int) * 5, stream);
  if (e != cudaSuccess) return check_cuda(e, "debug checks: report buffer");
  check_tables_kernel<<<(unsigned)batch, 128, 0, stream>>>(block_tables, max_pages, batch, num_pages, seq_lens, cu_new,
                                                           total_new, fixed_pages, page, mode);
  int h[5] = {0, 0, 0, 0, 0};
  e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaMemcpyAsync(h, rep, sizeof(h), cudaMemcpyDeviceToHost, stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
  if (e != cudaSuccess) return check_cuda(e, "debug checks (UQ_FLAG_DEBUG_CHECKS synchronises the stream; not capturable)");
  if (h[0] == 0) return UQ_OK;
  switch (h[1]) {
    case kBadLen:
      set_error("%s: debug check: sequence %d needs %d token positions, the block table holds %d (%d offenders in all)",
                who, h[2], h[4], h[3], h[0]);
      break;
    case kBadCount:
      set_error("%s: debug check: cu_new decreases at sequence %d (%d -> %d) (%d offenders in all)", who, h[2], h[3], h[4], h[0]);
      break;
    case kBadCu:
      set_error("%s: debug check: cu_new[%d] = %d, expected %d (%d offenders in all)", who, h[2], h[4], h[3], h[0]);
      break;
    case kPrefixDiffers:
      set_error("%s: debug check: block_tables[%d][%d] = %d differs from sequence 0's entry: the prefix is not shared "
                "(%d offenders in all)", who, h[2], h[3], h[4], h[0]);
      break;
    default:
      set_error("%s: debug check: block_tables[%d][%d] = %d is outside [0, %lld) (%d offenders in all)", who, h[2], h[3],
                h[4], num_pages, h[0]);
  }
  return UQ_ERR_INVALID_ARG;
}

}  // namespace uq
