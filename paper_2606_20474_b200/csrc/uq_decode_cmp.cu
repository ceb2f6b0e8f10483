// uq_decode_cmp.cu — the paper's COMPARISON caches on the CTA skeleton of uq_decode.cu: paged split-K
// decode attention over an FP8-E4M3 KV cache ("hardware FP8 KV", Table 3 :293-301) and over a BF16 KV cache
// (the BF16 baseline, :163), so that the paper's RELATIVE kernel claims — 4-bit moves about half the bytes of FP8, the
// FP4 kernel within 1.18 x of FP8 at 32K (:188, :295-301) — can be restated on B200 with everything else equal: same
// schedule (uq_sched.cuh), same TMA / mbarrier rings, same softmax warps with lazy references, same Vhat^T-in-TMEM PV
// product, same partial format (include/uq.h), same merge.  What differs is what the bytes are:
//   FP8   record = K [16 tok][128 B E4M3] | V [128 ch][16 tok E4M3]: QK by tcgen05.mma kind::f8f6f4 (E4M3 x E4M3, no
//         scale operand), V warps convert with cvt.rn.f16x2.e4m3x2 (no multiply); the query is cast_e4m3(q), unrotated;
//   BF16  record = K [16 tok][128 bf16] | V [128 ch][16 tok bf16]: QK by kind::f16 (bf16 x bf16), V warps move the
//         bf16 pairs to TMEM unchanged and P is rounded to bf16 as well (the instruction takes one 16-bit type for A and
//         B; it is also what BF16 attention kernels do); the query is the bf16 query itself.
// Readings: DESIGN.md G19.  head_dim 128 only.  CUDA path only; the oracle shares nothing with this file.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include <type_traits>

#include "uq_sched.cuh"
#include "uq_tc.cuh"

namespace uq {
namespace {

constexpr int kSoftmaxWarps = 4, kVWarps = 4, kIssuerWarps = 4;
constexpr int kComputeWarps = kSoftmaxWarps + kVWarps;
constexpr int kPBytes = 4096;                        // one P operand buffer (as uq_decode.cu)
constexpr float kThresh = 12.0f;
constexpr int kMaxBatch = 2048;

template <int KV>                                    // UQ_KV_FP8_E4M3 = 1, UQ_KV_BF16 = 2, UQ_KV_ULTRA_TQ = 3
struct CmpGeo {
  static_assert(KV == UQ_KV_FP8_E4M3 || KV == UQ_KV_BF16 || KV == UQ_KV_ULTRA_TQ, "comparison cache format");
  // Ultra-TQ (Alg. 2): the records arrive as they are (the "V" ring holds whole records), four more warps decode the K
  // codes through the codebook into the bf16 K operand buffers (the "K" ring), everything behind that is the BF16 path
  static constexpr bool kTq = KV == UQ_KV_ULTRA_TQ;
  static constexpr bool kBf16 = KV == UQ_KV_BF16 || kTq;            // operands of the two products are bf16
  static constexpr int kElem = kBf16 ? 2 : 1;                       // bytes per operand element
  static constexpr int kKPage = 16 * 128 * kElem;                   // K rows of a page in the operand: 2048 / 4096
  static constexpr int kVPage = kTq ? kTqRecord : kKPage;           // bytes a page puts into the V ring
  static constexpr int kVSrc = kTq ? 0 : kKPage;                    // ... from this offset of its record
  static constexpr int kRecordBytes = kTq ? kTqRecord : 2 * kKPage; // 4096 / 8192 / 2432
  static constexpr int kDequantWarps = kTq ? 4 : 0;
  static constexpr int kThreads = (kComputeWarps + kIssuerWarps + kDequantWarps) * 32;
  static constexpr int kBlocks = kElem;                             // 128-byte-wide swizzled blocks of a K row
  static constexpr int kKBlockBytes = 128 * 128;                    // [128 tokens][128 B]
  static constexpr int kKStageBytes = kBlocks * kKBlockBytes;       // 16384 / 32768
  static constexpr int kVStageBytes = kTilePages * kVPage;          // 16384 / 32768
  static constexpr int kKStages = KV == UQ_KV_BF16 ? 3 : 2;
  static constexpr int kVStages = 3;
  static constexpr int kCtasPerSm = kBf16 ? 1 : 2;
  static constexpr int kQBlockBytes = 16 * 128;                     // [16 heads][128 B]
  static constexpr int kQBytes = kBlocks * kQBlockBytes;
  static constexpr int kQKMmas = 4 * kElem;                         // 32 bytes of a row per instruction
  static constexpr int kOffK = 0;
  static constexpr int kOffV = kOffK + kKStages * kKStageBytes;
  static constexpr int kOffQ = kOffV + kVStages * kVStageBytes;
  static constexpr int kOffP = kOffQ + 2 * kQBytes;
  static constexpr int kOffLut = kOffP + 2 * kPBytes;               // Ultra-TQ: 256 x bf16x2, the codebook by code byte
  static constexpr int kOffEnd = kOffLut + (kTq ? 1024 : 0);
  static constexpr int kSmemBytes = kOffEnd + 1024;
  static_assert(kOffQ % 1024 == 0, "swizzled tiles need 1024-byte alignment");
  static constexpr uint32_t kColS = 0, kColO = 32, kColV = 64, kTmemCols = 256;
};

template <int KV>
struct CmpShared {
  using Geo = CmpGeo<KV>;
  uint64_t full_k[Geo::kKStages], empty_k[Geo::kKStages], full_v[Geo::kVStages], empty_v[Geo::kVStages];
  uint64_t s_full[2], s_free[2], ready[2], done[2], q_full[2];
  uint32_t tmem_base;
  float wmax[kSoftmaxWarps][16];
  float lsum[kSoftmaxWarps][16];
  float mref[16];
  int total_tiles, max_tiles;
  int pre[kMaxBatch + 1];
};

// D[tmem] (+)= A[smem, E4M3] . B[smem, E4M3]^T, fp32 accumulation, no scale operand
__device__ __forceinline__ void umma_f8f6f4_ss(uint32_t d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], %1, %2, %3, p;\n}\n"
      ::"r"(d), "l"(da), "l"(db), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void umma_f16_ss(uint32_t d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n}\n"
      ::"r"(d), "l"(da), "l"(db), "r"(idesc), "r"(acc) : "memory");
}
// two E4M3 bytes (a 16-bit half of w) -> f16x2
__device__ __forceinline__ uint32_t cvt_e4m3x2(uint32_t w, int hi) {
  uint32_t r;
  asm("{\n.reg .b16 lo, up;\nmov.b32 {lo, up}, %1;\n"
      "cvt.rn.f16x2.e4m3x2 %0, lo;\n}\n" : "=r"(r) : "r"(hi ? (w >> 16) : w));
  return r;
}

// ---------------------------------------------------------------- the kernel
template <int KV>
__global__ void __launch_bounds__(CmpGeo<KV>::kThreads, CmpGeo<KV>::kCtasPerSm)
decode_cmp_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ CUtensorMap tmap_q,
                  const uint8_t* __restrict__ cache, const int32_t* __restrict__ block_tables, int max_pages,
                  const int32_t* __restrict__ seq_lens, int batch, int Hq, int Hkv, int num_splits,
                  float score_scale /* sm_scale * log2(e) */, float* __restrict__ partial_acc,
                  float* __restrict__ partial_ml, const TqCodebook tq) {
  using Geo = CmpGeo<KV>;
  constexpr int kThreads = Geo::kThreads;
  constexpr int kKStages = Geo::kKStages, kVStages = Geo::kVStages, kKStageBytes = Geo::kKStageBytes,
                kVStageBytes = Geo::kVStageBytes, kKBlockBytes = Geo::kKBlockBytes, kQBytes = Geo::kQBytes,
                kQBlockBytes = Geo::kQBlockBytes, kKPage = Geo::kKPage, kVPage = Geo::kVPage, kBlocks = Geo::kBlocks;
  constexpr uint32_t kColS = Geo::kColS, kColO = Geo::kColO, kColV = Geo::kColV;
  extern __shared__ uint8_t smem_raw[];
  __shared__ __align__(8) CmpShared<KV> sh;

  const int G = Hq / Hkv;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  // warps 0..3 softmax, 4..7 V warps, 8..11 issuers (role 0 QK, 1 PV, 2 K producer, 3 V producer), as uq_decode.cu
  // (Ultra-TQ: warps 12..15 are the K dequantisers, role 100 + their index)
  const int role = warp < kComputeWarps ? warp + kIssuerWarps
                   : (warp < kComputeWarps + kIssuerWarps ? warp - kComputeWarps : 100 + warp - kComputeWarps - kIssuerWarps);

  const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sQ = base + Geo::kOffQ, sP = base + Geo::kOffP;
  const uint32_t bar_fullk = smem_u32(&sh.full_k[0]), bar_emptyk = smem_u32(&sh.empty_k[0]),
                 bar_fullv = smem_u32(&sh.full_v[0]), bar_emptyv = smem_u32(&sh.empty_v[0]),
                 bar_sfull = smem_u32(&sh.s_full[0]), bar_sfree = smem_u32(&sh.s_free[0]),
                 bar_ready = smem_u32(&sh.ready[0]), bar_done = smem_u32(&sh.done[0]),
                 bar_qfull = smem_u32(&sh.q_full[0]);

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < kKStages; ++s) { mbar_init(bar_fullk + 8 * s, Geo::kTq ? 4 : 1); mbar_init(bar_emptyk + 8 * s, 1); }
#pragma unroll
    for (int s = 0; s < kVStages; ++s) { mbar_init(bar_fullv + 8 * s, 1); mbar_init(bar_emptyv + 8 * s, kVWarps + Geo::kDequantWarps); }
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      mbar_init(bar_sfull + 8 * h, 1);
      mbar_init(bar_sfree + 8 * h, kSoftmaxWarps);
      mbar_init(bar_done + 8 * h, 1);
      mbar_init(bar_qfull + 8 * h, 1);
      mbar_init(bar_ready + 8 * h, kComputeWarps);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (role == 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&sh.tmem_base)),
                 "r"(Geo::kTmemCols));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  if constexpr (Geo::kTq) {                            // codebook by code byte: low nibble = even channel = low half
    for (int e = tid; e < 256; e += kThreads) {
      const uint32_t lo = __bfloat16_as_ushort(__float2bfloat16_rn(tq.c[e & 15])), hi = __bfloat16_as_ushort(__float2bfloat16_rn(tq.c[e >> 4]));
      asm volatile("st.shared.u32 [%0], %1;" ::"r"(base + Geo::kOffLut + 4 * e), "r"(lo | (hi << 16)) : "memory");
    }
  }
  pdl_launch_dependents();
  pdl_wait();
  for (int b = tid; b < batch; b += kThreads) {
    const int L = seq_lens[b];
    sh.pre[b + 1] = ((L + kPage - 1) / kPage + kTilePages - 1) / kTilePages;
  }
  if (tid == 0) sh.pre[0] = 0;
  __syncthreads();
  if (warp == 0) {
    int carry = 0, mx = 0;
    for (int b0 = 0; b0 < batch; b0 += 32) {
      const int b = b0 + lane;
      const int v = b < batch ? sh.pre[b + 1] : 0;
      int x = v;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(kFull, x, o);
        if (lane >= o) x += y;
      }
      if (b < batch) sh.pre[b + 1] = carry + x;
      carry += __shfl_sync(kFull, x, 31);
      mx = max(mx, __reduce_max_sync(kFull, v));
    }
    if (lane == 0) { sh.total_tiles = carry * Hkv; sh.max_tiles = mx; }
  }
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = sh.tmem_base;

  Sched sc;
  sc.seq_lens = seq_lens; sc.pre = sh.pre; sc.B = batch; sc.Hq = Hq; sc.Hkv = Hkv; sc.G = G; sc.S = num_splits;
  sc.total = sh.total_tiles;
  sc.tpc = 1;
  if (num_splits > 1) {
    const int even = (sc.total + (int)gridDim.x - 1) / (int)gridDim.x;
    const int fit = (sh.max_tiles + num_splits - 2) / (num_splits - 1);
    sc.tpc = max(1, max(even, fit));
  }

  if (role == 0) {
    // ================================================================ QK warp: S[128 tok x 16 heads] = K . Q^T
    // instruction descriptors: fp32 accumulate (bit 4), A / B format at bits 7 / 10 (kind::f8f6f4: 0 = E4M3;
    // kind::f16: 1 = BF16), N >> 3 at bit 17, M >> 4 at bit 24; both operands K-major
    const uint32_t idesc_qk = Geo::kBf16 ? ((1u << 4) | (1u << 7) | (1u << 10) | (2u << 17) | (8u << 24))
                                                : ((1u << 4) | (2u << 17) | (8u << 24));
    auto load_q = [&](const Unit& un, int k) {
      if (elect_one()) {
        mbar_expect_tx(bar_qfull + 8 * (k & 1), kQBytes);
#pragma unroll
        for (int c = 0; c < kBlocks; ++c)               // a 128-byte-wide block of the 16 query rows per copy
          tma_load_2d(sQ + kQBytes * (k & 1) + kQBlockBytes * c, &tmap_q, (128 / Geo::kElem) * c, un.b * Hq + un.kvh * G,
                      bar_qfull + 8 * (k & 1));
      }
    };
    Cursor cur, cur_nx;
    sc.start(cur);
    cur_nx = cur;
    Unit un, nx;
    bool have_nx = sc.next(cur_nx, nx);
    int gt = 0, sk = 0, phk = 0;
    int k = 0, k_q = -1;
    while (have_nx) {
      un = nx;
      have_nx = sc.next(cur_nx, nx);
      for (int i = 0; i < un.n_tiles; ++i) {
        const int sb = gt & 1;
        if (gt >= 2) mbar_wait(bar_sfree + 8 * sb, ((gt >> 1) - 1) & 1);
        if (i == 0 && k_q < k) { load_q(un, k); k_q = k; }
        if (i == 1 && have_nx) { load_q(nx, k + 1); k_q = k + 1; }
        if (i == 0) mbar_wait(bar_qfull + 8 * (k & 1), (k >> 1) & 1);
        const uint32_t st = base + Geo::kOffK + sk * kKStageBytes;
        mbar_wait(bar_fullk + 8 * sk, phk);
        tc_fence_after();
        if (elect_one()) {
          const uint32_t qb = sQ + kQBytes * (k & 1);
#pragma unroll
          for (int kb = 0; kb < Geo::kQKMmas; ++kb) {
            const uint64_t da = make_desc(st + (kb >> 2) * kKBlockBytes + 32 * (kb & 3), 16, 1024, 2);
            const uint64_t db = make_desc(qb + (kb >> 2) * kQBlockBytes + 32 * (kb & 3), 16, 1024, 2);
            if constexpr (Geo::kBf16) umma_f16_ss(tmem + kColS + 16 * sb, da, db, idesc_qk, kb > 0);
            else umma_f8f6f4_ss(tmem + kColS + 16 * sb, da, db, idesc_qk, kb > 0);
          }
          umma_commit(bar_sfull + 8 * sb);
          umma_commit(bar_emptyk + 8 * sk);
        }
        __syncwarp();
        ++gt;
        if (++sk == kKStages) { sk = 0; phk ^= 1; }
      }
      ++k;
    }
  } else if (role == 1) {
    // ================================================================ PV warp: O^T[128 d x 16 heads] += Vhat^T . P^T
    // A = Vhat^T from TMEM, B = P from smem (MN-major): both f16 (FP8 cache) or both bf16 (BF16 cache: the instruction
    // takes one 16-bit type for A and B — a mixed descriptor is an illegal instruction)
    const uint32_t idesc_pv = (1u << 4) | (Geo::kBf16 ? ((1u << 7) | (1u << 10)) : 0u) | (1u << 16) | (2u << 17) | (8u << 24);
    Cursor cur;
    sc.start(cur);
    Unit un;
    int gt = 0;
    while (sc.next(cur, un)) {
      for (int i = 0; i < un.n_tiles; ++i, ++gt) {
        mbar_wait(bar_ready + 8 * (gt & 1), (gt >> 1) & 1);
        tc_fence_after();
        if (lane == 0) {
          const uint32_t pbuf = sP + kPBytes * (gt & 1), vbuf = tmem + kColV + 64 * (gt & 1);
#pragma unroll
          for (int j = 0; j < 8; ++j)
            umma_f16_ts(tmem + kColO, vbuf + 8 * j, make_desc(pbuf + 512 * j, 256, 128, 0), idesc_pv,
                        (i > 0 || j > 0) ? 1u : 0u);
          umma_commit(bar_done + 8 * (gt & 1));
        }
        __syncwarp();
      }
    }
  } else if (role == 2 || role == 3) {
    // ================================================================ producers: K rows by TMA (swizzled), V by bulk copy
    const bool is_k = (role == 2);
    const bool idle = Geo::kTq && is_k;                 // Ultra-TQ: the K operand is written by the dequantiser warps
    const int n_stages = is_k ? kKStages : kVStages;
    const uint32_t bar_e = is_k ? bar_emptyk : bar_emptyv, bar_f = is_k ? bar_fullk : bar_fullv;
    const uint32_t page_tx = is_k ? (uint32_t)kKPage : (uint32_t)kVPage;
    const int pl = lane & 7, hl = lane >> 3;             // page of the tile, 128-byte block of the K row
    const bool copier = is_k ? lane < kTilePages * kBlocks : lane < kTilePages;
    const uint64_t pol = l2_evict_first_policy();
    Cursor cur;
    sc.start(cur);
    Unit un;
    int s = 0, ph = 1;
    while (!idle && sc.next(cur, un)) {
      const int32_t* bt = block_tables + (long long)un.b * max_pages + un.p0 + pl;
      int page_next = (copier && un.p0 + pl < un.p1) ? bt[0] : 0;
      for (int i = 0; i < un.n_tiles; ++i) {
        const int page = page_next;
        const int npg = min(kTilePages, un.p1 - (un.p0 + kTilePages * i));
        const int nb = un.p0 + kTilePages * (i + 1) + pl;
        page_next = (copier && nb < un.p1) ? bt[kTilePages * (i + 1)] : 0;
        mbar_wait(bar_e + 8 * s, ph);
        if (lane == 0) mbar_expect_tx(bar_f + 8 * s, (uint32_t)npg * page_tx);
        __syncwarp();
        if (copier && pl < npg) {
          if (is_k)
            tma_load_3d(base + Geo::kOffK + s * kKStageBytes + hl * kKBlockBytes + 2048 * pl, &tmap, (128 / Geo::kElem) * hl, 0,
                        page * Hkv + un.kvh, bar_f + 8 * s, pol);
          else
            bulk_g2s(base + Geo::kOffV + s * kVStageBytes + kVPage * pl,
                     cache + ((long long)page * Hkv + un.kvh) * Geo::kRecordBytes + Geo::kVSrc, kVPage, bar_f + 8 * s, pol);
        }
        if (++s == n_stages) { s = 0; ph ^= 1; }
      }
    }
  } else if (role >= 100) {
    // ================================================================ Ultra-TQ: K dequantiser warps (Alg. 2 l.7, "K:
    // dequant via C_K . norm"): thread = token row of the tile.  Its 64 code bytes go through the 256-entry table in
    // shared memory (one load per byte = two channels, the paper's "LDS gather"), times the block norm
    // (bf16 x bf16 -> bf16, one rounding), into the row of the K operand buffer (K-major, 128-byte swizzle: what the TMA
    // unit writes for the BF16 cache).
    if constexpr (Geo::kTq) {
      const int row = 32 * (role - 100) + lane;
      const uint32_t lut = base + Geo::kOffLut;
      Cursor cur;
      sc.start(cur);
      Unit un;
      int s = 0, ph_full = 0, sk = 0, phk = 1;
      while (sc.next(cur, un)) {
        for (int i = 0; i < un.n_tiles; ++i) {
          mbar_wait(bar_fullv + 8 * s, ph_full);       // the tile's records have landed
          mbar_wait(bar_emptyk + 8 * sk, phk);         // the product that read operand buffer sk last is complete
          const uint32_t rec = base + Geo::kOffV + s * kVStageBytes + kTqRecord * (row >> 4);
          const uint32_t dst = base + Geo::kOffK + sk * kKStageBytes + 128 * row;
          uint32_t nw[2];                              // the row's four block norms (bf16)
          asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(nw[0]), "=r"(nw[1]) : "r"(rec + 1024 + 8 * (row & 15)));
#pragma unroll
          for (int g = 0; g < 4; ++g) {                // 16 code bytes = 32 channels = one norm block
            const uint4 cw4 = lds128(rec + 64 * (row & 15) + 16 * g);
            const uint32_t w[4] = {cw4.x, cw4.y, cw4.z, cw4.w};
            const uint32_t n2 = __byte_perm(nw[g >> 1], 0, (g & 1) ? 0x3232 : 0x1010);   // (norm, norm)
            uint32_t o[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) {
              const uint32_t byte = (w[j >> 2] >> (8 * (j & 3))) & 0xFFu;
              uint32_t e;
              asm volatile("ld.shared.u32 %0, [%1];" : "=r"(e) : "r"(lut + 4 * byte));
              asm("mul.rn.bf16x2 %0, %1, %2;" : "=r"(o[j]) : "r"(e), "r"(n2));
            }
#pragma unroll
            for (int c = 0; c < 4; ++c)                // four 16-byte chunks of the row: chunk 4 (g & 1) + c of block g >> 1
              sts128(dst + (g >> 1) * kKBlockBytes + (((4 * (g & 1) + c) ^ (row & 7)) << 4),
                     make_uint4(o[4 * c], o[4 * c + 1], o[4 * c + 2], o[4 * c + 3]));
          }
          fence_async_smem();
          __syncwarp();
          if (lane == 0) {
            mbar_arrive(bar_fullk + 8 * sk);
            mbar_arrive(bar_emptyv + 8 * s);
          }
          if (++s == kVStages) { s = 0; ph_full ^= 1; }
          if (++sk == kKStages) { sk = 0; phk ^= 1; }
        }
      }
    }
  } else {
    const int cw = role - kIssuerWarps;                // 0..7
    const int q = warp & 3;                            // TMEM lane quarter
    const uint32_t lane_sel = (uint32_t)(32 * q) << 16;
    const int r = 32 * q + lane;                       // softmax: token row of the tile; V warps: channel d

    if (cw < kSoftmaxWarps) {
      // ============================================================== softmax warps
      const int atid = 32 * cw + lane;                 // 0..127
      float2* const ml_out = reinterpret_cast<float2*>(partial_ml);

      // items without any token: all their slots are empty, (m, l) = (-inf, 0)
      for (int it = blockIdx.x; it < batch * Hkv; it += gridDim.x) {
        const int b = it / Hkv;
        if (sc.tiles(b) == 0) {
          const long long row = ((long long)b * Hq + (long long)(it - b * Hkv) * G) * num_splits;
          for (int e = atid; e < G * num_splits; e += 32 * kSoftmaxWarps) ml_out[row + e] = make_float2(-INFINITY, 0.f);
        }
      }

      auto run = [&](auto nh_tag) {
        constexpr int NH = decltype(nh_tag)::value;    // head columns this thread handles: 8 (G <= 8) or 16
        Cursor cur;
        sc.start(cur);
        Unit un;
        int gt = 0;                                    // global tile counter
        const uint32_t p_row = sP + (r >> 3) * 256 + (r & 7) * 16;
        while (sc.next(cur, un)) {
          float nmref[NH], lsum[NH];                   // nmref = minus the per-head reference logit
#pragma unroll
          for (int j = 0; j < NH; ++j) { nmref[j] = INFINITY; lsum[j] = 0.f; }
          int rem = un.tok_end - un.p0 * kPage;        // valid tokens from the first row of the tile on

          for (int i = 0; i < un.n_tiles; ++i, rem -= kTilePages * kPage) {
            const int sb = gt & 1, ph2 = (gt >> 1) & 1;
            const bool tile_partial = rem < kTilePages * kPage;
            const bool tok_ok = r < rem;
            const uint32_t t_s = tmem + lane_sel + kColS + 16 * sb;
            const uint32_t p_addr = p_row + kPBytes * sb;

            mbar_wait(bar_sfull + 8 * sb, ph2);        // S(gt) is in TMEM
            if (gt >= 2) mbar_wait(bar_done + 8 * sb, ph2 ^ 1);   // PV(gt-2) has read P buffer gt&1 (the PV warp commits
                                                                   // once per tile: its issue stream bounds the tile period)
            tc_fence_after();

            float lt[NH];
            // softmax of this thread's row against the current references -> P (fp16, MN-major operand)
            auto softmax_pass = [&]() -> bool {
              float t[NH];
              tmem_ld<NH>(t_s, t);
#pragma unroll
              for (int j = 0; j < NH; j += 2) ffma2(t[j], t[j + 1], t[j], t[j + 1], score_scale, nmref[j], nmref[j + 1]);
              if (tile_partial) {
#pragma unroll
                for (int j = 0; j < NH; ++j) t[j] = tok_ok ? t[j] : -INFINITY;
              }
              float tmax = t[0];
#pragma unroll
              for (int j = 1; j < NH; ++j) tmax = fmaxf(tmax, t[j]);
#pragma unroll
              for (int j = 0; j < NH; ++j) lt[j] = ex2(t[j]);
#pragma unroll
              for (int c = 0; c < NH / 8; ++c) {
                uint4 o;
                if constexpr (Geo::kBf16) {                // kind::f16 wants A and B of one type: P as bf16, like V
                  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(o.x) : "f"(lt[8 * c + 1]), "f"(lt[8 * c + 0]));
                  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(o.y) : "f"(lt[8 * c + 3]), "f"(lt[8 * c + 2]));
                  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(o.z) : "f"(lt[8 * c + 5]), "f"(lt[8 * c + 4]));
                  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(o.w) : "f"(lt[8 * c + 7]), "f"(lt[8 * c + 6]));
                } else {
                  asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(o.x) : "f"(lt[8 * c + 1]), "f"(lt[8 * c + 0]));
                  asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(o.y) : "f"(lt[8 * c + 3]), "f"(lt[8 * c + 2]));
                  asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(o.z) : "f"(lt[8 * c + 5]), "f"(lt[8 * c + 4]));
                  asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(o.w) : "f"(lt[8 * c + 7]), "f"(lt[8 * c + 6]));
                }
                sts128(p_addr + 128 * c, o);
              }
              return tmax > kThresh;
            };

            bool rebase = (i == 0);
            if (!rebase) {
              const bool ex = softmax_pass();
              rebase = bar_softmax_or(1, ex);
            }
            if (__builtin_expect(rebase, 0)) {
              // ---- per-head maximum score of the tile -> new references; O and l rescaled
              float tm[NH];
              {
                float sv[NH];
                tmem_ld<NH>(t_s, sv);
#pragma unroll
                for (int j = 0; j < NH; ++j) {
                  float x = tok_ok ? sv[j] * score_scale : -INFINITY;
#pragma unroll
                  for (int o = 16; o; o >>= 1) x = fmaxf(x, __shfl_xor_sync(kFull, x, o));
                  tm[j] = x;
                }
              }
              if (lane == 0) {
#pragma unroll
                for (int j = 0; j < NH; ++j) sh.wmax[cw][j] = tm[j];
              }
              tc_fence_before();
              bar_softmax(1);
              float f[NH];
#pragma unroll
              for (int j = 0; j < NH; ++j) {
                float m = sh.wmax[0][j];
#pragma unroll
                for (int w = 1; w < kSoftmaxWarps; ++w) m = fmaxf(m, sh.wmax[w][j]);
                const float mold = -nmref[j], mnew = fmaxf(mold, m);
                const float fm = (mold == -INFINITY) ? 0.f : ex2(mold - mnew);
                nmref[j] = -mnew;
                lsum[j] *= fm;
                f[j] = fm;
              }
              if (i > 0) {  // every PV of this unit issued so far has to be in O before it is rescaled
                mbar_wait(bar_done + 8 * (sb ^ 1), ((gt - 1) >> 1) & 1);
                tc_fence_after();
                float ov[NH];
                const uint32_t t_o = tmem + lane_sel + kColO;      // channel r, heads 0..NH-1
                tmem_ld<NH>(t_o, ov);
#pragma unroll
                for (int j = 0; j < NH; ++j) ov[j] *= f[j];
                tmem_st<NH>(t_o, ov);
              }
              (void)softmax_pass();
              bar_softmax(1);                            // wmax may be rewritten only after every warp read it
            }
#pragma unroll
            for (int j = 0; j < NH; j += 2) fadd2(lsum[j], lsum[j + 1], lsum[j], lsum[j + 1], lt[j], lt[j + 1]);

            // ---- S has been read (QK may overwrite the buffer), P is written, O is consistent with mref
            fence_async_smem();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) {
              mbar_arrive(bar_sfree + 8 * sb);
              mbar_arrive(bar_ready + 8 * sb);
            }
            ++gt;
          }

          // ============================================================ the unit's (m, l)
#pragma unroll
          for (int j = 0; j < NH; ++j) {
            float v = lsum[j];
#pragma unroll
            for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
            lsum[j] = v;
          }
          if (lane == 0) {
#pragma unroll
            for (int j = 0; j < NH; ++j) {
              sh.lsum[cw][j] = lsum[j];
              if (cw == 0) sh.mref[j] = -nmref[j];
            }
          }
          bar_softmax(1);
          if (atid < G) {                              // one thread per query head
            float l = 0.f;
#pragma unroll
            for (int w = 0; w < kSoftmaxWarps; ++w) l += sh.lsum[w][atid];
            ml_out[un.row0 + (long long)atid * num_splits] = make_float2(sh.mref[atid] * 0.6931471805599453f, l);   // natural log
          }
          if (un.slots_used > 0) {                     // item finished: its remaining slots are empty
            const long long row_item = un.row0 - (un.slots_used - 1);
            const int n_empty = num_splits - un.slots_used;
            for (int e = atid; e < G * n_empty; e += 32 * kSoftmaxWarps) {
              const int head = e / n_empty, sl = un.slots_used + (e - head * n_empty);
              ml_out[row_item + (long long)head * num_splits + sl] = make_float2(-INFINITY, 0.f);
            }
          }
          bar_softmax(1);                                // sh.lsum / sh.mref are reused by the next unit
        }
      };
      if (G > 8) run(std::integral_constant<int, 16>{});
      else run(std::integral_constant<int, 8>{});
    } else {
      // ============================================================== V warps: thread = channel d, all 128 tokens
      // FP8: cvt.rn.f16x2.e4m3x2 per token pair; BF16: the pairs as they are.  No scales, hence no reference exponent.
      const uint32_t t_o = tmem + lane_sel + kColO;
      Cursor cur;
      sc.start(cur);
      Unit un;
      int gt = 0, s = 0, ph_full = 0;
      while (sc.next(cur, un)) {
        int rem = un.tok_end - un.p0 * kPage;
        for (int i = 0; i < un.n_tiles; ++i, rem -= kTilePages * kPage) {
          const int sb = gt & 1;
          // this channel's 16 tokens of page 0 (Ultra-TQ: its 8 code bytes; scale / zero of its block q from kTqVMeta on)
          const uint32_t vst = base + Geo::kOffV + s * kVStageBytes + (Geo::kTq ? kTqVCodes + 8 * r : (16 * Geo::kElem) * r);
          mbar_wait(bar_fullv + 8 * s, ph_full);
          if (gt >= 2) {                               // PV(gt-2) has read Vhat buffer gt&1
            mbar_wait(bar_done + 8 * sb, ((gt >> 1) - 1) & 1);
            tc_fence_after();
          }
          const uint32_t t_v = tmem + lane_sel + kColV + 64 * sb;
          const bool partial = rem < kTilePages * kPage;
#pragma unroll
          for (int h = 0; h < 4; ++h) {                // 32 tokens = two pages = 16 TMEM columns at a time
            uint32_t o[16];
#pragma unroll
            for (int pp = 0; pp < 2; ++pp) {
              const int pg = 2 * h + pp;
              if constexpr (Geo::kTq) {
                // Alg. 2 l.7 "V: scale . code + zero": nibbles j and j + 4 of an octet word are tokens 2j, 2j + 1; with
                // 0x4300 (bf16 128.0) below them they read 128 + code exactly; (x - 128) * scale + zero in bf16, one rounding
                uint32_t cw2[2];
                asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(cw2[0]), "=r"(cw2[1]) : "r"(vst + kVPage * pg));
                const uint32_t meta = base + Geo::kOffV + s * kVStageBytes + kVPage * pg + kTqVMeta + 64 * q;
                const uint4 s0 = lds128(meta), s1 = lds128(meta + 16), z0 = lds128(meta + 32), z1 = lds128(meta + 48);
                const uint32_t sc2[8] = {s0.x, s0.y, s0.z, s0.w, s1.x, s1.y, s1.z, s1.w};
                const uint32_t ze2[8] = {z0.x, z0.y, z0.z, z0.w, z1.x, z1.y, z1.z, z1.w};
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                  const uint32_t x = ((cw2[j >> 2] >> (4 * (j & 3))) & 0x000F000Fu) | 0x43004300u;
                  uint32_t cpair;
                  asm("sub.rn.bf16x2 %0, %1, %2;" : "=r"(cpair) : "r"(x), "r"(0x43004300u));
                  asm("fma.rn.bf16x2 %0, %1, %2, %3;" : "=r"(o[8 * pp + j]) : "r"(cpair), "r"(sc2[j]), "r"(ze2[j]));
                }
              } else if constexpr (KV == UQ_KV_BF16) {
                const uint4 a = lds128(vst + kVPage * pg), b = lds128(vst + kVPage * pg + 16);
                o[8 * pp + 0] = a.x; o[8 * pp + 1] = a.y; o[8 * pp + 2] = a.z; o[8 * pp + 3] = a.w;
                o[8 * pp + 4] = b.x; o[8 * pp + 5] = b.y; o[8 * pp + 6] = b.z; o[8 * pp + 7] = b.w;
              } else {
                const uint4 a = lds128(vst + kVPage * pg);
                const uint32_t w[4] = {a.x, a.y, a.z, a.w};
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                  o[8 * pp + 2 * j] = cvt_e4m3x2(w[j], 0);
                  o[8 * pp + 2 * j + 1] = cvt_e4m3x2(w[j], 1);
                }
              }
              if (partial) {                           // tokens past the end: stale bytes (NaN patterns included) -> 0
                const int nv = rem - 16 * pg;          // valid tokens of this page
#pragma unroll
                for (int j = 0; j < 8; ++j)
                  o[8 * pp + j] = (2 * j + 1 < nv) ? o[8 * pp + j] : ((2 * j < nv) ? (o[8 * pp + j] & 0xFFFFu) : 0u);
              }
            }
            tmem_st16_nowait(t_v + 16 * h, o);
          }
          tmem_wait_st();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) {
            mbar_arrive(bar_ready + 8 * sb);
            mbar_arrive(bar_emptyv + 8 * s);
          }
          ++gt;
          if (++s == kVStages) { s = 0; ph_full ^= 1; }
        }
        // the unit's accumulator
        mbar_wait(bar_done + 8 * ((gt - 1) & 1), ((gt - 1) >> 1) & 1);
        tc_fence_after();
        {
          float ov[16];
          tmem_ld<16>(t_o, ov);
#pragma unroll
          for (int j = 0; j < 16; ++j)
            if (j < G) partial_acc[(un.row0 + (long long)j * num_splits) * kHeadDim + r] = ov[j];
        }
        tc_fence_before();
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (role == 1) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(Geo::kTmemCols));
  }
}

// ---------------------------------------------------------------- append for the comparison caches
// One warp per new (token, kv head) row [and per query row for FP8]; a lane owns 4 channels.  FP8: OCP E4M3 of the
// bf16 value itself — the hardware conversion from the exact float32 is one rounding to nearest even, saturating at
// 448, i.e. the oracle's rule; a result of -0 is stored as +0 (reading G7).  BF16: the bits as they are.
__device__ __forceinline__ uint32_t e4m3x4_of_bf16(uint2 raw) {
  const float x0 = __uint_as_float(raw.x << 16), x1 = __uint_as_float(raw.x & 0xFFFF0000u);
  const float x2 = __uint_as_float(raw.y << 16), x3 = __uint_as_float(raw.y & 0xFFFF0000u);
  uint32_t n;
  asm("{\n.reg .b16 h0, h1;\n"
      "cvt.rn.satfinite.e4m3x2.f32 h0, %2, %1;\n"
      "cvt.rn.satfinite.e4m3x2.f32 h1, %4, %3;\n"
      "mov.b32 %0, {h0, h1};\n}\n" : "=r"(n) : "f"(x0), "f"(x1), "f"(x2), "f"(x3));
  const uint32_t t = n & 0x7F7F7F7Fu;
  const uint32_t nz = ((t + 0x7F7F7F7Fu) | t) & 0x80808080u;       // bit 7 of a byte set iff its magnitude is not 0
  return n & (0x7F7F7F7Fu | nz);
}

template <int KV>
__global__ void __launch_bounds__(128)
append_cmp_kernel(const uint16_t* __restrict__ k_new, const uint16_t* __restrict__ v_new,
                  const int32_t* __restrict__ cu_new, const int32_t* __restrict__ seq_lens,
                  const int32_t* __restrict__ block_tables, int max_pages, int batch, int total_new, int Hq, int Hkv,
                  uint8_t* __restrict__ cache, const uint16_t* __restrict__ q, uint8_t* __restrict__ q_out) {
  using Geo = CmpGeo<KV>;
  pdl_launch_dependents();
  pdl_wait();
  const int lane = threadIdx.x & 31;
  const long long u = (long long)blockIdx.x * 4 + (threadIdx.x >> 5);
  const long long n_kv = (long long)total_new * Hkv;
  if (u < n_kv) {
    const int row = (int)(u / Hkv), h = (int)(u - (long long)row * Hkv);
    int lo = 0, hi = batch;                            // the sequence of new row `row`: largest b with cu_new[b] <= row
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (cu_new[mid] <= row) lo = mid; else hi = mid;
    }
    const int b = lo, pos = seq_lens[b] + (row - cu_new[b]), t = pos & 15;
    const int page = block_tables[(long long)b * max_pages + (pos >> 4)];
    uint8_t* rec = cache + ((long long)page * Hkv + h) * Geo::kRecordBytes;
    const long long src = ((long long)row * Hkv + h) * kHeadDim + 4 * lane;
    const uint2 kr = *reinterpret_cast<const uint2*>(k_new + src), vr = *reinterpret_cast<const uint2*>(v_new + src);
    if constexpr (KV == UQ_KV_BF16) {
      *reinterpret_cast<uint2*>(rec + 256 * t + 8 * lane) = kr;
      const uint16_t vv[4] = {(uint16_t)(vr.x & 0xFFFFu), (uint16_t)(vr.x >> 16), (uint16_t)(vr.y & 0xFFFFu), (uint16_t)(vr.y >> 16)};
#pragma unroll
      for (int c = 0; c < 4; ++c)
        *reinterpret_cast<uint16_t*>(rec + Geo::kKPage + 32 * (4 * lane + c) + 2 * t) = vv[c];
    } else {
      *reinterpret_cast<uint32_t*>(rec + 128 * t + 4 * lane) = e4m3x4_of_bf16(kr);
      const uint32_t vb = e4m3x4_of_bf16(vr);
#pragma unroll
      for (int c = 0; c < 4; ++c) rec[Geo::kKPage + 16 * (4 * lane + c) + t] = (uint8_t)(vb >> (8 * c));
    }
    return;
  }
  if constexpr (KV == UQ_KV_FP8_E4M3) {
    const long long qu = u - n_kv;
    if (q != nullptr && qu < (long long)batch * Hq)
      *reinterpret_cast<uint32_t*>(q_out + qu * kHeadDim + 4 * lane) =
          e4m3x4_of_bf16(*reinterpret_cast<const uint2*>(q + qu * kHeadDim + 4 * lane));
  }
}

// ---------------------------------------------------------------- host
int32_t cmp_maps(int kv, const void* cache, long long records, const void* q_enc, long long q_rows, CUtensorMap* tk,
                 CUtensorMap* tq) {
  const EncodeTiledFn encode = encode_tiled_fn();
  if (!encode) return UQ_ERR_CUDA;
  const bool bf = (kv != UQ_KV_FP8_E4M3), no_k = (kv == UQ_KV_ULTRA_TQ);   // Ultra-TQ: no K map (its records are bulk-copied)
  const cuuint64_t rec = bf ? 8192 : 4096, rowb = bf ? 256 : 128;
  const cuuint64_t gdim[3] = {128, 16, (cuuint64_t)records};
  const cuuint64_t gstr[2] = {rowb, rec};
  const cuuint32_t box[3] = {bf ? 64u : 128u, 16, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  CUresult cr = CUDA_SUCCESS;
  if (no_k) *tk = CUtensorMap{};
  else cr = encode(tk, bf ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<void*>(cache),
                   gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                   CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (cr == CUDA_SUCCESS) {
    const cuuint64_t qdim[2] = {128, (cuuint64_t)q_rows};
    const cuuint64_t qstr[1] = {rowb};
    const cuuint32_t qbox[2] = {bf ? 64u : 128u, 16};
    cr = encode(tq, bf ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void*>(q_enc), qdim,
                qstr, qbox, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  }
  if (cr != CUDA_SUCCESS) {
    set_error("baseline decode: cuTensorMapEncodeTiled failed with CUresult %d", (int)cr);
    return UQ_ERR_CUDA;
  }
  return UQ_OK;
}

template <int KV>
int32_t launch_cmp(const uq_config* cfg, const CUtensorMap& tk, const CUtensorMap& tq, const void* cache,
                   const int32_t* block_tables, int32_t max_pages, const int32_t* seq_lens, int32_t batch,
                   int32_t num_splits, float* partial_acc, float* partial_ml, cudaStream_t stream,
                   const TqCodebook& cb = TqCodebook{}) {
  using Geo = CmpGeo<KV>;
  int sm_count = 0;
  int32_t st = current_device_sms(&sm_count);
  if (st != UQ_OK) return st;
  const long long slots = (long long)sm_count * Geo::kCtasPerSm, items = (long long)batch * cfg->num_kv_heads;
  const dim3 grid((unsigned)((num_splits == 1 && items < slots) ? items : slots));
  st = opt_in_dynamic_smem((const void*)decode_cmp_kernel<KV>, Geo::kSmemBytes, "baseline decode: cudaFuncSetAttribute");
  if (st != UQ_OK) return st;
  const float score_scale = resolved_sm_scale(cfg) * 1.4426950408889634f;
  return check_cuda(launch_pdl(decode_cmp_kernel<KV>, grid, dim3(Geo::kThreads), (size_t)Geo::kSmemBytes, stream, tk, tq,
                               (const uint8_t*)cache, block_tables, (int)max_pages, seq_lens, (int)batch,
                               (int)cfg->num_q_heads, (int)cfg->num_kv_heads, (int)num_splits, score_scale, partial_acc,
                               partial_ml, cb),
                    "uq_baseline_decode_attention launch");
}

int32_t check_kv(const uq_config* cfg, int32_t kv, const char* who) {
  int32_t st = check_config(cfg);
  if (st != UQ_OK) return st;
  st = require_head_dim_128(cfg, who);
  if (st != UQ_OK) return st;
  if (kv != UQ_KV_FP8_E4M3 && kv != UQ_KV_BF16 && kv != UQ_KV_ULTRA_TQ) {
    set_error("%s: kv_format must be UQ_KV_FP8_E4M3 (1), UQ_KV_BF16 (2) or UQ_KV_ULTRA_TQ (3)", who);
    return UQ_ERR_INVALID_ARG;
  }
  return UQ_OK;
}

}  // namespace
}  // namespace uq

extern "C" size_t uq_baseline_record_bytes(const uq_config* cfg, int32_t kv_format) {
  if (uq::check_kv(cfg, kv_format, "uq_baseline_record_bytes") != UQ_OK) return 0;
  return kv_format == UQ_KV_ULTRA_TQ ? (size_t)uq::kTqRecord : (kv_format == UQ_KV_BF16 ? 8192 : 4096);
}

extern "C" int32_t uq_baseline_append(const uq_config* cfg, int32_t kv_format, const void* k_new, const void* v_new,
                                      const int32_t* cu_new, const int32_t* seq_lens, const int32_t* block_tables,
                                      int32_t max_pages, int32_t batch, int32_t total_new, void* cache, int64_t num_pages,
                                      const void* q, void* q_out, void* stream) {
  using namespace uq;
  NvtxRange nvtx_range("uq_baseline_append");
  int32_t st = check_kv(cfg, kv_format, "uq_baseline_append");
  if (st != UQ_OK) return st;
  if (kv_format == UQ_KV_ULTRA_TQ) {
    set_error("uq_baseline_append: the Ultra-TQ cache takes a codebook: call uq_tq_append");
    return UQ_ERR_INVALID_ARG;
  }
  if (batch <= 0 || total_new < 0 || max_pages <= 0 || num_pages <= 0) {
    set_error("baseline append: batch/max_pages/num_pages must be positive, total_new >= 0");
    return UQ_ERR_INVALID_ARG;
  }
  if (total_new > 0 && (!k_new || !v_new || !cu_new || !seq_lens || !block_tables || !cache)) {
    set_error("baseline append: NULL pointer");
    return UQ_ERR_INVALID_ARG;
  }
  if (kv_format == UQ_KV_FP8_E4M3 && (q == nullptr) != (q_out == nullptr)) {
    set_error("baseline append: q and q_out must both be given or both be NULL");
    return UQ_ERR_INVALID_ARG;
  }
  if ((((uintptr_t)k_new | (uintptr_t)v_new | (uintptr_t)q) & 7u) || ((uintptr_t)cache & 15u) || ((uintptr_t)q_out & 3u)) {
    set_error("baseline append: misaligned pointer (k/v/q 8 B, cache 16 B, q_out 4 B)");
    return UQ_ERR_INVALID_ARG;
  }
  if ((cfg->flags & UQ_FLAG_DEBUG_CHECKS) && total_new > 0) {
    st = debug_check_tables("uq_baseline_append", block_tables, max_pages, batch, num_pages, seq_lens, cu_new, total_new, 0,
                            cfg->page_size, 1, (cudaStream_t)stream);
    if (st != UQ_OK) return st;
  }
  const long long q_rows = (kv_format == UQ_KV_FP8_E4M3 && q) ? (long long)batch * cfg->num_q_heads : 0;
  const long long units = (long long)total_new * cfg->num_kv_heads + q_rows;
  if (units == 0) return UQ_OK;
  const long long blocks = (units + 3) / 4;
  if (blocks > 0x7fffffffLL) {
    set_error("baseline append: too many work units");
    return UQ_ERR_INVALID_ARG;
  }
  auto kern = kv_format == UQ_KV_BF16 ? append_cmp_kernel<UQ_KV_BF16> : append_cmp_kernel<UQ_KV_FP8_E4M3>;
  return check_cuda(launch_pdl(kern, dim3((unsigned)blocks), dim3(128), 0, (cudaStream_t)stream, (const uint16_t*)k_new,
                               (const uint16_t*)v_new, cu_new, seq_lens, block_tables, (int)max_pages, (int)batch,
                               (int)total_new, (int)cfg->num_q_heads, (int)cfg->num_kv_heads, (uint8_t*)cache,
                               (const uint16_t*)q, (uint8_t*)q_out),
                    "uq_baseline_append launch");
}

extern "C" int32_t uq_baseline_decode_attention(const uq_config* cfg, int32_t kv_format, const void* q_enc, const void* cache,
                                                int64_t num_pages, const int32_t* block_tables, int32_t max_pages,
                                                const int32_t* seq_lens, int32_t batch, int32_t num_splits,
                                                float* partial_acc, float* partial_ml, void* stream) {
  using namespace uq;
  NvtxRange nvtx_range("uq_baseline_decode_attention");
  int32_t st = check_kv(cfg, kv_format, "uq_baseline_decode_attention");
  if (st != UQ_OK) return st;
  if (kv_format == UQ_KV_ULTRA_TQ) {
    set_error("uq_baseline_decode_attention: the Ultra-TQ cache takes a codebook: call uq_tq_decode_attention");
    return UQ_ERR_INVALID_ARG;
  }
  if (!q_enc || !cache || !block_tables || !seq_lens || !partial_acc || !partial_ml || batch <= 0 || num_splits <= 0 ||
      max_pages <= 0 || num_pages <= 0) {
    set_error("baseline decode: NULL pointer or non-positive size");
    return UQ_ERR_INVALID_ARG;
  }
  if (((uintptr_t)cache & 127u) || ((uintptr_t)q_enc & 15u) || ((uintptr_t)partial_acc & 15u) || ((uintptr_t)partial_ml & 7u)) {
    set_error("baseline decode: misaligned pointer (cache 128 B, q 16 B, partial_acc 16 B, partial_ml 8 B)");
    return UQ_ERR_INVALID_ARG;
  }
  if (batch > kMaxBatch) {
    set_error("baseline decode: batch %d exceeds the supported maximum of %d sequences per call", batch, kMaxBatch);
    return UQ_ERR_UNSUPPORTED;
  }
  const long long records = (long long)num_pages * cfg->num_kv_heads;
  if (records > 0x7fffffffLL) {
    set_error("baseline decode: num_pages * num_kv_heads must be < 2^31");
    return UQ_ERR_INVALID_ARG;
  }
  if (cfg->flags & UQ_FLAG_DEBUG_CHECKS) {
    st = debug_check_tables("uq_baseline_decode_attention", block_tables, max_pages, batch, num_pages, seq_lens, nullptr, 0, 0,
                            cfg->page_size, 0, (cudaStream_t)stream);
    if (st != UQ_OK) return st;
  }
  CUtensorMap tk, tq;
  st = cmp_maps(kv_format, cache, records, q_enc, (long long)batch * cfg->num_q_heads, &tk, &tq);
  if (st != UQ_OK) return st;
  if (kv_format == UQ_KV_BF16)
    return launch_cmp<UQ_KV_BF16>(cfg, tk, tq, cache, block_tables, max_pages, seq_lens, batch, num_splits, partial_acc,
                                  partial_ml, (cudaStream_t)stream);
  return launch_cmp<UQ_KV_FP8_E4M3>(cfg, tk, tq, cache, block_tables, max_pages, seq_lens, batch, num_splits, partial_acc,
                                    partial_ml, (cudaStream_t)stream);
}

// Ultra-TQ (Alg. 2): the decode of uq_baseline_decode_attention over the codebook cache.
extern "C" int32_t uq_tq_decode_attention(const uq_config* cfg, const float* codebook_k, const void* q_rot, const void* cache,
                                          int64_t num_pages, const int32_t* block_tables, int32_t max_pages,
                                          const int32_t* seq_lens, int32_t batch, int32_t num_splits, float* partial_acc,
                                          float* partial_ml, void* stream) {
  using namespace uq;
  NvtxRange nvtx_range("uq_tq_decode_attention");
  int32_t st = check_kv(cfg, UQ_KV_ULTRA_TQ, "uq_tq_decode_attention");
  if (st != UQ_OK) return st;
  if (!codebook_k || !q_rot || !cache || !block_tables || !seq_lens || !partial_acc || !partial_ml || batch <= 0 ||
      num_splits <= 0 || max_pages <= 0 || num_pages <= 0) {
    set_error("uq_tq_decode_attention: NULL pointer or non-positive size");
    return UQ_ERR_INVALID_ARG;
  }
  if (((uintptr_t)cache & 15u) || ((uintptr_t)q_rot & 15u) || ((uintptr_t)partial_acc & 15u) || ((uintptr_t)partial_ml & 7u)) {
    set_error("uq_tq_decode_attention: misaligned pointer (cache 16 B, q_rot 16 B, partial_acc 16 B, partial_ml 8 B)");
    return UQ_ERR_INVALID_ARG;
  }
  if (batch > kMaxBatch) {
    set_error("uq_tq_decode_attention: batch %d exceeds the supported maximum of %d sequences per call", batch, kMaxBatch);
    return UQ_ERR_UNSUPPORTED;
  }
  if ((long long)num_pages * cfg->num_kv_heads > 0x7fffffffLL) {
    set_error("uq_tq_decode_attention: num_pages * num_kv_heads must be < 2^31");
    return UQ_ERR_INVALID_ARG;
  }
  TqCodebook cb;
  for (int i = 0; i < 16; ++i) {
    cb.c[i] = codebook_k[i];
    if (!(cb.c[i] == cb.c[i]) || (i > 0 && !(cb.c[i] > cb.c[i - 1]))) {
      set_error("uq_tq_decode_attention: codebook_k must be 16 finite values in ascending order");
      return UQ_ERR_INVALID_ARG;
    }
  }
  if (cfg->flags & UQ_FLAG_DEBUG_CHECKS) {
    st = debug_check_tables("uq_tq_decode_attention", block_tables, max_pages, batch, num_pages, seq_lens, nullptr, 0, 0,
                            cfg->page_size, 0, (cudaStream_t)stream);
    if (st != UQ_OK) return st;
  }
  CUtensorMap tk, tq;
  st = cmp_maps(UQ_KV_ULTRA_TQ, cache, 0, q_rot, (long long)batch * cfg->num_q_heads, &tk, &tq);
  if (st != UQ_OK) return st;
  return launch_cmp<UQ_KV_ULTRA_TQ>(cfg, tk, tq, cache, block_tables, max_pages, seq_lens, batch, num_splits, partial_acc,
                                    partial_ml, (cudaStream_t)stream, cb);
}
