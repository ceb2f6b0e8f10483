// uq_decode_prefix_m.cu — decode attention over a SHARED PREFIX, second design ("cascade"; the
// agent workloads of the paper share a long prompt): the query rows of many sequences on the M side.
//
// The first design (uq_decode_prefix.cu, round 1) kept the decode kernel's orientation — tokens on the TMEM lanes, the
// 16 heads of each of four sequences on the columns — and paid for it in the softmax: a thread owned one token of one
// sequence (16 scores), every row maximum / sum crossed 128 threads, each sequence needed its own group of four warps
// and its own consensus barrier: 925 warp instructions per (sequence, 128-token tile), 0.3 of the MUFU / tensor bound.
// Here the score tile is S^T = Q K^T with M = 128 = NSEQ sequences x HS head slots (8 x 16 or, for GQA groups <= 8,
// 16 x 8) on the TMEM lanes and the tile's 128 tokens on the columns:
//   * a softmax thread owns one (sequence, head) row: 128 scores per tile, its reference / running sum are private —
//     no cross-thread reduction, no consensus (a row's reference scales that row of O only), ~3 instructions a score;
//   * P (fp16) goes back to TMEM and is the A operand of the PV product; Vhat (fp16, [channel][token], 128-byte swizzle)
//     is written to shared memory ONCE per tile for all NSEQ sequences and is the B operand; O[128 rows x 128 channels]
//     accumulates in TMEM;
//   * the row sums of P come out of the same product: 16 constant rows of ones behind the 128 channel rows of Vhat
//     (N = 144) put sum_t P[row][t] into accumulator columns 128..143 — the sum of exactly the fp16 values the numerator
//     uses, and 64 additions per thread and tile less in the softmax warps (4 % of the kernel's time);
//   * K codes x FP8 queries by tcgen05.mma kind::mxf8f6f4.block_scale with the K group scales as the B-side scale
//     factors (the paper's FP8 x FP4 scaled MMA), the query-side factors constant 1.
// V's reference exponent: a V warp (one 32-channel scale group) scans the scale bytes of its unit's tile range first —
// the prefix is L2 resident — and converts against the maximum it found, so O never has to be rescaled for V.
// head_dim 128.  Partial format, schedule (equal tile ranges per CTA) and merge as uq_decode.cu / include/uq.h.
#include <cuda.h>
#include <cuda_fp16.h>

#include "uq_tc.cuh"

namespace uq {
namespace {

#ifndef UQ_PREFIX_SW
#define UQ_PREFIX_SW 2
#endif
constexpr int kSW = UQ_PREFIX_SW;                    // softmax warps per TMEM lane quarter: each takes 128 / kSW token columns
static_assert(kSW == 2 || kSW == 4, "softmax warps per lane quarter");
constexpr int kSoftmaxWarps = 4 * kSW, kVWarps = 4, kIssuerWarps = 4;
constexpr int kComputeWarps = kSoftmaxWarps + kVWarps;
constexpr int kThreads = (kComputeWarps + kIssuerWarps) * 32;
constexpr int kCP = 8 / kSW;                         // 16-token chunks per softmax warp
constexpr int kColsPart = 128 / kSW;                 // score / accumulator columns per softmax warp
constexpr int kKStages = 3, kVStages = 4;
constexpr int kTilePages = 8;                        // 128 tokens per tile
constexpr int kRestBytes = kRecordBytes - 1024;      // V codes + K scales + V scales = 1152
constexpr int kKStageBytes = kTilePages * 2048;      // K codes, one byte per code
constexpr int kVStageBytes = kTilePages * kRestBytes;
constexpr int kVhRows = 144;                         // 128 channels + 16 rows of ones: the PV product also sums each row of P
constexpr int kVhBlock = kVhRows * 128;              // one block of 64 tokens: [144 rows][128 B], 128-byte swizzle
constexpr int kVhBytes = 2 * kVhBlock;               // Vhat of a tile: two blocks of 64 tokens
constexpr int kQBytes = 128 * 128;                   // the query rows of a unit: [128 rows][128 B E4M3]
constexpr float kThresh = 12.0f;
#ifdef UQ_TRACE
__device__ unsigned long long g_trace_prefix[UQ_TRACE_TILES * 16];
#endif
// trace events of CTA 3 (UQ_TR): 0 QK issue, 6 the QK warp sees PV(gt-2) done, 9 / 5 PV warp: Vhat ready / issue, softmax
// warp (part 0, quarter 0): 1 S seen, 10 pass 1 done, 2 maxima exchanged, 3 pass 2 done; V warp of quarter 0: 7 tile
// bytes seen, 12 Vhat buffer free, 4 tile converted
#define TRP(ev, tile) UQ_TR(g_trace_prefix, 3, ev, tile)

constexpr int kOffK = 0;                                        // kKStages x 16384, SW128
constexpr int kOffVh = kOffK + kKStages * kKStageBytes;         // 2 x 32768, SW128
constexpr int kOffQ = kOffVh + 2 * kVhBytes;                    // 2 x 16384, SW128
constexpr int kOffV = kOffQ + 2 * kQBytes;                      // kVStages x 9216
constexpr int kOffSFB = kOffV + kVStages * kVStageBytes;        // 4 x 512: K scales of a tile (ring of four atoms)
constexpr int kOffSFA = kOffSFB + 2048;                         // 512: query-side factors, constant
constexpr int kOffMul = kOffSFA + 512;                          // 4 V warps x 256 B of fp16 multipliers
constexpr int kOffEnd = kOffMul + kVWarps * 256;
constexpr int kSmemBytes = kOffEnd + 1024;
static_assert(kOffVh % 1024 == 0 && kOffQ % 1024 == 0, "swizzled tiles need 1024-byte alignment");

// TMEM columns (512 allocated, one CTA per SM)
constexpr uint32_t kColS = 0;      // 2 x 128: scores, lane = (sequence, head) row, column = token.  P (f16x2, column c =
                                   // tokens 2c, 2c+1) overwrites the first 64 columns of its score buffer IN PLACE, chunk
                                   // after chunk behind the softmax thread's reads: P is double-buffered for free
constexpr uint32_t kColO = 256;    // 144: accumulator, column = channel; columns 128..143 = the row sum of P (the ones rows)
constexpr uint32_t kColL = kColO + 128;
constexpr uint32_t kColSFA = 400;  // 4
constexpr uint32_t kColSFB = 404;  // 2 x 4
constexpr uint32_t kTmemCols = 512;

struct Shared {
  uint64_t full_k[kKStages], empty_k[kKStages], full_v[kVStages], empty_v[kVStages];
  uint64_t s_full[2];              // QK commit -> softmax warps: S(gt) is in TMEM buffer gt & 1
  uint64_t p_ready[2];             // 4 softmax warps -> PV warp: P(gt) has replaced S(gt) in buffer gt & 1
  uint64_t v_ready[2];             // 4 V warps -> PV warp: Vhat buffer gt & 1 is written
  uint64_t done[2];                // PV commit of tile gt -> done[gt & 1]: O up to date; score buffer / Vhat buffer gt & 1 free
  uint64_t q_full[2];
  uint32_t tmem_base;
  float vscale[4][4];              // [unit ordinal & 3][group]: 2^(eref - 13 - 127), for the epilogue of that unit
  float pmax[2][kSW][128];         // [tile parity][part][row]: partial row maxima of a tile (pass 1)
};

// Items = (group of NSEQ consecutive sequences, kv head), kv head fastest, PT tiles each; the tiles of all items form
// one sequence cut into equal ranges, one per CTA; a CTA walks UNITS (item, tile range); the CTAs sharing an item fill
// consecutive partial slots of it (the same slot for each of its sequences).
struct Unit {
  int b0, kvh, p0, n_tiles, slot, slots_used;
};
struct Sched {
  int NSEQ, Hkv, S, tpc, total, PT;
  int g, g1;                                           // cursor: global tile, range end
  __device__ void start() {
    g = min((int)blockIdx.x * tpc, total);
    g1 = min(g + tpc, total);
  }
  __device__ bool next(Unit& u) {
    if (g >= g1) return false;
    const int it = g / PT, t0 = g - it * PT, t1 = min(PT, t0 + (g1 - g));
    const int grp = it / Hkv;
    u.kvh = it - grp * Hkv;
    u.b0 = grp * NSEQ;
    u.slot = (int)blockIdx.x - (g - t0) / tpc;
    u.slots_used = (t1 == PT) ? u.slot + 1 : 0;
    u.p0 = kTilePages * t0;
    u.n_tiles = t1 - t0;
    g += t1 - t0;
    return true;
  }
};

// D[tmem] (+)= A[smem, E4M3] . B[smem, E2M1]^T with UE8M0 block scales in TMEM (both sides)
__device__ __forceinline__ void umma_mx(uint32_t d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t acc, uint32_t tsfa,
                                        uint32_t tsfb) {
  asm volatile(
      "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::mxf8f6f4.block_scale [%0], %1, %2, %3, [%5], [%6], p;\n}\n"
      ::"r"(d), "l"(da), "l"(db), "r"(idesc), "r"(acc), "r"(tsfa), "r"(tsfb) : "memory");
}
__device__ __forceinline__ void tmem_ld16_nowait(uint32_t taddr, uint32_t (&r)[16]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                 "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
               : "r"(taddr));
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_st8_nowait(uint32_t taddr, const uint32_t (&v)[8]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
               ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]) : "memory");
}

// ---------------------------------------------------------------- the kernel
template <int HS>                                      // head slots per sequence on the M side: 16 (GQA 9..16) or 8
__global__ void __launch_bounds__(kThreads, 1)
decode_prefix_m_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ CUtensorMap tmap_q,
                       const uint8_t* __restrict__ cache, const int32_t* __restrict__ block_tables, int max_pages,
                       int prefix_tiles, int batch, int Hq, int Hkv, int num_splits,
                       float score_scale /* sm_scale * log2(e) */, float* __restrict__ partial_acc,
                       float* __restrict__ partial_ml) {
  constexpr int NSEQ = 128 / HS;
  extern __shared__ uint8_t smem_raw[];
  __shared__ __align__(8) Shared sh;

  const int G = Hq / Hkv;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  // warps 0..3 softmax, 4..7 V warps, 8..11 issuers (role 0 QK, 1 PV, 2 K producer, 3 V producer)
  const int role = warp < kComputeWarps ? warp + kIssuerWarps : warp - kComputeWarps;

  const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sQ = base + kOffQ, sSFA = base + kOffSFA, sSFB = base + kOffSFB, sVh = base + kOffVh;
  const uint32_t bar_fullk = smem_u32(&sh.full_k[0]), bar_emptyk = smem_u32(&sh.empty_k[0]),
                 bar_fullv = smem_u32(&sh.full_v[0]), bar_emptyv = smem_u32(&sh.empty_v[0]),
                 bar_sfull = smem_u32(&sh.s_full[0]), bar_pready = smem_u32(&sh.p_ready[0]),
                 bar_vready = smem_u32(&sh.v_ready[0]),
                 bar_done = smem_u32(&sh.done[0]), bar_qfull = smem_u32(&sh.q_full[0]);

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < kKStages; ++s) { mbar_init(bar_fullk + 8 * s, 1); mbar_init(bar_emptyk + 8 * s, 1); }
#pragma unroll
    for (int s = 0; s < kVStages; ++s) { mbar_init(bar_fullv + 8 * s, 1); mbar_init(bar_emptyv + 8 * s, kVWarps + 1); }
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      mbar_init(bar_sfull + 8 * h, 1);
      mbar_init(bar_pready + 8 * h, kSoftmaxWarps);
      mbar_init(bar_vready + 8 * h, kVWarps);
      mbar_init(bar_done + 8 * h, 1);
      mbar_init(bar_qfull + 8 * h, 1);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (role == 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&sh.tmem_base)),
                 "r"(kTmemCols));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  if (tid < 128) {  // query-side scale factors: UE8M0 byte 127 = 2^0
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(sSFA + 4 * tid), "r"(0x7F7F7F7Fu) : "memory");
  }
  // the ones rows (f16 1.0) of both Vhat buffers: rows 128..143 of each 64-token block — the swizzle permutes equal chunks
  for (int e = tid; e < 2 * 2 * 16 * 32; e += kThreads) {
    const int blk = e >> 9, w = e & 511;
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(sVh + kVhBytes * (blk >> 1) + kVhBlock * (blk & 1) + 128 * 128 + 4 * w),
                 "r"(0x3C003C00u) : "memory");
  }
  pdl_launch_dependents();
  pdl_wait();
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = sh.tmem_base;

  Sched sc;
  sc.NSEQ = NSEQ; sc.Hkv = Hkv; sc.S = num_splits; sc.PT = prefix_tiles;
  sc.total = ((batch + NSEQ - 1) / NSEQ) * Hkv * prefix_tiles;
  {
    const int even = (sc.total + (int)gridDim.x - 1) / (int)gridDim.x;
    const int fit = (prefix_tiles + num_splits - 2) / (num_splits - 1);   // an item spans at most num_splits ranges
    sc.tpc = max(1, max(even, fit));
  }
  sc.start();

  if (role == 0) {
    // ================================================================ QK warp: S[128 rows x 128 tokens] = Q . K^T
    // A = the unit's query rows (E4M3; one 3-D TMA copy per unit: [NSEQ sequences][HS heads][128 B]), B = the tile's K
    // codes (E2M1), SFA = 1, SFB = the K group scales (gathered into a 512-byte atom, smem -> TMEM by tcgen05.cp).
    // idesc: b_sf_id [4,6), A format E4M3 (0) at 7, B format E2M1 (5) at 10, N >> 3 at 17, UE8M0 at 23, M >> 4 at 24
    const uint32_t idesc_qk = (0u << 7) | (5u << 10) | (16u << 17) | (1u << 23) | (8u << 24);
    if (elect_one()) umma_cp_sf(tmem + kColSFA, make_desc(sSFA, 16, 128, 0));
    auto load_q = [&](const Unit& un, int k) {
      if (elect_one()) {
        mbar_expect_tx(bar_qfull + 8 * (k & 1), kQBytes);
        tma_load_3d_plain(sQ + kQBytes * (k & 1), &tmap_q, 0, un.kvh * G, un.b0, bar_qfull + 8 * (k & 1));
      }
    };
    Sched nxs = sc;
    Unit un, nx;
    bool have_nx = nxs.next(nx);
    int gt = 0, sk = 0, phk = 0, sv = 0, phv = 0, k = 0, k_q = -1;
    while (have_nx) {
      un = nx;
      have_nx = nxs.next(nx);
      for (int i = 0; i < un.n_tiles; ++i) {
        const int sb = gt & 1;
        // the tile's K scales first (the V stage is released early): atom gt & 3 was last read by the tcgen05.cp of
        // tile gt-4, complete since the wait for PV(gt-3) in the iteration before
        mbar_wait(bar_fullv + 8 * sv, phv);
        const uint32_t st = base + kOffK + sk * kKStageBytes, rest = base + kOffV + sv * kVStageBytes;
        uint32_t v[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) {                  // token r = 32 c + lane -> 16-byte line `lane`, word c
          const int r = 32 * c + lane;
          asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v[c]) : "r"(rest + kRestBytes * (r >> 4) + 1024 + 4 * (r & 15)));
        }
        sts128(sSFB + 512 * (gt & 3) + 16 * lane, make_uint4(v[0], v[1], v[2], v[3]));
        fence_async_smem();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_emptyv + 8 * sv);
        if (gt >= 2) {
          mbar_wait(bar_done + 8 * sb, ((gt >> 1) - 1) & 1);   // PV(gt-2) has read P out of this score buffer
          TRP(6, gt - 2);
        }
        if (i == 0 && k_q < k) { load_q(un, k); k_q = k; }
        if (i == 1 && have_nx) { load_q(nx, k + 1); k_q = k + 1; }
        if (i == 0) mbar_wait(bar_qfull + 8 * (k & 1), (k >> 1) & 1);
        mbar_wait(bar_fullk + 8 * sk, phk);
        TRP(0, gt);
        tc_fence_after();
        if (elect_one()) {
          const uint32_t t_sfb = tmem + kColSFB + 4 * sb, qb = sQ + kQBytes * (k & 1);
          umma_cp_sf(t_sfb, make_desc(sSFB + 512 * (gt & 3), 16, 128, 0));
#pragma unroll
          for (int kb = 0; kb < 4; ++kb)
            umma_mx(tmem + kColS + 128 * sb, make_desc(qb + 32 * kb, 16, 1024, 2), make_desc(st + 32 * kb, 16, 1024, 2),
                    idesc_qk | ((uint32_t)kb << 4), kb > 0, tmem + kColSFA, t_sfb + ((uint32_t)kb << 30));
          umma_commit(bar_sfull + 8 * sb);
          umma_commit(bar_emptyk + 8 * sk);
        }
        __syncwarp();
        ++gt;
        if (++sk == kKStages) { sk = 0; phk ^= 1; }
        if (++sv == kVStages) { sv = 0; phv ^= 1; }
      }
      ++k;
    }
  } else if (role == 1) {
    // ================================================================ PV warp: O[128 rows x 128 ch] += P . Vhat
    // A = P from TMEM (f16), B = Vhat from smem ([channel][token]: K-major, 128-byte swizzle), N = 128
    const uint32_t idesc_pv = (1u << 4) | ((uint32_t)(kVhRows >> 3) << 17) | (8u << 24);   // N = 144
    Unit un;
    int gt = 0;
    while (sc.next(un)) {
      for (int i = 0; i < un.n_tiles; ++i, ++gt) {
        const int sb = gt & 1;
        mbar_wait(bar_vready + 8 * sb, (gt >> 1) & 1);
        TRP(9, gt);
        mbar_wait(bar_pready + 8 * sb, (gt >> 1) & 1);
        TRP(5, gt);
        tc_fence_after();
        if (lane == 0) {
          const uint32_t vb = sVh + kVhBytes * sb;
#pragma unroll
          for (int j = 0; j < 8; ++j)                    // 16 tokens per MMA = 8 columns of P, 32 bytes of a Vhat row
            umma_f16_ts(tmem + kColO, tmem + kColS + 128 * sb + kColsPart * (j / kCP) + 8 * (j % kCP), make_desc(vb + (j >> 2) * kVhBlock + 32 * (j & 3), 16, 1024, 2),
                        idesc_pv, (i > 0 || j > 0) ? 1u : 0u);
          umma_commit(bar_done + 8 * sb);
        }
        __syncwarp();
      }
    }
  } else if (role == 2 || role == 3) {
    // ================================================================ producers (as uq_decode.cu; the prefix pages are
    // the same in every block table: the first sequence of the group names them)
    const bool is_k = (role == 2);
    const int n_stages = is_k ? kKStages : kVStages;
    const uint32_t bar_e = is_k ? bar_emptyk : bar_emptyv, bar_f = is_k ? bar_fullk : bar_fullv;
    const uint32_t page_tx = is_k ? 1024u : (uint32_t)kRestBytes;
    const uint64_t pol = l2_evict_first_policy();      // (the prefix is re-read by other CTAs soon: L2 keeps it anyway)
    Unit un;
    int s = 0, ph = 1;
    while (sc.next(un)) {
      const int32_t* bt = block_tables + (long long)un.b0 * max_pages + un.p0 + lane;
      int page_next = (lane < kTilePages) ? bt[0] : 0;
      for (int i = 0; i < un.n_tiles; ++i) {
        const int page = page_next;
        page_next = (lane < kTilePages && i + 1 < un.n_tiles) ? bt[kTilePages * (i + 1)] : 0;
        mbar_wait(bar_e + 8 * s, ph);
        if (lane == 0) mbar_expect_tx(bar_f + 8 * s, (uint32_t)kTilePages * page_tx);
        __syncwarp();
        if (lane < kTilePages) {
          if (is_k)
            tma_load_3d(base + kOffK + s * kKStageBytes + 2048 * lane, &tmap, 0, 0, page * Hkv + un.kvh, bar_f + 8 * s, pol);
          else
            bulk_g2s(base + kOffV + s * kVStageBytes + kRestBytes * lane,
                     cache + ((long long)page * Hkv + un.kvh) * kRecordBytes + 1024, kRestBytes, bar_f + 8 * s, pol);
        }
        if (++s == n_stages) { s = 0; ph ^= 1; }
      }
    }
  } else {
    // ================================================================ compute warps
    const int q = warp & 3;                            // TMEM lane quarter
    const uint32_t lane_sel = (uint32_t)(32 * q) << 16;
    const int r = 32 * q + lane;                       // softmax: (sequence, head) row; V warps: channel

    if (role < kIssuerWarps + kSoftmaxWarps) {
      // ============================================================== softmax warps: thread = one (sequence, head) row x
      // one part of the tile's columns (kSW warps share a lane quarter: a single warp per scheduler cannot hide its own
      // ALU / MUFU latencies).  The parts of a row meet once a tile, to agree on the row maximum.
      const int part = (role - kIssuerWarps) >> 2;     // 0..kSW-1: token columns [kColsPart * part, + kColsPart)
      const int bar_id = 1 + q;                        // named barrier of the lane quarter's kSW warps
      const int si = r / HS, hh = r % HS;
      float2* const ml_out = reinterpret_cast<float2*>(partial_ml);
      Unit un;
      int gt = 0, k = 0;
      while (sc.next(un)) {
        const int b = un.b0 + si;
        const bool valid = (b < batch) && (hh < G);
        const long long prow = (((long long)b * Hq + (long long)un.kvh * G + hh) * num_splits) + un.slot;
        float nref = 0.f;                              // minus the row's reference logit (log2 units)
        for (int i = 0; i < un.n_tiles; ++i, ++gt) {
          const int sb = gt & 1;
          // this part's columns of the score buffer; its P (f16 pairs) overwrites their first half in place
          const uint32_t t_s = tmem + lane_sel + kColS + 128 * sb + kColsPart * part;
          mbar_wait(bar_sfull + 8 * sb, (gt >> 1) & 1);
          if (part == 0 && q == 0) TRP(1, gt);
          tc_fence_after();
          uint32_t sv[kCP][16];                        // the part's raw scores of the tile: kept for both passes
#pragma unroll
          for (int c = 0; c < kCP; ++c) tmem_ld16_nowait(t_s + 16 * c, sv[c]);
          tmem_wait_ld();
          // ---- pass 1: the row maximum (the scale is positive).  On the unit's first tile it becomes the row's
          // reference; later a row gets a new one only when a score exceeds the old by 2^12 (lazy: P is fp16) —
          // per row: its O row and running sums are scaled down, no other row is concerned
          float mx = -INFINITY;
#pragma unroll
          for (int c = 0; c < kCP; ++c)
#pragma unroll
            for (int j = 0; j < 16; j += 2) mx = fmaxf(mx, fmaxf(__uint_as_float(sv[c][j]), __uint_as_float(sv[c][j + 1])));
          sh.pmax[sb][part][r] = mx;
          if (part == 0 && q == 0) TRP(10, gt);
          asm volatile("bar.sync %0, %1;" ::"r"(bar_id), "n"(32 * kSW) : "memory");
          if (part == 0 && q == 0) TRP(2, gt);
#pragma unroll
          for (int pp = 0; pp < kSW; ++pp) mx = fmaxf(mx, sh.pmax[sb][pp][r]);
          mx *= score_scale;
          if (i == 0) {
            nref = -mx;
          } else if (__builtin_expect(__any_sync(kFull, mx + nref > kThresh), 0)) {
            const float add = (mx + nref > kThresh) ? mx + nref : 0.f;   // factor 1 for the rows that stay
            const float f = ex2(-add);
            mbar_wait(bar_done + 8 * ((gt - 1) & 1), ((gt - 1) >> 1) & 1);   // every PV issued so far has to be in O
            tc_fence_after();
#pragma unroll 1
            for (int cc = 0; cc < kCP + (part == 0 ? 1 : 0); ++cc) {   // this part's columns of the O row (part 0: + the row sum)
              const uint32_t t_oc = tmem + lane_sel + kColO + (cc < kCP ? kColsPart * part + 16 * cc : 128);
              float ov[16];
              tmem_ld<16>(t_oc, ov);
#pragma unroll
              for (int j = 0; j < 16; ++j) ov[j] *= f;
              tmem_st<16>(t_oc, ov);
            }
            nref -= add;
          }
          // ---- pass 2: P = 2^(s * scale - ref) as f16 pairs, written over the scores read above
#pragma unroll
          for (int c = 0; c < kCP; ++c) {
            float t[16];
#pragma unroll
            for (int j = 0; j < 16; j += 2)
              ffma2(t[j], t[j + 1], __uint_as_float(sv[c][j]), __uint_as_float(sv[c][j + 1]), score_scale, nref, nref);
            uint32_t o[8];
#pragma unroll
            for (int j = 0; j < 16; j += 2) {
              const float e0 = ex2(t[j]), e1 = ex2(t[j + 1]);
              asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(o[j >> 1]) : "f"(e1), "f"(e0));
            }
            tmem_st8_nowait(t_s + 8 * c, o);
          }
          tmem_wait_st();
          if (part == 0 && q == 0) TRP(3, gt);
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(bar_pready + 8 * sb);
        }
        // ============================================================ the unit's partial: (m, l) and the accumulator row
        mbar_wait(bar_done + 8 * ((gt - 1) & 1), ((gt - 1) >> 1) & 1);
        tc_fence_after();
        float lv[16];
        if (part == 0) tmem_ld<16>(tmem + lane_sel + kColL, lv);   // 16 copies of the row sum (warp-uniform branch)
        if (valid && part == 0) {
          ml_out[prow] = make_float2(-nref * 0.6931471805599453f, lv[0]);
          if (un.slots_used > 0)                       // item finished: its remaining slots are empty
            for (int sl = un.slots_used; sl < num_splits; ++sl) ml_out[prow - un.slot + sl] = make_float2(-INFINITY, 0.f);
        }
#pragma unroll
        for (int c = 0; c < kCP; ++c) {                // this part's channels of the row
          const int col = kColsPart * part + 16 * c;
          float ov[16];
          tmem_ld<16>(tmem + lane_sel + kColO + col, ov);
          if (valid) {
            float4* dst = reinterpret_cast<float4*>(partial_acc + prow * kHeadDim + col);
            const float sc_ = sh.vscale[k & 3][col >> 5];
#pragma unroll
            for (int j = 0; j < 4; ++j)
              dst[j] = make_float4(ov[4 * j] * sc_, ov[4 * j + 1] * sc_, ov[4 * j + 2] * sc_, ov[4 * j + 3] * sc_);
          }
        }
        tc_fence_before();                             // (the next unit's first PV needs every softmax warp's P: it cannot
                                                       //  overwrite O before all of them are through here)
        ++k;
      }
    } else {
      // ============================================================== V warps: thread = channel, one 32-channel group a warp
      const int g = q;
      const uint32_t scratch = base + kOffMul + 256 * g;
      Unit un;
      int gt = 0, s = 0, ph_full = 0, k = 0;
      while (sc.next(un)) {
        // ---- the largest scale byte of group g over the unit's tiles -> the reference exponent of the whole unit
        uint32_t m4 = 0u;
        {
          const int32_t* bt = block_tables + (long long)un.b0 * max_pages + un.p0;
          const int p = (lane >> 1) & 7, o = lane & 1;
          for (int i2 = 0; i2 < un.n_tiles; i2 += 2) {
            const int tile = i2 + (lane >> 4);
            if (tile < un.n_tiles) {
              const int page = bt[kTilePages * tile + p];
              const uint2 w = *reinterpret_cast<const uint2*>(cache + ((long long)page * Hkv + un.kvh) * kRecordBytes +
                                                              kOffVScales + 32 * o + 8 * g);
              m4 = __vmaxu4(m4, __vmaxu4(w.x, w.y));
            }
          }
        }
        int mxb = (int)max(max(m4 & 0xFFu, (m4 >> 8) & 0xFFu), max((m4 >> 16) & 0xFFu, m4 >> 24));
        mxb = __reduce_max_sync(kFull, mxb);
        const int eref = max(mxb, 28);
        if (lane == 0) sh.vscale[k & 3][g] = pow2i(eref - 13 - 127);    // stored Vhat = code * 2^(byte - eref + 13)
        const int kbase = eref - 28;                   // fp16 exponent field of a multiplier = byte - kbase

        for (int i = 0; i < un.n_tiles; ++i) {
          const int sb = gt & 1;
          const uint32_t rest = base + kOffV + s * kVStageBytes;
          mbar_wait(bar_fullv + 8 * s, ph_full);
          if (q == 0) TRP(7, gt);
          uint32_t sw;                                 // the tile's scale bytes of group g: lane <-> tokens 4 lane .. 4 lane + 3
          asm volatile("ld.shared.u32 %0, [%1];" : "=r"(sw)
                       : "r"(rest + kRestBytes * (lane >> 2) + 1088 + 32 * ((lane >> 1) & 1) + 8 * g + 4 * (lane & 1)));
          {
            const int b0_ = (int)(sw & 0xFFu), b1 = (int)((sw >> 8) & 0xFFu), b2 = (int)((sw >> 16) & 0xFFu), b3 = (int)(sw >> 24);
            const uint32_t e0 = (uint32_t)max(b0_ - kbase, 0), e1 = (uint32_t)max(b1 - kbase, 0),
                           e2 = (uint32_t)max(b2 - kbase, 0), e3 = (uint32_t)max(b3 - kbase, 0);
            asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(scratch + 8 * lane), "r"((e0 << 10) | (e1 << 26)),
                         "r"((e2 << 10) | (e3 << 26)) : "memory");
          }
          __syncwarp();
          if (gt >= 2) mbar_wait(bar_done + 8 * sb, ((gt >> 1) - 1) & 1);   // PV(gt-2) has read Vhat buffer gt & 1
          if (q == 0) TRP(12, gt);
          const uint32_t vrow = sVh + kVhBytes * sb + 128 * r;
          const uint32_t code0 = rest + 128 * g + 4 * lane;
#pragma unroll
          for (int h = 0; h < 4; ++h) {                // 32 tokens = four 16-byte chunks of the channel's row
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) {           // token octet kq: page kq >> 1, half kq & 1
              const int kq = 4 * h + kk;
              uint32_t cwd;
              asm volatile("ld.shared.u32 %0, [%1];" : "=r"(cwd) : "r"(code0 + kRestBytes * (kq >> 1) + 512 * (kq & 1)));
              const uint4 m4w = lds128(scratch + 16 * kq);
              uint32_t f[4];
              cvt_e2m1x8(cwd, f);
              const uint4 o4 = make_uint4(hmul2(f[0], m4w.x), hmul2(f[1], m4w.y), hmul2(f[2], m4w.z), hmul2(f[3], m4w.w));
              const int chunk = 4 * (h & 1) + kk;
              sts128(vrow + (h >> 1) * kVhBlock + (((chunk ^ (r & 7))) << 4), o4);
            }
          }
          if (q == 0) TRP(4, gt);
          fence_async_smem();
          __syncwarp();                                // also: every lane has read the scratch of this tile
          if (lane == 0) {
            mbar_arrive(bar_vready + 8 * sb);
            mbar_arrive(bar_emptyv + 8 * s);
          }
          ++gt;
          if (++s == kVStages) { s = 0; ph_full ^= 1; }
        }
        ++k;
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (role == 1) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(kTmemCols));
  }
}

}  // namespace

// 3-D view of q_fp8 for the M-side query tile: [batch][Hq][128 B]; box = NSEQ sequences x HS heads x 128 bytes.
static int32_t q_map_m(const void* q_fp8, int batch, int Hq, int HS, CUtensorMap* out) {
  const EncodeTiledFn encode = encode_tiled_fn();
  if (!encode) return UQ_ERR_CUDA;
  const cuuint64_t gdim[3] = {128, (cuuint64_t)Hq, (cuuint64_t)batch};
  const cuuint64_t gstr[2] = {128, (cuuint64_t)128 * Hq};
  const cuuint32_t box[3] = {128, (cuuint32_t)HS, (cuuint32_t)(128 / HS)};
  const cuuint32_t estr[3] = {1, 1, 1};
  const CUresult cr = encode(out, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<void*>(q_fp8), gdim, gstr, box, estr,
                             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (cr != CUDA_SUCCESS) {
    set_error("decode_prefix: cuTensorMapEncodeTiled (q_fp8, 3-D) failed with CUresult %d", (int)cr);
    return UQ_ERR_CUDA;
  }
  return UQ_OK;
}

// launcher used by uq_decode_prefix_attention (uq_decode_prefix.cu validates the arguments)
int32_t launch_prefix_m(const uq_config* cfg, const void* q_fp8, const void* cache, long long records,
                        const int32_t* block_tables, int32_t max_pages, int32_t batch, int32_t prefix_len,
                        int32_t num_splits, float* partial_acc, float* partial_ml, cudaStream_t stream) {
  const int G = cfg->num_q_heads / cfg->num_kv_heads;
  const int HS = G > 8 ? 16 : 8, NSEQ = 128 / HS;
  CUtensorMap tmap, tmap_q;
  int32_t st = k_code_map(cache, records, 128, &tmap);
  if (st != UQ_OK) return st;
  st = q_map_m(q_fp8, batch, cfg->num_q_heads, HS, &tmap_q);
  if (st != UQ_OK) return st;
  int sm_count = 0;
  st = current_device_sms(&sm_count);
  if (st != UQ_OK) return st;
  const long long total = (long long)((batch + NSEQ - 1) / NSEQ) * cfg->num_kv_heads * (prefix_len / 128);
  const dim3 grid((unsigned)(total < sm_count ? total : sm_count));    // one wave, one balanced tile range per CTA
  const float score_scale = resolved_sm_scale(cfg) * 1.4426950408889634f;
  auto kern = HS == 16 ? decode_prefix_m_kernel<16> : decode_prefix_m_kernel<8>;
  st = opt_in_dynamic_smem((const void*)kern, kSmemBytes, "decode_prefix: cudaFuncSetAttribute");
  if (st != UQ_OK) return st;
  return check_cuda(launch_pdl(kern, grid, dim3(kThreads), (size_t)kSmemBytes, stream, tmap, tmap_q, (const uint8_t*)cache,
                               block_tables, (int)max_pages, (int)(prefix_len / 128), (int)batch, (int)cfg->num_q_heads,
                               (int)cfg->num_kv_heads, (int)num_splits, score_scale, partial_acc, partial_ml),
                    "uq_decode_prefix_attention launch");
}

}  // namespace uq

#ifdef UQ_TRACE
// debug builds only (not part of include/uq.h): the [UQ_TRACE_TILES][16] clock64 table of the prefix kernel's traced CTA
extern "C" int uq_debug_trace_read_prefix(void* host, size_t bytes) {
  return (int)cudaMemcpyFromSymbol(host, uq::g_trace_prefix, bytes);
}
#endif
