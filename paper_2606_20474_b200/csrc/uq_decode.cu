// uq_decode.cu — paged split-K decode attention over the FP4+UE8M0 cache: Alg. 1 "Decode"
// l.7-8 of arxiv/paper_2606_20474 (Eq.(1) :104).  Paging / split-K / partial
// format follow include/uq.h.
//
// Design: the 128-token tiles (8 pages) of all (sequence, kv head) items form one
// sequence that is cut into equal contiguous ranges, one per resident CTA (one wave, 2 CTAs per SM); a
// range is walked as units (item, tile range), each unit writing one partial slot of its item.
// Warp roles (384 threads = 12 warps, one role each; the tile period is set by the longest serial instruction
// stream of the CTA, so the roles are cut to keep every stream short):
//   K producer   per page one TMA tensor copy of the packed FP4 K codes (CU_TENSOR_MAP_DATA_TYPE_16U4_ALIGN16B +
//                SWIZZLE_128B: the TMA unit lays the nibbles out in the 8-bit containers tcgen05 reads) into a
//                3-stage ring; L2 evict-first;
//   V producer   per page one cp.async.bulk of the rest of the record (V codes, K scales, V scales) into a
//                4-stage ring of its own;
//   QK issuer    S[128 tok x 16 heads] = K . Q^T with tcgen05.mma.kind::mxf8f6f4.block_scale — E2M1 keys x E4M3
//                queries with the UE8M0 group scales applied by the tensor core (the paper's FP8xFP4 scaled MMA,
//                PAPER.md:281), K scales staged smem -> TMEM with tcgen05.cp; S double-buffered in TMEM;
//   PV issuer    O^T[128 d x 16 heads] += Vhat^T . P^T with tcgen05.mma.kind::f16 (A = Vhat^T from TMEM, B = P from
//                smem); accumulators in TMEM;
//   4 softmax warps   thread = token row: S from TMEM (tcgen05.ld), base-2 softmax against a LAZY per-head
//                reference (a "rebase" — new reference, O rescaled in TMEM, tile's P redone — happens on the first
//                tile and whenever a score exceeds the reference by 2^12), P -> fp16 operand in smem;
//   4 V warps    thread = channel: V codes -> fp16 (cvt.rn.f16x2.e2m1x2 x exact power-of-two scale against the
//                warp's own reference exponent: its 32 channels are one scale group) written with tcgen05.st
//                straight into TMEM, where the PV MMA reads it as its A operand (no shared-memory round trip).
// The FP8 query tile is copied to smem by TMA once per unit ("hoisted").
// Every K/V byte is read from HBM exactly once.
#include <cuda.h>
#include <cuda_fp16.h>

#include <mutex>
#include <type_traits>

#include "uq_sched.cuh"
#include "uq_tc.cuh"

namespace uq {
namespace {

constexpr int kSoftmaxWarps = 4;                     // one per TMEM lane quarter
constexpr int kIssuerWarps = 4;                      // QK issuer, PV issuer, K producer, V producer
#ifndef UQ_KSTAGES
#define UQ_KSTAGES 3
#endif
#ifndef UQ_VSTAGES
#define UQ_VSTAGES 4
#endif
#ifndef UQ_CTAS_PER_SM
#define UQ_CTAS_PER_SM 2
#endif
#ifndef UQ_VBUFS
#define UQ_VBUFS 2
#endif
// Two rings: the K codes of a tile (16 KB at head_dim 128 once the TMA unit has expanded the nibbles) are needed by
// the QK MMA only and leave early; the rest of the records (V codes, K scales, V scales: 9 KB) stays until the V
// warps have converted it.  Separate rings let the small one run deep (bytes in flight hide HBM latency).
constexpr int kKStages = UQ_KSTAGES;
constexpr int kVStages = UQ_VSTAGES;
constexpr int kPBytes = 4096;                        // one P operand buffer: [token-core 16][head-core 2][8 tok][8 heads] f16
#ifdef UQ_TRACE
__device__ unsigned long long g_trace_decode[UQ_TRACE_TILES * 16];
#endif
// trace events of CTA 5 (UQ_TR): 0 QK issue, 8 / 9 QK warp before / after the wait for a free score buffer, 5 PV issue,
// 10 / 1 softmax warp 0 before / after the wait for S, 3 its tile done, 6 / 7 V warp 0 before / after the wait for the
// tile's bytes, 11 / 12 before / after the wait for a free Vhat buffer, 4 its tile done
#define TRD(ev, tile) UQ_TR(g_trace_decode, 5, ev, tile)
constexpr float kThresh = 12.0f;                     // lazy-reference threshold (log2 units)
constexpr int kMaxBatch = 2048;                      // sequences per call (tile prefix sums live in shared memory)
constexpr int kVBufs = UQ_VBUFS;                     // Vhat^T buffers in TMEM

// Everything that depends on head_dim D (include/uq.h: 64, 128 or 256).  D = 128 is the geometry the kernel was tuned
// on (one M = 128 PV product, 12 warps, 2 CTAs per SM); D = 64 runs the same CTA with the upper 64 accumulator rows
// fed zeros (two V warps idle; the tensor pipe has the room), D = 256 splits the head into two 128-channel halves:
// two K blocks per stage, two PV products per tile into two accumulators, eight V warps, one CTA of 16 warps per SM.
template <int D>
struct DecodeGeo {
  using R = RecordGeo<D>;
  static constexpr int kHalves = D == 256 ? 2 : 1;                  // 128-channel halves of the head
  static constexpr int kVWarps = 4 * kHalves;                       // one per (half, TMEM lane quarter)
  static constexpr int kComputeWarps = kSoftmaxWarps + kVWarps;
  static constexpr int kThreads = (kComputeWarps + kIssuerWarps) * 32;   // 12 warps: registers are allocated per 4 warps anyway
  static constexpr int kCtasPerSm = D == 256 ? 1 : UQ_CTAS_PER_SM;
  static constexpr int kRecordBytes = R::kBytes;
  static constexpr int kKPacked = 8 * D;                            // K codes of a page in HBM (1024 at D = 128)
  static constexpr int kRestBytes = R::kRest;                       // V codes + K scales + V scales = 1152
  static constexpr int kKRow = D < 128 ? D : 128;                   // bytes of a token row of a K block in smem (one per code)
  static constexpr int kKPageBytes = 16 * kKRow;                    // a page inside a block: 2048
  static constexpr int kKBlockBytes = kTilePages * kKPageBytes;     // 128 tokens x <= 128 channels: 16384
  static constexpr int kKStageBytes = kHalves * kKBlockBytes;
  static constexpr int kVStageBytes = kTilePages * kRestBytes;      // 9216
  static constexpr int kQBlockBytes = 16 * kKRow;                   // 16 heads x <= 128 channels: 2048
  static constexpr int kQBytes = kHalves * kQBlockBytes;
  // head_dim 128 / 256: K-major tiles with the 128-byte swizzle, as the TMA unit writes them.  head_dim 64: the packed
  // 4-bit tensor type of TMA takes 128-wide boxes only, so the packed codes arrive by plain bulk copies and an otherwise
  // idle warp spreads them into the unswizzled core-matrix layout [16-byte chunk c][row r] (chunk = 16 codes, 8 bytes of
  // nibbles + 8 of padding, as the tensor core reads 4-bit operands of kind::mxf8f6f4): LBO = the chunk stride.
  static constexpr uint32_t kSwz = D == 64 ? 0u : 2u;               // UMMA layout type: none / SWIZZLE_128B
  static constexpr uint32_t kSBO = D == 64 ? 128u : 1024u;          // eight rows
  static constexpr uint32_t kLBOk = D == 64 ? 128u * 16u : 16u;     // K block: next chunk (ignored with a swizzle)
  static constexpr uint32_t kLBOq = D == 64 ? 16u * 16u : 16u;      // Q block
  static constexpr int kQKMmas = D / 32;                            // one block-scaled MMA per 32-channel scale group
  static constexpr int kSfaAtoms = (kQKMmas + 3) / 4;               // 512-byte scale-factor atoms (4 groups each) per tile
  static constexpr int kSfaBytes = 512 * kSfaAtoms;
  // dynamic shared memory map (offsets from a 1024-byte aligned base)
  static constexpr int kOffK = 0;                                   // kKStages x 16384, SW128
  static constexpr int kOffV = kOffK + kKStages * kKStageBytes;     // kVStages x 9216
  static constexpr int kOffQ = kOffV + kVStages * kVStageBytes;     // 2 x 2048, SW128 (one per unit in flight)
  static constexpr int kOffSFA = kOffQ + 2 * kQBytes;               // 2 x 512
  static constexpr int kOffSFB = kOffSFA + 2 * kSfaBytes;           // 512
  static constexpr int kOffP = kOffSFB + 512;                       // 2 x 4096 (double-buffered)
  static constexpr int kOffMul = kOffP + 2 * kPBytes;               // V warps x 256 B of fp16 multipliers
  static constexpr int kOffKP = kOffMul + kVWarps * 256;            // head_dim 64: kKStages x 4096 of packed K codes
  static constexpr int kKPStage = D == 64 ? kTilePages * 8 * D : 0;
  static constexpr int kOffEnd = kOffKP + kKStages * kKPStage;
  static constexpr int kSmemBytes = kOffEnd + 1024;                 // + alignment slack
  static_assert(kOffQ % 1024 == 0 && kKStageBytes % 1024 == 0, "swizzled tiles need 1024-byte alignment");
  // TMEM columns
  static constexpr uint32_t kColS = 0;                              // 2 x 16
  static constexpr uint32_t kColO = 32;                             // 16 per half
  static constexpr uint32_t kColSFA = kColO + 16 * kHalves;         // 2 x 4 per atom
  static constexpr uint32_t kSfaCols = 4 * kSfaAtoms;
  static constexpr uint32_t kColSFB = kColSFA + 2 * kSfaCols;       // 4
  static constexpr uint32_t kColV = D == 256 ? 128 : 64;            // kVBufs x 64 per half: Vhat^T operand, lane = channel d,
  static constexpr uint32_t kVBufCols = 64 * kHalves;               //   column c = tokens 2c, 2c+1 (f16x2)
  static constexpr uint32_t kTmemCols = D == 256 ? 512 : (kVBufs == 1 ? 128 : 256);
  static_assert(kColSFB + 4 <= kColV && kColV + kVBufs * kVBufCols <= kTmemCols, "TMEM columns");
};

// ---------------------------------------------------------------- per-CTA shared bookkeeping
struct Shared {
  uint64_t full_k[kKStages];  // K producer (expect_tx) + TMA bytes -> QK warp
  uint64_t empty_k[kKStages]; // QK commit -> K producer
  uint64_t full_v[kVStages];  // V producer (expect_tx) + bulk-copy bytes -> QK warp (K scales), V warps
  uint64_t empty_v[kVStages]; // 4 V warps + QK warp -> V producer
  uint64_t s_full[2];         // QK commit -> softmax warps: S(gt) is in TMEM buffer gt&1
  uint64_t s_free[2];         // 8 compute warps -> QK warp: S buffer read, may be overwritten
  uint64_t ready[2];          // 4 softmax + 4 V warps -> PV warp: P (smem) and Vhat (TMEM) buffer gt&1 are written
                              // (two barriers: a V warp may be one tile ahead of the softmax warps)
  uint64_t done[2];           // PV commit of tile i -> done[i&1]: P / Vhat buffer i&1 free, O up to date
  uint64_t q_full[2];         // TMA: the FP8 query tile of a work unit landed (buffer = unit ordinal & 1)
  uint32_t tmem_base;
  float wmax[kSoftmaxWarps][16];
  float lsum[kSoftmaxWarps][16];
  float mref[16];
  int total_tiles, max_tiles;  // sum (x kv heads) and max over sequences of the tiles per (sequence, kv head)
  int pre[kMaxBatch + 1];      // pre[b] = tiles of sequences 0..b-1 (per kv head)
  uint64_t full_kp[kKStages];  // head_dim 64 only: bulk-copy bytes of the PACKED K codes -> the expander warp
};

// ---------------------------------------------------------------- the kernel
template <int D>
__global__ void __launch_bounds__(DecodeGeo<D>::kThreads, DecodeGeo<D>::kCtasPerSm)
decode_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ CUtensorMap tmap_q,
              const __grid_constant__ CUtensorMap tmap_v,
              const uint8_t* __restrict__ cache, const int32_t* __restrict__ block_tables, int max_pages,
              const int32_t* __restrict__ seq_lens, int batch, int Hq, int Hkv, int num_splits,
              float score_scale /* sm_scale * log2(e) */, float* __restrict__ partial_acc,
              float* __restrict__ partial_ml, int early /* UQ_FLAG_SMALL_APPEND_AHEAD */) {
  using Geo = DecodeGeo<D>;
  constexpr int kHalves = Geo::kHalves, kComputeWarps = Geo::kComputeWarps, kThreads = Geo::kThreads;
  constexpr int kRecordBytes = Geo::kRecordBytes, kRestBytes = Geo::kRestBytes, kKStageBytes = Geo::kKStageBytes,
                kVStageBytes = Geo::kVStageBytes, kKBlockBytes = Geo::kKBlockBytes, kKPageBytes = Geo::kKPageBytes,
                kQBytes = Geo::kQBytes, kQBlockBytes = Geo::kQBlockBytes, kSfaBytes = Geo::kSfaBytes;
  constexpr int kOffK = Geo::kOffK, kOffV = Geo::kOffV, kOffQ = Geo::kOffQ, kOffSFA = Geo::kOffSFA, kOffSFB = Geo::kOffSFB,
                kOffP = Geo::kOffP, kOffMul = Geo::kOffMul;
  constexpr uint32_t kColS = Geo::kColS, kColO = Geo::kColO, kColSFA = Geo::kColSFA, kColSFB = Geo::kColSFB,
                     kColV = Geo::kColV, kVBufCols = Geo::kVBufCols, kSfaCols = Geo::kSfaCols, kTmemCols = Geo::kTmemCols;
  extern __shared__ uint8_t smem_raw[];
  __shared__ __align__(8) Shared sh;

  const int G = Hq / Hkv;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
#ifndef UQ_ISSUERS_HIGH
#define UQ_ISSUERS_HIGH 1
#endif
  // role 0 QK issuer, 1 PV issuer, 2 K producer, 3 V producer, 4..7 softmax warps, 8..11 V warps
#if UQ_ISSUERS_HIGH
  const int role = warp < kComputeWarps ? warp + kIssuerWarps : warp - kComputeWarps;
#else
  const int role = warp;
#endif

  // The two shared-memory base addresses go through an opaque move: as plain expressions of a symbol the compiler
  // rematerialises them at every use (S2R CgaCtaId + MOV + LEA per mbarrier operation, ~140 instructions a tile).
  uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u, sh_base = smem_u32(&sh);
  asm volatile("mov.u32 %0, %0;" : "+r"(base));
  asm volatile("mov.u32 %0, %0;" : "+r"(sh_base));
  const uint32_t sQ = base + kOffQ, sSFA = base + kOffSFA, sSFB = base + kOffSFB, sP = base + kOffP;
  const uint32_t bar_fullk = sh_base + offsetof(Shared, full_k), bar_emptyk = sh_base + offsetof(Shared, empty_k),
                 bar_fullv = sh_base + offsetof(Shared, full_v), bar_emptyv = sh_base + offsetof(Shared, empty_v),
                 bar_sfull = sh_base + offsetof(Shared, s_full), bar_sfree = sh_base + offsetof(Shared, s_free),
                 bar_ready = sh_base + offsetof(Shared, ready), bar_done = sh_base + offsetof(Shared, done),
                 bar_qfull = sh_base + offsetof(Shared, q_full);

  // ---------------- setup
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < kKStages; ++s) {
      mbar_init(bar_fullk + 8 * s, 1);
      mbar_init(bar_emptyk + 8 * s, 1);
      if constexpr (D == 64) mbar_init(smem_u32(&sh.full_kp[s]), 1);
    }
#pragma unroll
    for (int s = 0; s < kVStages; ++s) {
      mbar_init(bar_fullv + 8 * s, 1);
      mbar_init(bar_emptyv + 8 * s, (kComputeWarps - kSoftmaxWarps) + 1);
    }
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
                 "r"(kTmemCols));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  if (tid < 128) {  // query-side scale factors: UE8M0 byte 127 = 2^0
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(sSFB + 4 * tid), "r"(0x7F7F7F7Fu) : "memory");
  }
  // Barriers, TMEM and scale constants are set up under the tail of the kernel before this one in the stream;
  // everything below reads global memory it may have written (programmatic dependent launch, uq_common.cuh).
  pdl_launch_dependents();
  // UQ_FLAG_SMALL_APPEND_AHEAD (include/uq.h): the caller guarantees that what still runs ahead of this kernel in the
  // stream writes q_fp8, the partial buffers and at most the last two pages of every sequence — nothing else this
  // kernel reads.  Then only the accesses that could meet those writes wait for the grid ahead (the Q tiles, a tile
  // holding one of a sequence's last two pages, every write of partials), and the K / V rings fill — the V warps
  // convert — under the append kernel: the HBM latency of the first tiles is off the step's critical path.
  if (!early) pdl_wait();
  // tiles per sequence -> inclusive prefix sums in shared memory (every CTA computes the same schedule)
  for (int b = tid; b < batch; b += kThreads) {
    const int L = seq_lens[b];
    sh.pre[b + 1] = ((L + kPage - 1) / kPage + kTilePages - 1) / kTilePages;
  }
  if (tid == 0) sh.pre[0] = 0;
  __syncthreads();
  if (warp == 0) {                                     // warp scan over chunks of 32 with a running carry
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
    const int fit = (sh.max_tiles + num_splits - 2) / (num_splits - 1);   // an item spans at most num_splits ranges
    sc.tpc = max(1, max(even, fit));
  }

  if (role == 0) {
    // ================================================================ QK warp
    // Per unit: the FP8 query tile (16 rows x 128 B, 128-byte swizzle) arrives by TMA into Q buffer
    // (unit ordinal & 1) — "hoisted", once per unit; rows past the unit's G heads belong to
    // the next kv head (or are zero past the tensor end) and only feed score columns nobody reads.
    // Per tile: S(gt)[128 tok x 16 heads] = K . Q^T once the tile's bytes have landed, the S buffer was read
    // by the softmax of global tile gt-2.
    const uint32_t idesc_qk = (5u << 7) | (0u << 10) | (2u << 17) | (1u << 23) | (8u << 24);   // E2M1 x E4M3, UE8M0, N=16, M=128
    if (early) pdl_wait();                             // q_fp8 comes from the kernel ahead
    if (elect_one()) umma_cp_sf(tmem + kColSFB, make_desc(sSFB, 16, 128, 0));
    auto load_q = [&](const Unit& un, int k) {         // lane 0: Q tile of unit ordinal k
      if (elect_one()) {
        mbar_expect_tx(bar_qfull + 8 * (k & 1), kQBytes);
        if constexpr (D == 64)                           // [chunk][row][16 B]: the unswizzled core-matrix order
          tma_load_3d_plain(sQ + kQBytes * (k & 1), &tmap_q, 0, un.b * Hq + un.kvh * G, 0, bar_qfull + 8 * (k & 1));
        else
          tma_load_2d(sQ + kQBytes * (k & 1), &tmap_q, 0, un.b * Hq + un.kvh * G, bar_qfull + 8 * (k & 1));
        if constexpr (kHalves == 2)                      // channels 128..255: a second 128-byte-wide block
          tma_load_2d(sQ + kQBytes * (k & 1) + kQBlockBytes, &tmap_q, 128, un.b * Hq + un.kvh * G, bar_qfull + 8 * (k & 1));
      }
    };
    Cursor cur, cur_nx;
    sc.start(cur);
    cur_nx = cur;
    Unit un, nx;
    bool have_nx = sc.next(cur_nx, nx);                // nx runs one unit ahead of un
    int gt = 0, sk = 0, phk = 0, sv = 0, phv = 0;      // global tile counter; its K / V stage and full-barrier parity
    int k = 0, k_q = -1;                               // ordinal of the current unit; last ordinal whose Q load was issued
    while (have_nx) {
      un = nx;
      have_nx = sc.next(cur_nx, nx);
      for (int i = 0; i < un.n_tiles; ++i) {
        const int sb = gt & 1;
        TRD(8, gt);
        if (gt >= 2) mbar_wait(bar_sfree + 8 * sb, ((gt >> 1) - 1) & 1);
        TRD(9, gt);
        // here every QK up to global tile gt-2 has completed (its S was read): at i == 0 the Q buffer of
        // unit k-2 (= buffer k & 1), at i == 1 that of unit k-1 (= buffer (k+1) & 1) may be refilled
        if (i == 0 && k_q < k) { load_q(un, k); k_q = k; }
        if (i == 1 && have_nx) { load_q(nx, k + 1); k_q = k + 1; }
        if (i == 0) mbar_wait(bar_qfull + 8 * (k & 1), (k >> 1) & 1);
        mbar_wait(bar_fullv + 8 * sv, phv);
        const uint32_t st = base + kOffK + sk * kKStageBytes, rest = base + kOffV + sv * kVStageBytes;
        // scale-factor atom: row r = 32 c + lane of the tile -> 16-byte line `lane`, word c (a word = the row's scale
        // bytes of four groups; head_dim 64 fills two of them, head_dim 256 a second atom with groups 4..7)
        uint32_t v[4], v2[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const int r = 32 * c + lane;
          const uint32_t a = rest + kRestBytes * (r >> 4) + 8 * D + (D / 32) * (r & 15);
          if constexpr (D == 64) asm volatile("ld.shared.u16 %0, [%1];" : "=r"(v[c]) : "r"(a));
          else if constexpr (D == 128) asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v[c]) : "r"(a));
          else asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v[c]), "=r"(v2[c]) : "r"(a));
        }
        sts128(sSFA + kSfaBytes * sb + 16 * lane, make_uint4(v[0], v[1], v[2], v[3]));
        if constexpr (D == 256) sts128(sSFA + kSfaBytes * sb + 512 + 16 * lane, make_uint4(v2[0], v2[1], v2[2], v2[3]));
        fence_async_smem();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_emptyv + 8 * sv);   // the K scales are copied: this warp is done with the V stage
        mbar_wait(bar_fullk + 8 * sk, phk);
        TRD(0, gt);
        tc_fence_after();
        if (elect_one()) {
          const uint32_t t_sfa = tmem + kColSFA + kSfaCols * sb, qb = sQ + kQBytes * (k & 1);
          umma_cp_sf(t_sfa, make_desc(sSFA + kSfaBytes * sb, 16, 128, 0));
          if constexpr (D == 256) umma_cp_sf(t_sfa + 4, make_desc(sSFA + kSfaBytes * sb + 512, 16, 128, 0));
#pragma unroll
          for (int kb = 0; kb < Geo::kQKMmas; ++kb)       // one scale group (32 channels) per instruction
            umma_mxf8f6f4(tmem + kColS + 16 * sb,
                          make_desc(st + (kb >> 2) * kKBlockBytes + (D == 64 ? 2 * Geo::kLBOk : 32u) * (kb & 3), Geo::kLBOk,
                                    Geo::kSBO, Geo::kSwz),
                          make_desc(qb + (kb >> 2) * kQBlockBytes + (D == 64 ? 2 * Geo::kLBOq : 32u) * (kb & 3), Geo::kLBOq,
                                    Geo::kSBO, Geo::kSwz),
                          idesc_qk | ((uint32_t)(kb & 3) << 29), kb > 0,
                          t_sfa + 4 * (kb >> 2) + ((uint32_t)(kb & 3) << 30), tmem + kColSFB);
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
    // ================================================================ PV warp
    // O^T[128 d x 16 heads] += Vhat^T (TMEM, buffer gt&1) . P^T (smem, buffer gt&1); f16 x f16 -> f32, B MN-major
    const uint32_t idesc_pv = (1u << 4) | (1u << 16) | (2u << 17) | (8u << 24);
    Cursor cur;
    sc.start(cur);
    Unit un;
    int gt = 0;
    while (sc.next(cur, un)) {
      for (int i = 0; i < un.n_tiles; ++i, ++gt) {
        mbar_wait(bar_ready + 8 * (gt & 1), (gt >> 1) & 1);
        TRD(5, gt);
        tc_fence_after();
        if (lane == 0) {
          const uint32_t pbuf = sP + kPBytes * (gt & 1), vbuf = tmem + kColV + kVBufCols * ((gt & 1) % kVBufs);
#pragma unroll
          for (int c = 0; c < kHalves; ++c)              // 128 channels per accumulator
#pragma unroll
            for (int j = 0; j < 8; ++j)                  // 16 tokens per MMA = 8 columns of Vhat^T
              umma_f16_ts(tmem + kColO + 16 * c, vbuf + 64 * c + 8 * j, make_desc(pbuf + 512 * j, 256, 128, 0), idesc_pv,
                          (i > 0 || j > 0) ? 1u : 0u);
          umma_commit(bar_done + 8 * (gt & 1));
        }
        __syncwarp();
      }
    }
  } else if (role == 2 || role == 3) {
    // ================================================================ producer warps
    // Warp 2 streams the K codes (one TMA tensor copy per page: the TMA unit expands the packed nibbles to
    // one byte per code), warp 3 the rest of the records (one 1152-byte bulk copy per page), each into its own
    // ring and at its own pace.  Lanes 0..7 issue one page each (the copies of a warp serialise at ~55 cycles:
    // ~450 cycles per tile and warp); the rings run across units.
    // (Measured: issuing a tile's eight copies back to back from one elected thread is slower, 131.7 us against
    // 119.7 us on config 2, than one copy per lane — see elect_one().)
    const bool is_k = (role == 2);
    const int n_stages = is_k ? kKStages : kVStages;
    const uint32_t bar_e = is_k ? bar_emptyk : bar_emptyv,
                   bar_f = is_k ? (D == 64 ? smem_u32(&sh.full_kp[0]) : bar_fullk) : bar_fullv;
    // head_dim <= 128: the rest of FOUR records (V codes, K scales, V scales) per copy — cp.async.bulk.tensor ...
    // tile::gather4 over the cache seen as [record][9 D bytes] rows of 8-byte elements: two copies a tile instead of eight
    constexpr bool kGather = (D <= 128);
    const uint32_t page_tx = is_k ? (uint32_t)Geo::kKPacked : (uint32_t)kRestBytes;
    const int pl = (kHalves == 2) ? (lane & 7) : lane;  // the lane's page of the tile; head_dim 256: lanes 8..15 of the
    const int hl = (kHalves == 2) ? (lane >> 3) : 0;    // K producer copy the second 128-channel block of pages 0..7
    const bool copier = (kHalves == 2 && is_k) ? lane < 2 * kTilePages : lane < kTilePages;
    const uint64_t pol = l2_evict_first_policy();
    Cursor cur;
    sc.start(cur);
    Unit un;
    int s = 0, ph = 1;                                 // stage, parity to wait for on empty[s]
    bool waited = !early;                              // has this warp waited for the grid ahead
    while (sc.next(cur, un)) {
      const int last_safe = ((un.L + kPage - 1) / kPage) - 2;   // pages from here on may still be written by the append ahead
      const int32_t* bt = block_tables + (long long)un.b * max_pages + un.p0 + pl;
      int page_next = (copier && un.p0 + pl < un.p1) ? bt[0] : 0;
      for (int i = 0; i < un.n_tiles; ++i) {
        const int page = page_next;
        const int npg = min(kTilePages, un.p1 - (un.p0 + kTilePages * i));
        const int nb = un.p0 + kTilePages * (i + 1) + pl;
        page_next = (copier && nb < un.p1) ? bt[kTilePages * (i + 1)] : 0;
        if (!waited && un.p0 + kTilePages * (i + 1) > last_safe) { pdl_wait(); waited = true; }
        mbar_wait(bar_e + 8 * s, ph);
        if (kGather && !is_k) {
          const int nops = (npg + 3) >> 2;             // pages past the end name record 0: copied, never read
          if (lane == 0) mbar_expect_tx(bar_f + 8 * s, (uint32_t)nops * 4u * page_tx);
          const int l4 = 4 * (lane & 1);
          const int r0 = __shfl_sync(kFull, page, l4) * Hkv + un.kvh, r1 = __shfl_sync(kFull, page, l4 + 1) * Hkv + un.kvh,
                    r2 = __shfl_sync(kFull, page, l4 + 2) * Hkv + un.kvh, r3 = __shfl_sync(kFull, page, l4 + 3) * Hkv + un.kvh;
          if (lane < nops)
            tma_gather4(base + kOffV + s * kVStageBytes + 4 * kRestBytes * lane, &tmap_v, 0, r0, r1, r2, r3, bar_f + 8 * s, pol);
          if (++s == n_stages) { s = 0; ph ^= 1; }
          continue;
        }
        if (lane == 0) mbar_expect_tx(bar_f + 8 * s, (uint32_t)npg * page_tx);
        __syncwarp();
        if ((kHalves == 2 && is_k) ? (copier && pl < npg) : (lane < npg)) {
          if (is_k) {
            if constexpr (D == 64)
              bulk_g2s(base + Geo::kOffKP + s * Geo::kKPStage + Geo::kKPacked * lane,
                       cache + ((long long)page * Hkv + un.kvh) * kRecordBytes, Geo::kKPacked, bar_f + 8 * s, pol);
            else
              tma_load_3d(base + kOffK + s * kKStageBytes + hl * kKBlockBytes + kKPageBytes * pl, &tmap, 128 * hl, 0,
                          page * Hkv + un.kvh, bar_f + 8 * s, pol);
          } else
            bulk_g2s(base + kOffV + s * kVStageBytes + kRestBytes * lane,
                     cache + ((long long)page * Hkv + un.kvh) * kRecordBytes + 8 * D, kRestBytes, bar_f + 8 * s, pol);
        }
        if (++s == n_stages) { s = 0; ph ^= 1; }
      }
    }
  } else {
    // ================================================================ compute warps (warp ids 4..11)
    // Two role-pure groups of four warps, one warp of each per TMEM lane quarter (hardware: warp id % 4):
    //   softmax warps (4..7):  thread = token row of the tile, all query heads of the kv head;
    //   V warps (8..11):       thread = channel d, all 128 tokens of the tile.
    // A V warp needs the tile's bytes but not its scores, so it may run ahead of the softmax warps; the
    // two groups meet only at the `ready` barrier of the PV warp.  The issuer warps sit on the lowest
    // warp ids so that the scheduler's highest-warp-id-first arbitration favours the compute warps.
    const int cw = role - kIssuerWarps;                // 0..7
    const int q = warp & 3;                            // TMEM lane quarter
    const uint32_t lane_sel = (uint32_t)(32 * q) << 16;
    const int r = 32 * q + lane;                       // softmax: token row of the tile; V warps: channel d

    if (cw < kSoftmaxWarps) {
      // ============================================================== softmax warps
      const int atid = 32 * cw + lane;                 // 0..127
      float2* const ml_out = reinterpret_cast<float2*>(partial_ml);
      if (early) pdl_wait();                           // the partial buffers may still be read by the merge ahead

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

            if (cw == 0) TRD(10, gt);
            mbar_wait(bar_sfull + 8 * sb, ph2);        // S(gt) is in TMEM
            if (cw == 0) TRD(1, gt);
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
                asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(o.x) : "f"(lt[8 * c + 1]), "f"(lt[8 * c + 0]));
                asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(o.y) : "f"(lt[8 * c + 3]), "f"(lt[8 * c + 2]));
                asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(o.z) : "f"(lt[8 * c + 5]), "f"(lt[8 * c + 4]));
                asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(o.w) : "f"(lt[8 * c + 7]), "f"(lt[8 * c + 6]));
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
#pragma unroll
                for (int c = 0; c < kHalves; ++c) {
                  float ov[NH];
                  const uint32_t t_o = tmem + lane_sel + kColO + 16 * c;   // channel 128 c + r, heads 0..NH-1
                  tmem_ld<NH>(t_o, ov);
#pragma unroll
                  for (int j = 0; j < NH; ++j) ov[j] *= f[j];
                  tmem_st<NH>(t_o, ov);
                }
              }
              (void)softmax_pass();
              bar_softmax(1);                            // wmax may be rewritten only after every warp read it
            }
#pragma unroll
            for (int j = 0; j < NH; j += 2) fadd2(lsum[j], lsum[j + 1], lsum[j], lsum[j + 1], lt[j], lt[j + 1]);

            // ---- S has been read (QK may overwrite the buffer), P is written, O is consistent with mref
            if (cw == 0) TRD(3, gt);
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
      // ============================================================== V warps
      // Warp of lane quarter q converts channel group g = q (channels 32 q .. 32 q + 31 = one UE8M0 scale
      // group of V): its reference exponent eref is its own, so the four V warps never have to agree on
      // anything.  Stored Vhat = code * 2^(byte - eref + 13) in fp16, written straight into TMEM.
      // head_dim 256: warps 4..7 of the compute warps take channels 0..127, warps 8..11 channels 128..255 (half hc,
      // group 4 hc + q); head_dim 64: the warps of lane quarters 2 and 3 have no channels — they zero their rows of
      // both Vhat^T buffers once (the PV product runs M = 128 with those accumulator rows unused) and only keep the
      // barrier counts.
      const int hc = (kHalves == 2) ? ((cw - kSoftmaxWarps) >> 2) : 0;   // 128-channel half
      const int g = 4 * hc + q;
      const bool active = (D >= 128) ? true : (q < 2);
      const uint32_t scratch = base + kOffMul + 256 * (cw - kSoftmaxWarps);
      const uint32_t t_o = tmem + lane_sel + kColO + 16 * hc;    // channel 128 hc + r, heads 0..15
      if constexpr (D == 64) {
        if (!active) {
          const uint32_t z[16] = {0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
#pragma unroll
          for (int c16 = 0; c16 < (int)(kVBufs * kVBufCols) / 16; ++c16) tmem_st16_nowait(tmem + lane_sel + kColV + 16 * c16, z);
          tmem_wait_st();
          tc_fence_before();
        }
      }
      Cursor cur;
      sc.start(cur);
      Unit un;
      int gt = 0, s = 0, ph_full = 0;                  // global tile counter, its V stage and full-barrier parity
      [[maybe_unused]] int xk = 0, xph = 0;            // head_dim 64, expander warp: K stage and packed-full parity
      while (sc.next(cur, un)) {
        int eref = 28;
        int rem = un.tok_end - un.p0 * kPage;          // valid tokens from the first token of the tile on

        for (int i = 0; i < un.n_tiles; ++i, rem -= kTilePages * kPage) {
          const int sb = gt & 1;
          const uint32_t rest = base + kOffV + s * kVStageBytes;   // [V codes | K scales | V scales] of page 0
          if (cw == kSoftmaxWarps) TRD(6, gt);
          mbar_wait(bar_fullv + 8 * s, ph_full);       // the tile's bytes have landed
          if (cw == kSoftmaxWarps) TRD(7, gt);
          if constexpr (D == 64) {
            if (!active) {                             // no channels: nothing to convert, the barriers still count this warp
              if (q == 2) {
                // the K expander: packed codes of the tile [128 tokens][32 B] -> [chunk c][row r][8 B codes + 8 B pad]
                mbar_wait(smem_u32(&sh.full_kp[xk]), xph);
                const uint32_t src = base + Geo::kOffKP + xk * Geo::kKPStage, dstk = base + kOffK + xk * kKStageBytes;
#pragma unroll
                for (int rr = 0; rr < 4; ++rr) {
                  const int row = lane + 32 * rr;
                  const uint4 lo = lds128(src + 32 * row), hi = lds128(src + 32 * row + 16);
                  asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(dstk + 16 * row), "r"(lo.x), "r"(lo.y) : "memory");
                  asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(dstk + 2048 + 16 * row), "r"(lo.z), "r"(lo.w) : "memory");
                  asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(dstk + 4096 + 16 * row), "r"(hi.x), "r"(hi.y) : "memory");
                  asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(dstk + 6144 + 16 * row), "r"(hi.z), "r"(hi.w) : "memory");
                }
                fence_async_smem();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_fullk + 8 * xk);
                if (++xk == kKStages) { xk = 0; xph ^= 1; }
              }
              // arrive for tile gt only once the `ready` phase of tile gt-2 (same buffer) is over, as the converting
              // warps do: an early arrival would be counted into that phase
              if (gt >= 2) mbar_wait(bar_done + 8 * sb, ((gt >> 1) - 1) & 1);
              __syncwarp();
              if (lane == 0) {
                mbar_arrive(bar_ready + 8 * sb);
                mbar_arrive(bar_emptyv + 8 * s);
              }
              ++gt;
              if (++s == kVStages) { s = 0; ph_full ^= 1; }
              continue;
            }
          }

          // ---- the tile's 128 scale bytes of group g: lane <-> tokens 4 lane .. 4 lane + 3
          uint32_t sw;
          asm volatile("ld.shared.u32 %0, [%1];" : "=r"(sw)
                       : "r"(rest + kRestBytes * (lane >> 2) + (8 * D + D / 2) + (D / 4) * ((lane >> 1) & 1) + 8 * g + 4 * (lane & 1)));
          if (rem < kTilePages * kPage) {              // bytes of tokens past the end (stale shared memory) -> 0
            const int nv = rem - 4 * lane;             // valid tokens among this lane's four
            sw = nv >= 4 ? sw : (nv <= 0 ? 0u : (sw & (0xFFFFFFFFu >> (8 * (4 - nv)))));
          }
          const int b0 = (int)(sw & 0xFFu), b1 = (int)((sw >> 8) & 0xFFu), b2 = (int)((sw >> 16) & 0xFFu), b3 = (int)(sw >> 24);
          if (__builtin_expect(__any_sync(kFull, max(max(b0, b1), max(b2, b3)) > eref), 0)) {   // warp-uniform
            const int enew = __reduce_max_sync(kFull, max(max(b0, b1), max(b2, b3))) + 2;
            if (i > 0) {
              // O rows of this lane quarter change unit: after the softmax warps are through with the tile
              // (their own rescale of O included) and every PV issued so far has landed
              mbar_wait(bar_sfree + 8 * sb, (gt >> 1) & 1);
              mbar_wait(bar_done + 8 * (sb ^ 1), ((gt - 1) >> 1) & 1);
              tc_fence_after();
              float ov[16];
              tmem_ld<16>(t_o, ov);
              const float fe = pow2i(eref - enew);
#pragma unroll
              for (int j = 0; j < 16; ++j) ov[j] *= fe;
              tmem_st<16>(t_o, ov);
            }
            eref = enew;
          }
          {   // four fp16 power-of-two multipliers (two f16x2: token pairs 2 lane, 2 lane + 1); byte 0 -> 0
            const int kbase = eref - 28;               // fp16 exponent field = byte - kbase (2^13 at byte = eref)
            const uint32_t e0 = (uint32_t)max(b0 - kbase, 0), e1 = (uint32_t)max(b1 - kbase, 0),
                           e2 = (uint32_t)max(b2 - kbase, 0), e3 = (uint32_t)max(b3 - kbase, 0);
            asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(scratch + 8 * lane), "r"((e0 << 10) | (e1 << 26)),
                         "r"((e2 << 10) | (e3 << 26)) : "memory");
          }
          __syncwarp();

          if (cw == kSoftmaxWarps) TRD(11, gt);
          if (gt >= 2) {                               // PV(gt-2) has read Vhat buffer gt&1
            mbar_wait(bar_done + 8 * sb, ((gt >> 1) - 1) & 1);
            tc_fence_after();
          }
          if (cw == kSoftmaxWarps) TRD(12, gt);
          // ---- V codes -> Vhat^T in TMEM buffer gt&1: lane = channel, column c = tokens 2c, 2c+1
          const uint32_t t_v = tmem + lane_sel + kColV + kVBufCols * sb + 64 * hc;
          const uint32_t code0 = rest + 128 * g + 4 * lane;
#pragma unroll
          for (int h = 0; h < 4; ++h) {                // 32 tokens (16 TMEM columns) at a time
            uint32_t o[16];
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) {           // token octet k: page k>>1, half k&1
              const int k = 4 * h + kk;
              uint32_t cwd;
              asm volatile("ld.shared.u32 %0, [%1];" : "=r"(cwd) : "r"(code0 + kRestBytes * (k >> 1) + 4 * D * (k & 1)));
              const uint4 m4 = lds128(scratch + 16 * k);
              uint32_t f[4];
              cvt_e2m1x8(cwd, f);
              o[4 * kk + 0] = hmul2(f[0], m4.x);
              o[4 * kk + 1] = hmul2(f[1], m4.y);
              o[4 * kk + 2] = hmul2(f[2], m4.z);
              o[4 * kk + 3] = hmul2(f[3], m4.w);
            }
            tmem_st16_nowait(t_v + 16 * h, o);
          }
          tmem_wait_st();
          if (cw == kSoftmaxWarps) TRD(4, gt);
          tc_fence_before();
          __syncwarp();                                 // also: every lane has read the scratch of this tile
          if (lane == 0) {
            mbar_arrive(bar_ready + 8 * sb);
            mbar_arrive(bar_emptyv + 8 * s);           // this warp is done with the stage's V codes and scales
          }
          ++gt;
          if (++s == kVStages) { s = 0; ph_full ^= 1; }
        }

        // ============================================================== the unit's accumulator
        mbar_wait(bar_done + 8 * ((gt - 1) & 1), ((gt - 1) >> 1) & 1);
        tc_fence_after();
        if (early) pdl_wait();                         // (returns at once after the first time)
        if (active) {
          float ov[16];
          tmem_ld<16>(t_o, ov);
          const float vscale = pow2i(eref - 13 - 127);  // stored Vhat = code * 2^(byte - eref + 13)
#pragma unroll
          for (int j = 0; j < 16; ++j)
            if (j < G) partial_acc[(un.row0 + (long long)j * num_splits) * D + 128 * hc + r] = ov[j] * vscale;
        }
        tc_fence_before();                              // the next unit's first PV overwrites O
      }
    }
  }

  // ---------------- teardown
  tc_fence_before();
  __syncthreads();
  if (role == 1) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(kTmemCols));
  }
}

}  // namespace

// ---------------------------------------------------------------- host: TMA descriptors (shared with uq_decode_prefix.cu)
namespace {
struct MapEntry {
  const void* cache;
  long long records;
  int device, head_dim;
  CUtensorMap map, rest;
};
std::mutex g_map_mu;
MapEntry g_maps[8];
int g_map_n = 0, g_map_next = 0;

}  // namespace

// 3-D view of the cache for TMA: [record][16 tokens][head_dim x 4-bit]; box = one page of K codes, 128 channels wide
// (head_dim 256: two copies per page; head_dim 64 does not use it).
int32_t k_code_map(const void* cache, long long records, int head_dim, CUtensorMap* out, CUtensorMap* out_rest) {
  int dev = 0;
  (void)cudaGetDevice(&dev);                           // the same virtual address may be another allocation on another device
  const EncodeTiledFn encode = encode_tiled_fn();
  if (!encode) return UQ_ERR_CUDA;
  std::lock_guard<std::mutex> lock(g_map_mu);
  for (int i = 0; i < g_map_n; ++i)
    if (g_maps[i].cache == cache && g_maps[i].records == records && g_maps[i].device == dev && g_maps[i].head_dim == head_dim) {
      *out = g_maps[i].map;
      if (out_rest) *out_rest = g_maps[i].rest;
      return UQ_OK;
    }
  const cuuint64_t gdim[3] = {(cuuint64_t)head_dim, 16, (cuuint64_t)records};
  const cuuint64_t gstr[2] = {(cuuint64_t)head_dim / 2, (cuuint64_t)17 * head_dim};
  const cuuint32_t box[3] = {128, 16, 1};              // the packed 4-bit tensor type takes 128-wide boxes only
  const cuuint32_t estr[3] = {1, 1, 1};
  CUtensorMap m = {}, mr = {};
  CUresult cr = CUDA_SUCCESS;
  if (head_dim <= 128) {
    // the rest of a record (9 D bytes from byte 8 D on) as a row of 8-byte elements: the source of the gather4 copies
    const cuuint64_t rdim[2] = {(cuuint64_t)(9 * head_dim / 8), (cuuint64_t)records};
    const cuuint64_t rstr[1] = {(cuuint64_t)17 * head_dim};
    const cuuint32_t rbox[2] = {(cuuint32_t)(9 * head_dim / 8), 1};
    const cuuint32_t rest_[2] = {1, 1};
    cr = encode(&mr, CU_TENSOR_MAP_DATA_TYPE_UINT64, 2, const_cast<uint8_t*>((const uint8_t*)cache) + 8 * head_dim, rdim, rstr,
                rbox, rest_, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (cr != CUDA_SUCCESS) {
      set_error("decode: cuTensorMapEncodeTiled (record rest, gather4) failed with CUresult %d", (int)cr);
      return UQ_ERR_CUDA;
    }
  }
  if (head_dim >= 128)
  cr = encode(&m, CU_TENSOR_MAP_DATA_TYPE_16U4_ALIGN16B, 3, const_cast<void*>(cache), gdim, gstr, box,
                             estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                             CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (cr != CUDA_SUCCESS) {
    set_error("decode: cuTensorMapEncodeTiled failed with CUresult %d", (int)cr);
    return UQ_ERR_CUDA;
  }
  MapEntry& e = g_maps[g_map_next];
  e.cache = cache;
  e.records = records;
  e.device = dev;
  e.head_dim = head_dim;
  e.map = m;
  e.rest = mr;
  g_map_next = (g_map_next + 1) % 8;
  if (g_map_n < 8) ++g_map_n;
  *out = m;
  if (out_rest) *out_rest = mr;
  return UQ_OK;
}

// View of q_fp8 for TMA: [batch * Hq rows][head_dim bytes]; box = 16 rows (the heads of one kv head, padded) x 128
// bytes, 128-byte swizzle; head_dim 64: 3-D, see below.
int32_t q_map(const void* q_fp8, long long rows, int head_dim, CUtensorMap* out) {
  const EncodeTiledFn encode = encode_tiled_fn();
  if (!encode) return UQ_ERR_CUDA;
  CUresult cr;
  if (head_dim == 64) {
    // [16-byte chunk][row][16 B]: the copy lands in the unswizzled core-matrix order the MMA descriptor names
    const cuuint64_t gdim[3] = {16, (cuuint64_t)rows, 4};
    const cuuint64_t gstr[2] = {64, 16};
    const cuuint32_t box[3] = {16, 16, 4};
    const cuuint32_t estr[3] = {1, 1, 1};
    cr = encode(out, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<void*>(q_fp8), gdim, gstr, box, estr,
                CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  } else {
    const cuuint64_t gdim[2] = {(cuuint64_t)head_dim, (cuuint64_t)rows};
    const cuuint64_t gstr[1] = {(cuuint64_t)head_dim};
    const cuuint32_t box[2] = {128, 16};
    const cuuint32_t estr[2] = {1, 1};
    cr = encode(out, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void*>(q_fp8), gdim, gstr, box, estr,
                CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  }
  if (cr != CUDA_SUCCESS) {
    set_error("decode: cuTensorMapEncodeTiled (q_fp8) failed with CUresult %d", (int)cr);
    return UQ_ERR_CUDA;
  }
  return UQ_OK;
}

namespace {
template <int D>
int32_t launch_decode(const uq_config* cfg, const CUtensorMap& tmap, const CUtensorMap& tmap_q, const CUtensorMap& tmap_v,
                      const void* cache,
                      const int32_t* block_tables, int32_t max_pages, const int32_t* seq_lens, int32_t batch,
                      int32_t num_splits, float score_scale, float* partial_acc, float* partial_ml, int sm_count,
                      cudaStream_t stream) {
  using Geo = DecodeGeo<D>;
  const long long slots = (long long)sm_count * Geo::kCtasPerSm;
  const long long items = (long long)batch * cfg->num_kv_heads;
  // num_splits == 1: a CTA per item (round-robin beyond the resident set); otherwise one balanced tile range per CTA
  const dim3 grid((unsigned)((num_splits == 1 && items < slots) ? items : slots));
  int32_t st = opt_in_dynamic_smem((const void*)decode_kernel<D>, Geo::kSmemBytes, "decode: cudaFuncSetAttribute");
  if (st != UQ_OK) return st;
  return check_cuda(launch_pdl(decode_kernel<D>, grid, dim3(Geo::kThreads), (size_t)Geo::kSmemBytes, stream, tmap, tmap_q, tmap_v,
                               (const uint8_t*)cache, block_tables, (int)max_pages, seq_lens, (int)batch,
                               (int)cfg->num_q_heads, (int)cfg->num_kv_heads, (int)num_splits, score_scale, partial_acc,
                               partial_ml, (int)((cfg->flags & UQ_FLAG_SMALL_APPEND_AHEAD) != 0)),
                    "uq_decode_attention launch");
}
}  // namespace

}  // namespace uq


extern "C" int32_t uq_decode_attention(const uq_config* cfg, const void* q_fp8, const void* cache,
                                       int64_t num_pages, const int32_t* block_tables, int32_t max_pages,
                                       const int32_t* seq_lens, int32_t batch, int32_t num_splits,
                                       float* partial_acc, float* partial_ml, void* stream) {
  using namespace uq;
  NvtxRange nvtx_range("uq_decode_attention");
  int32_t st = check_config(cfg);
  if (st != UQ_OK) return st;
  if (!q_fp8 || !cache || !block_tables || !seq_lens || !partial_acc || !partial_ml || batch <= 0 ||
      num_splits <= 0 || max_pages <= 0 || num_pages <= 0) {
    set_error("decode: NULL pointer or non-positive size");
    return UQ_ERR_INVALID_ARG;
  }
  if (((uintptr_t)cache & 31u) || ((uintptr_t)q_fp8 & 15u) || ((uintptr_t)partial_acc & 15u) ||
      ((uintptr_t)partial_ml & 7u)) {
    set_error("decode: misaligned pointer (cache 32 B, q_fp8 16 B, partial_acc 16 B, partial_ml 8 B)");
    return UQ_ERR_INVALID_ARG;
  }
  const long long records = (long long)num_pages * cfg->num_kv_heads;
  if (records > 0x7fffffffLL) {
    set_error("decode: num_pages * num_kv_heads must be < 2^31");
    return UQ_ERR_INVALID_ARG;
  }
  if (cfg->flags & UQ_FLAG_DEBUG_CHECKS) {
    st = debug_check_tables("uq_decode_attention", block_tables, max_pages, batch, num_pages, seq_lens, nullptr, 0, 0,
                            cfg->page_size, 0, (cudaStream_t)stream);
    if (st != UQ_OK) return st;
  }
  CUtensorMap tmap = {}, tmap_v = {};                  // head_dim 64 copies the packed K codes without a tensor map
  st = k_code_map(cache, records, cfg->head_dim, &tmap, &tmap_v);
  if (st != UQ_OK) return st;
  CUtensorMap tmap_q;
  st = q_map(q_fp8, (long long)batch * cfg->num_q_heads, cfg->head_dim, &tmap_q);
  if (st != UQ_OK) return st;
  const float score_scale = resolved_sm_scale(cfg) * 1.4426950408889634f;
  if (batch > kMaxBatch) {
    set_error("decode: batch %d exceeds the supported maximum of %d sequences per call", batch, kMaxBatch);
    return UQ_ERR_UNSUPPORTED;
  }
  int sm_count = 0;
  st = current_device_sms(&sm_count);
  if (st != UQ_OK) return st;
  switch (cfg->head_dim) {
    case 64:
      return launch_decode<64>(cfg, tmap, tmap_q, tmap_v, cache, block_tables, max_pages, seq_lens, batch, num_splits, score_scale,
                               partial_acc, partial_ml, sm_count, (cudaStream_t)stream);
    case 256:
      return launch_decode<256>(cfg, tmap, tmap_q, tmap_v, cache, block_tables, max_pages, seq_lens, batch, num_splits, score_scale,
                                partial_acc, partial_ml, sm_count, (cudaStream_t)stream);
    default:
      return launch_decode<128>(cfg, tmap, tmap_q, tmap_v, cache, block_tables, max_pages, seq_lens, batch, num_splits, score_scale,
                                partial_acc, partial_ml, sm_count, (cudaStream_t)stream);
  }
}

#ifdef UQ_TRACE
// debug builds only (not part of include/uq.h): the [UQ_TRACE_TILES][16] clock64 table of the decode kernel's traced CTA
extern "C" int uq_debug_trace_read_decode(void* host, size_t bytes) {
  return (int)cudaMemcpyFromSymbol(host, uq::g_trace_decode, bytes);
}
#endif
