// uq_decode_prefix.cu — decode attention over a SHARED PREFIX ("cascade"): the first prefix_len
// tokens of every sequence of the call are the same physical pages (the agent workloads of the paper share a long
// prompt), so a 128-token tile of the prefix is staged, its V codes converted and its MMAs issued
// once for kNS sequences at a time instead of once per sequence.  Same CTA design as uq_decode.cu (read that file
// first): TMA K / V rings, tcgen05 block-scaled QK, softmax warps with lazy per-head references, V warps writing
// Vhat^T to TMEM, PV from TMEM — with the score tile widened from 16 to 16 kNS columns (the query tiles of kNS
// sequences side by side), one group of four softmax warps per sequence (each with its own named barrier, references
// and running sums), and one CTA of 24 warps per SM (the TMEM columns and shared memory of two).  All items have the
// same length, so the schedule is plain arithmetic.
// Measured on config 4 (256 sequences, 30,000-token prefix): this kernel 334 us for the prefix of all
// sequences (0.83 us per four-sequence tile), the whole step 721 us against 989 us with the plain kernel.  One softmax
// group for all four sequences was 1.8 x slower, two sequences per tile 1.6 x.
#include <cuda.h>
#include <cuda_fp16.h>

#include <mutex>
#include <type_traits>

#include "uq_tc.cuh"

namespace uq {
namespace {

#ifndef UQ_PREFIX_GROUPS
#define UQ_PREFIX_GROUPS 4
#endif
constexpr int kSoftGroups = UQ_PREFIX_GROUPS;        // softmax warp groups: each takes kNS / kSoftGroups of the sequences
constexpr int kSoftmaxWarps = 4;                     // per group: one warp per TMEM lane quarter
constexpr int kVWarps = 4;
constexpr int kComputeWarps = kSoftGroups * kSoftmaxWarps + kVWarps;
constexpr int kIssuerWarps = 4;                      // QK issuer, PV issuer, K producer, V producer
constexpr int kThreads = (kComputeWarps + kIssuerWarps) * 32;
#ifndef UQ_PREFIX_NSEQ
#define UQ_PREFIX_NSEQ 4
#endif
constexpr int kNS = UQ_PREFIX_NSEQ;                   // sequences per prefix tile
constexpr int kNCols = 16 * kNS;                      // score columns: 16 head slots per sequence
constexpr int kSeqPerGroup = kNS / UQ_PREFIX_GROUPS;
static_assert(kSeqPerGroup * UQ_PREFIX_GROUPS == kNS, "sequences per tile must divide over the softmax groups");
#undef UQ_KSTAGES
#undef UQ_VSTAGES
#undef UQ_CTAS_PER_SM
#ifndef UQ_PREFIX_CTAS
#define UQ_PREFIX_CTAS 1
#endif
#if UQ_PREFIX_CTAS == 2
#define UQ_KSTAGES 3
#define UQ_VSTAGES 4
#else
#define UQ_KSTAGES 4
#define UQ_VSTAGES 6
#endif
#define UQ_CTAS_PER_SM UQ_PREFIX_CTAS
// Two rings: the K codes of a tile (16 KB once the TMA unit has expanded the nibbles) are needed by the QK
// MMA only and leave early; the rest of the records (V codes, K scales, V scales: 9 KB) stays until the V
// warps have converted it.  Separate rings let the small one run deep (bytes in flight hide HBM latency).
constexpr int kKStages = UQ_KSTAGES;
constexpr int kVStages = UQ_VSTAGES;
constexpr int kTilePages = 8;                        // 128 tokens per tile
constexpr int kRestBytes = kRecordBytes - 1024;      // V codes + K scales + V scales = 1152
constexpr int kKStageBytes = kTilePages * 2048;      // K codes, one byte per code: 16384
constexpr int kVStageBytes = kTilePages * kRestBytes;   // 9216
constexpr int kPBytes = 4096 * kNS;                  // one P operand buffer: [token-core 16][head-core 2 kNS][8 tok][8 heads] f16
constexpr float kThresh = 12.0f;                     // lazy-reference threshold (log2 units)

// dynamic shared memory map (offsets from a 1024-byte aligned base)
constexpr int kOffK = 0;                                       // kKStages x 16384, SW128
constexpr int kOffV = kOffK + kKStages * kKStageBytes;         // kVStages x 9216
constexpr int kOffQ = kOffV + kVStages * kVStageBytes;         // 2 x 2048, SW128 (one per unit in flight)
constexpr int kOffSFA = kOffQ + 4096 * kNS;                    // 2 x 512
constexpr int kOffSFB = kOffSFA + 1024;                        // 512
constexpr int kOffP = kOffSFB + 512;                           // 2 x 4096 (double-buffered)
constexpr int kOffMul = kOffP + 2 * kPBytes;                   // 4 V warps x 256 B of fp16 multipliers
constexpr int kOffEnd = kOffMul + kComputeWarps * 128;
constexpr int kSmemBytes = kOffEnd + 1024;                     // + alignment slack

// TMEM columns
constexpr uint32_t kColS = 0;                   // 2 x kNCols
constexpr uint32_t kColO = 2 * kNCols;          // kNCols
constexpr uint32_t kColSFA = 3 * kNCols;        // 2 x 4
constexpr uint32_t kColSFB = 3 * kNCols + 8;    // 4
#ifndef UQ_VBUFS
#define UQ_VBUFS 2
#endif
constexpr int kVBufs = UQ_VBUFS;   // Vhat^T buffers in TMEM
constexpr uint32_t kColV = UQ_PREFIX_CTAS == 2 ? 128 : (3 * kNCols + 12 + 31) / 32 * 32;    // kVBufs x 64: Vhat^T operand, lane = channel d, column c = tokens 2c, 2c+1 (f16x2)
constexpr uint32_t kTmemCols = UQ_PREFIX_CTAS == 2 ? 256 : 512;
static_assert(kColV + 128 <= kTmemCols, "TMEM columns");
static_assert(3 * kNCols + 12 <= kColV, "score / accumulator / scale columns must stay below the Vhat buffers");

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
  float wmax[kSoftGroups][kSoftmaxWarps][16];
  float lsum[kSoftGroups][kSoftmaxWarps][16];
  float mref[kSoftGroups][16];
};

// ---------------------------------------------------------------- work schedule
// Items = (group of kNS consecutive sequences, kv head), kv head fastest, every item PT = prefix_len / 128 tiles
// long.  The tiles of all items form one sequence that is cut into equal contiguous ranges, one per CTA; a range may
// end inside an item and start inside the next one, so a CTA works through a few UNITS (item, tile range).  The CTAs
// that share an item write consecutive partial slots of it (the same slot for each of its sequences); tpc is raised
// if needed so that no item spans more than num_splits CTAs.
struct Unit {
  int b, kvh, p0, p1, n_tiles, tok_end;               // b: first sequence of the group
  int slots_used;                                      // > 0 on the unit holding the item's last tile: slots the item uses
  long long row0;                                      // partial row of (sequence b, head 0) in this unit's slot:
};                                                     // + head * num_splits, + hs * Hq * num_splits for sequence b + hs
struct Cursor {
  int it, t, g, g1;                                    // item, tile inside it, global tile, range end
};

struct Sched {
  int B, Hq, Hkv, G, S, tpc, total, PT;

  __device__ void start(Cursor& c) const {
    c.g = min((int)blockIdx.x * tpc, total);
    c.g1 = min(c.g + tpc, total);
    c.it = c.g / PT;
    c.t = c.g - c.it * PT;
  }
  // next unit of this CTA, false when there is none
  __device__ bool next(Cursor& c, Unit& u) const {
    if (c.g >= c.g1) return false;
    const int grp = c.it / Hkv;
    u.kvh = c.it - grp * Hkv;
    u.b = grp * kNS;
    const int t0 = c.t, t1 = min(PT, t0 + (c.g1 - c.g));
    const int item_start = c.g - t0;                   // global tile index of the item's first tile
    const int slot = (int)blockIdx.x - item_start / tpc;
    u.slots_used = (t1 == PT) ? slot + 1 : 0;
    u.row0 = ((long long)u.b * Hq + (long long)u.kvh * G) * S + slot;
    c.g += t1 - t0;
    c.t = t1;
    if (t1 == PT) { c.t = 0; ++c.it; }
    u.p0 = kTilePages * t0;
    u.p1 = kTilePages * t1;
    u.n_tiles = t1 - t0;
    u.tok_end = u.p1 * kPage;
    return true;
  }
};

// ---------------------------------------------------------------- the kernel
__global__ void __launch_bounds__(kThreads, UQ_CTAS_PER_SM)
decode_prefix_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ CUtensorMap tmap_q,
              const uint8_t* __restrict__ cache, const int32_t* __restrict__ block_tables, int max_pages,
              int prefix_tiles, int batch, int Hq, int Hkv, int num_splits,
              float score_scale /* sm_scale * log2(e) */, float* __restrict__ partial_acc,
              float* __restrict__ partial_ml) {
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

  const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sQ = base + kOffQ, sSFA = base + kOffSFA, sSFB = base + kOffSFB, sP = base + kOffP;
  const uint32_t bar_fullk = smem_u32(&sh.full_k[0]), bar_emptyk = smem_u32(&sh.empty_k[0]),
                 bar_fullv = smem_u32(&sh.full_v[0]), bar_emptyv = smem_u32(&sh.empty_v[0]),
                 bar_sfull = smem_u32(&sh.s_full[0]), bar_sfree = smem_u32(&sh.s_free[0]),
                 bar_ready = smem_u32(&sh.ready[0]), bar_done = smem_u32(&sh.done[0]),
                 bar_qfull = smem_u32(&sh.q_full[0]);

  // ---------------- setup
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < kKStages; ++s) {
      mbar_init(bar_fullk + 8 * s, 1);
      mbar_init(bar_emptyk + 8 * s, 1);
    }
#pragma unroll
    for (int s = 0; s < kVStages; ++s) {
      mbar_init(bar_fullv + 8 * s, 1);
      mbar_init(bar_emptyv + 8 * s, kVWarps + 1);
    }
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      mbar_init(bar_sfull + 8 * h, 1);
      mbar_init(bar_sfree + 8 * h, kSoftGroups * kSoftmaxWarps);
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
  pdl_wait();
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = sh.tmem_base;

  Sched sc;
  sc.B = batch; sc.Hq = Hq; sc.Hkv = Hkv; sc.G = G; sc.S = num_splits; sc.PT = prefix_tiles;
  sc.total = ((batch + kNS - 1) / kNS) * Hkv * prefix_tiles;
  {
    const int even = (sc.total + (int)gridDim.x - 1) / (int)gridDim.x;
    const int fit = (prefix_tiles + num_splits - 2) / (num_splits - 1);   // an item spans at most num_splits ranges (>= 2)
    sc.tpc = max(1, max(even, fit));
  }

  if (role == 0) {
    // ================================================================ QK warp
    // Per unit: the FP8 query tile (16 rows x 128 B, 128-byte swizzle) arrives by TMA into Q buffer
    // (unit ordinal & 1) — "hoisted", once per unit; rows past the unit's G heads belong to
    // the next kv head (or are zero past the tensor end) and only feed score columns nobody reads.
    // Per tile: S(gt)[128 tok x 16 heads] = K . Q^T once the tile's bytes have landed, the S buffer was read
    // by the softmax of global tile gt-2.
    const uint32_t idesc_qk = (5u << 7) | (0u << 10) | ((uint32_t)(kNCols >> 3) << 17) | (1u << 23) | (8u << 24);   // E2M1 x E4M3, UE8M0, N=16 kNS, M=128
    if (elect_one()) umma_cp_sf(tmem + kColSFB, make_desc(sSFB, 16, 128, 0));
    auto load_q = [&](const Unit& un, int k) {         // lane 0: Q tile of unit ordinal k
      if (elect_one()) {
        mbar_expect_tx(bar_qfull + 8 * (k & 1), 2048 * kNS);
#pragma unroll
        for (int hs = 0; hs < kNS; ++hs)               // rows past the last sequence are zero-filled by the TMA unit
          tma_load_2d(sQ + 2048 * kNS * (k & 1) + 2048 * hs, &tmap_q, 0, (un.b + hs) * Hq + un.kvh * G, bar_qfull + 8 * (k & 1));
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
        if (gt >= 2) mbar_wait(bar_sfree + 8 * sb, ((gt >> 1) - 1) & 1);
        // here every QK up to global tile gt-2 has completed (its S was read): at i == 0 the Q buffer of
        // unit k-2 (= buffer k & 1), at i == 1 that of unit k-1 (= buffer (k+1) & 1) may be refilled
        if (i == 0 && k_q < k) { load_q(un, k); k_q = k; }
        if (i == 1 && have_nx) { load_q(nx, k + 1); k_q = k + 1; }
        if (i == 0) mbar_wait(bar_qfull + 8 * (k & 1), (k >> 1) & 1);
        mbar_wait(bar_fullv + 8 * sv, phv);
        const uint32_t st = base + kOffK + sk * kKStageBytes, rest = base + kOffV + sv * kVStageBytes;
        // scale-factor atom: row r = 32 c + lane of the tile -> 16-byte line `lane`, word c
        uint32_t v[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const int r = 32 * c + lane;
          asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v[c]) : "r"(rest + kRestBytes * (r >> 4) + 1024 + 4 * (r & 15)));
        }
        sts128(sSFA + 512 * sb + 16 * lane, make_uint4(v[0], v[1], v[2], v[3]));
        fence_async_smem();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_emptyv + 8 * sv);   // the K scales are copied: this warp is done with the V stage
        mbar_wait(bar_fullk + 8 * sk, phk);
        tc_fence_after();
        if (elect_one()) {
          const uint32_t t_sfa = tmem + kColSFA + 4 * sb, qb = sQ + 2048 * kNS * (k & 1);
          umma_cp_sf(t_sfa, make_desc(sSFA + 512 * sb, 16, 128, 0));
#pragma unroll
          for (int kb = 0; kb < 4; ++kb)
            umma_mxf8f6f4(tmem + kColS + kNCols * sb, make_desc(st + 32 * kb, 16, 1024, 2), make_desc(qb + 32 * kb, 16, 1024, 2),
                          idesc_qk | ((uint32_t)kb << 29), kb > 0, t_sfa + ((uint32_t)kb << 30), tmem + kColSFB);
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
    const uint32_t idesc_pv = (1u << 4) | (1u << 16) | ((uint32_t)(kNCols >> 3) << 17) | (8u << 24);
    Cursor cur;
    sc.start(cur);
    Unit un;
    int gt = 0;
    while (sc.next(cur, un)) {
      for (int i = 0; i < un.n_tiles; ++i, ++gt) {
        mbar_wait(bar_ready + 8 * (gt & 1), (gt >> 1) & 1);
        tc_fence_after();
        if (lane == 0) {
          const uint32_t pbuf = sP + kPBytes * (gt & 1), vbuf = tmem + kColV + 64 * ((gt & 1) % kVBufs);
#pragma unroll
          for (int j = 0; j < 8; ++j)                    // 16 tokens per MMA = 8 columns of Vhat^T
            umma_f16_ts(tmem + kColO, vbuf + 8 * j, make_desc(pbuf + 512 * kNS * j, 256 * kNS, 128, 0), idesc_pv,
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
    const uint32_t bar_e = is_k ? bar_emptyk : bar_emptyv, bar_f = is_k ? bar_fullk : bar_fullv;
    const uint32_t page_tx = is_k ? 1024u : (uint32_t)kRestBytes;
    const uint64_t pol = l2_evict_first_policy();
    Cursor cur;
    sc.start(cur);
    Unit un;
    int s = 0, ph = 1;                                 // stage, parity to wait for on empty[s]
    while (sc.next(cur, un)) {
      const int32_t* bt = block_tables + (long long)un.b * max_pages + un.p0 + lane;
      int page_next = (lane < kTilePages && un.p0 + lane < un.p1) ? bt[0] : 0;
      for (int i = 0; i < un.n_tiles; ++i) {
        const int page = page_next;
        const int npg = min(kTilePages, un.p1 - (un.p0 + kTilePages * i));
        const int nb = un.p0 + kTilePages * (i + 1) + lane;
        page_next = (lane < kTilePages && nb < un.p1) ? bt[kTilePages * (i + 1)] : 0;
        mbar_wait(bar_e + 8 * s, ph);
        if (lane == 0) mbar_expect_tx(bar_f + 8 * s, (uint32_t)npg * page_tx);
        __syncwarp();
        if (lane < npg) {
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

    if (cw < kSoftGroups * kSoftmaxWarps) {
      // ============================================================== softmax warps
      const int grp = cw >> 2, cwl = cw & 3;           // softmax group, warp inside it
      const int bar_id = 1 + grp;                      // the group's named barrier
      const int atid = 32 * cwl + lane;                // 0..127 inside the group
      float2* const ml_out = reinterpret_cast<float2*>(partial_ml);
      const long long seq_rows = (long long)Hq * num_splits;   // partial rows of one sequence

      auto run = [&](auto nh_tag) {
        constexpr int NH = decltype(nh_tag)::value;    // head columns per sequence this thread handles: 8 (G <= 8) or 16
        Cursor cur;
        sc.start(cur);
        Unit un;
        int gt = 0;                                    // global tile counter
        const uint32_t p_row = sP + (r >> 3) * (256 * kNS) + (r & 7) * 16;
        while (sc.next(cur, un)) {
          float nmref[kSeqPerGroup][NH], lsum[kSeqPerGroup][NH];         // nmref = minus the per-head reference logit, per sequence
#pragma unroll
          for (int hq = 0; hq < kSeqPerGroup; ++hq) {
#pragma unroll
            for (int j = 0; j < NH; ++j) { nmref[hq][j] = INFINITY; lsum[hq][j] = 0.f; }
          }

          for (int i = 0; i < un.n_tiles; ++i) {       // every tile of the prefix is whole: no token mask
            const int sb = gt & 1, ph2 = (gt >> 1) & 1;
            mbar_wait(bar_sfull + 8 * sb, ph2);        // S(gt) is in TMEM
            if (gt >= 2) mbar_wait(bar_done + 8 * sb, ph2 ^ 1);   // PV(gt-2) has read P buffer gt&1
            tc_fence_after();

#pragma unroll
            for (int hq = 0; hq < kSeqPerGroup; ++hq) { // this warp group's sequences one after the other
              const int hs = grp * kSeqPerGroup + hq;
              const uint32_t t_s = tmem + lane_sel + kColS + kNCols * sb + 16 * hs;
              const uint32_t p_addr = p_row + kPBytes * sb + 256 * hs;   // head-cores 2 hs, 2 hs + 1
              float lt[NH];
              // softmax of this thread's row against the current references -> P (fp16, MN-major operand)
              auto softmax_pass = [&]() -> bool {
                float t[NH];
                tmem_ld<NH>(t_s, t);
#pragma unroll
                for (int j = 0; j < NH; j += 2)
                  ffma2(t[j], t[j + 1], t[j], t[j + 1], score_scale, nmref[hq][j], nmref[hq][j + 1]);
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
                rebase = bar_softmax_or(bar_id, ex);
              }
              if (__builtin_expect(rebase, 0)) {
                // ---- per-head maximum score of the tile -> new references; O and l of this sequence rescaled
                float tm[NH];
                {
                  float sv[NH];
                  tmem_ld<NH>(t_s, sv);
#pragma unroll
                  for (int j = 0; j < NH; ++j) {
                    float x = sv[j] * score_scale;
#pragma unroll
                    for (int o = 16; o; o >>= 1) x = fmaxf(x, __shfl_xor_sync(kFull, x, o));
                    tm[j] = x;
                  }
                }
                if (lane == 0) {
#pragma unroll
                  for (int j = 0; j < NH; ++j) sh.wmax[grp][cwl][j] = tm[j];
                }
                tc_fence_before();
                bar_softmax(bar_id);
                float f[NH];
#pragma unroll
                for (int j = 0; j < NH; ++j) {
                  float m = sh.wmax[grp][0][j];
#pragma unroll
                  for (int w = 1; w < kSoftmaxWarps; ++w) m = fmaxf(m, sh.wmax[grp][w][j]);
                  const float mold = -nmref[hq][j], mnew = fmaxf(mold, m);
                  const float fm = (mold == -INFINITY) ? 0.f : ex2(mold - mnew);
                  nmref[hq][j] = -mnew;
                  lsum[hq][j] *= fm;
                  f[j] = fm;
                }
                if (i > 0) {  // every PV of this unit issued so far has to be in O before it is rescaled
                  mbar_wait(bar_done + 8 * (sb ^ 1), ((gt - 1) >> 1) & 1);
                  tc_fence_after();
                  float ov[NH];
                  const uint32_t t_o = tmem + lane_sel + kColO + 16 * hs;   // channel r, heads of sequence hs
                  tmem_ld<NH>(t_o, ov);
#pragma unroll
                  for (int j = 0; j < NH; ++j) ov[j] *= f[j];
                  tmem_st<NH>(t_o, ov);
                }
                (void)softmax_pass();
                bar_softmax(bar_id);                          // wmax may be rewritten only after every warp read it
              }
#pragma unroll
              for (int j = 0; j < NH; j += 2)
                fadd2(lsum[hq][j], lsum[hq][j + 1], lsum[hq][j], lsum[hq][j + 1], lt[j], lt[j + 1]);
            }

            // ---- S has been read (QK may overwrite the buffer), P is written, O is consistent with the references
            fence_async_smem();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) {
              mbar_arrive(bar_sfree + 8 * sb);
              mbar_arrive(bar_ready + 8 * sb);
            }
            ++gt;
          }

          // ============================================================ the unit's (m, l), sequence by sequence
#pragma unroll
          for (int hq = 0; hq < kSeqPerGroup; ++hq) {
            const int hs = grp * kSeqPerGroup + hq;
#pragma unroll
            for (int j = 0; j < NH; ++j) {
              float v = lsum[hq][j];
#pragma unroll
              for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
              lsum[hq][j] = v;
            }
            if (lane == 0) {
#pragma unroll
              for (int j = 0; j < NH; ++j) {
                sh.lsum[grp][cwl][j] = lsum[hq][j];
                if (cwl == 0) sh.mref[grp][j] = -nmref[hq][j];
              }
            }
            bar_softmax(bar_id);
            if (un.b + hs < batch) {
              const long long row0 = un.row0 + hs * seq_rows;
              if (atid < G) {                            // one thread per query head
                float l = 0.f;
#pragma unroll
                for (int w = 0; w < kSoftmaxWarps; ++w) l += sh.lsum[grp][w][atid];
                ml_out[row0 + (long long)atid * num_splits] = make_float2(sh.mref[grp][atid] * 0.6931471805599453f, l);   // natural log
              }
              if (un.slots_used > 0) {                   // item finished: its remaining slots are empty
                const long long row_item = row0 - (un.slots_used - 1);
                const int n_empty = num_splits - un.slots_used;
                for (int e = atid; e < G * n_empty; e += 32 * kSoftmaxWarps) {
                  const int head = e / n_empty, sl = un.slots_used + (e - head * n_empty);
                  ml_out[row_item + (long long)head * num_splits + sl] = make_float2(-INFINITY, 0.f);
                }
              }
            }
            bar_softmax(bar_id);                              // sh.lsum / sh.mref are reused by the next sequence / unit
          }
        }
      };
      if (G > 8) run(std::integral_constant<int, 16>{});
      else run(std::integral_constant<int, 8>{});
    } else {
      // ============================================================== V warps
      // Warp of lane quarter q converts channel group g = q (channels 32 q .. 32 q + 31 = one UE8M0 scale
      // group of V): its reference exponent eref is its own, so the four V warps never have to agree on
      // anything.  Stored Vhat = code * 2^(byte - eref + 13) in fp16, written straight into TMEM.
      const int g = q;
      const uint32_t scratch = base + kOffMul + 256 * (cw - kSoftGroups * kSoftmaxWarps);
      const uint32_t t_o = tmem + lane_sel + kColO;    // channel r, heads 0..15 of sequence 0 of the group
      Cursor cur;
      sc.start(cur);
      Unit un;
      int gt = 0, s = 0, ph_full = 0;                  // global tile counter, its V stage and full-barrier parity
      while (sc.next(cur, un)) {
        int eref = 28;
        int rem = un.tok_end - un.p0 * kPage;          // valid tokens from the first token of the tile on

        for (int i = 0; i < un.n_tiles; ++i, rem -= kTilePages * kPage) {
          const int sb = gt & 1;
          const uint32_t rest = base + kOffV + s * kVStageBytes;   // [V codes | K scales | V scales] of page 0
          mbar_wait(bar_fullv + 8 * s, ph_full);       // the tile's bytes have landed

          // ---- the tile's 128 scale bytes of group g: lane <-> tokens 4 lane .. 4 lane + 3
          uint32_t sw;
          asm volatile("ld.shared.u32 %0, [%1];" : "=r"(sw)
                       : "r"(rest + kRestBytes * (lane >> 2) + 1088 + 32 * ((lane >> 1) & 1) + 8 * g + 4 * (lane & 1)));
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
              const float fe = pow2i(eref - enew);
#pragma unroll
              for (int hs = 0; hs < kNS; ++hs) {
                float ov[16];
                tmem_ld<16>(t_o + 16 * hs, ov);
#pragma unroll
                for (int j = 0; j < 16; ++j) ov[j] *= fe;
                tmem_st<16>(t_o + 16 * hs, ov);
              }
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

          if (gt >= 2) {                               // PV(gt-2) has read Vhat buffer gt&1
            mbar_wait(bar_done + 8 * sb, ((gt >> 1) - 1) & 1);
            tc_fence_after();
          }
          // ---- V codes -> Vhat^T in TMEM buffer gt&1: lane = channel, column c = tokens 2c, 2c+1
          const uint32_t t_v = tmem + lane_sel + kColV + 64 * sb;
          const uint32_t code0 = rest + 128 * g + 4 * lane;
#pragma unroll
          for (int h = 0; h < 4; ++h) {                // 32 tokens (16 TMEM columns) at a time
            uint32_t o[16];
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) {           // token octet k: page k>>1, half k&1
              const int k = 4 * h + kk;
              uint32_t cwd;
              asm volatile("ld.shared.u32 %0, [%1];" : "=r"(cwd) : "r"(code0 + kRestBytes * (k >> 1) + 512 * (k & 1)));
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
        {
          const float vscale = pow2i(eref - 13 - 127);  // stored Vhat = code * 2^(byte - eref + 13)
#pragma unroll
          for (int hs = 0; hs < kNS; ++hs) {
            float ov[16];
            tmem_ld<16>(t_o + 16 * hs, ov);
            if (un.b + hs < batch) {
              const long long row0 = un.row0 + (long long)hs * Hq * num_splits;
#pragma unroll
              for (int j = 0; j < 16; ++j)
                if (j < G) partial_acc[(row0 + (long long)j * num_splits) * kHeadDim + r] = ov[j] * vscale;
            }
          }
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
}  // namespace uq

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
  CUtensorMap tmap, tmap_q;
  st = k_code_map(cache, records, 128, &tmap);
  if (st != UQ_OK) return st;
  st = q_map(q_fp8, (long long)batch * cfg->num_q_heads, 128, &tmap_q);
  if (st != UQ_OK) return st;
  const float score_scale = resolved_sm_scale(cfg) * 1.4426950408889634f;
  int sm_count = 0;
  st = current_device_sms(&sm_count);
  if (st != UQ_OK) return st;
  const long long total = (long long)((batch + kNS - 1) / kNS) * cfg->num_kv_heads * (prefix_len / 128);
  const long long slots = (long long)sm_count * UQ_CTAS_PER_SM;
  const dim3 grid((unsigned)(total < slots ? total : slots));   // one wave, one balanced tile range per CTA
  st = opt_in_dynamic_smem((const void*)decode_prefix_kernel, kSmemBytes, "decode_prefix: cudaFuncSetAttribute");
  if (st != UQ_OK) return st;
  return check_cuda(launch_pdl(decode_prefix_kernel, grid, dim3(kThreads), (size_t)kSmemBytes, (cudaStream_t)stream, tmap,
                               tmap_q, (const uint8_t*)cache, block_tables, (int)max_pages, (int)(prefix_len / 128),
                               (int)batch, (int)cfg->num_q_heads, (int)cfg->num_kv_heads, (int)num_splits, score_scale,
                               partial_acc, partial_ml),
                    "uq_decode_prefix_attention launch");
}
