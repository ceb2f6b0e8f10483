// uq_decode.cu — paged split-K decode attention over the FP4+UE8M0 cache: Alg. 1 "Decode"
// l.7-8 of arxiv/paper_2606_20474 (Eq.(1) :104).  Paging / split-K / partial
// format follow include/uq.h.
//
// Design: one CTA per (sequence, kv head, split); each of its warps is an
// independent stream processor over 16-token page records:
//   * lane 0 brings whole 2176-byte records into a per-warp shared-memory ring with
//     cp.async.bulk + mbarrier (no CTA-wide barrier in the loop);
//   * S^T[16 tok x 8 heads] = Kcodes . Q^T on tensor cores (mma.sync m16n8k32 e4m3): the FP4
//     codes become E4M3 bytes by pure bit placement (E2M1 value * 2^-6 is an E4M3 bit pattern,
//     subnormals included), the FP8 query fragments are loaded once per CTA ("hoisted",
//     PAPER.md:285), products are exact, and the UE8M0 group scale (one MMA k-step = one
//     32-channel group) is applied to the fp32 accumulator: S += 2^(byte-127) * acc;
//   * online softmax in fp32 with a LAZY reference maximum (rescale only when a score exceeds
//     the reference by more than 8 in log2 units);
//   * O^T[128 d x 8 heads] += Vhat^T . P^T (mma.sync m16n8k16 f16): token-pair-interleaved V
//     codes convert with cvt.rn.f16x2.e2m1x2 straight into A fragments, V scales are applied as
//     exact power-of-two fp16 multipliers relative to a running reference exponent.
// Every K/V byte is read from HBM once and touched by exactly one warp.
#include <cuda_fp16.h>

#include "uq_common.cuh"

namespace uq {
namespace {

constexpr int kWarps = 4;
constexpr int kStages = 4;
constexpr int kHeadStride = 132;  // padded fp32 row (128 + 4) of the CTA combine staging
constexpr unsigned kFull = 0xffffffffu;

// ---------------------------------------------------------------- PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ uint4 lds128(uint32_t a) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
  return v;
}
__device__ __forceinline__ uint2 lds64(uint32_t a) {
  uint2 v;
  asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a));
  return v;
}
__device__ __forceinline__ float ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel) {
  uint32_t d;
  asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));
  return d;
}
__device__ __forceinline__ uint32_t max_u16x2(uint32_t a, uint32_t b) {
  uint32_t d;
  asm("max.u16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
  return d;
}
__device__ __forceinline__ uint32_t pack_f16x2(float lo, float hi) {
  uint32_t d;
  asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
  return d;
}
__device__ __forceinline__ uint32_t movm_trans(uint32_t a) {
  uint32_t d;
  asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(d) : "r"(a));
  return d;
}
__device__ __forceinline__ uint32_t hmul2(uint32_t a, uint32_t b) {
  uint32_t d;
  asm("mul.rn.f16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
  return d;
}
// four packed byte pairs of E2M1 codes -> four f16x2 registers (low nibble -> low half)
__device__ __forceinline__ void cvt_e2m1x8(uint32_t w, uint32_t (&h)[4]) {
  asm("{\n"
      ".reg .b8 b0, b1, b2, b3;\n"
      "mov.b32 {b0, b1, b2, b3}, %4;\n"
      "cvt.rn.f16x2.e2m1x2 %0, b0;\n"
      "cvt.rn.f16x2.e2m1x2 %1, b1;\n"
      "cvt.rn.f16x2.e2m1x2 %2, b2;\n"
      "cvt.rn.f16x2.e2m1x2 %3, b3;\n"
      "}\n" : "=r"(h[0]), "=r"(h[1]), "=r"(h[2]), "=r"(h[3]) : "r"(w));
}
__device__ __forceinline__ void mma_e4m3(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                         uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k32.row.col.f32.e4m3.e4m3.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, "
               "{%10,%11,%12,%13};"
               : "=f"(d[0]), "=f"(d[1]), "=f"(d[2]), "=f"(d[3])
               : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1), "f"(0.f), "f"(0.f), "f"(0.f), "f"(0.f));
}
__device__ __forceinline__ void mma_f16(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                        uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, "
               "{%0,%1,%2,%3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
               : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

// E2M1 nibbles -> E4M3 bytes holding value * 2^-6:  byte = sign<<7 | (e1 e0 m)<<2.
// lo: the four low nibbles of w (even channels), hi: the four high nibbles (odd channels).
__device__ __forceinline__ uint32_t e2m1_lo_to_e4m3(uint32_t w) {
  return ((w << 2) & 0x1C1C1C1Cu) | ((w << 4) & 0x80808080u);
}
__device__ __forceinline__ uint32_t e2m1_hi_to_e4m3(uint32_t w) {
  return ((w >> 2) & 0x1C1C1C1Cu) | (w & 0x80808080u);
}
// fp32 2^(byte-127) for byte `i` of word w (byte 0 -> +0.0, which is what an all-zero group needs)
template <int I>
__device__ __forceinline__ float ue8m0_to_f32(uint32_t w) {
  const uint32_t bits = (I < 3 ? (w << (23 - 8 * I)) : (w >> 1)) & 0x7F800000u;
  return __uint_as_float(bits);
}

// ---------------------------------------------------------------- the kernel
// NT = number of 8-head tiles (1 for GQA group <= 8, 2 for <= 16).
template <int NT>
__global__ void __launch_bounds__(kWarps * 32, 3)
decode_kernel(const uint8_t* __restrict__ q_fp8, const uint8_t* __restrict__ cache,
              const int32_t* __restrict__ block_tables, int max_pages,
              const int32_t* __restrict__ seq_lens, int Hq, int Hkv, int num_splits,
              float score_scale /* sm_scale * log2(e) * 2^6 */,
              float* __restrict__ partial_acc, float* __restrict__ partial_ml) {
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ __align__(8) uint64_t s_bar[kWarps][kStages];
  __shared__ float s_m[kWarps][16];
  __shared__ float s_l[kWarps][16];
  __shared__ int s_e[kWarps];

  const int split = blockIdx.x, kvh = blockIdx.y, b = blockIdx.z;
  const int G = Hq / Hkv;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int g = lane >> 2, c = lane & 3;

  const int L = seq_lens[b];
  const int n_pages = (L + kPage - 1) / kPage;
  const int pps = (n_pages + num_splits - 1) / num_splits;
  const int p0 = split * pps;
  const int p1 = min(p0 + pps, n_pages);
  const long long row0 = ((long long)b * Hq + (long long)kvh * G) * num_splits + split;  // + head*num_splits
  if (p0 >= p1) {  // empty split: (m, l) = (-inf, 0); acc is never read by the merge
    if (threadIdx.x < G) {
      float2* ml = reinterpret_cast<float2*>(partial_ml) + row0 + (long long)threadIdx.x * num_splits;
      *ml = make_float2(-INFINITY, 0.f);
    }
    return;
  }

  // ---- hoisted FP8 query fragments (B operand of S^T = K Q^T)
  uint32_t qb[NT][4][2];
#pragma unroll
  for (int nt = 0; nt < NT; ++nt) {
    const int head = 8 * nt + g;
    const uint8_t* qrow = q_fp8 + ((long long)b * Hq + (long long)kvh * G + head) * kHeadDim;
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
      uint2 w = make_uint2(0u, 0u);
      if (head < G) w = *reinterpret_cast<const uint2*>(qrow + 32 * ks + 8 * c);
      qb[nt][ks][0] = prmt(w.x, w.y, 0x6420);  // even channels 8c+{0,2,4,6}  <-> k = 4c+i
      qb[nt][ks][1] = prmt(w.x, w.y, 0x7531);  // odd channels               <-> k = 16+4c+i
    }
  }

  // ---- per-warp page pipeline
  uint8_t* ring = smem + (size_t)warp * kStages * kRecordBytes;
  const uint32_t ring_u32 = smem_u32(ring);
  const uint32_t bar_u32 = smem_u32(&s_bar[warp][0]);
  if (lane == 0) {
#pragma unroll
    for (int s = 0; s < kStages; ++s) mbar_init(bar_u32 + 8 * s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncwarp();
  const int n_my = (p1 - p0 - warp + kWarps - 1) / kWarps;  // pages p0+warp, p0+warp+kWarps, ...
  const int32_t* bt = block_tables + (long long)b * max_pages;
  const uint8_t* cache_h = cache + (long long)kvh * kRecordBytes;
  const long long page_stride = (long long)Hkv * kRecordBytes;

  // block-table window: lane j holds the physical page of this warp's page index (32*win + j)
  int bt_win = 0;
  int bt_reg = (lane < n_my) ? bt[p0 + warp + kWarps * lane] : 0;
  auto issue = [&](int i) {  // all lanes call; lane 0 issues the copy of warp-page i
    if ((i >> 5) != bt_win) {
      bt_win = i >> 5;
      const int j = 32 * bt_win + lane;
      bt_reg = (j < n_my) ? bt[p0 + warp + kWarps * j] : 0;
    }
    const int page = __shfl_sync(kFull, bt_reg, i & 31);
    if (lane == 0) {
      const int st = i % kStages;
      mbar_expect_tx(bar_u32 + 8 * st, kRecordBytes);
      bulk_g2s(ring_u32 + st * kRecordBytes, cache_h + (long long)page * page_stride, kRecordBytes,
               bar_u32 + 8 * st);
    }
  };
  for (int i = 0; i < kStages && i < n_my; ++i) issue(i);

  // ---- running state
  float O[8][NT][4];
#pragma unroll
  for (int mt = 0; mt < 8; ++mt)
#pragma unroll
    for (int nt = 0; nt < NT; ++nt)
#pragma unroll
      for (int j = 0; j < 4; ++j) O[mt][nt][j] = 0.f;
  float mref[NT][2], lsum[NT][2];
#pragma unroll
  for (int nt = 0; nt < NT; ++nt) {
    mref[nt][0] = mref[nt][1] = -INFINITY;
    lsum[nt][0] = lsum[nt][1] = 0.f;
  }
  // Reference UE8M0 byte for V.  A group with scale byte B enters the PV product as
  // code * 2^(B - eref + 13) in fp16 (exact for B >= eref - 27, flushed to zero below), so the
  // largest value is 6 * 2^13 < 65504; eref >= 28 keeps B - (eref - 28) a valid exponent field.
  int eref = 28;

  // ================================================================ main loop over pages
  for (int i = 0; i < n_my; ++i) {
    const int st = i % kStages;
    const uint32_t rec = ring_u32 + st * kRecordBytes;
    mbar_wait(bar_u32 + 8 * st, (i / kStages) & 1);

    const uint4 kA = lds128(rec + kOffKCodes + 64 * g + 16 * c);        // token g,   groups 0..3
    const uint4 kB = lds128(rec + kOffKCodes + 64 * (g + 8) + 16 * c);  // token g+8
    uint2 ksc = lds64(rec + kOffKScales + 8 * g);                       // scale words of g, g+8
    const uint4 v0 = lds128(rec + kOffVCodes + 16 * lane);              // d tiles 0..3
    const uint4 v1 = lds128(rec + kOffVCodes + 512 + 16 * lane);        // d tiles 4..7
    uint4 vsc = lds128(rec + kOffVScales + 16 * c);                     // V scales of this lane's 4 tokens

    // tokens past the sequence end (last page only): neutralise their scales, mask their scores
    const int page_idx = p0 + warp + kWarps * i;
    const int n_valid = L - page_idx * kPage;  // >= 1
    const bool partial = n_valid < kPage;
    if (partial) {
      if (g >= n_valid) ksc.x = 0u;
      if (g + 8 >= n_valid) ksc.y = 0u;
      const uint32_t mA0 = (2 * c < n_valid) ? 0x0000FFFFu : 0u, mB0 = (2 * c + 1 < n_valid) ? 0xFFFF0000u : 0u;
      const uint32_t mA1 = (2 * c + 8 < n_valid) ? 0x0000FFFFu : 0u, mB1 = (2 * c + 9 < n_valid) ? 0xFFFF0000u : 0u;
      vsc.x &= (mA0 | mB0);
      vsc.y &= (mA0 | mB0);
      vsc.z &= (mA1 | mB1);
      vsc.w &= (mA1 | mB1);
    }

    // ---------------- S^T = K Q^T, one MMA k-step per 32-channel group, scale on the accumulator
    float S[NT][4];
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) S[nt][0] = S[nt][1] = S[nt][2] = S[nt][3] = 0.f;
    const uint32_t kAw[4] = {kA.x, kA.y, kA.z, kA.w};
    const uint32_t kBw[4] = {kB.x, kB.y, kB.z, kB.w};
    const float sA[4] = {ue8m0_to_f32<0>(ksc.x), ue8m0_to_f32<1>(ksc.x), ue8m0_to_f32<2>(ksc.x), ue8m0_to_f32<3>(ksc.x)};
    const float sB[4] = {ue8m0_to_f32<0>(ksc.y), ue8m0_to_f32<1>(ksc.y), ue8m0_to_f32<2>(ksc.y), ue8m0_to_f32<3>(ksc.y)};
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
      const uint32_t a0 = e2m1_lo_to_e4m3(kAw[ks]), a1 = e2m1_lo_to_e4m3(kBw[ks]);
      const uint32_t a2 = e2m1_hi_to_e4m3(kAw[ks]), a3 = e2m1_hi_to_e4m3(kBw[ks]);
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) {
        float acc[4];
        mma_e4m3(acc, a0, a1, a2, a3, qb[nt][ks][0], qb[nt][ks][1]);
        S[nt][0] = fmaf(acc[0], sA[ks], S[nt][0]);
        S[nt][1] = fmaf(acc[1], sA[ks], S[nt][1]);
        S[nt][2] = fmaf(acc[2], sB[ks], S[nt][2]);
        S[nt][3] = fmaf(acc[3], sB[ks], S[nt][3]);
      }
    }
    // log2-domain scores; S[nt][0..1]: token g, heads 8nt+2c, +1;  S[nt][2..3]: token g+8
    bool exceed = false;
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        float x = S[nt][j] * score_scale;
        if (partial && ((j < 2 ? g : g + 8) >= n_valid)) x = -INFINITY;
        S[nt][j] = x;
        exceed |= x > mref[nt][j & 1] + 8.0f;
      }
    }
    if (__any_sync(kFull, exceed)) {  // rare: raise the reference maximum, rescale O and l
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) {
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          float mx = fmaxf(S[nt][j], S[nt][j + 2]);
          mx = fmaxf(mx, __shfl_xor_sync(kFull, mx, 4));
          mx = fmaxf(mx, __shfl_xor_sync(kFull, mx, 8));
          mx = fmaxf(mx, __shfl_xor_sync(kFull, mx, 16));
          const float mnew = fmaxf(mref[nt][j], mx);
          const float f = (mref[nt][j] == -INFINITY) ? 0.f : ex2(mref[nt][j] - mnew);
          mref[nt][j] = mnew;
          lsum[nt][j] *= f;
#pragma unroll
          for (int mt = 0; mt < 8; ++mt) {
            O[mt][nt][j] *= f;
            O[mt][nt][j + 2] *= f;
          }
        }
      }
    }
    // P = 2^(x - mref); accumulate l; pack to f16 and transpose into B fragments of P^T
    uint32_t pb[NT][2];
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
      const float p0v = ex2(S[nt][0] - mref[nt][0]), p1v = ex2(S[nt][1] - mref[nt][1]);
      const float p2v = ex2(S[nt][2] - mref[nt][0]), p3v = ex2(S[nt][3] - mref[nt][1]);
      lsum[nt][0] += p0v + p2v;
      lsum[nt][1] += p1v + p3v;
      pb[nt][0] = movm_trans(pack_f16x2(p0v, p1v));  // -> (tokens 2c,2c+1 ; head g)
      pb[nt][1] = movm_trans(pack_f16x2(p2v, p3v));  // -> (tokens 2c+8,2c+9 ; head g)
    }

    // ---------------- V scales -> fp16 power-of-two multipliers relative to eref
    // word (p, hf) holds bytes [tokA gr=2hf, tokA gr=2hf+1, tokB gr=2hf, tokB gr=2hf+1]
    const uint32_t vw[4] = {vsc.x, vsc.y, vsc.z, vsc.w};
    uint32_t vraw[2][4];  // [pair][group] as u16x2 (byte of token A, byte of token B)
#pragma unroll
    for (int p = 0; p < 2; ++p)
#pragma unroll
      for (int gr = 0; gr < 4; ++gr) vraw[p][gr] = prmt(vw[2 * p + (gr >> 1)], 0u, (gr & 1) ? 0x4341u : 0x4240u);
    {
      uint32_t mx = vraw[0][0];
#pragma unroll
      for (int p = 0; p < 2; ++p)
#pragma unroll
        for (int gr = 0; gr < 4; ++gr) mx = max_u16x2(mx, vraw[p][gr]);
      const int top = max((int)(mx & 0xFFFFu), (int)(mx >> 16));
      if (__any_sync(kFull, top > eref)) {  // rare: raise the reference exponent, rescale O
        int e = top;
        e = max(e, __shfl_xor_sync(kFull, e, 1));
        e = max(e, __shfl_xor_sync(kFull, e, 2));
        e = max(e, eref);
        const int fe = 127 + eref - e;  // 2^(eref - e); flushes to 0 beyond fp32 range
        const float f = fe > 0 ? __uint_as_float((uint32_t)fe << 23) : 0.f;
        eref = e;
#pragma unroll
        for (int mt = 0; mt < 8; ++mt)
#pragma unroll
          for (int nt = 0; nt < NT; ++nt)
#pragma unroll
            for (int j = 0; j < 4; ++j) O[mt][nt][j] *= f;
      }
    }
    const uint32_t kbase = (uint32_t)(eref - 28) * 0x00010001u;
    uint32_t vmul[2][4];
#pragma unroll
    for (int p = 0; p < 2; ++p)
#pragma unroll
      for (int gr = 0; gr < 4; ++gr) vmul[p][gr] = (max_u16x2(vraw[p][gr], kbase) - kbase) << 10;  // fp16 2^(byte-eref+13); 0 below 2^-14

    // ---------------- O^T += Vhat^T P^T
    const uint32_t vword[8] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w};
#pragma unroll
    for (int mt = 0; mt < 8; ++mt) {
      uint32_t h[4];
      cvt_e2m1x8(vword[mt], h);  // h0: pair0 d=16mt+g, h1: pair0 d+8, h2: pair1 d, h3: pair1 d+8
      const uint32_t a0 = hmul2(h[0], vmul[0][mt >> 1]), a1 = hmul2(h[1], vmul[0][mt >> 1]);
      const uint32_t a2 = hmul2(h[2], vmul[1][mt >> 1]), a3 = hmul2(h[3], vmul[1][mt >> 1]);
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) mma_f16(O[mt][nt], a0, a1, a2, a3, pb[nt][0], pb[nt][1]);
    }

    // ---------------- release the stage and refill it
    __syncwarp();
    if (i + kStages < n_my) issue(i + kStages);
  }

  // ================================================================ CTA combine of the warps
  // l: sum the lanes that share the same heads (same c) over g
#pragma unroll
  for (int nt = 0; nt < NT; ++nt)
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      float v = lsum[nt][j];
      v += __shfl_xor_sync(kFull, v, 4);
      v += __shfl_xor_sync(kFull, v, 8);
      v += __shfl_xor_sync(kFull, v, 16);
      lsum[nt][j] = v;
    }
  if (g == 0) {
#pragma unroll
    for (int nt = 0; nt < NT; ++nt)
#pragma unroll
      for (int j = 0; j < 2; ++j) s_m[warp][8 * nt + 2 * c + j] = mref[nt][j];
  }
  if (lane == 0) s_e[warp] = eref;
  __syncthreads();  // also: every warp is done with its ring, which becomes the staging buffer

  int emax = s_e[0];
#pragma unroll
  for (int w = 1; w < kWarps; ++w) emax = max(emax, s_e[w]);
  const int fe = 127 + eref - emax;
  const float fexp = fe > 0 ? __uint_as_float((uint32_t)fe << 23) : 0.f;
  float* stage = reinterpret_cast<float*>(smem) + (size_t)warp * 16 * kHeadStride;
#pragma unroll
  for (int nt = 0; nt < NT; ++nt)
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      const int head = 8 * nt + 2 * c + j;
      float M = s_m[0][head];
#pragma unroll
      for (int w = 1; w < kWarps; ++w) M = fmaxf(M, s_m[w][head]);
      const float fm = (mref[nt][j] == -INFINITY) ? 0.f : ex2(mref[nt][j] - M);
      if (g == 0) s_l[warp][head] = lsum[nt][j] * fm;
      const float f = fm * fexp;
#pragma unroll
      for (int mt = 0; mt < 8; ++mt) {
        stage[head * kHeadStride + 16 * mt + g] = O[mt][nt][j] * f;
        stage[head * kHeadStride + 16 * mt + g + 8] = O[mt][nt][j + 2] * f;
      }
    }
  __syncthreads();

  // sum over warps, undo the reference exponent, write the split's partial (coalesced)
  const int ve = emax - 13;  // true value = acc * 2^(emax - 13 - 127)
  const float vscale = __uint_as_float((uint32_t)max(ve, 0) << 23) * (ve < 0 ? 0.f : 1.f);
  const float* stg = reinterpret_cast<const float*>(smem);
  for (int idx = threadIdx.x; idx < G * kHeadDim; idx += kWarps * 32) {
    const int head = idx >> 7, d = idx & 127;
    float v = 0.f;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) v += stg[(w * 16 + head) * kHeadStride + d];
    partial_acc[(row0 + (long long)head * num_splits) * kHeadDim + d] = v * vscale;
  }
  if (threadIdx.x < G) {
    const int head = threadIdx.x;
    float M = s_m[0][head], l = 0.f;
#pragma unroll
    for (int w = 1; w < kWarps; ++w) M = fmaxf(M, s_m[w][head]);
#pragma unroll
    for (int w = 0; w < kWarps; ++w) l += s_l[w][head];
    float2* ml = reinterpret_cast<float2*>(partial_ml) + row0 + (long long)head * num_splits;
    *ml = make_float2(M * 0.6931471805599453f, l);  // natural-log units
  }
}

}  // namespace
}  // namespace uq

extern "C" int32_t uq_decode_attention(const uq_config* cfg, const void* q_fp8, const void* cache,
                                       int64_t num_pages, const int32_t* block_tables, int32_t max_pages,
                                       const int32_t* seq_lens, int32_t batch, int32_t num_splits,
                                       float* partial_acc, float* partial_ml, void* stream) {
  using namespace uq;
  int32_t st = check_config(cfg);
  if (st != UQ_OK) return st;
  if (!q_fp8 || !cache || !block_tables || !seq_lens || !partial_acc || !partial_ml || batch <= 0 ||
      num_splits <= 0 || max_pages <= 0 || num_pages <= 0) {
    set_error("decode: NULL pointer or non-positive size");
    return UQ_ERR_INVALID_ARG;
  }
  if (batch > 65535 || cfg->num_kv_heads > 65535) {
    set_error("decode: batch and num_kv_heads must be <= 65535");
    return UQ_ERR_INVALID_ARG;
  }
  if (((uintptr_t)cache & 15u) || ((uintptr_t)q_fp8 & 7u) || ((uintptr_t)partial_acc & 15u) ||
      ((uintptr_t)partial_ml & 7u)) {
    set_error("decode: misaligned pointer (cache 16 B, q_fp8 8 B, partial_acc 16 B, partial_ml 8 B)");
    return UQ_ERR_INVALID_ARG;
  }
  const int G = cfg->num_q_heads / cfg->num_kv_heads;
  const size_t ring = (size_t)kWarps * kStages * kRecordBytes;
  const size_t staging = (size_t)kWarps * 16 * kHeadStride * sizeof(float);
  const size_t smem = ring > staging ? ring : staging;
  const float score_scale = resolved_sm_scale(cfg) * 1.4426950408889634f * 64.0f;
  const dim3 grid((unsigned)num_splits, (unsigned)cfg->num_kv_heads, (unsigned)batch);
  cudaError_t e;
  if (G <= 8) {
    e = cudaFuncSetAttribute(decode_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return check_cuda(e, "decode: cudaFuncSetAttribute");
    decode_kernel<1><<<grid, kWarps * 32, smem, (cudaStream_t)stream>>>(
        (const uint8_t*)q_fp8, (const uint8_t*)cache, block_tables, max_pages, seq_lens, cfg->num_q_heads,
        cfg->num_kv_heads, num_splits, score_scale, partial_acc, partial_ml);
  } else {
    e = cudaFuncSetAttribute(decode_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return check_cuda(e, "decode: cudaFuncSetAttribute");
    decode_kernel<2><<<grid, kWarps * 32, smem, (cudaStream_t)stream>>>(
        (const uint8_t*)q_fp8, (const uint8_t*)cache, block_tables, max_pages, seq_lens, cfg->num_q_heads,
        cfg->num_kv_heads, num_splits, score_scale, partial_acc, partial_ml);
  }
  return check_cuda(cudaGetLastError(), "uq_decode_attention launch");
}
