/*
 * uq.h — C ABI of libuq.so: UltraQuant's data-parallel hot path on NVIDIA B200 (sm_100a).
 *
 * Implements Algorithm 1 of arxiv/paper_2606_20474 ("UltraQuant: 4-bit KV Caching for
 * Context-Heavy Agents"), /root/reference/PAPER.md:245-261:
 *
 *   Write  (l.1-5): K <- R*K (Walsh-Hadamard over head_dim; V unrotated); 32-channel groups;
 *                   per group m = max|x|, E = round(log2(c*m)) (UE8M0 exponent, byte = E+127);
 *                   per coordinate code = nearest level of x/2^E in
 *                   F = {0,+-.5,+-1,+-1.5,+-2,+-3,+-4,+-6} (E2M1); store 2 codes/byte + 1 scale
 *                   byte per group (17 B / 32 elements).
 *   Decode (l.6-8): Q <- cast_fp8_e4m3(R*Q); xhat = code * 2^(byte-127) (Eq.(1));
 *                   softmax(sm_scale * Q Khat^T) Vhat for every query head of a KV head.
 *
 * Paging, block tables, split-K and the merge are not in the paper; they follow
 * BASELINE.json's north_star.  Readings of everything the paper leaves open: DESIGN.md.
 *
 * CONVENTIONS
 *  - Every pointer is a DEVICE pointer owned by the caller unless it says "host".  The library
 *    never allocates, frees or keeps device memory, never synchronises the device, and only
 *    enqueues work on the caller's stream (a cudaStream_t passed as void*; NULL = legacy stream).
 *  - Every function returns a status code; no C++ exception crosses the boundary.
 *    uq_last_error_string() (host, thread-local) describes the last failure.
 *  - Arguments are validated on the host only.  Block-table entries outside [0, num_pages),
 *    seq_lens beyond max_pages*page_size, NaN/Inf inputs: undefined behaviour — unless
 *    UQ_FLAG_DEBUG_CHECKS is set (below), which validates the tables on the device first.
 *  - The library may be used on several devices of one process: a call runs on the CURRENT device
 *    (cudaSetDevice), which must own every pointer passed; per-device state (SM count, shared-memory
 *    opt-in of the kernels, TMA descriptors) is kept per device and guarded by mutexes.
 *  - Supported geometry in this version: head_dim in {64, 128, 256} (the head sizes the paper validates,
 *    PAPER.md:322), group_size = 32, page_size = 16, num_q_heads / num_kv_heads in 1..16, batch <= 2048 for
 *    uq_decode_attention (UQ_ERR_UNSUPPORTED otherwise).  head_dim 128 — the geometry of every BASELINE.json
 *    config — is the tuned path; at 64 and 256 uq_rotate_quantize_append runs its float64 kernel only (no float32
 *    fast path, no bulk kernel), uq_decode_attention the same CTA design re-sized, and
 *    uq_decode_prefix_attention / uq_calibrate_c return UQ_ERR_UNSUPPORTED.
 *  - GQA map: query head h reads KV head h / (num_q_heads/num_kv_heads).
 *
 * PHYSICAL CACHE LAYOUT (uint8), written out for head_dim 128; for head_dim D the record has 17 D bytes
 * (uq_cache_record_bytes) and the four regions are [0, 8D) K codes (token t at (D/2) t), [8D, 16D) V codes (word at
 * 8D + 4D (t>>3) + 128 (d>>5) + 4 (d&31)), [16D, 16D + D/2) K scales (token t's D/32 bytes at 16D + (D/32) t) and
 * [16D + D/2, 17D) V scales (token t, group g at 16D + D/2 + (D/4)(t>>3) + 8 g + (t&7)).
 * cache[num_pages][num_kv_heads][UQ_RECORD_BYTES]; the record
 * of (page p, kv head h) starts at byte (p*num_kv_heads + h)*2176 and holds 16 tokens with
 * exactly 4.25 bit/element and no padding.  The cache base must be 32-byte aligned (the K
 * codes are fetched by TMA as packed 4-bit tensors).  With t = token slot in the page
 * (0..15), d = channel (0..127), g = d / 32 (group):
 *
 *   [   0,1024)  K codes, LOGICAL order: token t at 64*t, byte j holds channel 2j in bits 0-3
 *                and channel 2j+1 in bits 4-7 (what Alg. 1 l.5 writes; the tensor cores read
 *                it directly as E2M1).
 *   [1024,2048)  V codes, token-major nibbles.  The 32-bit word at
 *                   1024 + 512*(t>>3) + 128*(d>>5) + 4*(d&31)
 *                holds channel d of the eight tokens 8*(t>>3) .. 8*(t>>3)+7; token t sits in
 *                bits 4*(t&7) .. 4*(t&7)+3.
 *   [2048,2112)  K scale bytes: token t's four group bytes (group 0 first) at 2048 + 4*t.
 *   [2112,2176)  V scale bytes: token t, group g at 2112 + 32*(t>>3) + 8*g + (t&7).
 *
 * tests/uq_layout.py holds an independent unpacker written from this description.
 */
#ifndef UQ_H_
#define UQ_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define UQ_OK 0
#define UQ_ERR_INVALID_ARG 1  /* null pointer, non-positive size, Hq % Hkv != 0, misaligned pointer */
#define UQ_ERR_UNSUPPORTED 2  /* geometry outside the supported set above */
#define UQ_ERR_WORKSPACE 3    /* reserved: no entry point takes a workspace (uq_decode_workspace_bytes reports 0) */
#define UQ_ERR_CUDA 4         /* launch / driver error */

#define UQ_RECORD_BYTES 2176  /* 16 tokens * (64 + 4 + 64 + 4) bytes */

/* uq_config.flags: keep uq_rotate_quantize_append on the one-warp-per-octet kernel even for prefill-sized calls
 * (the bytes written do not depend on it; tests use it to cover both kernels on the same inputs). */
#define UQ_FLAG_NO_BULK_APPEND 1u
/* uq_config.flags: debug mode.  uq_rotate_quantize_append, uq_decode_attention and uq_decode_prefix_attention first run a
 * small kernel over exactly the table entries and lengths the call is going to use — decode: 0 <= seq_lens[b] <=
 * max_pages*page_size and every entry of pages [0, ceil(seq_lens[b]/page_size)) inside [0, num_pages); append: cu_new
 * starts at 0, ends at total_new and does not decrease, seq_lens[b] + count fits the table, the entries of the pages
 * written are in range; shared prefix: the prefix entries are in range AND equal to sequence 0's — then copy a five-word
 * report to the host and SYNCHRONISE the stream (the one exception to "never synchronises"; such a call cannot be captured
 * into a CUDA graph).  On an offender the call returns UQ_ERR_INVALID_ARG, names the first one in uq_last_error_string()
 * and launches nothing else.  Without the flag none of this runs. */
#define UQ_FLAG_DEBUG_CHECKS 2u
/* uq_config.flags, read by uq_decode_attention only: a promise about what runs AHEAD of the call in its stream.  The
 * library's kernels are launched with programmatic stream serialization: a kernel's CTAs may become resident while the
 * kernel before it still runs and normally wait for it before they touch global memory.  With this flag the caller
 * guarantees that the work still running ahead (the step's uq_rotate_quantize_append and, before it, the previous step's
 * merge) writes nothing this call reads except q_fp8, the partial buffers and the LAST TWO pages of each sequence's
 * block-table range — i.e. the append adds at most 16 tokens per sequence, and seq_lens / block_tables were final before
 * it started.  The decode kernel then waits only where it could meet those writes (query tiles, tiles holding one of a
 * sequence's last two pages, every write of partials) and streams the rest of the cache under the append kernel: the
 * fill of its pipelines leaves the step's critical path.  Results are identical with and without the flag. */
#define UQ_FLAG_SMALL_APPEND_AHEAD 4u

typedef struct {
  int32_t num_q_heads;   /* e.g. 64 */
  int32_t num_kv_heads;  /* e.g. 4  */
  int32_t head_dim;      /* 128 */
  int32_t page_size;     /* 16 */
  int32_t group_size;    /* 32 */
  float c_k;             /* global constant c for keys   (0.156f); used as (double)c_k */
  float c_v;             /* global constant c for values (0.156f; same rule, reading G3) */
  float sm_scale;        /* softmax scale; 0 => 1/sqrt(head_dim) */
  uint32_t flags;        /* UQ_FLAG_* bits; unknown bits are an error */
} uq_config;

/* Host.  Static, thread-local description of the last error returned on this thread. */
const char* uq_last_error_string(void);

/* Host.  Bytes of one (page, kv_head) record: page_size*(d/2 + d/32)*2 = 17 d = 2176 at d = 128; 0 if unsupported. */
size_t uq_cache_record_bytes(const uq_config* cfg);

/* Host.  Device scratch uq_decode_attention / uq_decode_prefix_attention need beyond the caller's partial buffers for
 * `batch` sequences and `num_splits` slots: *bytes = 0 in this version — the schedule (tile prefix sums of up to 2048
 * sequences), the K / V rings, the operands and the accumulators live in shared memory and TMEM, which is why those
 * entry points take no workspace argument.  Kept so that a caller sizing its arena does not have to know that. */
int32_t uq_decode_workspace_bytes(const uq_config* cfg, int32_t batch, int32_t num_splits, size_t* bytes);

/*
 * Alg. 1 "Write" l.1-5 and "Decode" l.6: quantize-on-append.
 *
 *  k_new, v_new  bf16 [total_new, num_kv_heads, head_dim].  Rows cu_new[b] .. cu_new[b+1]-1 are
 *                the new tokens of sequence b, written at positions seq_lens[b] + j through
 *                block_tables[b][pos / page_size], slot pos % page_size.
 *  cu_new        int32 [batch+1], cu_new[0] = 0.       seq_lens  int32 [batch], lengths BEFORE
 *                the append (read-only: the caller advances them).
 *  block_tables  int32 [batch, max_pages].             cache: layout above, num_pages pages.
 *  total_new     host int: cu_new[batch] (rows in k_new / v_new); may be 0.
 *  q             bf16 [batch, num_q_heads, head_dim] or NULL.  If given, q_fp8 (uint8, same
 *                shape) receives cast_fp8_e4m3(R*q): OCP E4M3, round-to-nearest-even,
 *                saturating at +-448, zero stored as 0x00.
 *
 * Two kernels, one result: calls with on average >= 64 new tokens per sequence (and >= 1024 in all, k_new / v_new
 * 16-byte aligned) take the bulk kernel (one warp per page, rows staged in shared memory by TMA, the rotation
 * done in registers with two lanes per token); all other calls, and the partly covered first / last page of a bulk
 * call's ranges, one warp per aligned octet of positions.
 *
 * Every rounding decision (scale exponent, E2M1 code, E4M3 byte) is taken on float64 values of
 * the exactly-computed rotation (reading G1), so codes, scale bytes and q_fp8 are
 * bit-identical to the float64 oracle.  (A float32 fast path computes the same vector with a proven error bound
 * and accepts a decision only if the whole error interval lies on one side of every rounding boundary; any other
 * vector is redone in float64: the bytes written are those of the float64 path.)  Tokens of one sequence that share a V-code byte (slots
 * 2i, 2i+1) may arrive in one call or in successive calls on the same stream; two concurrent
 * calls must not append to the same page.  Appending to a page shared by several block tables
 * is the caller's error.
 */
int32_t uq_rotate_quantize_append(const uq_config* cfg, const void* k_new, const void* v_new,
                                  const int32_t* cu_new, const int32_t* seq_lens,
                                  const int32_t* block_tables, int32_t max_pages, int32_t batch,
                                  int32_t total_new, void* cache, int64_t num_pages,
                                  const void* q, void* q_fp8, void* stream);

/*
 * Alg. 1 "Decode" l.7-8 for one decode step, split-K over the sequence.
 *
 *  q_fp8        uint8 [batch, num_q_heads, head_dim] (E4M3 bytes of the rotated query).
 *  seq_lens     int32 [batch]: lengths INCLUDING any token appended in this step.
 *  num_splits   >= 1: the number of partial SLOTS per (sequence, query head).  The kernel cuts the
 *               128-token tiles of all (sequence, kv head) items of the call, taken one item after
 *               the other, into equal contiguous ranges, one per resident CTA (the same HBM traffic
 *               per CTA whatever the sequence lengths are); a range may end inside an item, and the
 *               CTAs that share an item fill consecutive slots of it, starting at slot 0.  Ranges are
 *               made longer when needed so that no item spans more than num_splits of them; slots
 *               an item does not use are written as empty.  With num_splits = 1 every item is
 *               processed whole by one CTA.  Which tokens a slot covers is therefore an
 *               implementation detail; uq_merge_splits needs only the format below.
 *               batch <= 2048 per call.
 *  partial_acc  float32 [batch, num_q_heads, num_splits, head_dim]
 *  partial_ml   float32 [batch, num_q_heads, num_splits, 2] = (m_s, l_s)
 *
 * Partial format: with z_t = sm_scale * q8 . khat_t (natural-log units),
 *     m_s   = a reference logit of split s (>= every z_t of the split minus 12*ln2; it need
 *             not be the exact maximum),  l_s = sum_t exp(z_t - m_s),
 *     acc_s = sum_t exp(z_t - m_s) * vhat_t   (unnormalised).
 * An empty split (a slot its item does not use, or any slot of a sequence of length 0) writes m_s = -inf, l_s = 0;
 * its acc_s row is NOT written and must not be read: a merge skips every slot with l_s = 0 (uq_merge_splits does),
 * it must not multiply a weight of 0 into the row (stale memory may hold NaN).
 *
 * Arithmetic: S = K Q^T by tcgen05.mma kind::mxf8f6f4.block_scale (E2M1 x E4M3 products exact,
 * UE8M0 group scales applied by the tensor core, fp32 accumulation in TMEM); exp in fp32
 * (ex2.approx); P and Vhat enter the PV product (tcgen05.mma kind::f16) as fp16, Vhat relative to
 * a running reference exponent (values more than 2^25 below the largest V scale seen so far
 * flush to zero); accumulation in fp32 in TMEM.
 *
 * Accuracy domain.  With p_t the softmax weights and A[h,d] = sum_t p_t |vhat[t,d]| the ABSOLUTE attention mass of an
 * output element, the merged output satisfies
 *     |out - ref| <= 2^-8 |ref| + 2^-10 A[h,d]        (ref = the float64 oracle on the same codes)
 * — bf16 output rounding, fp32 accumulation and ex2.approx in the first term, the fp16 rounding of P (2^-11 per term,
 * which cancelling terms do not cancel) in the second.  The north-star bound |out - ref| <= 2e-3 + 1e-2 |ref| is
 * therefore GUARANTEED for A <= 2 (values of unit scale, the case of every BASELINE.json config: A ~ 0.8 for N(0,1)
 * values) and for outputs that dominate their own mass (|ref| >= 0.2 A: peaked attention at any scale); it is not
 * guaranteed where terms much larger than 2 cancel to a small output (V scaled by 2^12 with diffuse attention:
 * measured errors of 0.05 on outputs of 1.3 with A = 279).  Softmax weights below 2^-24 of a split's reference weight
 * underflow in fp16 and are dropped from the numerator: harmless unless more than 2^-10 of a row's mass sits on such
 * tokens (a single token dominating > 10^4 others by exactly 2^24..2^25).  DESIGN.md "Tolerance" derives both.
 */
int32_t uq_decode_attention(const uq_config* cfg, const void* q_fp8, const void* cache,
                            int64_t num_pages, const int32_t* block_tables, int32_t max_pages,
                            const int32_t* seq_lens, int32_t batch, int32_t num_splits,
                            float* partial_acc, float* partial_ml, void* stream);

/*
 * Merge of split partials (exact reassociation of the softmax):
 *     M = max_s m_s;  out = sum_s e^(m_s-M) acc_s / sum_s e^(m_s-M) l_s,  cast to bf16 (RNE).
 * Splits with l_s = 0 are ignored; if all are empty (seq_len 0) the output row is zeros.
 *  out_bf16     bf16 [batch, num_q_heads, head_dim]
 */
int32_t uq_merge_splits(const uq_config* cfg, const float* partial_acc, const float* partial_ml,
                        int32_t batch, int32_t num_splits, void* out_bf16, void* stream);

/*
 * Shared-prefix ("cascade") decode: the first prefix_len tokens of ALL `batch` sequences are the same physical pages
 * (block_tables[b][p] is the same for every b and p < prefix_len / page_size: the caller's guarantee — the long
 * shared prompt of the paper's agent workloads).  Computes the partials of exactly those tokens
 * for every sequence, each 128-token tile staged, converted and multiplied once for 8 sequences at a time (16 for GQA groups <= 8); the
 * remaining tokens of a sequence go through uq_decode_attention with block_tables + prefix_len / page_size and
 * seq_lens - prefix_len, and uq_merge_splits2 combines the two sets.
 *  prefix_len   a positive multiple of 128, <= every sequence's length.      num_splits >= 2.
 *  partial_acc / partial_ml: as for uq_decode_attention, [batch, num_q_heads, num_splits, ...].
 * Arithmetic and error bound as uq_decode_attention.
 */
int32_t uq_decode_prefix_attention(const uq_config* cfg, const void* q_fp8, const void* cache,
                                   int64_t num_pages, const int32_t* block_tables, int32_t max_pages,
                                   int32_t batch, int32_t prefix_len, int32_t num_splits,
                                   float* partial_acc, float* partial_ml, void* stream);

/* uq_merge_splits over two sets of partials of the same rows (splits_a and splits_b slots per row). */
int32_t uq_merge_splits2(const uq_config* cfg, const float* acc_a, const float* ml_a, int32_t splits_a,
                         const float* acc_b, const float* ml_b, int32_t splits_b, int32_t batch,
                         void* out_bf16, void* stream);

/*
 * The objective of Eq.(2) on a grid of constants — "solved once, offline, on captured rotated key
 * activations" (:128).  For every c_j of the grid:
 *     sq_err[j] = sum over all elements z of (z - zhat_j(z))^2,        sq_norm[0] = sum z^2,
 * z = the rotated vector H x / sqrt(head_dim) if rotate != 0 (keys, Alg. 1 l.1), else x itself (values); m = the
 * absmax of z's 32-channel group;
 *     scale_mode 0:  zhat = s * q(z / s) with s = c_j * m and q the nearest level               (Eq.(2) as printed);
 *     scale_mode 1:  zhat = Eq.(1) of the code Alg. 1 l.3-5 stores: s = 2^round(log2(c_j * m)) (the deployed
 *                    quantiser; ties and clamping as in uq_rotate_quantize_append; E2M1 levels only);
 *     scale_mode 2:  s = c_j, no absmax: a fixed grid for vectors of known norm (the per-token-norm schemes the
 *                    paper compares with, Fig. 2).
 *  levels   NULL: F = {0,.5,1,1.5,2,3,4,6} (E2M1); else float32 [8] (device), ascending magnitudes of another
 *           symmetric codebook (uniform INT4: 0..7; Lloyd-Max centroids), nearest level, a tie to the smaller one.
 * E[.] of Eq.(2) is sq_err[j] / (n_vec * head_dim); the calibrated constant is the c_j with the smallest sq_err[j].
 *  x        bf16 [n_vec, head_dim], 8-byte aligned.     c_grid  float32 [n_c] (device), used as (double)c_j.
 *  sq_err   float64 [n_c], sq_norm float64 [1] (device): zeroed on the stream, then accumulated.
 * Arithmetic: float64 throughout, on the exactly computed rotation (the decisions are the oracle's); the sums are
 * accumulated per warp and combined with atomic float64 additions, so they equal the oracle's up to the order of
 * the additions (relative difference ~1e-13) and may differ in the last bits from run to run.
 */
int32_t uq_calibrate_c(const uq_config* cfg, const void* x, int64_t n_vec, int32_t rotate,
                       const float* c_grid, int32_t n_c, int32_t scale_mode, const float* levels,
                       double* sq_err, double* sq_norm, void* stream);

/*
 * COMPARISON CACHES — not UltraQuant: the two systems the paper compares it with at kernel level,
 * "hardware FP8 KV" and the BF16 baseline (PAPER.md:163; Table 3, :293-301), as paged caches under the same decode
 * CTA design, so that the paper's relative claims (4-bit reads about half the bytes of FP8, :188; the FP4 kernel within
 * 1.18 x of FP8 at 32K, :295-301) can be restated on B200.  The paper only names them; reading G19:
 *   UQ_KV_FP8_E4M3  K and V stored as OCP E4M3 bytes of the bf16 values themselves (no rotation, scale 1, round to
 *                   nearest even, saturating at 448, +0 only); the query is cast the same way (q_out of the append);
 *   UQ_KV_BF16      K and V stored as they are; the query is the bf16 query (the append does not touch it).
 * Record of (page, kv head): K rows [16 tokens][128 elements] then V [128 channels][16 tokens], 4096 / 8192 bytes; cache
 * base 128-byte aligned.  head_dim 128 only.  uq_baseline_decode_attention writes the partial format of
 * uq_decode_attention (same schedule, same num_splits meaning); uq_merge_splits finishes.  Scores: E4M3 x E4M3 by
 * kind::f8f6f4 / bf16 x bf16 by kind::f16, fp32 accumulation; P enters the PV product as fp16, V as fp16 (from E4M3:
 * exact) / bf16: the accuracy domain stated for uq_decode_attention applies.
 */
#define UQ_KV_FP8_E4M3 1
#define UQ_KV_BF16 2
size_t uq_baseline_record_bytes(const uq_config* cfg, int32_t kv_format);
/* k_new, v_new, cu_new, seq_lens, block_tables, total_new: as uq_rotate_quantize_append.  q bf16 [batch, Hq, 128] and
 * q_out uint8 [batch, Hq, 128] (FP8 only; both NULL or both given; ignored for BF16). */
int32_t uq_baseline_append(const uq_config* cfg, int32_t kv_format, const void* k_new, const void* v_new,
                           const int32_t* cu_new, const int32_t* seq_lens, const int32_t* block_tables,
                           int32_t max_pages, int32_t batch, int32_t total_new, void* cache, int64_t num_pages,
                           const void* q, void* q_out, void* stream);
/* q_enc: uint8 E4M3 [batch, Hq, 128] (FP8) or bf16 [batch, Hq, 128] (BF16); everything else as uq_decode_attention. */
int32_t uq_baseline_decode_attention(const uq_config* cfg, int32_t kv_format, const void* q_enc, const void* cache,
                                     int64_t num_pages, const int32_t* block_tables, int32_t max_pages,
                                     const int32_t* seq_lens, int32_t batch, int32_t num_splits,
                                     float* partial_acc, float* partial_ml, void* stream);

/*
 * ULTRA-TQ (the paper's Algorithm 2, "Calibrated LUT int4 KV encoding") — the codebook path that
 * UltraQuant replaces, as the third comparison cache (last item): rotated keys as 4-bit indices
 * into a 16-entry codebook C_K with a bf16 l2 norm per 32-channel block; values as 4-bit uniform codes with a bf16
 * (scale, zero) per block; dequantisation on read.  Readings of what Algorithm 2 leaves open: DESIGN.md G20.
 *   codebook_k   HOST float32 [16], finite, ascending: the algorithm's input C_K (for block coordinates scaled to unit
 *                l2 norm; calibrating it is out of scope).  Passed by value into the kernels.
 * Record of (page, kv head), 2432 bytes (uq_baseline_record_bytes(cfg, UQ_KV_ULTRA_TQ)), cache base 16-byte aligned:
 *   [0, 1024)      K indices: token slot t at 64 t, byte j = channels 2j (bits 0-3), 2j + 1 (bits 4-7)
 *   [1024, 1152)   K block norms: bf16, token t block g at 1024 + 8 t + 2 g
 *   [1152, 2176)   V codes: channel c at 1152 + 8 c, 32-bit word t >> 3; inside an octet token 2n in nibble n, token
 *                  2n + 1 in nibble n + 4
 *   [2176, 2432)   V block g at 2176 + 64 g: bf16 scale of tokens 0..15, then bf16 zero of tokens 0..15
 * uq_tq_append: Alg. 2 l.1-4 for the new rows (arguments as uq_rotate_quantize_append) and l.5 for the query: q bf16
 * [batch, Hq, 128] -> q_rot bf16 [batch, Hq, 128] = bf16(R q) (both NULL or both given).  Every decision in float64:
 * the cache image and q_rot are bit-exact against the oracle.  head_dim 128 only.
 * uq_tq_decode_attention: Alg. 2 l.6-8, partial format / schedule / num_splits of uq_decode_attention, uq_merge_splits
 * finishes.  K = bf16(bf16(C_K[idx]) * norm) through a 256-entry table in shared memory (a load per code byte), V =
 * bf16(scale * code + zero) with one rounding; both products bf16 x bf16 with fp32 accumulation, P as bf16 (as the BF16
 * comparison cache).
 */
#define UQ_KV_ULTRA_TQ 3
int32_t uq_tq_append(const uq_config* cfg, const float* codebook_k, const void* k_new, const void* v_new,
                     const int32_t* cu_new, const int32_t* seq_lens, const int32_t* block_tables, int32_t max_pages,
                     int32_t batch, int32_t total_new, void* cache, int64_t num_pages, const void* q, void* q_rot,
                     void* stream);
int32_t uq_tq_decode_attention(const uq_config* cfg, const float* codebook_k, const void* q_rot, const void* cache,
                               int64_t num_pages, const int32_t* block_tables, int32_t max_pages, const int32_t* seq_lens,
                               int32_t batch, int32_t num_splits, float* partial_acc, float* partial_ml, void* stream);

/*
 * Decode without allocation: uq_decode_attention followed by uq_merge_splits with the split partials held in a static
 * device array inside libuq.so instead of caller buffers — for callers that cannot call cudaMalloc (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid it).  The call itself allocates nothing either: no
 * cudaMalloc / cudaFree, no allocating library routine.
 *
 *  UQ_STATIC_SCRATCH_BYTES   size of that array: every GPU that loads the library holds this much until the process
 *                            exits.  A call needs  round_up(batch * num_q_heads * num_splits * head_dim * 4, 256)
 *                            + batch * num_q_heads * num_splits * 8  bytes (uq_decode_static_scratch_needed); config 2
 *                            (32 x 64 heads, head_dim 128) needs 1.02 MiB per split.  A call that needs more returns
 *                            UQ_ERR_UNSUPPORTED with the sizes in uq_last_error_string() and launches nothing.
 *  q_fp8, cache, num_pages, block_tables, max_pages, seq_lens, batch, num_splits, stream: as uq_decode_attention.
 *  out_bf16                  bf16 [batch, num_q_heads, head_dim], as uq_merge_splits.
 *
 * Result: identical to uq_decode_attention + uq_merge_splits with the same num_splits (the same kernels run).
 * The array is shared by EVERY call on a device and keeps the last call's contents.  Nothing in it has to start at
 * zero (the decode kernel writes (m, l) of every slot on every call and the merge reads an acc row only where l != 0),
 * so no clear is issued.  Calls that may overlap on the GPU — two streams, two threads, two graphs replayed
 * concurrently — RACE on it: serialise them on one stream or with events.  Each device has its own copy; the address
 * is looked up once per device (cudaGetSymbolAddress, with that device current) on the first call there.
 */
#define UQ_STATIC_SCRATCH_BYTES (32u << 20)
size_t uq_static_scratch_bytes(void);
int32_t uq_decode_static_scratch_needed(const uq_config* cfg, int32_t batch, int32_t num_splits, size_t* bytes);
int32_t uq_decode_attention_static(const uq_config* cfg, const void* q_fp8, const void* cache, int64_t num_pages,
                                   const int32_t* block_tables, int32_t max_pages, const int32_t* seq_lens,
                                   int32_t batch, int32_t num_splits, void* out_bf16, void* stream);

/* Host.  A num_splits (slot count) that lets uq_decode_attention balance `batch` sequences of about
 * `avg_seq_len` tokens over the current device with room for sequences twice that long (never below 1). */
int32_t uq_suggest_num_splits(const uq_config* cfg, int32_t batch, int32_t avg_seq_len);

/* Host.  The same with the longest sequence of the call known: enough slots for it at the balanced range length
 * (a skewed length mix — e.g. the private suffixes of a shared-prefix batch — otherwise stretches every CTA's range). */
int32_t uq_suggest_num_splits_max(const uq_config* cfg, int32_t batch, int32_t avg_seq_len, int32_t max_seq_len);

/* Host.  A slot count for uq_decode_prefix_attention (>= 2) that lets every SM take an equal tile range of the prefix. */
int32_t uq_suggest_prefix_splits(const uq_config* cfg, int32_t batch, int32_t prefix_len);

#ifdef __cplusplus
}
#endif
#endif /* UQ_H_ */
