// uq_sched.cuh — the balanced one-wave work schedule of the paged decode kernels (uq_decode.cu, uq_decode_cmp.cu):
// units (item, tile range) of 128-token tiles, computed identically by every CTA from seq_lens.  Device code only.
#pragma once
#include "uq_common.cuh"

namespace uq {
namespace {

constexpr int kTilePages = 8;                        // 128 tokens per tile

// ---------------------------------------------------------------- work schedule
// The tiles (128 tokens) of all (sequence, kv head) items form one sequence, item after item.  With
// num_splits >= 2 every CTA of the grid takes one contiguous range of `tpc` tiles of it (balanced: the
// same amount of HBM traffic per CTA whatever the lengths are); a range may end inside an item and
// start inside the next one, so a CTA works through a few UNITS (item, tile range), keeping its TMA /
// MMA pipelines running across unit boundaries.  The CTAs that share an item write consecutive partial
// slots of it; tpc is raised if needed so that no item spans more than num_splits CTAs.  With
// num_splits == 1 a unit is a whole item and CTA c takes items c, c + gridDim.x, ...
struct Unit {
  int b, kvh, p0, p1, n_tiles, tok_end, L;
  int slots_used;                                      // > 0 on the unit holding the item's last tile: slots the item uses
  long long row0;                                      // partial row of head 0 in this unit's slot: + head * num_splits
};
struct Cursor {
  int b, kvh, t, g, g1, it;                            // balanced: position (b, kvh, tile t), global tile g, range end g1; items: it
};

struct Sched {
  const int32_t* seq_lens;
  const int* pre;                                      // shared: pre[b] = tiles of sequences < b (per kv head)
  int B, Hq, Hkv, G, S, tpc, total;
  __device__ __forceinline__ int tiles(int b) const { return pre[b + 1] - pre[b]; }

  __device__ void start(Cursor& c) const {
    if (S == 1) { c.it = blockIdx.x; return; }
    c.g = min((int)blockIdx.x * tpc, total);
    c.g1 = min(c.g + tpc, total);
    if (c.g >= c.g1) return;
    int lo = 0, hi = B;                                // largest b with Hkv * pre[b] <= g (and tiles(b) > 0 follows)
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (Hkv * pre[mid] <= c.g) lo = mid; else hi = mid;
    }
    c.b = lo;
    const int off = c.g - Hkv * pre[lo], tb = tiles(lo);
    c.kvh = off / tb;
    c.t = off - c.kvh * tb;
  }
  // next unit of this CTA, false when there is none
  __device__ bool next(Cursor& c, Unit& u) const {
    int t0, t1, tb;
    if (S == 1) {
      for (;; c.it += gridDim.x) {
        if (c.it >= B * Hkv) return false;
        u.b = c.it / Hkv;
        tb = tiles(u.b);
        if (tb > 0) break;
      }
      u.kvh = c.it - u.b * Hkv;
      c.it += gridDim.x;
      t0 = 0; t1 = tb;
      u.slots_used = 1;
      u.row0 = ((long long)u.b * Hq + (long long)u.kvh * G) * S;
    } else {
      if (c.g >= c.g1) return false;
      u.b = c.b; u.kvh = c.kvh;
      tb = tiles(c.b);
      t0 = c.t;
      t1 = min(tb, t0 + (c.g1 - c.g));
      const int item_start = c.g - t0;                 // global tile index of the item's first tile
      const int slot = (int)blockIdx.x - item_start / tpc;
      u.slots_used = (t1 == tb) ? slot + 1 : 0;
      u.row0 = ((long long)u.b * Hq + (long long)u.kvh * G) * S + slot;
      c.g += t1 - t0;
      c.t = t1;
      if (t1 == tb) {                                  // on to the next item with tiles
        c.t = 0;
        if (++c.kvh == Hkv) {
          c.kvh = 0;
          do { ++c.b; } while (c.b < B && tiles(c.b) == 0);
        }
      }
    }
    u.L = seq_lens[u.b];
    const int n_pages = (u.L + kPage - 1) / kPage;
    u.p0 = kTilePages * t0;
    u.p1 = min(kTilePages * t1, n_pages);
    u.n_tiles = t1 - t0;
    u.tok_end = min(u.L, u.p1 * kPage);
    return true;
  }
};

}  // namespace
}  // namespace uq
