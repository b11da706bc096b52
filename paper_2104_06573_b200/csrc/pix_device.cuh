// pix_device.cuh -- device helpers shared by the cluster kernels (fused.cu, findrun.cu, cluster.cu): the word decode
// and the calibration (a1, a2), the union step, and the bucket position hash.  One definition each.
// PAPER.md:31 names the steps ("unpacks them, calibrates the individual pixels, and clusters the pixels on each
// detector module"); the arithmetic is fixed by readings S1-S10, S13 of DESIGN.md.  Nothing here is shared with oracle/.
#pragma once

#include "pix_common.cuh"

namespace pix {

// ------------------------------------------------------------------ a1: decode (S1-S6)
// With the pre-digested cabling entry (pix_common.cuh).  Returns the status; module/row/col are defined only for
// ST_OK.  fedbase = fed * 2048.
__device__ __forceinline__ uint32_t decode_word(const CabEntry* __restrict__ cab, uint32_t w, uint32_t fedbase,
                                                uint32_t& module, uint32_t& row, uint32_t& col) {
  const CabEntry e = __ldg(cab + fedbase + (w >> 21));  // index (fed*64 + link)*32 + roc
  const uint32_t dcol = (w >> 16) & 31u, pxid = (w >> 8) & 255u;
  const uint32_t bad = (e.x >> 16) & 0xFFu;
  uint32_t st = ST_OK;
  if (pxid >= 160u) st = ST_ERR_PXID;
  if (dcol >= 26u) st = ST_ERR_DCOL;
  if (bad) st = bad;
  if (w == 0u) st = ST_EMPTY;
  const int rr = (int)(pxid >> 1), cc = (int)(2u * dcol + (pxid & 1u));
  module = e.x & 0xFFFFu;
  row = (uint32_t)((int)(e.y & 0xFFu) + rr * ((int)e.y >> 24));
  col = (uint32_t)((int)((e.y >> 8) & 0x1FFu) + cc * ((int)e.x >> 24));
  return st;
}

// ------------------------------------------------------------------ a2: calibrate (S7)
// Four separately rounded binary32 RN operations (the _rn intrinsics are never contracted to FMA), then
// NaN/negative -> 0, clamp, truncate.
__device__ __forceinline__ int32_t calibrate(const Chunk& c, uint32_t adc, float2 gp) {
  const float f1 = __fsub_rn((float)adc, gp.y);
  const float f2 = __fmul_rn(f1, gp.x);
  const float f3 = __fmul_rn(f2, c.vcal_gain);
  const float f4 = __fadd_rn(f3, c.vcal_offset);
  if (!(f4 >= 0.0f)) return 0;
  return __float2int_rz(fminf(f4, c.max_e_f));
}

// sg / F (F is a power of two in both detector configurations: a shift)
__device__ __forceinline__ uint32_t div_F(const Chunk& c, uint32_t sg) { return c.F_shift != 0xFFFFFFFFu ? sg >> c.F_shift : sg / c.F; }

// a3: module_first / module_end are keyed by module id (S12).  Every run start also counts one run of its module:
// two or more runs make the event NONCONTIGUOUS (S11; offsets_kernel raises the flag).  None of the three atomics
// returns a value, so nothing waits for them.  key = event_rel << 16 | module, g = global word index.
__device__ __forceinline__ void run_start(const Chunk& c, uint32_t key, uint32_t g) {
  const uint32_t er = key >> 16, m = key & 0xFFFFu;
  atomicMin(c.module_first + ((size_t)(c.e0 + er) * c.M + m), g - c.segB[er * c.F]);
  atomicAdd(c.n_runs + ((size_t)er * c.M + m), 1u);
}
// true when module m of event er (launch-group relative) has more than one run: its range is not a run (S11)
__device__ __forceinline__ bool module_split(const Chunk& c, uint32_t er, uint32_t m) {
  return c.n_runs[(size_t)er * c.M + m] >= 2u;
}
__device__ __forceinline__ void run_end(const Chunk& c, uint32_t key, uint32_t g) {
  const uint32_t er = key >> 16, m = key & 0xFFFFu;
  atomicMax(c.module_end + ((size_t)(c.e0 + er) * c.M + m), g - c.segB[er * c.F] + 1u);
}

// A run the warp kernel cannot take goes to the warp-per-run kernel's list.  Every event may list at most M runs:
// an event with one run per module (S11) never needs more, and an event that asks for more is NONCONTIGUOUS, so
// the lists (E x M entries) cannot overflow and a bad event cannot take the room of its neighbours.
__device__ __forceinline__ void push_run(const Chunk& c, uint32_t* list, uint32_t ctl_count, uint32_t er, uint32_t m) {
  if (atomicAdd(c.ev_cnt + (size_t)er * EC_STRIDE + EC_PUSHED, 1u) >= c.M) return;
  const uint32_t i = atomicAdd(c.ctl + ctl_count, 1u);
  if (i < c.list_cap) list[i] = er * c.M + m;
}

// ------------------------------------------------------------------ union (S13, S14)
// Union on parent links L (L[x] <= x): hook-and-descend, no root searches.  For the edge (a, b) with hi = max,
// lo = min: p = atomicMin(&L[hi], lo).  p == hi: hi was a root and now hangs under lo; p == lo: already linked.
// Otherwise hi keeps the smaller of p and lo as its parent and the other one still has to be joined to it: go on
// with the edge (p, lo), whose larger end is below hi, so the descent ends.  Links only ever join digis of one
// component and point to smaller indices, so every component ends as one tree rooted at its lowest digi (S14).
__device__ __forceinline__ void hook(uint32_t* L, uint32_t a, uint32_t b) {
  bool done = a == b;  // single exit: the lanes of a warp reconverge after the loop
  while (!done) {
    const uint32_t hi = a > b ? a : b, lo = a > b ? b : a;
    const uint32_t p = atomicMin(L + hi, lo);
    if (p == hi || p == lo) done = true;
    else { a = p; b = lo; }
  }
}

// ------------------------------------------------------------------ position hash (S10, S13)
// 2^NB_LOG2 buckets of 4 slots: one 128-bit shared load per lookup and no probing loop on the common path.
// h = key * HASH_MUL mod 2^KEY_BITS is a bijection on the KEY_BITS-bit keys; bucket = top NB_LOG2 bits of h, tag =
// the rest, so (bucket, tag) names the key exactly.  A key whose home bucket is full goes to the next bucket(s)
// and records the displacement: slot = disp (2) | tag | digi (DIGI_BITS) | below_threshold (1).  Slots of a bucket
// fill in order and are never emptied; equal keys meet in one slot and keep the lowest digi (S10: first index wins).
template <uint32_t KEY_BITS, uint32_t NB_LOG2, uint32_t DIGI_BITS>
struct BucketHash {
  static constexpr uint32_t EMPTY = 0xFFFFFFFFu, HASH_MUL = 0x9E3779B1u, MAX_DISP = 3;
  static constexpr uint32_t KEY_MASK = (1u << KEY_BITS) - 1u, TAG_BITS = KEY_BITS - NB_LOG2, TAG_MASK = (1u << TAG_BITS) - 1u;
  static constexpr uint32_t NBUCKET = 1u << NB_LOG2, SLOTS = 4u * NBUCKET, SH = DIGI_BITS + 1u, DIGI_MASK = (1u << DIGI_BITS) - 1u;
  static_assert(2u + TAG_BITS + SH <= 32u, "slot: disp | tag | digi | below");

  static __device__ __forceinline__ uint32_t mix(uint32_t key) { return (key * HASH_MUL) & KEY_MASK; }
  // mixed value of key + d, given the mixed value of key
  static __device__ __forceinline__ uint32_t step(uint32_t h, uint32_t d) { return (h + d * HASH_MUL) & KEY_MASK; }

  // 0: inserted; 1: the key was already there (a duplicate pixel, S10); 2: no room within MAX_DISP buckets.
  // (Looking at the bucket first and aiming one atomicCAS at its first free slot was measured slower.)
  static __device__ __noinline__ uint32_t insert(uint32_t* tab, uint32_t key, uint32_t t, uint32_t below) {
    const uint32_t h = mix(key), tag = h & TAG_MASK;
    uint32_t p = (h >> TAG_BITS) * 4u, res = 2u;
#pragma unroll 1
    for (uint32_t i = 0; i < 4u * (MAX_DISP + 1u) && res == 2u; ++i, p = (p + 1u) & (SLOTS - 1u)) {
      const uint32_t want = ((i >> 2) << TAG_BITS) | tag, mine = (want << SH) | (t << 1) | below;
      const uint32_t old = atomicCAS(&tab[p], EMPTY, mine);
      if (old == EMPTY) res = 0u;
      else if ((old >> SH) == want) { atomicMin(&tab[p], mine); res = 1u; }  // same pixel: the lowest digi owns it
    }
    return res;
  }
  static __device__ __forceinline__ uint32_t match4(const uint4& e, uint32_t want) {
    uint32_t r = EMPTY;
    if ((e.w >> SH) == want) r = e.w;
    if ((e.z >> SH) == want) r = e.z;
    if ((e.y >> SH) == want) r = e.y;
    if ((e.x >> SH) == want) r = e.x;
    return r;
  }
  static __device__ __noinline__ uint32_t find_slow(const uint32_t* tab, uint32_t h) {
    const uint32_t tag = h & TAG_MASK;
    uint32_t b = h >> TAG_BITS, r = EMPTY;
    for (uint32_t i = 1; i <= MAX_DISP && r == EMPTY; ++i) {  // the buckets after the (full) home bucket
      b = (b + 1u) & (NBUCKET - 1u);
      const uint4 e = *reinterpret_cast<const uint4*>(&tab[b * 4u]);
      r = match4(e, (i << TAG_BITS) | tag);
      if (e.w == EMPTY) break;
    }
    return r;
  }
  // slot contents of the key whose mixed value is h, or EMPTY
  static __device__ __forceinline__ uint32_t find(const uint32_t* tab, uint32_t h) {
    const uint4 e = *reinterpret_cast<const uint4*>(&tab[(h >> TAG_BITS) * 4u]);
    uint32_t r = match4(e, h & TAG_MASK);
    if (r == EMPTY && e.w != EMPTY) r = find_slow(tab, h);  // home bucket full, no match (rare): displaced keys
    return r;
  }
  // the home bucket only; full = the bucket has no free slot, so a key that is not in it may sit in the next buckets
  static __device__ __forceinline__ uint32_t find_home(const uint32_t* tab, uint32_t h, bool& full) {
    const uint4 e = *reinterpret_cast<const uint4*>(&tab[(h >> TAG_BITS) * 4u]);
    const uint32_t r = match4(e, h & TAG_MASK);
    full = r == EMPTY && e.w != EMPTY;
    return r;
  }
  static __device__ __forceinline__ uint32_t digi(uint32_t e) { return (e >> 1) & DIGI_MASK; }
  static __device__ __forceinline__ bool live(uint32_t e) { return e != EMPTY && !(e & 1u); }
};

}  // namespace pix
