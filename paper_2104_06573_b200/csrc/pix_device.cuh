// pix_device.cuh -- device helpers shared by the kernels (runs.cu, tile.cu, cluster.cu): the word decode
// and the calibration (a1, a2), the run bookkeeping (a3) and the union step.  One definition each.
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

// Union for long clusters (hook-and-descend walks chains that grow with the cluster): tile.cu's items of long runs, cluster.cu.  After
// Jaiganesh & Burtscher's ECL-CC: find the representatives with intermediate pointer jumping (plain stores are safe
// here because a label is only ever replaced by an ancestor and only roots are hooked), hook the larger root under
// the smaller one by compare-and-swap, go on from the winner's parent when the root was taken meanwhile.
__device__ __forceinline__ uint32_t representative(uint32_t* L, uint32_t v) {
  uint32_t curr = L[v];
  if (curr != v) {
    uint32_t prev = v, next;
    while (curr > (next = L[curr])) { L[prev] = next; prev = curr; curr = next; }
  }
  return curr;
}
static __device__ __noinline__ void unite_roots(uint32_t* L, uint32_t a, uint32_t b) {
  uint32_t ra = representative(L, a), rb = representative(L, b);
  while (ra != rb) {
    const uint32_t hi = ra > rb ? ra : rb, lo = ra > rb ? rb : ra;
    const uint32_t old = atomicCAS(L + hi, hi, lo);
    if (old == hi) break;
    ra = representative(L, old); rb = lo;
  }
}

}  // namespace pix
