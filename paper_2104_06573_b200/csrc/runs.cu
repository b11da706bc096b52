// runs.cu -- a3 of the Clusters path ("clusters the pixels on each detector module": the module
// boundaries come first) as a streaming pre-pass, and the packing of module runs into work items for the tile
// kernel (tile.cu).  DESIGN.md S11, S12.
//
// runs_kernel: a warp walks ranges of sixteen 128-word chunks, two chunks at a time with eight consecutive words per
// lane (two 128-bit loads, the next pair's loads in flight meanwhile) while they lie in one (event, FED) segment and
// every word is decodable, else one chunk with four words per lane.  A word is decoded as
// far as its status and module (cabling gather only); a decodable word starts a run when its (event, module) differs
// from the previous decodable word's (when all 128 words of the chunk are decodable, the usual case, that is the
// word before it: one shuffle; otherwise a ballot / find-last-set scan).  Output: one start bit per word (bit g - T0
// of sbits, T0 = first word of the launch group rounded down to 128; the lanes' nibbles are folded into four words by
// three shuffles), module_first / module_end / the per-module run count (run_start, run_end), and one flag per chunk:
// every word decodable and the words of a run strictly ascending in (link, roc, dcol, pxid) -- read-out order, in which
// no pixel comes twice (tile.cu then skips its search for duplicates).
// The previous decodable word before a range is searched backwards, 32 words at a time, never beyond the start of the
// event (an earlier event's word never continues a run; segfill_kernel closes every event's last run).
//
// pack_kernel: one warp per event walks the event's start bits (staged in shared memory) and cuts it into items: maximal stretches of whole
// runs of at most ITEM_WIN words (greedy: the next item starts at the last run start inside the window), at most
// ITEM_RUNS runs each.  A run longer than TILE_WORDS words is cut into equal pieces that the tile kernel only decodes;
// the first piece carries ITEM_LONG_HEAD and the tile kernel hands the run to the block-per-run kernel (cluster.cu).
// An event is cut at up to seven run starts into pieces that different warps pack (the chain of a piece is short); any
// two consecutive items of a piece cover more than ITEM_WIN2 words, which bounds the item list.
// Nothing here is shared with oracle/.
#include "pix_common.cuh"
#include "pix_device.cuh"

namespace pix {

namespace {

constexpr uint32_t HC = CHUNK_WORDS, FULL = 0xFFFFFFFFu, NOKEY = 0xFFFFFFFFu;
constexpr uint32_t RANGE = 16;  // chunks a warp walks in one go (the look-back is done once per range)

// (event, module) of a decodable word, NOKEY otherwise (S4-S6: the same checks as decode_word, without the position)
__device__ __forceinline__ uint32_t run_key(const CabEntry* __restrict__ cab, uint32_t w, uint32_t fedbase, uint32_t er) {
  const uint32_t ex = __ldg(reinterpret_cast<const uint32_t*>(cab + fedbase + (w >> 21)));  // .x: module | bad << 16 | ...
  const bool ok = !(ex & 0xFF0000u) && ((w >> 16) & 31u) < 26u && ((w >> 8) & 255u) < 160u && w != 0u;
  return ok ? ((er << 16) | (ex & 0xFFFFu)) : NOKEY;
}

__global__ void __launch_bounds__(256, 4) runs_kernel(const __grid_constant__ Chunk c) {
  chain_begin();
  const uint32_t lane = threadIdx.x & 31u;
  const uint32_t F = c.F, S = (c.e1 - c.e0) * F;
  const uint32_t* __restrict__ segB = c.segB;
  const uint32_t gBeg = segB[0], gEnd = segB[S];
  if (gBeg >= gEnd) return;
  const uint32_t T0 = gBeg & ~(HC - 1u);
  const uint32_t n_chunks = (gEnd - T0 + HC - 1u) / HC;
  const uint32_t lt_mask = (1u << lane) - 1u;
  const uint32_t nwarp = (gridDim.x * blockDim.x) >> 5;
  for (uint32_t c0 = ((blockIdx.x * blockDim.x + threadIdx.x) >> 5) * RANGE; c0 < n_chunks; c0 += nwarp * RANGE) {
    const uint32_t c1 = c0 + RANGE < n_chunks ? c0 + RANGE : n_chunks;
    // ---- the last decodable word before the range, inside the event of the range's first word
    uint32_t carry_key = NOKEY, carry_g = 0u, carry_w = 0xFFFFFFFFu;  // carry_w: its raw word (all ones: unknown)
    {
      const uint32_t b = T0 + c0 * HC, cs = c.chunk_seg[c0], er0 = cs >> 16, sg0 = er0 * F + (cs & 0xFFFFu);
      const uint32_t gw = b < gBeg ? gBeg : b, evb = segB[er0 * F];
      uint32_t g = gw;  // words [evb, g) are still to be searched, backwards
      while (g > evb) {
        const bool in = lane < g - evb;
        const uint32_t gi = g - 1u - lane;
        uint32_t key = NOKEY, wi = 0u;
        if (in) {
          uint32_t sg = sg0;
          while (segB[sg] > gi) --sg;
          wi = __ldg(c.words + gi);
          key = run_key(c.cab, wi, (sg - er0 * F) << 11, er0);
        }
        const uint32_t bal = __ballot_sync(FULL, key != NOKEY);
        if (bal) {
          const int src = __ffs(bal) - 1;
          carry_key = __shfl_sync(FULL, key, src);
          carry_w = __shfl_sync(FULL, wi, src);
          carry_g = g - 1u - (uint32_t)src;
          break;
        }
        g = (g - evb > 32u) ? g - 32u : evb;
      }
    }
    auto load_chunk = [&](uint32_t ci) {  // the four words of this lane in chunk ci (0 where there is no word)
      const uint32_t b = T0 + ci * HC, g0 = b + 4u * lane;
      uint4 wv = make_uint4(0u, 0u, 0u, 0u);
      if (b >= gBeg && b + HC <= gEnd) wv = __ldg(reinterpret_cast<const uint4*>(c.words + g0));
      else {
        if (g0 >= gBeg && g0 < gEnd) wv.x = __ldg(c.words + g0);
        if (g0 + 1u >= gBeg && g0 + 1u < gEnd) wv.y = __ldg(c.words + g0 + 1u);
        if (g0 + 2u >= gBeg && g0 + 2u < gEnd) wv.z = __ldg(c.words + g0 + 2u);
        if (g0 + 3u >= gBeg && g0 + 3u < gEnd) wv.w = __ldg(c.words + g0 + 3u);
      }
      return wv;
    };
    // Two chunks at a time, eight consecutive words per lane, while they lie inside one (event, FED) segment and every
    // word is decodable (nearly always); the words of the next pair are in flight meanwhile.  Otherwise one chunk.
    bool pre = false;
    uint4 pa = make_uint4(0u, 0u, 0u, 0u), pb = pa;
    for (uint32_t ci = c0; ci < c1; ++ci) {
      const uint32_t b = T0 + ci * HC, g0 = b + 4u * lane;
      const uint32_t cs = c.chunk_seg[ci];
      const uint32_t er0 = cs >> 16, fed0 = cs & 0xFFFFu, sg0 = er0 * F + fed0;
      const uint32_t seg_end = segB[sg0 + 1u];
      if (ci + 1u < c1 && b >= gBeg && b + 2u * HC <= gEnd && b + 2u * HC <= seg_end) {
        const uint4* wp = reinterpret_cast<const uint4*>(c.words + b + 8u * lane);
        const uint4 wa = pre ? pa : __ldg(wp), wb = pre ? pb : __ldg(wp + 1);
        pre = ci + 3u < c1 && b + 4u * HC <= gEnd;
        if (pre) { pa = __ldg(wp + 64); pb = __ldg(wp + 65); }  // the pair after this one (2 x 128 words = 64 uint4 on)
        const uint32_t w8[8] = {wa.x, wa.y, wa.z, wa.w, wb.x, wb.y, wb.z, wb.w};
        uint32_t k[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) k[i] = run_key(c.cab, w8[i], fed0 << 11, er0);
        const uint32_t kmx = max(max(max(k[0], k[1]), max(k[2], k[3])), max(max(k[4], k[5]), max(k[6], k[7])));
        if (__all_sync(FULL, kmx != NOKEY)) {
          const uint32_t g8 = b + 8u * lane;
          uint32_t pkey = __shfl_up_sync(FULL, k[7], 1), pg = g8 - 1u, pw = __shfl_up_sync(FULL, w8[7], 1);
          if (lane == 0) { pkey = carry_key; pg = carry_g; pw = carry_w; }
          uint32_t sm = k[0] != pkey ? 1u : 0u;
          bool viol = k[0] == pkey && (w8[0] >> 8) <= (pw >> 8);  // words of a run that do not ascend (read-out order)
#pragma unroll
          for (int i = 1; i < 8; ++i) {
            sm |= k[i] != k[i - 1] ? 1u << i : 0u;
            viol |= k[i] == k[i - 1] && (w8[i] >> 8) <= (w8[i - 1] >> 8);
          }
          const bool pair_bad = __any_sync(FULL, viol);
          if (lane < 2) c.cbad[ci + lane] = pair_bad ? 1 : 0;
          carry_w = __shfl_sync(FULL, w8[7], 31);
          if (sm) {  // (one copy of the atomics for the usual case of one start per lane)
            const uint32_t j0 = (uint32_t)__ffs((int)sm) - 1u;
            uint32_t sk = k[0], sp = pkey;
#pragma unroll
            for (int i = 1; i < 8; ++i) if (j0 == (uint32_t)i) { sk = k[i]; sp = k[i - 1]; }
            run_start(c, sk, g8 + j0);
            if (sp != NOKEY) run_end(c, sp, j0 ? g8 + j0 - 1u : pg);
            if (sm & (sm - 1u)) {  // rare: more runs start inside the lane's eight words
              uint32_t pk = NOKEY;
#pragma unroll 1
              for (uint32_t i = 0; i < 8u; ++i) {
                const uint32_t ki = k[0];
#pragma unroll
                for (int t = 0; t < 7; ++t) k[t] = k[t + 1];
                k[7] = ki;  // rotate: ki is word i's key
                if (i > j0 && ((sm >> i) & 1u)) { run_start(c, ki, g8 + i); run_end(c, pk, g8 + i - 1u); }
                pk = ki;
              }
            }
          }
          carry_key = __shfl_sync(FULL, k[7], 31); carry_g = b + 2u * HC - 1u;
          // start bits: lane l's byte sits at bit 8 l of the 256-bit row; lanes 0, 4, 8 ... end up with the eight words
          uint32_t v = sm;
          v |= __shfl_down_sync(FULL, v, 1) << 8;
          v |= __shfl_down_sync(FULL, v, 2) << 16;
          if ((lane & 3u) == 0u) c.sbits[ci * 4u + (lane >> 2)] = v;
          ++ci;  // two chunks done
          continue;
        }
      }
      pre = false;
      const bool all_in = b >= gBeg && b + HC <= gEnd;
      const bool one_seg = all_in && b + HC <= seg_end;
      const uint4 wv = load_chunk(ci);
      const uint32_t w[4] = {wv.x, wv.y, wv.z, wv.w};
      uint32_t key[4];
      if (one_seg) {
#pragma unroll
        for (int j = 0; j < 4; ++j) key[j] = run_key(c.cab, w[j], fed0 << 11, er0);
      } else {  // a FED / event boundary inside the chunk, or a chunk at the edge of the launch group
#pragma unroll 1
        for (int j = 0; j < 4; ++j) {
          const uint32_t g = g0 + j;
          uint32_t k = NOKEY;
          if (g >= gBeg && g < gEnd) {
            uint32_t sg = sg0;
            while (sg + 1u < S && segB[sg + 1u] <= g) ++sg;
            const uint32_t er = div_F(c, sg);
            k = run_key(c.cab, w[j], (sg - er * F) << 11, er);
          }
          key[0] = key[1]; key[1] = key[2]; key[2] = key[3]; key[3] = k;  // after four turns key[j] is word j's
        }
      }
      // a word starts a run when its (event, module) differs from the previous decodable word's
      uint32_t startmask = 0u;
      uint32_t s_key = NOKEY, s_g = 0u, s_pkey = NOKEY, s_pg = 0u;  // the lane's first run start and its predecessor
      const uint32_t kmax = max(max(key[0], key[1]), max(key[2], key[3]));
      bool chunk_bad = true;  // an undecodable word, or words of a run that do not ascend
      if (__all_sync(FULL, kmax != NOKEY)) {  // the usual chunk: every word decodable, the previous word is the neighbour
        uint32_t pkey = __shfl_up_sync(FULL, key[3], 1), pg = g0 - 1u, pw = __shfl_up_sync(FULL, w[3], 1);
        if (lane == 0) { pkey = carry_key; pg = carry_g; pw = carry_w; }
        const bool viol = (key[0] == pkey && (w[0] >> 8) <= (pw >> 8)) || (key[1] == key[0] && (w[1] >> 8) <= (w[0] >> 8)) ||
                          (key[2] == key[1] && (w[2] >> 8) <= (w[1] >> 8)) || (key[3] == key[2] && (w[3] >> 8) <= (w[2] >> 8));
        chunk_bad = __any_sync(FULL, viol);
        carry_w = __shfl_sync(FULL, w[3], 31);
        startmask = (key[0] != pkey ? 1u : 0u) | (key[1] != key[0] ? 2u : 0u) | (key[2] != key[1] ? 4u : 0u) | (key[3] != key[2] ? 8u : 0u);
        if (startmask) {
          const uint32_t j0 = (uint32_t)__ffs((int)startmask) - 1u;
          s_key = j0 == 0u ? key[0] : j0 == 1u ? key[1] : j0 == 2u ? key[2] : key[3];
          s_pkey = j0 == 0u ? pkey : j0 == 1u ? key[0] : j0 == 2u ? key[1] : key[2];
          s_g = g0 + j0;
          s_pg = j0 == 0u ? pg : s_g - 1u;
        }
        carry_key = __shfl_sync(FULL, key[3], 31); carry_g = b + HC - 1u;
      } else {
        uint32_t tkey = NOKEY, tj = 0u;  // the lane's last decodable word
#pragma unroll
        for (int j = 0; j < 4; ++j) if (key[j] != NOKEY) { tkey = key[j]; tj = j; }
        const uint32_t has = __ballot_sync(FULL, tkey != NOKEY);
        const uint32_t below_l = has & lt_mask;
        const int src = below_l ? 31 - __clz(below_l) : 0;
        uint32_t pkey = __shfl_sync(FULL, tkey, src), pg = b + 4u * (uint32_t)src + __shfl_sync(FULL, tj, src);
        if (!below_l) { pkey = carry_key; pg = carry_g; }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          if (key[j] == NOKEY) continue;
          if (key[j] != pkey) {
            if (!startmask) { s_key = key[j]; s_g = g0 + j; s_pkey = pkey; s_pg = pg; }
            startmask |= 1u << j;
          }
          pkey = key[j]; pg = g0 + j;
        }
        if (has) {
          const int top = 31 - __clz(has);
          carry_key = __shfl_sync(FULL, tkey, top); carry_g = b + 4u * (uint32_t)top + __shfl_sync(FULL, tj, top);
        }
        carry_w = 0xFFFFFFFFu;
      }
      if (lane == 0) c.cbad[ci] = chunk_bad ? 1 : 0;
      if (s_key != NOKEY) {  // one copy of the atomics for the usual case of at most one start per lane
        run_start(c, s_key, s_g);
        if (s_pkey != NOKEY) run_end(c, s_pkey, s_pg);
      }
      if (startmask & (startmask - 1u)) {  // rare: several runs start inside the lane's four words
        uint32_t pk = NOKEY, pgg = 0u;
        bool first = true;
#pragma unroll 1
        for (int j = 0; j < 4; ++j) {
          const uint32_t kj = key[0];
          key[0] = key[1]; key[1] = key[2]; key[2] = key[3]; key[3] = kj;  // rotate: kj is word j's key
          if (kj == NOKEY) continue;
          if ((startmask >> j) & 1u) {
            if (!first) { run_start(c, kj, g0 + j); run_end(c, pk, pgg); }
            first = false;
          }
          pk = kj; pgg = g0 + j;
        }
      }
      // start bits of the chunk: lane l's nibble sits at bit 4 l of the 128-bit row
      // (three folding shuffles: lanes 0, 8, 16, 24 end up with the words of their eight lanes)
      uint32_t v = startmask;
      v |= __shfl_down_sync(FULL, v, 1) << 4;
      v |= __shfl_down_sync(FULL, v, 2) << 8;
      v |= __shfl_down_sync(FULL, v, 4) << 16;
      if ((lane & 7u) == 0u) c.sbits[ci * 4u + (lane >> 3)] = v;
    }
  }
}

// ---- pack_kernel: one warp per event.  The event's start bits are staged in shared memory, BUFW words at a time.
constexpr uint32_t BUFW = 288, NEED = 34;  // a step looks at the words [s >> 5, (s >> 5) + NEED)
constexpr int PACK_WARPS = 4;
constexpr uint32_t PACK_SEGS = 8;  // pieces of an event that are packed by different warps

struct PackWarp {
  uint32_t buf[BUFW];
  uint4 items[32];
};

struct Stage {  // a warp's window on the start bits
  const uint32_t* __restrict__ sbits;
  uint32_t* buf;
  uint32_t w0, w_end;  // first staged word; one past the last word of the launch group's bits that may be read
  uint32_t lane;
  __device__ __forceinline__ void ensure(uint32_t w_lo) {  // words [w_lo, w_lo + NEED) readable
    if (w_lo >= w0 && w_lo + NEED <= w0 + BUFW) return;
    __syncwarp();
    w0 = w_lo;
    for (uint32_t i = lane; i < BUFW; i += 32u) buf[i] = (w0 + i < w_end) ? sbits[w0 + i] : 0u;
    __syncwarp();
  }
  __device__ __forceinline__ uint32_t rd(uint32_t wi) const { return buf[wi - w0]; }
};

// highest start bit in (lo, hi] (bit indices relative to T0; hi - lo <= 992 so the range spans at most 32 words), or NO_INDEX
__device__ __forceinline__ uint32_t last_start(const Stage& st, uint32_t lo, uint32_t hi) {
  const int w_hi = (int)(hi >> 5), w_lo = (int)(lo >> 5), wi = w_hi - (int)st.lane;
  uint32_t v = 0u;
  if (wi >= w_lo) {
    v = st.rd((uint32_t)wi);
    if (wi == w_hi) v &= (2u << (hi & 31u)) - 1u;
    if (wi == w_lo) v &= ~((2u << (lo & 31u)) - 1u);
  }
  const uint32_t bal = __ballot_sync(FULL, v != 0u);
  if (!bal) return NO_INDEX;
  const int src = __ffs(bal) - 1;
  const uint32_t vv = __shfl_sync(FULL, v, src);
  return (uint32_t)(w_hi - src) * 32u + 31u - (uint32_t)__clz(vv);
}
// lowest start bit in (lo, hi], same limits
__device__ __forceinline__ uint32_t first_start(const Stage& st, uint32_t lo, uint32_t hi) {
  const int w_hi = (int)(hi >> 5), w_lo = (int)(lo >> 5), wi = w_lo + (int)st.lane;
  uint32_t v = 0u;
  if (wi <= w_hi) {
    v = st.rd((uint32_t)wi);
    if (wi == w_hi) v &= (2u << (hi & 31u)) - 1u;
    if (wi == w_lo) v &= ~((2u << (lo & 31u)) - 1u);
  }
  const uint32_t bal = __ballot_sync(FULL, v != 0u);
  if (!bal) return NO_INDEX;
  const int src = __ffs(bal) - 1;
  const uint32_t vv = __shfl_sync(FULL, v, src);
  return (uint32_t)(w_lo + src) * 32u + (uint32_t)__ffs(vv) - 1u;
}
// start bits in [lo, hi), hi - lo <= 1024
__device__ __forceinline__ uint32_t count_starts(const Stage& st, uint32_t lo, uint32_t hi) {
  if (hi <= lo) return 0u;
  const uint32_t last = hi - 1u;
  const int w_hi = (int)(last >> 5), w_lo = (int)(lo >> 5);
  uint32_t n = 0u;
  for (int wi = w_lo + (int)st.lane; wi <= w_hi; wi += 32) {
    uint32_t v = st.rd((uint32_t)wi);
    if (wi == w_hi) v &= (2u << (last & 31u)) - 1u;
    if (wi == w_lo) v &= ~((1u << (lo & 31u)) - 1u);
    n += __popc(v);
  }
  return __reduce_add_sync(FULL, n);
}

__global__ void __launch_bounds__(PACK_WARPS * 32) pack_kernel(const __grid_constant__ Chunk c) {
  chain_begin();
  __shared__ PackWarp sm[PACK_WARPS];
  const uint32_t lane = threadIdx.x & 31u;
  PackWarp& pw = sm[threadIdx.x >> 5];
  const uint32_t F = c.F, Ec = c.e1 - c.e0, S = Ec * F;
  const uint32_t* __restrict__ segB = c.segB;
  const uint32_t gBeg = segB[0], gEnd = segB[S];
  if (gBeg >= gEnd) return;
  const uint32_t T0 = gBeg & ~(HC - 1u);
  const uint32_t nwarp = (gridDim.x * blockDim.x) >> 5;
  Stage st;
  st.sbits = c.sbits; st.buf = pw.buf; st.lane = lane; st.w_end = ((gEnd - T0 + HC - 1u) / HC) * 4u;
  for (uint32_t task = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; task < Ec * PACK_SEGS; task += nwarp) {
    // An event is cut at PACK_SEGS - 1 run starts (the first one at or after each k/PACK_SEGS of its length) and the
    // pieces are packed by different warps: the greedy chain of a piece is short, and the seams cost at most one short
    // item each.
    const uint32_t er = task / PACK_SEGS, seg = task % PACK_SEGS;
    const uint32_t evb = segB[er * F], ev_end = segB[(er + 1u) * F];
    if (evb >= ev_end) continue;
    st.w0 = 0xFFFFFFFFu - BUFW;  // nothing staged
    auto first_start_from = [&](uint32_t lo, uint32_t limit) {  // first start bit in [lo, limit), or limit (bit indices; lo >= 1)
      uint32_t p = lo - 1u, nx = NO_INDEX;
      while (nx == NO_INDEX && p + 1u < limit) {
        const uint32_t q = (limit - 1u - p > 992u) ? p + 992u : limit - 1u;
        st.ensure(p >> 5);
        nx = first_start(st, p, q);
        p = q;
      }
      return nx == NO_INDEX ? limit : nx;
    };
    const uint32_t n_ev = ev_end - evb, rb = evb - T0, re = ev_end - T0;
    const uint32_t q0 = rb + (uint32_t)(((uint64_t)n_ev * seg) / PACK_SEGS), q1 = rb + (uint32_t)(((uint64_t)n_ev * (seg + 1u)) / PACK_SEGS);
    const uint32_t s_beg = T0 + ((seg == 0u || q0 == rb) ? rb : first_start_from(q0, re));
    const uint32_t eve = T0 + ((seg + 1u == PACK_SEGS) ? re : (q1 == rb ? rb : first_start_from(q1, re)));  // this piece ends here
    if (s_beg >= eve) continue;
    uint32_t sg = er * F;  // FED of the piece's first word: the last FED that begins at or before it
    for (uint32_t f0 = 0u; f0 < F; f0 += 32u) {
      const bool in = f0 + lane < F;
      const uint32_t v = in ? segB[er * F + f0 + lane] : 0xFFFFFFFFu;
      const uint32_t m = __ballot_sync(FULL, in && v <= s_beg);
      if (m) sg = er * F + f0 + 31u - (uint32_t)__clz(m);
      if (m != FULL) break;
    }
    uint32_t s = s_beg;
    uint32_t n_buf = 0u;  // items waiting in pw.items
    auto flush = [&]() {
      __syncwarp();
      uint32_t base = 0u;
      if (lane == 0 && n_buf) base = atomicAdd(c.ctl + CTL_ITEM_COUNT, n_buf);
      base = __shfl_sync(FULL, base, 0);
      if (lane < n_buf && base + lane < c.item_cap) c.items[base + lane] = pw.items[lane];
      n_buf = 0u;
      __syncwarp();
    };
    uint32_t sg_end = segB[sg + 1u];  // first word of the next FED (kept in a register: no global load per item)
    auto emit = [&](uint32_t g, uint32_t len, uint32_t flags) {
      while (sg + 1u < (er + 1u) * F && sg_end <= g) { ++sg; sg_end = segB[sg + 1u]; }
      if (lane == 0) pw.items[n_buf] = make_uint4(g, len | (flags << 16), er | ((sg - er * F) << 16), 0u);
      if (++n_buf == 32u) flush();
    };
    while (s < eve) {
      const uint32_t rs = s - T0, rlast = eve - 1u - T0;  // bit indices of the item's first word and of the event's last word
      st.ensure(rs >> 5);
      uint32_t win = ITEM_WIN;
      uint32_t nxt;  // bit index of the next item's first word
      while (true) {
        if (rlast - rs < win) nxt = rlast + 1u;  // the rest of the event fits
        else nxt = last_start(st, rs, rs + win);
        if (nxt == NO_INDEX || win == ITEM_WIN2) break;
        if (count_starts(st, rs, nxt) <= ITEM_RUNS) break;
        win = ITEM_WIN2;  // too many runs: a shorter item (at most ITEM_WIN2 + 1 <= ITEM_RUNS runs)
      }
      if (nxt != NO_INDEX) {
        emit(s, nxt - rs, 0u);
        s = T0 + nxt;
        continue;
      }
      // no run starts in (s, s + win]: one run (or a stretch of undecodable words) longer than that
      const bool head = (st.rd(rs >> 5) >> (rs & 31u)) & 1u;
      uint32_t p = rs + win;
      while (nxt == NO_INDEX && p < rlast) {
        const uint32_t q = (rlast - p > 992u) ? p + 992u : rlast;
        st.ensure(p >> 5);
        nxt = first_start(st, p, q);
        p = q;
      }
      if (nxt == NO_INDEX) nxt = rlast + 1u;
      const uint32_t L = nxt - rs;
      if (L <= TILE_WORDS) emit(s, L, 0u);
      else {
        const uint32_t pieces = (L + TILE_WORDS - 1u) / TILE_WORDS, plen = (L + pieces - 1u) / pieces;
        for (uint32_t k = 0, o = 0; o < L; ++k, o += plen)
          emit(s + o, (L - o < plen) ? L - o : plen, ITEM_DECODE_ONLY | ((k == 0 && head) ? ITEM_LONG_HEAD : 0u));
      }
      s = T0 + nxt;
    }
    flush();
  }
}

}  // namespace

void launch_runs(const Chunk& c, uint32_t words_bound, int n_sm, cudaStream_t stream) {
  uint64_t nb = ((uint64_t)words_bound + 2 * HC + 8 * RANGE * HC - 1) / (8 * RANGE * HC);  // 8 warps of RANGE chunks per block
  if (nb < 1) nb = 1;
  if (nb > (uint64_t)n_sm * 64) nb = (uint64_t)n_sm * 64;
  launch_chained(true, runs_kernel, (unsigned)nb, 256, 0, stream, c);
  const uint32_t Ec = c.e1 - c.e0;
  launch_chained(true, pack_kernel, (Ec * PACK_SEGS + PACK_WARPS - 1u) / PACK_WARPS, PACK_WARPS * 32, 0, stream, c);
}

}  // namespace pix
