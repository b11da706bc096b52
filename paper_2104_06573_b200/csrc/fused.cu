// fused.cu -- init, and the fused warp kernel: a1 decode (S1-S6), a2 calibrate (S7-S9), a3 module
// boundaries (S11, S12), a4 findClus (S10, S13) and a5 sums / charge cut / renumber / temp records (S9, S14,
// S18) of the path PAPER.md:31 describes ("unpacks them, calibrates the individual pixels, and clusters the
// pixels on each detector module"), in ONE pass over the raw words.
//
// The word stream is cut into home chunks of 128 words, one warp per chunk, 32 words (one per lane) per round.
// A module's decodable words form one run (S11); a run belongs to the warp whose home chunk holds its first
// word.  Warps never wait for each other (no block barrier); all tables are per-warp shared memory.  A warp
//   A  clears its position hash, finds the (event, FED) segment of its chunk, and looks back for the last
//      decodable word before the chunk (its run may continue into the chunk)
//   B  home rounds 0-3: decodes + calibrates its 128 words, stores module/row/col/charge (and the final status
//      of undecodable words), finds run starts with a ballot/shuffle "previous decodable word" scan (a3), and
//      inserts every owned digi into the position hash keyed by (run, row, col); equal keys keep the lowest digi
//   C  extension rounds 4-7: decodes on until the first word of another run, to complete its last run
//   D  looks up the forward neighbours of its digis, compacts the adjacent pairs into a dense edge list and
//      unites them (lock-free min-index union-find, all lanes busy)
//   E  every live digi adds charge | 1 << 24, charge*col, charge*row into its root's accumulators
//   F  surviving roots (Q >= cut) are numbered in digi order per run (ballot/popc), temp records written
//   G  final status and clus of every digi the warp owns; per-event counters
// Runs that do not fit the 256-word window, chunks with more than RC runs and charge sums that could overflow
// 32 bits go to the overflow list (cluster.cu).  Nothing here is shared with oracle/.
#include "pix_common.cuh"

namespace pix {

namespace {

constexpr uint32_t NOKEY = 0xFFFFFFFFu;

// ------------------------------------------------------------------ init
// One warp per event of the chunk builds the clamped, monotone segment table
//   segB[e_rel*F + f] = global word index where FED f of event e starts,  segB[Ec*F] = end of chunk.
// Offsets are clamped into [lo, hi] (lo = start of chunk, hi = min(n_total, lo + cap_words)) so that
// whatever the caller's offset arrays hold, every index derived later stays inside the buffers.
// Other threads initialise the per-(event,module) range sentinels and zero the counters.
__global__ void __launch_bounds__(256) init_kernel(const __grid_constant__ Chunk c, uint32_t n_total) {
  const uint32_t Ec = c.e1 - c.e0;
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
  uint32_t lo = ev_offset(c, c.e0);
  lo = lo < n_total ? lo : n_total;
  const uint32_t room = n_total - lo;
  const uint32_t hi = lo + (room < c.cap_words ? room : c.cap_words);
  if (tid < CTL_WORDS) c.ctl[tid] = 0;
  // one warp per event: lanes take FEDs, the running max over the clamped offsets is a warp max-scan
  const uint32_t lane = threadIdx.x & 31u, wid = tid >> 5, nwarp = nth >> 5;
  for (uint32_t er = wid; er < Ec; er += nwarp) {
    const uint32_t e = c.e0 + er;
    const uint32_t rb = ev_offset(c, e), re = ev_offset(c, e + 1);
    const uint32_t b = rb < lo ? lo : (rb > hi ? hi : rb);
    const uint32_t en = re < b ? b : (re > hi ? hi : re);
    const uint32_t nw = en - b;
    const uint32_t flags = (re > hi || rb > hi || re < rb || rb < lo) ? FLAG_TOO_LARGE : 0u;
    uint32_t carry = 0;
    for (uint32_t f0 = 0; f0 < c.F; f0 += 32u) {
      const uint32_t f = f0 + lane;
      uint32_t fo = (f == 0 || f >= c.F || !c.fed_off) ? 0u : c.fed_off[(size_t)e * (c.F + 1) + f];
      fo = fo > nw ? nw : fo;
      fo = fo > carry ? fo : carry;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const uint32_t o = __shfl_up_sync(0xFFFFFFFFu, fo, d);
        if (lane >= (uint32_t)d && o > fo) fo = o;
      }
      if (f < c.F) c.segB[er * c.F + f] = b + fo;  // monotone by construction
      carry = __shfl_sync(0xFFFFFFFFu, fo, 31);
    }
    if (er == Ec - 1 && lane == 0) c.segB[Ec * c.F] = en;
    if (lane < EC_STRIDE) c.ev_cnt[(size_t)er * EC_STRIDE + lane] = (lane == EC_FLAGS) ? flags : 0u;
  }
  const uint32_t nmod = Ec * c.M;
  uint32_t* mf = c.module_first + (size_t)c.e0 * c.M;
  uint32_t* me = c.module_end + (size_t)c.e0 * c.M;
  for (uint32_t t = tid; t < nmod; t += nth) { mf[t] = NO_INDEX; me[t] = 0u; c.n_clus[t] = 0u; }
}

// ------------------------------------------------------------------ decode / calibrate
// S1-S6 with the pre-digested cabling entry (pix_common.cuh).  Returns the status; module/row/col are defined
// only for ST_OK.  fedbase = fed * 2048.
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

// S7: four separately rounded binary32 RN operations (the _rn intrinsics are never contracted to FMA),
// then NaN/negative -> 0, clamp, truncate.
__device__ __forceinline__ int32_t calibrate(const Chunk& c, uint32_t adc, float2 gp) {
  const float f1 = __fsub_rn((float)adc, gp.y);
  const float f2 = __fmul_rn(f1, gp.x);
  const float f3 = __fmul_rn(f2, c.vcal_gain);
  const float f4 = __fadd_rn(f3, c.vcal_offset);
  if (!(f4 >= 0.0f)) return 0;
  return __float2int_rz(fminf(f4, c.max_e_f));
}

// last s in [0, S) with segB[s] <= g, given segB[0] <= g < segB[S]; warp-cooperative 32-ary search
__device__ __forceinline__ uint32_t warp_find_segment(const uint32_t* __restrict__ segB, uint32_t S, uint32_t g,
                                                      uint32_t lane) {
  uint32_t lo = 0, hi = S;  // invariant: segB[lo] <= g < segB[hi]
  while (hi - lo > 1) {
    const uint32_t step = (hi - lo + 31u) / 32u;
    const uint32_t p = lo + (lane + 1u) * step;
    const bool le = (p < hi) && (segB[p] <= g);
    const uint32_t cnt = __popc(__ballot_sync(0xFFFFFFFFu, le));
    const uint32_t nlo = lo + cnt * step;
    const uint32_t nhi = nlo + step;
    lo = nlo;
    hi = nhi < hi ? nhi : hi;
  }
  return lo;
}

// a3: module_first / module_end are keyed by module id (S12); a second run of a module flags the event (S11)
__device__ __forceinline__ uint32_t run_start(const Chunk& c, uint32_t key, uint32_t g) {
  const uint32_t er = key >> 16, m = key & 0xFFFFu;
  const uint32_t i = g - c.segB[er * c.F];
  const uint32_t old = atomicMin(c.module_first + ((size_t)(c.e0 + er) * c.M + m), i);
  if (old != NO_INDEX) atomicOr(c.ev_cnt + (size_t)er * EC_STRIDE + EC_FLAGS, FLAG_NONCONTIGUOUS);
  return i;
}
__device__ __forceinline__ void run_end(const Chunk& c, uint32_t key, uint32_t g) {
  const uint32_t er = key >> 16, m = key & 0xFFFFu;
  atomicMax(c.module_end + ((size_t)(c.e0 + er) * c.M + m), g - c.segB[er * c.F] + 1u);
}
__device__ __forceinline__ void push_overflow(const Chunk& c, uint32_t key) {
  const uint32_t i = atomicAdd(c.ctl + CTL_OVF_COUNT, 1u);
  if (i < c.ovf_cap) c.ovf_list[i] = (key >> 16) * c.M + (key & 0xFFFFu);
}

// ------------------------------------------------------------------ the fused warp kernel
constexpr int WPB = 4;                    // warps per block (they share nothing but the block)
constexpr int FT = WPB * 32;
constexpr uint32_t HC = 128;              // words of a home chunk (rounds 0-3)
constexpr uint32_t MAXT = 256;            // window: home chunk + up to 4 extension rounds
constexpr uint32_t WTAB = 512;            // hash slots per warp
constexpr uint32_t RC = 62;               // runs a warp can own
constexpr uint32_t ECAP = 3 * MAXT;       // at most 3 forward edges per digi
constexpr uint32_t EMPTY = 0xFFFFFFFFu, INVALID = 0xFFFFFFFFu;
constexpr uint32_t MARK_DUP = 0xFFFFFFFEu, MARK_BELOW = 0xFFFFFFFDu;  // label of a digi that is not live
constexpr uint32_t Q_SAFE = 0xFFFFFFFFu / 415u;  // sum(e*col), sum(e*row) fit 32 bits while sum(e) <= Q_SAFE
constexpr uint32_t HASH_MUL = 0x9E3779B1u;
constexpr uint32_t KEY_BITS = 23, KEY_MASK = (1u << KEY_BITS) - 1u, TAG_BITS = 14, TAG_MASK = (1u << TAG_BITS) - 1u;
static_assert(((RC + 1u) << 17) <= (1u << KEY_BITS) && (1u << (KEY_BITS - TAG_BITS)) == WTAB && MAXT <= 256,
              "key: run (6 bits) | row (8) | col (9); slot: disp (9) | tag (14) | digi (8) | below (1)");

// digi key inside the window: run (6 bits) | row (8 bits) | col (9 bits).  Neighbour keys are key+1 (col+1)
// and key+512-1, +512, +512+1 (row+1): col 416..511 and row 160..255 never occur, so no bounds checks (S13).
struct __align__(16) WarpSmem {
  uint32_t tab[WTAB];      // position hash, EMPTY-filled.  After phase D, tab + edge: qn = tab, sx = tab + 256, sy = tab + 512
  uint16_t edge[ECAP];     // a | b << 8
  uint32_t dkey[MAXT];     // key of the digi in window slot t (word b + t), INVALID if not owned / undecodable
  uint32_t label[MAXT];    // union-find parent, or MARK_*
  uint16_t chg[MAXT];      // charge; after phase E: local id of a root, or NO_ID
  uint32_t run_ifirst[RC + 2];  // event-relative index of the run's first digi
  uint32_t run_key[RC + 2];     // event_rel << 16 | module
  uint16_t run_first[RC + 2];   // window slot of the run's first digi
  uint16_t run_base[RC + 2];    // survivors before the run
  uint8_t run_bad[RC + 2];      // the run is left to the overflow kernel
};
static_assert(WTAB * 4 + ECAP * 2 >= 3 * MAXT * 4 + MAXT, "the sums and the root list fit in tab + edge");
static_assert(sizeof(WarpSmem) % 16 == 0, "per-warp slices stay 16-byte aligned");

// Position hash, open addressing, one word per slot.  h = key * HASH_MUL mod 2^23 is a bijection on the 23-bit
// keys; home slot = top 9 bits of h, tag = the other 14, so (home, tag) names the key exactly.  A key stored
// i slots after its home records the displacement: slot = disp (9) | tag (14) | digi (8) | below_threshold (1).
// Slots are never emptied; equal keys meet in one slot and keep the lowest digi (S10).
__device__ __forceinline__ uint32_t hmix(uint32_t key) { return (key * HASH_MUL) & KEY_MASK; }

// returns true when the key was already there (a duplicate pixel, S10)
__device__ __forceinline__ bool hinsert(WarpSmem& s, uint32_t key, uint32_t t, uint32_t below) {
  const uint32_t h = hmix(key);
  uint32_t p = h >> TAG_BITS, want = h & TAG_MASK;
#pragma unroll 1
  while (true) {
    const uint32_t mine = (want << 9) | (t << 1) | below;
    const uint32_t old = atomicCAS(&s.tab[p], EMPTY, mine);
    if (old == EMPTY) return false;
    if ((old >> 9) == want) { atomicMin(&s.tab[p], mine); return true; }  // same pixel: the lowest digi owns it
    p = (p + 1u) & (WTAB - 1u); want += 1u << TAG_BITS;  // at most 256 of the 512 slots are ever taken
  }
}
// slot contents of the key whose mixed value is h, or EMPTY
__device__ __forceinline__ uint32_t hfind(const WarpSmem& s, uint32_t h) {
  uint32_t p = h >> TAG_BITS, want = h & TAG_MASK;
  uint32_t e = s.tab[p];
#pragma unroll 1
  while (e != EMPTY && (e >> 9) != want) {
    p = (p + 1u) & (WTAB - 1u); want += 1u << TAG_BITS;
    e = s.tab[p];
  }
  return e;
}
__device__ __forceinline__ uint32_t slot_digi(uint32_t e) { return (e >> 1) & 0xFFu; }
__device__ __forceinline__ bool slot_live(uint32_t e) { return e != EMPTY && !(e & 1u); }

// union-find on s.label; labels strictly decrease along parents
__device__ __forceinline__ uint32_t uf_find(volatile uint32_t* L, uint32_t x) {
  uint32_t p = L[x];
  while (p != x) {
    const uint32_t gp = L[p];
    if (gp != p) L[x] = gp;  // path halving; a racing hook only ever lowers a parent inside the same component
    x = p; p = gp;
  }
  return x;
}
__device__ __forceinline__ void uf_unite(uint32_t* L, uint32_t a, uint32_t b) {
  bool done = false;  // single exit: the lanes of a warp reconverge after the loop
  while (!done) {
    a = uf_find(L, a); b = uf_find(L, b);
    if (a == b) { done = true; }
    else {
      if (a < b) { const uint32_t t = a; a = b; b = t; }
      const uint32_t old = atomicMin(L + a, b);  // hook the larger root under the smaller
      if (old == a) done = true;
      else a = old;                            // a was no longer a root: keep merging its parent with b
    }
  }
}

// (event, FED) of word g >= b, given the segment sg0 of the chunk's first word and the next boundary nextB0
__device__ __forceinline__ void seg_of(const uint32_t* __restrict__ segB, uint32_t S, uint32_t F, uint32_t g, uint32_t sg0,
                                       uint32_t nextB0, uint32_t er0, uint32_t fed0, uint32_t& er, uint32_t& fed) {
  er = er0; fed = fed0;
  if (g >= nextB0) {  // rare: a FED / event boundary inside the window (g < segB[S] always)
    uint32_t sg = sg0 + 1u;
    while (sg + 1u < S && segB[sg + 1u] <= g) ++sg;
    er = sg / F; fed = sg - er * F;
  }
}

__global__ void __launch_bounds__(FT, 8) fused_kernel(const __grid_constant__ Chunk c) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  WarpSmem& s = reinterpret_cast<WarpSmem*>(smem_raw)[warp];
  const uint32_t F = c.F, S = (c.e1 - c.e0) * F;
  const uint32_t* __restrict__ segB = c.segB;
  const uint32_t gBeg = segB[0], gEnd = segB[S];
  if (gBeg >= gEnd) return;
  const uint32_t T0 = gBeg & ~31u;  // rounds are 128-byte aligned
  const uint32_t n_chunks = (gEnd - T0 + HC - 1u) / HC;
  const uint32_t lt_mask = (1u << lane) - 1u, le_mask = lt_mask | (1u << lane);
  constexpr uint32_t FULL = 0xFFFFFFFFu;
  uint32_t* const w0 = reinterpret_cast<uint32_t*>(&s);  // tab + edge, reused after phase D
  uint32_t* const qn = w0; uint32_t* const sx = w0 + MAXT; uint32_t* const sy = w0 + 2 * MAXT;
  uint16_t* const lid = s.chg;
  uint8_t* const rlist = reinterpret_cast<uint8_t*>(w0 + 3 * MAXT);  // roots in digi order (after phase D)
  constexpr uint32_t NO_ID = 0xFFFFu;

  for (uint32_t ci = blockIdx.x * WPB + warp; ci < n_chunks; ci += gridDim.x * WPB) {
    const uint32_t b = T0 + ci * HC;
    // ================================================================== A: load; clear; segment; look-back
    uint32_t w[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const uint32_t g = b + 32u * k + lane;
      w[k] = (g >= gBeg && g < gEnd) ? __ldg(c.words + g) : 0u;
    }
    {
      uint4* t4 = reinterpret_cast<uint4*>(s.tab);
      const uint4 e4 = make_uint4(EMPTY, EMPTY, EMPTY, EMPTY);
#pragma unroll
      for (int k = 0; k < (int)(WTAB / 4 / 32); ++k) t4[lane + 32 * k] = e4;
      if (lane < (RC + 2u) / 4u) reinterpret_cast<uint32_t*>(s.run_bad)[lane] = 0u;
    }
    const uint32_t gw = b < gBeg ? gBeg : b;  // b < gEnd by the chunk count
    const uint32_t sg0 = warp_find_segment(segB, S, gw, lane);
    const uint32_t er0 = sg0 / F, fed0 = sg0 - er0 * F, nextB0 = segB[sg0 + 1u];
    uint32_t ckey = NOKEY, cg = 0u;  // last decodable word so far (warp-uniform)
    {
      uint32_t g = gw;  // words [gBeg, g) are still to be searched, backwards
      while (g > gBeg) {
        const bool in = lane < g - gBeg;
        const uint32_t gi = g - 1u - lane;
        uint32_t key = NOKEY;
        if (in) {
          uint32_t sg = sg0;
          while (segB[sg] > gi) --sg;  // segB[0] = gBeg <= gi
          const uint32_t er = sg / F, fed = sg - er * F;
          uint32_t m, r, cc;
          if (decode_word(c.cab, __ldg(c.words + gi), fed << 11, m, r, cc) == ST_OK) key = (er << 16) | m;
        }
        const uint32_t bal = __ballot_sync(FULL, key != NOKEY);
        if (bal) {
          const int src = __ffs(bal) - 1;
          ckey = __shfl_sync(FULL, key, src);
          cg = g - 1u - (uint32_t)src;
          break;
        }
        g = (g - gBeg > 32u) ? g - 32u : gBeg;
      }
    }
    __syncwarp();  // the cleared hash is visible

    // ================================================================== B: home rounds
    uint32_t R = 0u;        // runs started in the home chunk so far
    uint32_t f_t = MAXT;    // window slot of the first owned digi
    bool dup_seen = false;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const uint32_t t = 32u * k + lane, g = b + t;
      const bool in = g >= gBeg && g < gEnd;
      uint32_t er, fed;
      seg_of(segB, S, F, g, sg0, nextB0, er0, fed0, er, fed);
      uint32_t m = 0xFFFFu, row = 0xFFFFu, col = 0xFFFFu, st = 0xFFu;
      int32_t e = 0;
      bool dec = false;
      if (in) {
        uint32_t dm, dr, dc;
        st = decode_word(c.cab, w[k], fed << 11, dm, dr, dc);
        dec = st == ST_OK;
        if (dec) {
          m = dm; row = dr; col = dc;
          const float2 gp = __ldg(c.gp + (m * (uint32_t)COLS + col));  // S8: one pair per (module, col)
          e = calibrate(c, w[k] & 255u, gp);
          if (e < c.thr) st = ST_BELOW;                                // S9
        } else {  // undecodable: finished here
          atomicAdd(c.ev_cnt + (size_t)er * EC_STRIDE + (st - ST_EMPTY), 1u);
          c.d_status[g] = (uint8_t)st; c.d_clus[g] = -1;
        }
        c.d_module[g] = (uint16_t)m; c.d_row[g] = (uint16_t)row; c.d_col[g] = (uint16_t)col; c.d_charge[g] = e;
      }
      // ---- a3: previous decodable word of every lane (ballot + shuffle, carry across rounds)
      const uint32_t key = dec ? ((er << 16) | m) : NOKEY;
      const uint32_t has = __ballot_sync(FULL, dec);
      const uint32_t below_l = has & lt_mask;
      const int src = below_l ? 31 - __clz(below_l) : 0;
      uint32_t pkey = __shfl_sync(FULL, key, src), pg = b + 32u * k + (uint32_t)src;
      if (!below_l) { pkey = ckey; pg = cg; }
      const bool start = dec && key != pkey;
      uint32_t ifirst = 0u;
      if (start) {
        ifirst = run_start(c, key, g);
        if (pkey != NOKEY) run_end(c, pkey, pg);
      }
      const uint32_t sm = __ballot_sync(FULL, start);
      const uint32_t r = R + __popc(sm & le_mask);  // run of this word; 0: a run of an earlier chunk
      if (start) {
        if (r <= RC) { s.run_first[r] = (uint16_t)t; s.run_ifirst[r] = ifirst; s.run_key[r] = key; }
        else push_overflow(c, key);
      }
      const bool own = dec && r >= 1u && r <= RC;
      const uint32_t dk = own ? ((r << 17) | (row << 9) | col) : INVALID;
      s.dkey[t] = dk;
      s.label[t] = (own && st == ST_OK) ? t : MARK_BELOW;
      s.chg[t] = (uint16_t)e;
      if (own) dup_seen |= hinsert(s, dk, t, st == ST_BELOW ? 1u : 0u);
      if (has) {
        const int top = 31 - __clz(has);
        ckey = __shfl_sync(FULL, key, top); cg = b + 32u * k + (uint32_t)top;
      }
      if (R == 0u && sm) f_t = 32u * k + (uint32_t)(__ffs(sm) - 1);
      R += __popc(sm);
    }
    if (ci == n_chunks - 1u && lane == 0 && ckey != NOKEY) run_end(c, ckey, cg);  // the chunk's last run
    if (R == 0u) continue;  // nothing owned
    const uint32_t Rn = R < RC ? R : RC;

    // ================================================================== C: extension rounds for the last run
    uint32_t n_t = HC;  // window slots staged
    if (R <= RC) {
      const uint32_t keyR = ckey;  // the last decodable word of the home chunk is in the last run
      bool ended = b + HC >= gEnd;
#pragma unroll 1
      for (uint32_t k = 4; k < MAXT / 32u && !ended; ++k) {
        const uint32_t t = 32u * k + lane, g = b + t;
        const bool in = g < gEnd;
        bool dec = false, stop = true;  // the end of the data stops the run
        uint32_t key = NOKEY, m = 0, row = 0, col = 0, wv = 0;
        if (in) {
          uint32_t er, fed;
          seg_of(segB, S, F, g, sg0, nextB0, er0, fed0, er, fed);
          wv = __ldg(c.words + g);
          dec = decode_word(c.cab, wv, fed << 11, m, row, col) == ST_OK;
          key = (er << 16) | m;
          stop = dec && key != keyR;
        }
        const uint32_t stopmask = __ballot_sync(FULL, stop);
        const uint32_t first = stopmask ? (uint32_t)(__ffs(stopmask) - 1) : 32u;
        const bool own = dec && lane < first;
        uint32_t dk = INVALID, lb = MARK_BELOW;
        if (own) {
          const float2 gp = __ldg(c.gp + (m * (uint32_t)COLS + col));
          const int32_t e = calibrate(c, wv & 255u, gp);
          dk = (R << 17) | (row << 9) | col;
          const bool below = e < c.thr;
          if (!below) lb = t;
          s.chg[t] = (uint16_t)e;
          dup_seen |= hinsert(s, dk, t, below ? 1u : 0u);
        }
        s.dkey[t] = dk; s.label[t] = lb;
        n_t = 32u * (k + 1u);
        ended = stopmask != 0u;
      }
      if (!ended && b + MAXT < gEnd && lane == 0) s.run_bad[R] = 1;  // the run does not fit the window: the overflow kernel takes it
    }
    __syncwarp();  // hash, dkey, label, run tables complete
    const uint32_t k0 = f_t >> 5, k1 = n_t >> 5;  // rounds that hold owned digis

    // ================================================================== D: duplicates; neighbours -> edges -> unions
    if (__any_sync(FULL, dup_seen)) {  // rare: some pixel appears twice; the digi not in the slot is a DUPLICATE (S10)
      for (uint32_t k = k0; k < k1; ++k) {
        const uint32_t t = 32u * k + lane, key = s.dkey[t];
        if (key != INVALID && slot_digi(hfind(s, hmix(key))) != t) s.label[t] = MARK_DUP;
      }
      __syncwarp();
    }
    // Forward neighbours (S13): E (r, c+1), SW (r+1, c-1), S (r+1, c), SE (r+1, c+1).  When S is live, SW and SE are
    // joined to it by their own E edges, so d-S alone is enough.
    uint32_t ne = 0u;
#pragma unroll 1
    for (uint32_t k = k0; k < k1; ++k) {
      const uint32_t t = 32u * k + lane, key = s.dkey[t];
      const bool live = key != INVALID && s.label[t] == t;
      bool f0 = false, f1 = false, f2 = false;
      uint32_t n0 = 0, n1 = 0, n2 = 0;
      if (live) {
        const uint32_t h = hmix(key);
        const uint32_t eE = hfind(s, (h + HASH_MUL) & KEY_MASK), eS = hfind(s, (h + 512u * HASH_MUL) & KEY_MASK);
        const uint32_t eSW = hfind(s, (h + 511u * HASH_MUL) & KEY_MASK), eSE = hfind(s, (h + 513u * HASH_MUL) & KEY_MASK);
        const bool hS = slot_live(eS);
        f0 = slot_live(eE); n0 = slot_digi(eE);
        f1 = hS || slot_live(eSW); n1 = slot_digi(hS ? eS : eSW);
        f2 = !hS && slot_live(eSE); n2 = slot_digi(eSE);
      }
      const uint32_t m0 = __ballot_sync(FULL, f0), m1 = __ballot_sync(FULL, f1), m2 = __ballot_sync(FULL, f2);
      if (f0) s.edge[ne + __popc(m0 & lt_mask)] = (uint16_t)(t | (n0 << 8));
      ne += __popc(m0);
      if (f1) s.edge[ne + __popc(m1 & lt_mask)] = (uint16_t)(t | (n1 << 8));
      ne += __popc(m1);
      if (f2) s.edge[ne + __popc(m2 & lt_mask)] = (uint16_t)(t | (n2 << 8));
      ne += __popc(m2);
    }
    __syncwarp();
    for (uint32_t i0 = 0u; i0 < ne; i0 += 32u) {  // warp-uniform trip count: the lanes reconverge every iteration
      if (i0 + lane < ne) {
        const uint32_t e = s.edge[i0 + lane];
        uf_unite(s.label, e & 0xFFu, e >> 8);
      }
      __syncwarp();
    }
    __syncwarp();  // components complete; the hash is dead, its memory becomes qn / sx / sy / lid

    // ================================================================== E: cluster sums; dense list of the roots
    {
      uint4* t4 = reinterpret_cast<uint4*>(w0);
      const uint4 z4 = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
      for (int k = 0; k < (int)(3 * MAXT / 4 / 32); ++k) t4[lane + 32 * k] = z4;
    }
    __syncwarp();
    uint32_t nr = 0u;  // roots so far
#pragma unroll 1
    for (uint32_t k = k0; k < k1; ++k) {
      const uint32_t t = 32u * k + lane;
      volatile uint32_t* L = s.label;
      uint32_t r = L[t];
      const bool live = r < MAXT;  // else MARK_*
      if (live) {
        while (true) { const uint32_t n = L[r]; if (n == r) break; r = n; }
        L[t] = r;  // flatten: r is the root, so other walkers through t stay correct
        const uint32_t key = s.dkey[t], e = s.chg[t];
        atomicAdd(&qn[r], e | (1u << 24));  // charge sum (< 2^24: 256 * 65535) | pixel count (256 wraps to 0)
        atomicAdd(&sx[r], e * (key & 511u));
        atomicAdd(&sy[r], e * ((key >> 9) & 255u));
      }
      const bool root = live && r == t;
      const uint32_t rm = __ballot_sync(FULL, root);
      if (root) rlist[nr + __popc(rm & lt_mask)] = (uint8_t)t;  // digi order
      nr += __popc(rm);
    }
    __syncwarp();

    // ================================================================== F: cut, renumber, temp records (one root per lane)
    {
      uint32_t cnt = 0u;      // surviving roots before this iteration
      uint32_t crun = 0u;     // run of the last surviving root so far (runs 1 .. crun have their run_base)
      const uint32_t relb = b - gBeg;  // may wrap for the first chunk; only used added to a slot >= gBeg - b
#pragma unroll 1
      for (uint32_t i0 = 0u; i0 < nr; i0 += 32u) {
        const bool valid = i0 + lane < nr;
        uint32_t t = 0u, r = 0u, Q = 0u, np = 0u;
        if (valid) {
          t = rlist[i0 + lane];
          r = s.dkey[t] >> 17;
          const uint32_t v = qn[t];
          Q = v & 0xFFFFFFu; np = v >> 24;
          if (np == 0u) np = 256u;
          if (Q > Q_SAFE) s.run_bad[r] = 1;  // 32-bit weighted sums may have wrapped
        }
        const bool surv = valid && (int32_t)Q >= c.cut;  // S9: equality keeps
        const uint32_t sm = __ballot_sync(FULL, surv);
        const uint32_t before = sm & lt_mask;
        const uint32_t rank = cnt + __popc(before);
        const int pl = before ? 31 - __clz(before) : 0;
        uint32_t rp = __shfl_sync(FULL, r, pl);  // run of the previous surviving root
        if (!before) rp = crun;
        if (surv)
          for (uint32_t q = rp + 1u; q <= r; ++q) s.run_base[q] = (uint16_t)rank;  // first survivor of run r
        if (sm) crun = __shfl_sync(FULL, r, 31 - __clz(sm));
        cnt += __popc(sm);
        __syncwarp();
        if (valid) {
          uint32_t id = NO_ID;
          if (surv) {
            id = rank - s.run_base[r];
            const uint32_t rf = s.run_first[r];
            // S18: exact integer sums, one rounding each + a 2-ulp division (within 1e-5)
            const float fq = (float)Q;
            put_temp(c.t_rec + (relb + rf + id), s.run_ifirst[r] + (t - rf), np, Q, __fdividef((float)sx[t], fq),
                     __fdividef((float)sy[t], fq));
          }
          lid[t] = (uint16_t)id;
        }
      }
      for (uint32_t q = crun + 1u + lane; q <= Rn + 1u; q += 32u) s.run_base[q] = (uint16_t)cnt;
    }
    __syncwarp();  // run_base, run_bad, local ids final
    for (uint32_t r = 1u + lane; r <= Rn; r += 32u) {
      const uint32_t key = s.run_key[r];
      if (s.run_bad[r]) push_overflow(c, key);
      else c.n_clus[(key >> 16) * c.M + (key & 0xFFFFu)] = (uint32_t)s.run_base[r + 1u] - s.run_base[r];
    }

    // ================================================================== G: final status and clus, counters
    uint32_t cntA = 0u, cntB = 0u, n_pre = 0u;  // dup | below << 16 ; ok | cut << 16 ; roots
    uint32_t ev_lo = NOKEY, ev_hi = 0u;         // events of the digis this lane counted
#pragma unroll 1
    for (uint32_t k = k0; k < k1; ++k) {
      const uint32_t t = 32u * k + lane, key = s.dkey[t];
      if (key == INVALID) continue;
      const uint32_t r = key >> 17;
      if (s.run_bad[r]) continue;  // the overflow kernel finishes this run
      const uint32_t ev = s.run_key[r] >> 16;
      ev_lo = ev < ev_lo ? ev : ev_lo; ev_hi = ev > ev_hi ? ev : ev_hi;
      const uint32_t lab = s.label[t];
      uint32_t so; int32_t cl = -1;
      if (lab == MARK_DUP) { so = ST_DUP; cntA += 1u; }
      else if (lab == MARK_BELOW) { so = ST_BELOW; cntA += 0x10000u; }
      else {
        const uint32_t id = lid[lab];
        if (id != NO_ID) { so = ST_OK; cl = (int32_t)id; cntB += 1u; } else { so = ST_CUT; cntB += 0x10000u; }
        n_pre += lab == t ? 1u : 0u;
      }
      c.d_status[b + t] = (uint8_t)so; c.d_clus[b + t] = cl;
    }
    // counters: one event per warp in the common case -> warp sums, lane 0 adds; else every digi adds its own
    {
      const uint32_t lo = __reduce_min_sync(FULL, ev_lo), hi = __reduce_max_sync(FULL, ev_hi);
      if (lo == NOKEY) {
        // no counted digi in this warp
      } else if (lo == hi) {
        const uint32_t a = __reduce_add_sync(FULL, cntA), bb = __reduce_add_sync(FULL, cntB);
        const uint32_t p = __reduce_add_sync(FULL, n_pre);
        if (lane == 0) {
          uint32_t* ec = c.ev_cnt + (size_t)lo * EC_STRIDE;
          if (a & 0xFFFFu) atomicAdd(ec + EC_DUP, a & 0xFFFFu);
          if (a >> 16) atomicAdd(ec + EC_BELOW, a >> 16);
          if (bb & 0xFFFFu) atomicAdd(ec + EC_OK, bb & 0xFFFFu);
          if (bb >> 16) atomicAdd(ec + EC_CUT, bb >> 16);
          if (p) atomicAdd(ec + EC_PRECUT, p);
        }
      } else {
        for (uint32_t k = k0; k < k1; ++k) {
          const uint32_t t = 32u * k + lane, key = s.dkey[t];
          if (key == INVALID) continue;
          const uint32_t r = key >> 17;
          if (s.run_bad[r]) continue;
          uint32_t* ec = c.ev_cnt + (size_t)(s.run_key[r] >> 16) * EC_STRIDE;
          const uint32_t lab = s.label[t];
          if (lab == MARK_DUP) atomicAdd(ec + EC_DUP, 1u);
          else if (lab == MARK_BELOW) atomicAdd(ec + EC_BELOW, 1u);
          else {
            atomicAdd(ec + (lid[lab] != NO_ID ? EC_OK : EC_CUT), 1u);
            if (lab == t) atomicAdd(ec + EC_PRECUT, 1u);
          }
        }
      }
    }
    __syncwarp();  // shared state is rewritten by the next chunk
  }
}

}  // namespace

static inline int grid_for(uint32_t work_items, uint32_t per_block, int cap_blocks) {
  uint64_t b = ((uint64_t)work_items + per_block - 1) / per_block;
  if (b < 1) b = 1;
  return (int)(b < (uint64_t)cap_blocks ? b : (uint64_t)cap_blocks);
}

void launch_init(const Chunk& c, uint32_t n_total, int n_sm, cudaStream_t stream) {
  const uint32_t Ec = c.e1 - c.e0;
  init_kernel<<<grid_for(Ec * c.M, 256, n_sm * 8), 256, 0, stream>>>(c, n_total);
}

cudaError_t configure_fused_kernel() {
  return cudaFuncSetAttribute(fused_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(WPB * sizeof(WarpSmem)));
}

void launch_fused(const Chunk& c, uint32_t words_bound, int n_sm, cudaStream_t stream) {
  fused_kernel<<<grid_for(words_bound + 31u, WPB * HC, n_sm * 8), FT, WPB * sizeof(WarpSmem), stream>>>(c);
}

}  // namespace pix
