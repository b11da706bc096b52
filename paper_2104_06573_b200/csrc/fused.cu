// fused.cu -- init, and the fused tile kernel: a1 decode (S1-S6), a2 calibrate (S7-S9), a3 module
// boundaries (S11, S12), a4 findClus (S10, S13) and a5 sums / charge cut / renumber / temp records (S9, S14,
// S18) of the path PAPER.md:31 describes ("unpacks them, calibrates the individual pixels, and clusters the
// pixels on each detector module"), in ONE pass over the raw words.
//
// A block takes a tile of 1024 consecutive words (4 per thread, one 128-bit load).  A module's decodable words
// form one run (S11); a run belongs to the tile that holds its first word.  The block
//   A  clears its position hash; warp 0 looks back for the last decodable word before the tile (carry-in run)
//   B  decodes + calibrates its words, stores module/row/col/charge, finds run starts with a ballot/shuffle
//      "previous decodable word" scan, numbers the tile's runs with a block prefix sum, and inserts every owned
//      decodable digi into the position hash keyed by (run, row, col); equal keys keep the lowest digi (S10)
//   C  meanwhile warp 0 looks ahead (up to 512 more words) for the rest of the tile's last run
//   D  every warp looks up the forward neighbours of its digis, compacts the adjacent pairs into a dense edge
//      list and unites them (lock-free min-index union-find, all lanes busy)
//   E  roots store, members atomically add: charge, charge*col, charge*row (u32) and the pixel count
//   F  surviving roots (Q >= cut) are numbered in digi order per run (block prefix sum), temp records written
//   G  final status and clus of every word the tile owns
// Runs that do not fit the window or the hash, tiles with more than RCAP runs and charge sums that could
// overflow 32 bits go to the overflow list (cluster.cu).  Nothing here is shared with oracle/.
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

// ------------------------------------------------------------------ the fused tile kernel
constexpr int FT = 256;                   // threads per block
constexpr int FW = FT / 32;
constexpr uint32_t TW = FT * 4;           // words per tile
constexpr uint32_t AHEAD = 512;           // look-ahead for the tile's last run
constexpr uint32_t CW = TW + AHEAD;       // window
constexpr uint32_t TABN = 8192;           // hash slots
constexpr uint32_t RCAP = 254;            // runs a tile can own
constexpr uint32_t EDGE_CAP = CW / FW;    // edge slots per warp (in Smem::q)
constexpr uint32_t EMPTY = 0xFFFFFFFFu, INVALID = 0xFFFFFFFFu, NO_SLOT = 0xFFFFFFFFu;
constexpr uint32_t MARK_DUP = 0xFFFFFFFEu, MARK_BELOW = 0xFFFFFFFDu;  // label of a digi that is not live
constexpr uint32_t Q_SAFE = 0xFFFFFFFFu / 415u;  // sum(e*col), sum(e*row) fit 32 bits while sum(e) <= Q_SAFE
constexpr uint32_t HASH_MUL = 0x9E3779B1u;
static_assert(TABN == 8192 && CW <= 2048 && 2 * CW <= TABN, "slot layout: 11-bit bucket, 17-bit tag, 11-bit digi");

// digi key inside the window: run (11 bits) | row (8 bits) | col (9 bits).  Neighbour keys are key+1 (col+1)
// and key+512-1, +512, +512+1 (row+1): col 416..511 and row 160..255 never occur, so no bounds checks (S13).
struct __align__(16) Smem {
  uint32_t tab[TABN];    // position hash (see hinsert), EMPTY-filled.  After phase D: sx = tab, sy = tab + CW
  uint32_t dkey[CW];     // key of the digi in window slot d (word tBeg + d), INVALID if not owned / undecodable
  uint32_t label[CW];    // union-find parent (low 16 bits) | members added << 16, or MARK_*
  uint32_t q[CW];        // phase D: per-warp edge lists; then root: charge sum; after phase F: local id or NO_INDEX
  uint16_t chg[CW];      // charge; after phase E: the list of surviving roots
  uint32_t run_ifirst[RCAP + 2];  // event-relative index of the run's first digi
  uint16_t run_first[RCAP + 2];   // window slot of the run's first digi
  uint16_t run_base[RCAP + 2];    // survivors before the run
  uint8_t run_bad[RCAP + 2];      // the run is left to the overflow kernel
  uint2 warp_last[FW];
  uint32_t warp_sum[FW];
  uint2 carry;
  uint32_t n_tot;
};

// Position hash: 2048 buckets of 4 slots, one 128-bit shared load per lookup.  h = key * HASH_MUL mod 2^28 is a
// bijection on the 28-bit keys; bucket = top 11 bits of h, tag = the other 17, so (bucket, tag) names the key
// exactly and no second load is needed to verify a hit.  A key whose home bucket is full goes to the next
// bucket(s) and records the displacement.  Slot = 0 | disp (2) | tag (17) | digi (11) | below_threshold (1);
// slots of a bucket fill in order and are never emptied, equal keys meet in one slot and keep the lowest digi (S10).
constexpr uint32_t NBUCKET = TABN / 4, MAX_DISP = 3, TAG_BITS = 17, TAG_MASK = (1u << TAG_BITS) - 1u;
__device__ __forceinline__ uint32_t hmix(uint32_t key) { return (key * HASH_MUL) & 0x0FFFFFFFu; }

// returns the slot index, or NO_SLOT: no room within MAX_DISP buckets (the run then goes to the overflow kernel)
__device__ __forceinline__ uint32_t hinsert(Smem& s, uint32_t key, uint32_t d, uint32_t below) {
  const uint32_t h = hmix(key), tag = h & TAG_MASK;
  uint32_t p = (h >> TAG_BITS) * 4u;
#pragma unroll 1
  for (uint32_t i = 0; i < 4u * (MAX_DISP + 1u); ++i, p = (p + 1u) & (TABN - 1u)) {
    const uint32_t want = ((i >> 2) << TAG_BITS) | tag, mine = (want << 12) | (d << 1) | below;
    const uint32_t old = atomicCAS(&s.tab[p], EMPTY, mine);
    if (old == EMPTY) return p;
    if ((old >> 12) == want) { atomicMin(&s.tab[p], mine); return p; }  // same pixel: the lowest digi owns it
  }
  return NO_SLOT;
}
__device__ __forceinline__ uint32_t half_match(const uint4& e, uint32_t want) {
  uint32_t r = EMPTY;
  if ((e.w >> 12) == want) r = e.w;
  if ((e.z >> 12) == want) r = e.z;
  if ((e.y >> 12) == want) r = e.y;
  if ((e.x >> 12) == want) r = e.x;
  return r;
}
__device__ __noinline__ uint32_t hfind_slow(const Smem& s, uint32_t key) {
  const uint32_t h = hmix(key), tag = h & TAG_MASK;
  uint32_t b = h >> TAG_BITS;
  for (uint32_t i = 1; i <= MAX_DISP; ++i) {  // the buckets after the (full) home bucket
    b = (b + 1u) & (NBUCKET - 1u);
    const uint4 e = *reinterpret_cast<const uint4*>(&s.tab[b * 4u]);
    const uint32_t r = half_match(e, (i << TAG_BITS) | tag);
    if (r != EMPTY) return r;
    if (e.w == EMPTY) return EMPTY;
  }
  return EMPTY;
}
// slot contents of `key`, or EMPTY
__device__ __forceinline__ uint32_t hfind(const Smem& s, uint32_t key) {
  const uint32_t h = hmix(key), want = h & TAG_MASK;
  const uint4 e = *reinterpret_cast<const uint4*>(&s.tab[(h >> TAG_BITS) * 4u]);
  uint32_t r = half_match(e, want);
  if (r == EMPTY && e.w != EMPTY) r = hfind_slow(s, key);  // home bucket full, no match (rare): displaced keys
  return r;
}
__device__ __forceinline__ uint32_t slot_digi(uint32_t e) { return (e >> 1) & 0x7FFu; }

// union-find on s.label (phase D only: high halves are zero); labels strictly decrease along parents
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
  while (true) {
    a = uf_find(L, a); b = uf_find(L, b);
    if (a == b) return;
    if (a < b) { const uint32_t t = a; a = b; b = t; }
    const uint32_t old = atomicMin(L + a, b);  // hook the larger root under the smaller
    if (old == a) return;
    a = old;                                   // a was no longer a root: keep merging its parent with b
  }
}

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v, uint32_t lane) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, v, d);
    if (lane >= (uint32_t)d) v += t;
  }
  return v;
}

// phase D, part 1, for the 4 digis of window slots d0..d0+3 (active lanes; the call is warp-uniform): duplicate
// check and forward-neighbour lookups; the adjacent pairs go to the warp's edge list (ballot compaction).
// Forward neighbours (S13): E (r, c+1), SW (r+1, c-1), S (r+1, c), SE (r+1, c+1).  When S is live, SW and SE are
// joined to it by their own E edges, so d-S alone is enough.
template <bool NATIVE>
__device__ __forceinline__ void phase_edges(Smem& s, uint32_t d0, bool active, const uint32_t (&slot)[4], uint32_t* elist,
                                            uint32_t& ne, uint32_t lt_mask) {
  uint4 k4 = make_uint4(INVALID, INVALID, INVALID, INVALID);
  if (active) k4 = *reinterpret_cast<const uint4*>(&s.dkey[d0]);
  const uint32_t k[4] = {k4.x, k4.y, k4.z, k4.w};
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const uint32_t key = k[j], d = d0 + j;
    bool live = key != INVALID;
    // own pixel: a tile word remembers its slot; a look-ahead word (inserted by warp 0) looks itself up
    const uint32_t own = NATIVE ? s.tab[slot[j] & (TABN - 1u)] : hfind(s, key);
    const uint32_t eE = hfind(s, key + 1u), eSW = hfind(s, key + 511u), eS = hfind(s, key + 512u),
                   eSE = hfind(s, key + 513u);
    if (live && slot_digi(own) != d) { s.label[d] = MARK_DUP; live = false; }  // S10: an earlier word owns this pixel
    if (own & 1u) live = false;                                                // below threshold: joins nothing
    const bool hS = live && eS != EMPTY && !(eS & 1u);
    const bool f[3] = {live && eE != EMPTY && !(eE & 1u), hS || (live && eSW != EMPTY && !(eSW & 1u)),
                       live && !hS && eSE != EMPTY && !(eSE & 1u)};
    const uint32_t nb[3] = {slot_digi(eE), slot_digi(hS ? eS : eSW), slot_digi(eSE)};
#pragma unroll
    for (int t = 0; t < 3; ++t) {
      const uint32_t mask = __ballot_sync(0xFFFFFFFFu, f[t]);
      if (f[t]) {
        const uint32_t pos = ne + __popc(mask & lt_mask);
        if (pos < EDGE_CAP) elist[pos] = d | (nb[t] << 16);
        else uf_unite(s.label, d, nb[t]);  // list full (dense window): unite in place
      }
      ne += __popc(mask);
    }
  }
}

// phase E1: roots store their own contribution
__device__ __forceinline__ void phase_roots(Smem& s, uint32_t d0) {
  uint32_t* sx = s.tab; uint32_t* sy = s.tab + CW;
  const uint4 l4 = *reinterpret_cast<const uint4*>(&s.label[d0]);
  const uint32_t l[4] = {l4.x, l4.y, l4.z, l4.w};
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const uint32_t d = d0 + j;
    if (l[j] != d) continue;
    const uint32_t key = s.dkey[d], e = s.chg[d];
    s.q[d] = e; sx[d] = e * (key & 511u); sy[d] = e * ((key >> 9) & 255u);
  }
}
// phase E2: members find their root, flatten, and add their contribution
__device__ __forceinline__ void phase_members(Smem& s, uint32_t d0) {
  uint32_t* sx = s.tab; uint32_t* sy = s.tab + CW;
  volatile uint32_t* L = s.label;
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const uint32_t d = d0 + j;
    uint32_t p = L[d];
    if (p >= CW || p == d) continue;  // MARK_*, roots (their high half may already count members)
    uint32_t r = p;
    while (true) { const uint32_t n = L[r] & 0xFFFFu; if (n == r) break; r = n; }
    L[d] = r;
    const uint32_t key = s.dkey[d], e = s.chg[d];
    atomicAdd(&s.q[r], e);
    atomicAdd(&sx[r], e * (key & 511u));
    atomicAdd(&sy[r], e * ((key >> 9) & 255u));
    atomicAdd(&s.label[r], 0x10000u);
  }
}

__device__ __forceinline__ bool is_root(uint32_t lab, uint32_t d) { return (lab & 0xFFFFu) == d && (lab >> 16) < 0x8000u; }

__global__ void __launch_bounds__(FT, 4) fused_kernel(const __grid_constant__ Chunk c) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Smem& s = *reinterpret_cast<Smem*>(smem_raw);
  const uint32_t Ec = c.e1 - c.e0, S = Ec * c.F;
  const uint32_t* __restrict__ segB = c.segB;
  const uint32_t gBeg = segB[0], gEnd = segB[S];
  if (gBeg >= gEnd) return;
  const uint32_t T0 = gBeg & ~3u;
  const uint32_t n_tiles = (gEnd - T0 + TW - 1u) / TW;
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const uint32_t lt_mask = (1u << lane) - 1u;

  for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const uint32_t tBeg = T0 + tile * TW, tEnd = tBeg + TW;
    // ================================================================== A: load; clear; segment; look-back
    const uint32_t g0 = tBeg + tid * 4u;
    const bool any = (g0 + 4u > gBeg) && (g0 < gEnd);
    const bool full = (g0 >= gBeg) && (g0 + 4u <= gEnd);
    uint32_t w[4] = {0u, 0u, 0u, 0u};
    if (full) {
      const uint4 v = __ldg(reinterpret_cast<const uint4*>(c.words + g0));
      w[0] = v.x; w[1] = v.y; w[2] = v.z; w[3] = v.w;
    } else if (any) {
#pragma unroll
      for (int j = 0; j < 4; ++j) if (g0 + j >= gBeg && g0 + j < gEnd) w[j] = __ldg(c.words + g0 + j);
    }
    {
      uint4* t4 = reinterpret_cast<uint4*>(s.tab);
      const uint4 e4 = make_uint4(EMPTY, EMPTY, EMPTY, EMPTY);
#pragma unroll
      for (int k = 0; k < (int)(TABN / 4 / FT); ++k) t4[tid + k * FT] = e4;
      if (tid < (RCAP + 2u) / 4u) reinterpret_cast<uint32_t*>(s.run_bad)[tid] = 0u;
    }
    // segment (event, FED) of the warp's first word inside the chunk
    uint32_t gw = tBeg + warp * 128u;
    gw = gw < gBeg ? gBeg : (gw >= gEnd ? gEnd - 1u : gw);
    const uint32_t sgw = warp_find_segment(segB, S, gw, lane);
    if (warp == 0) {  // last decodable word before the tile: its run may continue into the tile
      uint2 carry = make_uint2(NOKEY, 0u);
      uint32_t g = gw;  // words [gBeg, g) are still to be searched, backwards
      while (g > gBeg) {
        const bool in = lane < g - gBeg;
        const uint32_t gi = g - 1u - lane;
        uint32_t key = NOKEY;
        if (in) {
          uint32_t sg = sgw;
          while (segB[sg] > gi) --sg;  // segB[0] = gBeg <= gi
          const uint32_t er = sg / c.F, fed = sg - er * c.F;
          uint32_t m, r, cc;
          if (decode_word(c.cab, c.words[gi], fed << 11, m, r, cc) == ST_OK) key = (er << 16) | m;
        }
        const uint32_t b = __ballot_sync(0xFFFFFFFFu, key != NOKEY);
        if (b) {
          const int src = __ffs(b) - 1;
          carry.x = __shfl_sync(0xFFFFFFFFu, key, src);
          carry.y = g - 1u - (uint32_t)src;
          break;
        }
        g = (g - gBeg > 32u) ? g - 32u : gBeg;
      }
      if (lane == 0) s.carry = carry;
    }

    // ================================================================== B: decode, calibrate, run starts
    uint32_t st[4], key[4], pos[4];
    int32_t chg[4];
    uint32_t tkey = NOKEY, tg = 0u;
    uint32_t inmask = 0u;  // words of this thread inside the chunk
    {
      uint32_t mod[4], row[4], col[4];
      uint32_t sg = sgw;
      if (any) {
        const uint32_t gf = g0 < gBeg ? gBeg : g0;
        while (sg + 1u < S && segB[sg + 1u] <= gf) ++sg;
      }
      uint32_t er = sg / c.F, fed = sg - er * c.F;
      uint32_t nextB = segB[sg + 1u];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const uint32_t g = g0 + j;
        st[j] = 0xFFu; key[j] = NOKEY; pos[j] = 0u; mod[j] = row[j] = col[j] = 0xFFFFu; chg[j] = 0;
        if (!any || g < gBeg || g >= gEnd) continue;
        inmask |= 1u << j;
        if (g >= nextB) {  // rare: the thread's words straddle a FED / event boundary
          while (sg + 1u < S && segB[sg + 1u] <= g) ++sg;
          er = sg / c.F; fed = sg - er * c.F; nextB = segB[sg + 1u];
        }
        uint32_t m, r, cc;
        st[j] = decode_word(c.cab, w[j], fed << 11, m, r, cc);
        if (st[j] == ST_OK) {
          mod[j] = m; row[j] = r; col[j] = cc;
          const float2 gp = __ldg(c.gp + (m * (uint32_t)COLS + cc));  // S8: one pair per (module, col)
          chg[j] = calibrate(c, w[j] & 255u, gp);
          if (chg[j] < c.thr) st[j] = ST_BELOW;                      // S9
          key[j] = (er << 16) | m;
          pos[j] = (r << 9) | cc;
          tkey = key[j]; tg = g;
        } else {
          atomicAdd(c.ev_cnt + (size_t)er * EC_STRIDE + (st[j] - ST_EMPTY), 1u);
        }
      }
      if (full) {
        *reinterpret_cast<ushort4*>(c.d_module + g0) = make_ushort4(mod[0], mod[1], mod[2], mod[3]);
        *reinterpret_cast<ushort4*>(c.d_row + g0) = make_ushort4(row[0], row[1], row[2], row[3]);
        *reinterpret_cast<ushort4*>(c.d_col + g0) = make_ushort4(col[0], col[1], col[2], col[3]);
        *reinterpret_cast<int4*>(c.d_charge + g0) = make_int4(chg[0], chg[1], chg[2], chg[3]);
      } else if (any) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          if (!(inmask >> j & 1u)) continue;
          const uint32_t g = g0 + j;
          c.d_module[g] = (uint16_t)mod[j]; c.d_row[g] = (uint16_t)row[j]; c.d_col[g] = (uint16_t)col[j];
          c.d_charge[g] = chg[j];
        }
      }
    }
    // ---- a3: previous decodable word of every thread (warp-shuffle last-valid scan + carries)
    const uint32_t has = __ballot_sync(0xFFFFFFFFu, tkey != NOKEY);
    const uint32_t below_l = has & lt_mask;
    {
      const int top = has ? 31 - __clz(has) : 0;
      const uint32_t lk = __shfl_sync(0xFFFFFFFFu, tkey, top), lg = __shfl_sync(0xFFFFFFFFu, tg, top);
      if (lane == 0) s.warp_last[warp] = has ? make_uint2(lk, lg) : make_uint2(NOKEY, 0u);
    }
    const int src = below_l ? 31 - __clz(below_l) : 0;
    uint32_t pkey = __shfl_sync(0xFFFFFFFFu, tkey, src);
    uint32_t pg = __shfl_sync(0xFFFFFFFFu, tg, src);
    __syncthreads();  // #1: warp_last, carry, cleared hash
    if (!below_l) {  // nothing decodable earlier in this warp: take the nearest earlier warp, else the look-back
      uint2 cin = s.carry;
      for (int wq = (int)warp - 1; wq >= 0; --wq) {
        const uint2 v = s.warp_last[wq];
        if (v.x != NOKEY) { cin = v; break; }
      }
      pkey = cin.x; pg = cin.y;
    }
    uint32_t startmask = 0u;
    uint32_t ifirst[4] = {0u, 0u, 0u, 0u};
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      if (key[j] == NOKEY) continue;
      if (key[j] != pkey) {
        startmask |= 1u << j;
        ifirst[j] = run_start(c, key[j], g0 + j);
        if (pkey != NOKEY) run_end(c, pkey, pg);
      }
      pkey = key[j]; pg = g0 + j;
    }
    // the tile's last decodable word: its run is the one the look-ahead completes
    uint2 lastv = s.carry;
    bool tile_has = false;
    for (int wq = FW - 1; wq >= 0; --wq) {
      const uint2 v = s.warp_last[wq];
      if (v.x != NOKEY) { lastv = v; tile_has = true; break; }
    }
    if (tile == n_tiles - 1u && tid == 0 && lastv.x != NOKEY) run_end(c, lastv.x, lastv.y);  // the chunk's last run
    // ---- number the tile's runs: block prefix sum of the run starts
    const uint32_t nst = __popc(startmask);
    const uint32_t incl = warp_incl_scan(nst, lane);
    if (lane == 31) s.warp_sum[warp] = incl;
    __syncthreads();  // #2
    uint32_t rbase = incl - nst, n_runs = 0;
#pragma unroll
    for (int q = 0; q < FW; ++q) { const uint32_t v = s.warp_sum[q]; if (q < (int)warp) rbase += v; n_runs += v; }
    const uint32_t R = n_runs < RCAP ? n_runs : RCAP;  // runs this tile owns; the last one may reach past the tile
    if (n_runs == 0u) {
      // nothing owned: only the undecodable words of the tile are finished here
      if (full && (st[0] >= ST_EMPTY) && (st[1] >= ST_EMPTY) && (st[2] >= ST_EMPTY) && (st[3] >= ST_EMPTY)) {
        *reinterpret_cast<uchar4*>(c.d_status + g0) = make_uchar4(st[0], st[1], st[2], st[3]);
        *reinterpret_cast<int4*>(c.d_clus + g0) = make_int4(-1, -1, -1, -1);
      } else {
#pragma unroll
        for (int j = 0; j < 4; ++j)
          if ((inmask >> j & 1u) && st[j] >= ST_EMPTY) { c.d_status[g0 + j] = (uint8_t)st[j]; c.d_clus[g0 + j] = -1; }
      }
      __syncthreads();
      continue;
    }
    // stage the window slots of this thread's words and insert the owned ones into the hash
    uint32_t runl[4], slot[4];
    {
      uint32_t r = rbase;
      uint32_t dk[4], lb[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        if (startmask >> j & 1u) {
          ++r;
          if (r <= RCAP) { s.run_first[r] = (uint16_t)(tid * 4u + j); s.run_ifirst[r] = ifirst[j]; }
          else push_overflow(c, key[j]);
        }
        runl[j] = (key[j] != NOKEY && r >= 1u && r <= RCAP) ? r : 0u;  // 0: not owned by this tile
        dk[j] = runl[j] ? ((runl[j] << 17) | pos[j]) : INVALID;
        lb[j] = (!runl[j] || st[j] == ST_BELOW) ? MARK_BELOW : tid * 4u + j;
      }
      *reinterpret_cast<uint4*>(&s.dkey[tid * 4u]) = make_uint4(dk[0], dk[1], dk[2], dk[3]);
      *reinterpret_cast<uint4*>(&s.label[tid * 4u]) = make_uint4(lb[0], lb[1], lb[2], lb[3]);
      *reinterpret_cast<uint2*>(&s.chg[tid * 4u]) =
          make_uint2((uint32_t)chg[0] | ((uint32_t)chg[1] << 16), (uint32_t)chg[2] | ((uint32_t)chg[3] << 16));
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        slot[j] = 0u;
        if (!runl[j]) continue;
        slot[j] = hinsert(s, dk[j], tid * 4u + j, st[j] == ST_BELOW ? 1u : 0u);
        if (slot[j] == NO_SLOT) s.run_bad[runl[j]] = 1;
      }
    }

    // ================================================================== C: look-ahead for the last run (warp 0)
    if (warp == 0) {
      uint32_t n_tot = TW;
      if (tile_has && n_runs <= RCAP && tEnd < gEnd) {
        const uint32_t keyR = lastv.x;
        uint32_t p = tEnd;
        bool ended = false;
        uint32_t sg = warp_find_segment(segB, S, tEnd, lane);
        while (!ended && p < gEnd && p < tEnd + AHEAD) {
          const uint32_t x0 = p + lane * 4u;
          uint32_t ww[4] = {0u, 0u, 0u, 0u};
          if (x0 + 4u <= gEnd) {
            const uint4 v = __ldg(reinterpret_cast<const uint4*>(c.words + x0));
            ww[0] = v.x; ww[1] = v.y; ww[2] = v.z; ww[3] = v.w;
          } else {
#pragma unroll
            for (int j = 0; j < 4; ++j) if (x0 + j < gEnd) ww[j] = __ldg(c.words + x0 + j);
          }
          uint32_t dk[4], lb[4], ch[4];
          int stop = 4;  // first word of this lane that ends the run (another run's decodable word, or chunk end)
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const uint32_t g = x0 + j;
            dk[j] = INVALID; lb[j] = MARK_BELOW; ch[j] = 0u;
            if (g >= gEnd) { if (stop == 4) stop = j; continue; }
            while (sg + 1u < S && segB[sg + 1u] <= g) ++sg;
            const uint32_t er = sg / c.F, fed = sg - er * c.F;
            uint32_t m, r, cc;
            const uint32_t stj = decode_word(c.cab, ww[j], fed << 11, m, r, cc);
            if (stj != ST_OK) continue;
            if (((er << 16) | m) != keyR) { if (stop == 4) stop = j; continue; }
            if (stop != 4) continue;
            const float2 gp = __ldg(c.gp + (m * (uint32_t)COLS + cc));
            const int32_t e = calibrate(c, ww[j] & 255u, gp);
            dk[j] = (R << 17) | (r << 9) | cc; ch[j] = (uint32_t)e;
            lb[j] = (e < c.thr) ? MARK_BELOW : (g - tBeg);
          }
          const uint32_t stopped = __ballot_sync(0xFFFFFFFFu, stop != 4);
          const uint32_t first_stop = stopped ? (uint32_t)(__ffs(stopped) - 1) : 32u;
          if (lane > first_stop) {
#pragma unroll
            for (int j = 0; j < 4; ++j) { dk[j] = INVALID; lb[j] = MARK_BELOW; }
          }
          const uint32_t d0 = x0 - tBeg;
          *reinterpret_cast<uint4*>(&s.dkey[d0]) = make_uint4(dk[0], dk[1], dk[2], dk[3]);
          *reinterpret_cast<uint4*>(&s.label[d0]) = make_uint4(lb[0], lb[1], lb[2], lb[3]);
          *reinterpret_cast<uint2*>(&s.chg[d0]) = make_uint2(ch[0] | (ch[1] << 16), ch[2] | (ch[3] << 16));
#pragma unroll
          for (int j = 0; j < 4; ++j)
            if (dk[j] != INVALID && hinsert(s, dk[j], d0 + j, lb[j] == MARK_BELOW ? 1u : 0u) == NO_SLOT) s.run_bad[R] = 1;
          if (stopped) { ended = true; n_tot = (p - tBeg) + (first_stop + 1u) * 4u; }
          else { p += 128u; n_tot = p - tBeg; }
        }
        if (!ended && p < gEnd) {  // the run does not fit the window: the overflow kernel takes it
          if (lane == 0) s.run_bad[R] = 1;
          n_tot = TW;
        }
      }
      if (lane == 0) s.n_tot = n_tot;
    }
    __syncthreads();  // #3: hash complete
    const uint32_t n_tot = s.n_tot;
    const uint32_t d0n = tid * 4u, d0x = TW + tid * 4u;
    const bool has_ext = d0x < n_tot;
    const bool warp_ext = TW + warp * 128u < n_tot;  // warp-uniform: some lane of this warp has look-ahead slots

    // ================================================================== D: neighbours -> edge list -> unions
    {
      uint32_t* elist = s.q + warp * EDGE_CAP;
      uint32_t ne = 0u;
      phase_edges<true>(s, d0n, true, slot, elist, ne, lt_mask);
      if (warp_ext) phase_edges<false>(s, d0x, has_ext, slot, elist, ne, lt_mask);
      __syncwarp();
      ne = ne < EDGE_CAP ? ne : EDGE_CAP;
      for (uint32_t i = lane; i < ne; i += 32u) {
        const uint32_t e = elist[i];
        uf_unite(s.label, e & 0xFFFFu, e >> 16);
      }
    }
    __syncthreads();  // #4: components complete; the hash is dead, its memory becomes sx / sy
    // ================================================================== E: cluster sums
    phase_roots(s, d0n);
    if (has_ext) phase_roots(s, d0x);
    __syncthreads();  // #5
    phase_members(s, d0n);
    if (has_ext) phase_members(s, d0x);
    __syncthreads();  // #6
    // ================================================================== F: cut, renumber, temp records
    uint32_t labn[4], labx[4] = {MARK_BELOW, MARK_BELOW, MARK_BELOW, MARK_BELOW};
    uint32_t survn = 0u, survx = 0u, rootn = 0u, rootx = 0u;
    {
      const uint4 l4 = *reinterpret_cast<const uint4*>(&s.label[d0n]);
      labn[0] = l4.x; labn[1] = l4.y; labn[2] = l4.z; labn[3] = l4.w;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        if (!runl[j] || !is_root(labn[j], d0n + j)) continue;
        rootn |= 1u << j;
        const uint32_t Q = s.q[d0n + j];
        if (Q > Q_SAFE) s.run_bad[runl[j]] = 1;                  // 32-bit weighted sums may have wrapped
        if ((long long)Q >= (long long)c.cut) survn |= 1u << j;  // S9: equality keeps
      }
      if (has_ext) {
        const uint4 x4 = *reinterpret_cast<const uint4*>(&s.label[d0x]);
        const uint4 k4 = *reinterpret_cast<const uint4*>(&s.dkey[d0x]);
        const uint32_t kx[4] = {k4.x, k4.y, k4.z, k4.w};
        labx[0] = x4.x; labx[1] = x4.y; labx[2] = x4.z; labx[3] = x4.w;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          if (kx[j] == INVALID) { labx[j] = INVALID; continue; }  // INVALID label: slot not in the run
          if (!is_root(labx[j], d0x + j)) continue;
          rootx |= 1u << j;
          const uint32_t Q = s.q[d0x + j];
          if (Q > Q_SAFE) s.run_bad[R] = 1;
          if ((long long)Q >= (long long)c.cut) survx |= 1u << j;
        }
      }
    }
    const uint32_t packed = __popc(survn) | (__popc(survx) << 16);
    const uint32_t pincl = warp_incl_scan(packed, lane);
    if (lane == 31) s.warp_sum[warp] = pincl;
    __syncthreads();  // #7
    uint32_t pbase = pincl - packed, ptot = 0;
#pragma unroll
    for (int q = 0; q < FW; ++q) { const uint32_t v = s.warp_sum[q]; if (q < (int)warp) pbase += v; ptot += v; }
    const uint32_t totN = ptot & 0xFFFFu, totAll = totN + (ptot >> 16);
    const uint32_t exclN = pbase & 0xFFFFu, exclX = totN + (pbase >> 16);
    {
      uint32_t r = rbase;
#pragma unroll
      for (int j = 0; j < 4; ++j)
        if (startmask >> j & 1u) {
          ++r;
          if (r <= RCAP) s.run_base[r] = (uint16_t)(exclN + __popc(survn & ((1u << j) - 1u)));
        }
      if (tid == 0) s.run_base[R + 1u] = (uint16_t)totAll;
    }
    // surviving roots, densely listed in digi order (the charge array is dead by now)
    uint16_t* slist = s.chg;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      if (rootn >> j & 1u) {
        if (survn >> j & 1u) slist[exclN + __popc(survn & ((1u << j) - 1u))] = (uint16_t)(d0n + j);
        else s.q[d0n + j] = NO_INDEX;
      }
      if (rootx >> j & 1u) {
        if (survx >> j & 1u) slist[exclX + __popc(survx & ((1u << j) - 1u))] = (uint16_t)(d0x + j);
        else s.q[d0x + j] = NO_INDEX;
      }
    }
    __syncthreads();  // #8: run_base, run_bad, survivor list final
    {
      uint32_t r = rbase;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        if (!(startmask >> j & 1u)) continue;
        ++r;
        if (r > RCAP) continue;
        if (s.run_bad[r]) push_overflow(c, key[j]);
        else c.n_clus[(key[j] >> 16) * c.M + (key[j] & 0xFFFFu)] = (uint32_t)s.run_base[r + 1u] - s.run_base[r];
      }
      // one survivor per thread: local id (S14) and temp record (S18)
      const uint32_t* sx = s.tab; const uint32_t* sy = s.tab + CW;
      const uint32_t relBeg = tBeg - gBeg;  // may wrap for the chunk's first tile; only used added to a slot >= gBeg - tBeg
      for (uint32_t i = tid; i < totAll; i += FT) {
        const uint32_t d = slist[i];
        const uint32_t rr = s.dkey[d] >> 17;
        const uint32_t id = i - s.run_base[rr];
        const uint32_t Q = s.q[d];
        s.q[d] = id;
        if (s.run_bad[rr]) continue;
        const uint32_t rf = s.run_first[rr];
        const uint32_t o = relBeg + rf + id;
        c.t_first[o] = s.run_ifirst[rr] + (d - rf);
        c.t_npix[o] = 1u + (s.label[d] >> 16);
        c.t_charge[o] = Q;
        c.t_x[o] = (float)sx[d] / (float)Q;   // S18; exact integer sums, one rounding each (within 1e-5)
        c.t_y[o] = (float)sy[d] / (float)Q;
      }
    }
    __syncthreads();  // #9: q holds the local ids
    // ================================================================== G: final status and clus, counters
    uint32_t cntA = 0u, cntB = 0u, n_pre = 0u;  // dup | below << 16 ; ok | cut << 16 ; roots
    uint32_t ev_lo = NOKEY, ev_hi = 0u;         // events of the digis this thread counted
    uint32_t cmask = 0u, cmaskx = 0u;           // digis counted (native, look-ahead)
    {
      int32_t cl[4];
      uint32_t so[4];
      bool mine_all = full;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        cl[j] = -1; so[j] = st[j];
        if (st[j] >= ST_EMPTY) continue;             // undecodable: status as decoded (0xFF outside the chunk)
        if (!runl[j] || s.run_bad[runl[j]]) { mine_all = false; so[j] = 0xFFu; continue; }
        cmask |= 1u << j;
        const uint32_t e = key[j] >> 16;
        ev_lo = e < ev_lo ? e : ev_lo; ev_hi = e > ev_hi ? e : ev_hi;
        const uint32_t lab = labn[j];
        if (lab == MARK_DUP) { so[j] = ST_DUP; cntA += 1u; }
        else if (lab == MARK_BELOW) { so[j] = ST_BELOW; cntA += 0x10000u; }
        else {
          const uint32_t id = s.q[lab & 0xFFFFu];
          if (id != NO_INDEX) { so[j] = ST_OK; cl[j] = (int32_t)id; cntB += 1u; } else { so[j] = ST_CUT; cntB += 0x10000u; }
          n_pre += rootn >> j & 1u;
        }
      }
      if (mine_all) {
        *reinterpret_cast<uchar4*>(c.d_status + g0) = make_uchar4(so[0], so[1], so[2], so[3]);
        *reinterpret_cast<int4*>(c.d_clus + g0) = make_int4(cl[0], cl[1], cl[2], cl[3]);
      } else {
#pragma unroll
        for (int j = 0; j < 4; ++j)
          if ((inmask >> j & 1u) && so[j] != 0xFFu) { c.d_status[g0 + j] = (uint8_t)so[j]; c.d_clus[g0 + j] = cl[j]; }
      }
    }
    const uint32_t er_x = lastv.x >> 16;  // the look-ahead digis belong to the run of the tile's last decodable word
    if (has_ext && !s.run_bad[R]) {
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const uint32_t lab = labx[j];
        if (lab == INVALID) continue;
        cmaskx |= 1u << j;
        uint32_t sj; int32_t cj = -1;
        if (lab == MARK_DUP) { sj = ST_DUP; cntA += 1u; }
        else if (lab == MARK_BELOW) { sj = ST_BELOW; cntA += 0x10000u; }
        else {
          const uint32_t id = s.q[lab & 0xFFFFu];
          if (id != NO_INDEX) { sj = ST_OK; cj = (int32_t)id; cntB += 1u; } else { sj = ST_CUT; cntB += 0x10000u; }
          n_pre += rootx >> j & 1u;
        }
        c.d_status[tBeg + d0x + j] = (uint8_t)sj; c.d_clus[tBeg + d0x + j] = cj;
      }
      if (cmaskx) { ev_lo = er_x < ev_lo ? er_x : ev_lo; ev_hi = er_x > ev_hi ? er_x : ev_hi; }
    }
    // counters: one event per warp in the common case -> warp sums, lane 0 adds; else every digi adds its own
    {
      const uint32_t lo = __reduce_min_sync(0xFFFFFFFFu, ev_lo), hi = __reduce_max_sync(0xFFFFFFFFu, ev_hi);
      if (lo == NOKEY) {
        // no counted digi in this warp
      } else if (lo == hi) {
        const uint32_t a = __reduce_add_sync(0xFFFFFFFFu, cntA), b = __reduce_add_sync(0xFFFFFFFFu, cntB);
        const uint32_t p = __reduce_add_sync(0xFFFFFFFFu, n_pre);
        if (lane == 0) {
          uint32_t* ec = c.ev_cnt + (size_t)lo * EC_STRIDE;
          if (a & 0xFFFFu) atomicAdd(ec + EC_DUP, a & 0xFFFFu);
          if (a >> 16) atomicAdd(ec + EC_BELOW, a >> 16);
          if (b & 0xFFFFu) atomicAdd(ec + EC_OK, b & 0xFFFFu);
          if (b >> 16) atomicAdd(ec + EC_CUT, b >> 16);
          if (p) atomicAdd(ec + EC_PRECUT, p);
        }
      } else {
#pragma unroll
        for (int half = 0; half < 2; ++half) {
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            if (!((half ? cmaskx : cmask) >> j & 1u)) continue;
            uint32_t* ec = c.ev_cnt + (size_t)(half ? er_x : (key[j] >> 16)) * EC_STRIDE;
            const uint32_t lab = half ? labx[j] : labn[j];
            if (lab == MARK_DUP) atomicAdd(ec + EC_DUP, 1u);
            else if (lab == MARK_BELOW) atomicAdd(ec + EC_BELOW, 1u);
            else {
              atomicAdd(ec + (s.q[lab & 0xFFFFu] != NO_INDEX ? EC_OK : EC_CUT), 1u);
              if ((half ? rootx : rootn) >> j & 1u) atomicAdd(ec + EC_PRECUT, 1u);
            }
          }
        }
      }
    }
    __syncthreads();  // #10: shared state is rewritten by the next tile
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
  return cudaFuncSetAttribute(fused_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem));
}

void launch_fused(const Chunk& c, uint32_t words_bound, int n_sm, cudaStream_t stream) {
  fused_kernel<<<grid_for(words_bound + 3u, TW, n_sm * 64), FT, sizeof(Smem), stream>>>(c);
}

}  // namespace pix
