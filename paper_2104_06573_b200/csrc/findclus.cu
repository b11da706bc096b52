// findclus.cu -- the warp cluster kernel: a4 findClus (S10, S13) and a5 sums / charge cut / renumber /
// temp records (S9, S14, S18) of the path PAPER.md:31 describes ("clusters the pixels on each detector module").
//
// The word stream is cut into home chunks of 128 words, one warp per chunk, 32 digis (one per lane) per round.
// A module's decodable words form one run (S11); a run belongs to the warp whose home chunk holds its first
// word (the start bits come from decode.cu).  Warps never wait for each other (no block barrier); all tables are
// per-warp shared memory.  A warp
//   A  clears its position hash and reads the start bits of its window (home chunk + up to 128 more words)
//   B  reads row / col / charge of the digis of its runs and inserts them into the position hash keyed by
//      (run, row, col); equal keys keep the lowest digi (S10)
//   D  looks up the forward neighbours of its digis, compacts the adjacent pairs into a dense edge list and
//      unites them (lock-free min-index union-find, all lanes busy)
//   E  every live digi adds charge | 1 << 24, charge*col, charge*row into its root's accumulators; dense root list
//   F  surviving roots (Q >= cut) are numbered in digi order per run (ballot/popc), temp records written
//   G  final status and clus of every digi the warp owns; per-event counters
// Runs that do not fit the 256-word window, chunks with more than RC runs and charge sums that could overflow
// 32 bits go to the overflow list (cluster.cu).  Nothing here is shared with oracle/.
#include "pix_common.cuh"

namespace pix {

namespace {

constexpr uint32_t NOKEY = 0xFFFFFFFFu;

__device__ __forceinline__ void push_overflow(const Chunk& c, uint32_t key) {
  const uint32_t i = atomicAdd(c.ctl + CTL_MID_COUNT, 1u);  // the warp-per-run kernel (findrun.cu) is next
  if (i < c.ovf_cap) c.mid_list[i] = (key >> 16) * c.M + (key & 0xFFFFu);
}

constexpr int WPB = 4;                    // warps per block (they share nothing but the block)
constexpr int FT = WPB * 32;
constexpr uint32_t HC = 128;              // words of a home chunk (rounds 0-3)
constexpr uint32_t MAXT = 256;            // window: home chunk + up to 4 extension rounds
constexpr uint32_t WTAB = 1024;           // hash slots per warp: 256 buckets of 4
constexpr uint32_t RC = 62;               // runs a warp can own
constexpr uint32_t ECAP = 256;            // edge list; flushed (united) when a round might not fit
constexpr uint32_t EMPTY = 0xFFFFFFFFu, INVALID = 0xFFFFFFFFu;
constexpr uint32_t MARK_DUP = 0xFFFFFFFEu, MARK_BELOW = 0xFFFFFFFDu;  // label of a digi that is not live
constexpr uint32_t Q_SAFE = 0xFFFFFFFFu / 415u;  // sum(e*col), sum(e*row) fit 32 bits while sum(e) <= Q_SAFE
constexpr uint32_t HASH_MUL = 0x9E3779B1u;
constexpr uint32_t KEY_BITS = 23, KEY_MASK = (1u << KEY_BITS) - 1u, TAG_BITS = 15, TAG_MASK = (1u << TAG_BITS) - 1u;
constexpr uint32_t NBUCKET = WTAB / 4, MAX_DISP = 3;
static_assert(((RC + 1u) << 17) <= (1u << KEY_BITS) && (1u << (KEY_BITS - TAG_BITS)) == NBUCKET && MAXT <= 256,
              "key: run (6 bits) | row (8) | col (9); slot: disp (2) | tag (15) | digi (8) | below (1)");

// digi key inside the window: run (6 bits) | row (8 bits) | col (9 bits).  Neighbour keys are key+1 (col+1)
// and key+512-1, +512, +512+1 (row+1): col 416..511 and row 160..255 never occur, so no bounds checks (S13).
struct __align__(16) WarpSmem {
  uint32_t tab[WTAB];      // position hash, EMPTY-filled.  After phase D: qn = tab, sx = tab + 256, sy = tab + 512, root list
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
static_assert(WTAB * 4 >= 3 * MAXT * 4 + MAXT, "the sums and the root list fit in tab");
static_assert(sizeof(WarpSmem) % 16 == 0, "per-warp slices stay 16-byte aligned");

// Position hash: 256 buckets of 4 slots, one 128-bit shared load per lookup and no probing loop on the common
// path.  h = key * HASH_MUL mod 2^23 is a bijection on the 23-bit keys; bucket = top 8 bits of h, tag = the
// other 15, so (bucket, tag) names the key exactly.  A key whose home bucket is full goes to the next bucket(s)
// and records the displacement: slot = 0 | disp (2) | tag (15) | digi (8) | below_threshold (1).  Slots of a
// bucket fill in order and are never emptied; equal keys meet in one slot and keep the lowest digi (S10).
__device__ __forceinline__ uint32_t hmix(uint32_t key) { return (key * HASH_MUL) & KEY_MASK; }

// 0: inserted; 1: the key was already there (a duplicate pixel, S10); 2: no room within MAX_DISP buckets.
// Not inlined: eight copies in the unrolled staging rounds cost more in instruction fetch than the call.
__device__ __noinline__ uint32_t hinsert(WarpSmem& s, uint32_t key, uint32_t t, uint32_t below) {
  const uint32_t h = hmix(key), tag = h & TAG_MASK;
  uint32_t p = (h >> TAG_BITS) * 4u, res = 2u;
#pragma unroll 1
  for (uint32_t i = 0; i < 4u * (MAX_DISP + 1u) && res == 2u; ++i, p = (p + 1u) & (WTAB - 1u)) {
    const uint32_t want = ((i >> 2) << TAG_BITS) | tag, mine = (want << 9) | (t << 1) | below;
    const uint32_t old = atomicCAS(&s.tab[p], EMPTY, mine);
    if (old == EMPTY) res = 0u;
    else if ((old >> 9) == want) { atomicMin(&s.tab[p], mine); res = 1u; }  // same pixel: the lowest digi owns it
  }
  return res;
}
__device__ __forceinline__ uint32_t half_match(const uint4& e, uint32_t want) {
  uint32_t r = EMPTY;
  if ((e.w >> 9) == want) r = e.w;
  if ((e.z >> 9) == want) r = e.z;
  if ((e.y >> 9) == want) r = e.y;
  if ((e.x >> 9) == want) r = e.x;
  return r;
}
__device__ __noinline__ uint32_t hfind_slow(const WarpSmem& s, uint32_t h) {
  const uint32_t tag = h & TAG_MASK;
  uint32_t b = h >> TAG_BITS, r = EMPTY;
  for (uint32_t i = 1; i <= MAX_DISP && r == EMPTY; ++i) {  // the buckets after the (full) home bucket
    b = (b + 1u) & (NBUCKET - 1u);
    const uint4 e = *reinterpret_cast<const uint4*>(&s.tab[b * 4u]);
    r = half_match(e, (i << TAG_BITS) | tag);
    if (e.w == EMPTY) break;
  }
  return r;
}
// slot contents of the key whose mixed value is h, or EMPTY
__device__ __forceinline__ uint32_t hfind(const WarpSmem& s, uint32_t h) {
  const uint4 e = *reinterpret_cast<const uint4*>(&s.tab[(h >> TAG_BITS) * 4u]);
  uint32_t r = half_match(e, h & TAG_MASK);
  if (r == EMPTY && e.w != EMPTY) r = hfind_slow(s, h);  // home bucket full, no match (rare): displaced keys
  return r;
}
__device__ __forceinline__ uint32_t slot_digi(uint32_t e) { return (e >> 1) & 0xFFu; }
__device__ __forceinline__ bool slot_live(uint32_t e) { return e != EMPTY && !(e & 1u); }

// Union on s.label (parent links, L[x] <= x): hook-and-descend, no root searches.  For the edge (a, b) with
// hi = max, lo = min: p = atomicMin(&L[hi], lo).  p == hi: hi was a root and now hangs under lo; p == lo: already
// linked.  Otherwise hi keeps the smaller of p and lo as its parent and the other one still has to be joined to it:
// go on with the edge (p, lo), whose larger end is below hi, so the descent ends.  Links only ever join digis of one
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

// (event, FED) of word g >= b, given the segment sg0 of the chunk's first word and the next boundary nextB0
// rare: word g lies beyond the segment of the chunk's first word (a FED / event boundary inside the window)
__device__ __noinline__ uint2 event_of(const Chunk& c, uint32_t S, uint32_t sg0, uint32_t g) {
  uint32_t sg = sg0 + 1u;
  while (sg + 1u < S && c.segB[sg + 1u] <= g) ++sg;
  const uint32_t er = sg / c.F;
  return make_uint2(er, c.segB[er * c.F]);  // event of the launch group, global index of its word 0
}

__global__ void __launch_bounds__(FT, 7) findclus_kernel(const __grid_constant__ Chunk c) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  WarpSmem& s = reinterpret_cast<WarpSmem*>(smem_raw)[warp];
  const uint32_t F = c.F, S = (c.e1 - c.e0) * F;
  const uint32_t* __restrict__ segB = c.segB;
  const uint32_t gBeg = segB[0], gEnd = segB[S];
  if (gBeg >= gEnd) return;
  const uint32_t T0 = gBeg & ~(CHUNK_WORDS - 1u);
  const uint32_t n_chunks = (gEnd - T0 + HC - 1u) / HC;
  const uint32_t lt_mask = (1u << lane) - 1u, le_mask = lt_mask | (1u << lane);
  constexpr uint32_t FULL = 0xFFFFFFFFu;
  uint32_t* const w0 = reinterpret_cast<uint32_t*>(&s);  // tab + edge, reused after phase D
  uint32_t* const qn = w0; uint32_t* const sx = w0 + MAXT; uint32_t* const sy = w0 + 2 * MAXT;
  uint16_t* const lid = s.chg;
  uint8_t* const rlist = reinterpret_cast<uint8_t*>(w0 + 3 * MAXT);  // roots in digi order (after phase D)
  constexpr uint32_t NO_ID = 0xFFFFu;

  const uint32_t stride = gridDim.x * WPB;
  uint32_t ci = blockIdx.x * WPB + warp;
  uint32_t sbv_n = 0u, sg_n = 0u;  // prefetched for the next chunk: start bits (lane k < 8: round k), segment
  if (ci < n_chunks) {
    if (lane < 8u && ci * 4u + lane < n_chunks * 4u) sbv_n = c.startbits[ci * 4u + lane];
    sg_n = c.chunk_seg[ci];
  }
  for (; ci < n_chunks; ci += stride) {
    const uint32_t b = T0 + ci * HC;
    // ================================================================== A: start bits of the window; clear
    const uint32_t sbv = sbv_n, sg0 = sg_n;
    const uint32_t nextB0 = segB[sg0 + 1u];  // segment of the chunk's first word: its end, its event, the event's base
    const uint32_t er0 = sg0 / F, ebase0 = segB[er0 * F];
    {
      const uint32_t cn = ci + stride;
      sbv_n = 0u;
      if (cn < n_chunks) {
        if (lane < 8u && cn * 4u + lane < n_chunks * 4u) sbv_n = c.startbits[cn * 4u + lane];
        sg_n = c.chunk_seg[cn];
      }
    }
    const uint32_t home = __ballot_sync(FULL, lane < 4u && sbv != 0u);
    if (!home) continue;  // no run starts here: nothing owned
    {
      uint4* t4 = reinterpret_cast<uint4*>(s.tab);
      const uint4 e4 = make_uint4(EMPTY, EMPTY, EMPTY, EMPTY);
#pragma unroll
      for (int k = 0; k < (int)(WTAB / 4 / 32); ++k) t4[lane + 32 * k] = e4;
      if (lane < (RC + 2u) / 4u) reinterpret_cast<uint32_t*>(s.run_bad)[lane] = 0u;
    }
    uint32_t sb[8], rb[8];  // start bits of round k; runs started before round k (warp-uniform)
    uint32_t R = 0u;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      sb[k] = __shfl_sync(FULL, sbv, k);
      rb[k] = R;
      if (k < 4) R += __popc(sb[k]);
    }
    const uint32_t kf = (uint32_t)__ffs(home) - 1u;
    const uint32_t f_t = 32u * kf + (uint32_t)__ffs(__shfl_sync(FULL, sbv, kf)) - 1u;  // first owned slot
    // end of the last run: the first start bit after the home chunk, the end of the data, or "does not fit"
    const uint32_t ext = __ballot_sync(FULL, lane >= 4u && lane < 8u && sbv != 0u);
    uint32_t e_t;
    bool fits = true;
    if (ext) {
      const uint32_t ke = (uint32_t)__ffs(ext) - 1u;
      e_t = 32u * ke + (uint32_t)__ffs(__shfl_sync(FULL, sbv, ke)) - 1u;
    } else if (b + MAXT >= gEnd) {
      e_t = gEnd - b;
    } else {
      fits = false; e_t = MAXT;
    }
    const uint32_t Rn = R < RC ? R : RC;
    __syncwarp();  // the cleared hash is visible

    // ================================================================== B: stage + insert the digis of the owned runs
    bool dup_seen = false;
    const uint32_t kl = (e_t + 31u) >> 5;  // rounds kf .. kl-1 hold the window
#pragma unroll
    for (uint32_t half = 0; half < 2; ++half) {
      const uint32_t ks = 4u * half;
      if (kl <= ks || kf >= ks + 4u) continue;  // warp-uniform
      // all global loads of the four rounds first, then the staging: one exposed latency per half
      uint32_t rw[4], cl[4], md[4];
      int32_t ch[4];
#pragma unroll
      for (uint32_t j = 0; j < 4; ++j) {
        const uint32_t k = ks + j, t = 32u * k + lane, g = b + t;
        const bool in0 = k >= kf && k < kl && t >= f_t && t < e_t;
        rw[j] = in0 ? (uint32_t)c.d_row[g] : 0xFFFFu;
        cl[j] = in0 ? (uint32_t)c.d_col[g] : 0u;
        ch[j] = in0 ? c.d_charge[g] : 0;
        md[j] = (in0 && half == 0u && (sb[k] >> lane & 1u)) ? (uint32_t)c.d_module[g] : 0xFFFFFFFFu;
      }
#pragma unroll
      for (uint32_t j = 0; j < 4; ++j) {
        const uint32_t k = ks + j;
        if (k < kf || k >= kl) continue;  // warp-uniform
        const uint32_t t = 32u * k + lane, g = b + t;
        const uint32_t r = (half == 0u ? rb[k] : R) + __popc(sb[k] & le_mask & (half == 0u ? FULL : 0u));
        const bool in = t >= f_t && t < e_t && r <= RC;
        const uint32_t row = rw[j], col = cl[j];
        const int32_t e = ch[j];
        if (in && md[j] != 0xFFFFFFFFu) {  // the first digi of run r
          uint32_t er = er0, eb = ebase0;
          if (g >= nextB0) { const uint2 ev = event_of(c, S, sg0, g); er = ev.x; eb = ev.y; }
          s.run_first[r] = (uint16_t)t; s.run_key[r] = (er << 16) | md[j]; s.run_ifirst[r] = g - eb;
        }
        const bool dec = in && row != 0xFFFFu;
        const bool below = e < c.thr;  // S9
        const uint32_t dk = dec ? ((r << 17) | (row << 9) | col) : INVALID;
        s.dkey[t] = dk;
        s.label[t] = (dec && !below) ? t : MARK_BELOW;
        s.chg[t] = (uint16_t)e;
        if (dec) {
          const uint32_t ins = hinsert(s, dk, t, below ? 1u : 0u);
          dup_seen |= ins == 1u;
          if (ins == 2u) s.run_bad[r] = 1;  // no room near the home bucket: the overflow kernel takes the run
        }
      }
    }
    __syncwarp();  // hash, dkey, label, run tables complete
    if (R > RC) {  // too many runs: the ones beyond RC go to the overflow kernel
#pragma unroll
      for (uint32_t k = 0; k < 4; ++k) {
        const uint32_t g = b + 32u * k + lane;
        if ((sb[k] >> lane & 1u) && rb[k] + __popc(sb[k] & le_mask) > RC) {
          const uint32_t er = g >= nextB0 ? event_of(c, S, sg0, g).x : er0;
          push_overflow(c, (er << 16) | c.d_module[g]);
        }
      }
    } else if (!fits && lane == 0) {
      s.run_bad[R] = 1;  // the last run does not fit the window: the overflow kernel takes it
    }
    __syncwarp();
    const uint32_t k0 = kf, k1 = kl;  // rounds that hold owned digis

    // ================================================================== D: duplicates; neighbours -> edges -> unions
    if (__any_sync(FULL, dup_seen)) {  // rare: some pixel appears twice; the digi not in the slot is a DUPLICATE (S10)
      for (uint32_t k = k0; k < k1; ++k) {
        const uint32_t t = 32u * k + lane, key = s.dkey[t];
        if (key != INVALID && slot_digi(hfind(s, hmix(key))) != t) s.label[t] = MARK_DUP;
      }
      __syncwarp();
    }
    // Forward neighbours (S13): E (r, c+1), SW (r+1, c-1), S (r+1, c), SE (r+1, c+1).  When S is live, SW and SE are
    // joined to it by their own E edges, so d-S alone is enough; when E is live, SE is E's S neighbour.
    uint32_t ne = 0u;
#pragma unroll 1
    for (uint32_t k = k0; k < k1; ++k) {
      const uint32_t t = 32u * k + lane, key = s.dkey[t];
      if (ne + 96u > ECAP) {  // the round's edges might not fit: unite what is listed (warp-uniform)
        __syncwarp();
        for (uint32_t i0 = 0u; i0 < ne; i0 += 32u) {
          if (i0 + lane < ne) {
            const uint32_t e = s.edge[i0 + lane];
            hook(s.label, e & 0xFFu, e >> 8);
          }
          __syncwarp();
        }
        ne = 0u;
      }
      const bool live = key != INVALID && s.label[t] < MAXT;
      bool f0 = false, f1 = false, f2 = false;
      uint32_t n0 = 0, n1 = 0, n2 = 0;
      if (live) {
        const uint32_t h = hmix(key);
        const uint32_t eE = hfind(s, (h + HASH_MUL) & KEY_MASK), eS = hfind(s, (h + 512u * HASH_MUL) & KEY_MASK);
        const uint32_t eSW = hfind(s, (h + 511u * HASH_MUL) & KEY_MASK), eSE = hfind(s, (h + 513u * HASH_MUL) & KEY_MASK);
        const bool hS = slot_live(eS);
        f0 = slot_live(eE); n0 = slot_digi(eE);
        f1 = hS || slot_live(eSW); n1 = slot_digi(hS ? eS : eSW);
        f2 = !hS && !f0 && slot_live(eSE); n2 = slot_digi(eSE);  // with E live, SE is E's S: E joins it
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
        hook(s.label, e & 0xFFu, e >> 8);
      }
      __syncwarp();
    }
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {  // two pointer-jumping rounds: the chains shrink 4x before the sums
      for (uint32_t k = k0; k < k1; ++k) {
        const uint32_t t = 32u * k + lane;
        const uint32_t l = s.label[t];
        if (l < MAXT) { const uint32_t ll = s.label[l]; if (ll != l) s.label[t] = ll; }
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

cudaError_t configure_findclus_kernel() {
  return cudaFuncSetAttribute(findclus_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(WPB * sizeof(WarpSmem)));
}

void launch_findclus(const Chunk& c, uint32_t words_bound, int n_sm, cudaStream_t stream) {
  uint64_t nb = ((uint64_t)words_bound + CHUNK_WORDS + WPB * HC - 1) / (WPB * HC);
  if (nb < 1) nb = 1;
  if (nb > (uint64_t)n_sm * 7) nb = (uint64_t)n_sm * 7;
  findclus_kernel<<<(int)nb, FT, WPB * sizeof(WarpSmem), stream>>>(c);
}

}  // namespace pix
