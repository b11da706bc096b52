// tile.cu -- the tile kernel of the Clusters path ("unpacks them, calibrates the individual pixels, and
// clusters the pixels on each detector module"): a1 decode (S1-S6), a2 calibrate (S7-S9), a4 findClus (S10,
// S13) and a5 sums / charge cut / renumber / temp records (S9, S14, S18) for one work item per block.
//
// A work item (runs.cu) is a stretch of at most 1024 raw words holding whole module runs.  A block of 256 threads
// takes it with four words per thread (word p = tid + 256 j, so every access is coalesced); the word's key, flags,
// charge and root stay in registers through all phases (the loop of the neighbour search, the largest body, is rolled
// and its registers turned, ROT4: fully unrolled the kernel lost 15 % to instruction fetch), only the tables live in
// shared memory:
//   P0  clear the tables; the item's run-start bits (fetched at the top of the item by the last warp, whose fourth
//       word lies beyond every item, and worked up after its share of the decoding)
//   P1  decode, calibrate, store module / row / col / charge (in front of P0's barrier: none of it needs the tables);
//       then run index from the start bits; insert into the position hash: key = run | row | col -> bucket (11 bits) + tag (14 bits), exact; a bucket holds four 32-bit
//       entries tag | below | word (one 128-bit load per lookup; the smallest of the four entry ^ tag is the answer)
//       plus a second level (4 entries per 32 buckets) that is only read when the first is full; slots are handed
//       out by a per-bucket counter (one shared atomicAdd, no probing, no CAS)
//   P2  duplicates (S10) from the list of words that were not first in their bucket (exact pass only when a candidate
//       turns up; list and pass are skipped for an item whose words come in the detector's read-out order, which the
//       pre-pass certifies per 128-word chunk: such words are all different pixels), four forward-neighbour lookups
//       per word, at most two edges per pixel and none that other pixels' edges imply, into a per-warp list, lock-free
//       unions on the labels: hook-and-descend, or by representatives when the item's runs are long (pix_device.cuh)
//   P3  root of every live pixel; roots start their accumulators (in the memory of the dead hash) and are listed in
//       word order; the other pixels add charge | pixel count, charge*col, charge*row by shared atomics
//   P4  one root per thread: Q >= cut survives (ballot bitmap, per-warp scan), numbered per run; temp records
//   P5  final status and clus, per-run cluster count and temp base, per-event counters
// Phases are separated by block barriers (seven per item); five blocks per SM; a block's first item is its own index,
// the following ones come from a counter (so that the blocks of the grid end together).
// What the kernel cannot take goes to the block-per-run kernel (cluster.cu): runs longer than 1024 words (decoded
// here, ITEM_DECODE_ONLY), items whose hash overflows a bucket (8 keys), runs with a cluster charge beyond Q_SAFE.
// Nothing here is shared with oracle/.
#include <cstddef>

#include "pix_common.cuh"
#include "pix_device.cuh"

namespace pix {

namespace {

#ifndef TILE_NT
#define TILE_NT 256
#endif
#ifndef TILE_BLOCKS
#define TILE_BLOCKS 5
#endif
constexpr int NT = TILE_NT, NJ = TILE_WORDS / NT, BLOCKS_PER_SM = TILE_BLOCKS, NWARP = NT / 32;
static_assert(TILE_WORDS == 1024 && NJ == 4, "the kernel is written for 1024-word items and four words per thread (ROT4, the 32-word bitmaps)");
constexpr uint32_t FULL = 0xFFFFFFFFu, NOKEY = 0xFFFFFFFFu;
// buckets of 4 entries, 0.5 keys per bucket: a bucket is full for 0.2 % of the lookups
constexpr uint32_t NBK = 2 * TILE_WORDS, NBK_LOG2 = 11, TAG_BITS = 25 - NBK_LOG2, TAG_MASK = (1u << TAG_BITS) - 1u;
// key: run (8) | row (8) | col (9) = 25 bits.  h = (key << 7) * HMUL mod 2^32: the top 25 bits are key * HMUL mod 2^25,
// a bijection of the key; bucket = top 11 bits, tag = the next 14, so (bucket, tag) names the key exactly, and the hash
// of a neighbour is h + a constant.
constexpr uint32_t HMUL = 0x9E3779B1u;
constexpr uint32_t D_E = (1u << 7) * HMUL, D_SW = (511u << 7) * HMUL, D_S = (512u << 7) * HMUL, D_SE = (513u << 7) * HMUL;
constexpr uint32_t MARK = 0xFFFFFFFDu;               // label of a word that is not a live pixel
// A word's state word: key (25 bits: run | row | col) and flags.  The hash shifts the flags out (key << 7).
constexpr uint32_t K_BELOW = 1u << 25, K_DUP = 1u << 26, K_SLOT = 27;  // K_SLOT: 4 bits, the word's slot in its bucket
#define ROT4(a) do { const uint32_t t_ = a[0]; a[0] = a[1]; a[1] = a[2]; a[2] = a[3]; a[3] = t_; } while (0)
constexpr uint32_t NONE = 0xFFFFu, NO_ID = 0xFFFFu;
constexpr uint32_t Q_SAFE = 0xFFFFFFFFu / 415u;      // sum(e*col), sum(e*row) fit 32 bits while sum(e) <= Q_SAFE
constexpr uint32_t BIG_RUN = 256u;                   // runs this long count their pixels in a word of their own
constexpr uint32_t ECAP = 3 * 32;                    // edges a warp lists before it unites them (one word per lane)
constexpr uint32_t BB_SHIFT = 5, BB_MASK = (1u << BB_SHIFT) - 1u;  // first-level buckets per second-level bucket
constexpr uint32_t B_KEY = (1u << (16 + BB_SHIFT)) - 1u, B_WORD = 16 + BB_SHIFT, B_BELOW = B_WORD + 10;  // fields of a second-level entry

// A first-level entry: tag << 11 | below_threshold << 10 | word; FREE matches no tag.  x ^ tag_word(h) is below 2048
// exactly for the entries of the pixel with hash h, and then it is below << 10 | word: the smallest of a bucket's four
// differences is the lookup's result (live pixel: below 1024).
constexpr uint32_t FREE = 0xFFFFFFFFu, E_TAG = TAG_MASK << 11, E_BELOW = 1u << 10;

struct __align__(16) TileSmem {
  union {
    uint4 ent[NBK];          // first level: four entries per bucket
    struct { uint32_t qn[TILE_WORDS], sx[TILE_WORDS], sy[TILE_WORDS], npx[TILE_WORDS]; } sum;  // after P2: the roots' accumulators
  };
  uint32_t tagsB[4 * (NBK >> BB_SHIFT)];  // second level, 4 entries per 32 buckets: tag + 1 | (bucket & 31) << 16 | word << 21 | below << 31
  uint32_t cnt[NBK / 4];     // entries per bucket, one byte each
  uint32_t cntB[(NBK >> BB_SHIFT) / 4];  // entries per second-level bucket, one byte each (tagsB is never cleared)
  uint32_t edge[NT / 32][ECAP];  // per warp: the edges its words found, a | b << 16
  uint32_t label[TILE_WORDS];        // after P3: lid, 16 bits each (local id of a root, or NO_ID)
  uint32_t bits[32], pre[32];        // run-start bits of the item, run starts before each word of bits
  uint32_t survb[32];                // roots that survive the cut, in root order
  uint32_t rootb[32];                // words that are roots
  uint16_t run_pos[256], run_mod[256];
  uint8_t run_big[256];
  uint8_t run_bad[2][256];           // by item parity: the next item's P0 clears the other one while P5 still reads this one
  uint32_t n_runs, wbase, next_item, pad[1];
};
static_assert(sizeof(TileSmem) <= 233472 / BLOCKS_PER_SM - 1024, "BLOCKS_PER_SM blocks per SM");

__device__ __forceinline__ uint32_t hash_of(uint32_t key) { return (key << 7) * HMUL; }
__device__ __forceinline__ bool k_live(uint32_t k) { return (k & (K_BELOW | K_DUP)) == 0u; }  // NOKEY has every bit set
__device__ __forceinline__ uint32_t k_run(uint32_t k) { return (k >> 17) & 0xFFu; }
__device__ __forceinline__ uint32_t bucket_of(uint32_t h) { return h >> (32 - NBK_LOG2); }
__device__ __forceinline__ uint32_t want_of(uint32_t h) { return ((h >> 7) & TAG_MASK) + 1u; }  // the tag in a second-level entry
__device__ __forceinline__ uint32_t tag_word(uint32_t h) { return (h << 4) & E_TAG; }
__device__ __forceinline__ uint32_t min4(const uint4& x, uint32_t tw) {
  return min(min(x.x ^ tw, x.y ^ tw), min(x.z ^ tw, x.w ^ tw));
}
__device__ __forceinline__ uint32_t entries_of(const uint4& x, uint32_t tw) {  // how many entries of the bucket belong to the pixel
  return ((x.x ^ tw) < 2048u ? 1u : 0u) + ((x.y ^ tw) < 2048u ? 1u : 0u) + ((x.z ^ tw) < 2048u ? 1u : 0u) + ((x.w ^ tw) < 2048u ? 1u : 0u);
}
__device__ __forceinline__ uint32_t countB(const TileSmem& s, uint32_t bB) {
  const uint32_t n = (s.cntB[bB >> 2] >> ((bB & 3u) * 8u)) & 0xFFu;
  return n > 4u ? 4u : n;
}
// second level (rare): the live pixel, or NONE
__device__ __noinline__ uint32_t lookup_B(const TileSmem& s, uint32_t b, uint32_t want) {
  const uint32_t bB = b >> BB_SHIFT, n = countB(s, bB), w19 = want | ((b & BB_MASK) << 16);
  for (uint32_t i = 0; i < n; ++i) {
    const uint32_t e = s.tagsB[bB * 4u + i];
    if ((e & B_KEY) == w19) return (e >> B_BELOW) ? NONE : ((e >> B_WORD) & 0x3FFu);
  }
  return NONE;
}
// second level (rare): entries of the pixel
__device__ __noinline__ uint32_t matches_B(const TileSmem& s, uint32_t b, uint32_t want) {
  const uint32_t bB = b >> BB_SHIFT, n = countB(s, bB), w19 = want | ((b & BB_MASK) << 16);
  uint32_t k = 0u;
  for (uint32_t i = 0; i < n; ++i) k += (s.tagsB[bB * 4u + i] & B_KEY) == w19 ? 1u : 0u;
  return k;
}

// Lookup of four pixels at once (the four loads are in flight together).  The result is the word of the live pixel
// with hash h[i], or a value >= 1024 (no such pixel, or below threshold).
__device__ __forceinline__ void lookup4(const TileSmem& s, const uint32_t (&h)[4], uint32_t (&res)[4]) {
  uint4 x[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) x[i] = s.ent[bucket_of(h[i])];
  bool rare = false;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    res[i] = min4(x[i], tag_word(h[i]));
    rare |= res[i] >= 2048u && x[i].w != FREE;
  }
  if (rare) {  // a miss in a bucket whose first level is full
#pragma unroll
    for (int i = 0; i < 4; ++i)
      if (res[i] >= 2048u && x[i].w != FREE) res[i] = lookup_B(s, bucket_of(h[i]), want_of(h[i]));
  }
}

// rare: the pixel of word p appears more than once in its bucket.  The lowest word owns it (S10); every entry of the
// pixel is made to name the owner, so a lookup may take any of them.  Returns true when p is not the owner.
__device__ __noinline__ bool resolve_dup(TileSmem& s, uint32_t b, uint32_t h, uint32_t p, uint32_t k_own) {
  uint32_t* const eA = reinterpret_cast<uint32_t*>(s.ent + b);
  const uint32_t tw = tag_word(h), want = want_of(h);
  const uint32_t bB = b >> BB_SHIFT, nB = eA[3] != FREE ? countB(s, bB) : 0u, w19 = want | ((b & BB_MASK) << 16);
  uint32_t best = 0xFFFFFFFFu;  // word << 1 | below
  for (uint32_t i = 0; i < 4u; ++i) {
    const uint32_t d = eA[i] ^ tw;
    if (d >= 2048u) continue;
    const uint32_t v = ((d & 0x3FFu) << 1) | (d >> 10);
    best = v < best ? v : best;
  }
  for (uint32_t i = 0; i < nB; ++i) {
    const uint32_t e = s.tagsB[bB * 4u + i];
    if ((e & B_KEY) != w19) continue;
    const uint32_t v = (((e >> B_WORD) & 0x3FFu) << 1) | (e >> B_BELOW);
    best = v < best ? v : best;
  }
  if ((best >> 1) == p) return false;
  if (k_own < 4u) eA[k_own] = tw | (best >> 1) | ((best & 1u) ? E_BELOW : 0u);
  else s.tagsB[bB * 4u + k_own - 4u] = w19 | ((best >> 1) << B_WORD) | ((best & 1u) << B_BELOW);
  return true;
}

__global__ void __launch_bounds__(NT, BLOCKS_PER_SM) tile_kernel(const __grid_constant__ Chunk c) {
  chain_begin();
  extern __shared__ __align__(16) unsigned char smem_raw[];
  TileSmem& s = *reinterpret_cast<TileSmem*>(smem_raw);
  uint32_t tid;
  asm volatile("mov.u32 %0, %%tid.x;" : "=r"(tid));  // read once: the compiler would re-read the special register all over the kernel
  const uint32_t lane = tid & 31u, warp = tid >> 5;
  const uint32_t F = c.F, S = (c.e1 - c.e0) * F;
  const uint32_t* __restrict__ segB = c.segB;
  const uint32_t gBeg = segB[0], gEnd = segB[S];
  if (gBeg >= gEnd) return;
  const uint32_t T0 = gBeg & ~(CHUNK_WORDS - 1u);
  uint32_t n_items = c.ctl[CTL_ITEM_COUNT];
  n_items = n_items < c.item_cap ? n_items : c.item_cap;
  const uint32_t lt_mask = (1u << lane) - 1u, le_mask = lt_mask | (1u << lane);
  uint32_t* const ent32 = reinterpret_cast<uint32_t*>(s.ent);
  uint16_t* const lid = reinterpret_cast<uint16_t*>(s.label);  // not in the hash: the next item's P0 clears that while P5 still reads lid

  uint32_t par = 0u;
  uint32_t nxt;
  for (uint32_t it = blockIdx.x; it < n_items; it = nxt) {
    // The block's first item is its own index, the others come from a counter: asked for now, handed to the block with
    // the barrier after P1 (blocks that drew cheap items go on drawing, so the grid ends together).
    uint32_t nxt_t0 = 0u;
    if (tid == 0) nxt_t0 = gridDim.x + atomicAdd(c.ctl + CTL_ITEM_NEXT, 1u);
    const uint4 item = c.items[it];
    const uint32_t g0 = item.x, len = item.y & 0xFFFFu, iflags = item.y >> 16, er = item.z & 0xFFFFu, fed0 = item.z >> 16;
    const bool cluster_it = !(iflags & ITEM_DECODE_ONLY);
    uint32_t w[NJ];
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
      const uint32_t p = tid + NT * j;
      w[j] = p < len ? __ldg(c.words + g0 + p) : 0u;
    }
    const uint32_t ebase = segB[er * F];
    const uint32_t nextB = segB[er * F + fed0 + 1u];        // first word of the next FED
    // the item's stretch of the temp record area, one slot per word: asked for now, needed in P4
    uint32_t wbase_t0 = 0u;
    if (tid == 0 && cluster_it) wbase_t0 = alloc_temp(c, len);
    // Words in read-out order (every 128-word chunk the item touches is clean, runs.cu) are all different pixels
    bool off_t = false;
    if (tid <= ((g0 + len - 1u - T0) >> 7) - ((g0 - T0) >> 7)) off_t = c.cbad[((g0 - T0) >> 7) + tid] != 0;
    // No barrier here: what P0 writes (hash, counters, start bits, the run_bad of this item's parity) is not read by
    // the previous item's P5, and nothing else is written before the barrier at the end of P0.
    uint8_t* const rbad = s.run_bad[par];
    par ^= 1u;
    // ================================================================== P0: clear; start bits of the item
    {
      const uint4 z4 = make_uint4(0u, 0u, 0u, 0u), f4 = make_uint4(FREE, FREE, FREE, FREE);
#pragma unroll
      for (int k = 0; k < (int)(NBK / NT); ++k) s.ent[tid + NT * k] = f4;
      if (tid < (NBK / 4 + (NBK >> BB_SHIFT) / 4) / 4) reinterpret_cast<uint4*>(s.cnt)[tid] = z4;  // cnt and cntB
      if (tid < 64) reinterpret_cast<uint32_t*>(rbad)[tid] = 0u;
      if (tid < 32) s.survb[tid] = 0u;
    }
    // the item's start bits: warp NWARP - 1 (its fourth word lies beyond every item: it has the least to do) fetches
    // them now and works them up after its share of the decoding, just before the barrier
    uint32_t sb_lo = 0u, sb_hi = 0u;
    if (warp == NWARP - 1u) { const uint32_t wq = (g0 - T0) >> 5; sb_lo = c.sbits[wq + lane]; sb_hi = c.sbits[wq + lane + 1u]; }
    auto start_bits = [&]() {
      {
        uint32_t v = __funnelshift_r(sb_lo, sb_hi, (g0 - T0) & 31u);
        const uint32_t nb = len > 32u * lane ? len - 32u * lane : 0u;
        v &= nb >= 32u ? FULL : ((1u << nb) - 1u);
        s.bits[lane] = v;
        uint32_t pc = __popc(v), inc = pc;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
          const uint32_t o = __shfl_up_sync(FULL, inc, d);
          if (lane >= (uint32_t)d) inc += o;
        }
        s.pre[lane] = inc - pc;
        if (lane == 31) s.n_runs = inc;
      }
    };
    // ================================================================== P1: decode, calibrate, insert
    // The words' state stays in registers and is turned by one place per iteration (ROT4), so that the word at hand is
    // always [0]: free in the unrolled loops (register renaming), three moves in the rolled one of P2.
    // First what needs neither the cleared tables nor the start bits -- decode, calibration, the four stores -- so that
    // nobody waits at P0's barrier for the warp that fetches the start bits; the module waits in cr's upper half.
    const uint32_t fed_split = g0 + len <= nextB ? 0xFFFFFFFFu : nextB;  // words from here on belong to a later FED (rare)
    uint32_t key[NJ];  // K_* below; NOKEY: not decodable
    uint32_t cr[NJ];   // charge | root << 16
    bool fail = false;
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
      const uint32_t p = tid + NT * j, g = g0 + p;
      const bool valid = p < len;
      uint32_t fed = fed0;
      if (g >= fed_split && valid) {  // a FED boundary inside the item
        uint32_t sg = er * F + fed0 + 1u;
        while (sg + 1u < (er + 1u) * F && segB[sg + 1u] <= g) ++sg;
        fed = sg - er * F;
      }
      uint32_t m, row, col;
      const uint32_t st = decode_word(c.cab, w[0], fed << 11, m, row, col);
      const bool ok = valid && st == ST_OK;
      int32_t e = 0;
      if (ok) e = calibrate(c, w[0] & 255u, __ldg(c.gp + (m * (uint32_t)COLS + col)));  // S8: one pair per (module, col)
      else { m = row = col = 0xFFFFu; }
      if (valid) {
        __stcs(c.d_module + g, (uint16_t)m); __stcs(c.d_row + g, (uint16_t)row); __stcs(c.d_col + g, (uint16_t)col); __stcs(c.d_charge + g, e);
        if (!ok) {  // undecodable words are finished here
          c.d_status[g] = (uint8_t)st; c.d_clus[g] = -1;
          atomicAdd(c.ev_cnt + (size_t)er * EC_STRIDE + (st - ST_EMPTY), 1u);
        }
      }
      key[0] = ok ? ((row << 9) | col | (e < c.thr ? K_BELOW : 0u)) : NOKEY;  // S9; the run comes after the barrier
      cr[0] = (uint32_t)e | (m << 16);
      ROT4(w); ROT4(key); ROT4(cr);
    }
    if (warp == NWARP - 1u) start_bits();
    const bool ordered = !__syncthreads_or(off_t) && c.geom_unique != 0u;  // P0 is done
    // Words that are not the first entry of their bucket go to a per-warp list (bucket | slot | tag): only they can be
    // the later copy of a pixel that appears twice (S10), and after the barrier the list is checked with all lanes busy.
    uint32_t* const dl = s.edge[warp];  // (the edge lists are not in use yet)
    uint32_t nd = 0u;
    bool cand = false;  // some pixel of the item may appear twice
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
      const uint32_t p = tid + NT * j;
      const uint32_t kj = key[0];
      const bool ok = kj != NOKEY, below = (kj & K_BELOW) != 0u;
      const uint32_t bw = s.bits[j * NWARP + warp];
      const uint32_t r = s.pre[j * NWARP + warp] + __popc(bw & le_mask) - 1u;  // a decodable word lies in a run: r >= 0
      uint32_t k0 = NOKEY, chk = 0u;
      if (ok) {
        k0 = kj | (r << 17);
        if ((bw >> lane) & 1u) { s.run_pos[r] = (uint16_t)p; s.run_mod[r] = (uint16_t)(cr[0] >> 16); }
        if (cluster_it) {
          const uint32_t h = hash_of(k0), b = bucket_of(h), sh8 = (b & 3u) * 8u;
          const uint32_t k = (atomicAdd(&s.cnt[b >> 2], 1u << sh8) >> sh8) & 0xFFu;
          const uint32_t tag = want_of(h);
          uint32_t kk = k;
          if (k < 4u) ent32[b * 4u + k] = tag_word(h) | (below ? E_BELOW : 0u) | p;
          else {  // rare: the bucket's first level is full
            const uint32_t bB = b >> BB_SHIFT, shB = (bB & 3u) * 8u;
            const uint32_t kb = (atomicAdd(&s.cntB[bB >> 2], 1u << shB) >> shB) & 0xFFu;
            if (kb < 4u) s.tagsB[bB * 4u + kb] = tag | ((b & BB_MASK) << 16) | (p << B_WORD) | (below ? 1u << B_BELOW : 0u);
            else fail = true;
            kk = 4u + (kb < 4u ? kb : 0u);
          }
          k0 |= kk << K_SLOT;
          if (k >= 1u && !ordered) chk = b | ((k < 7u ? k : 7u) << 11) | (tag << 14);
        }
      }
      if (!ordered) {
        const uint32_t mc = __ballot_sync(FULL, chk != 0u);
        const uint32_t at = nd + __popc(mc & lt_mask);
        if (chk != 0u) { if (at < ECAP) dl[at] = chk; else cand = true; }  // a full list: take the exact path
        nd += __popc(mc);
      }
      s.label[p] = (ok && !below) ? p : MARK;
      key[0] = k0; cr[0] &= 0xFFFFu;
      ROT4(key); ROT4(cr);
    }
    if (!cluster_it) {  // a piece of a run longer than the tile: the block-per-run kernel clusters it
      if ((iflags & ITEM_LONG_HEAD) && tid == 0 && key[0] != NOKEY) push_run(c, c.ovf_list, CTL_OVF_COUNT, er, s.run_mod[0]);
      if (tid == 0) s.next_item = nxt_t0;
      __syncthreads();  // P1 read the start bits: the next item's P0 rewrites them
      nxt = s.next_item;
      continue;
    }
    if (tid == 0) { s.wbase = wbase_t0; s.next_item = nxt_t0; }
    const uint32_t R = s.n_runs;
    const bool failed = __syncthreads_or(fail);
    nxt = s.next_item;
    if (failed) {  // a bucket with more than 8 keys: the block-per-run kernel takes the runs of the item
      if (tid < R) push_run(c, c.ovf_list, CTL_OVF_COUNT, er, s.run_mod[tid]);
      continue;
    }
    if (nxt < n_items) {  // the next item: its words on their way into L2 while this one is clustered
      const uint4 nx = c.items[nxt];
      const uint32_t* q = c.words + nx.x + 32u * tid;  // one 128-byte line per thread covers up to 8192 words
      if (32u * tid < (nx.y & 0xFFFFu)) asm volatile("prefetch.global.L2 [%0];" :: "l"(q));
    }
    // ================================================================== P2: neighbours -> edges -> unions; duplicates
    if (tid < R) {
      const uint32_t e1 = tid + 1u < R ? s.run_pos[tid + 1u] : len;
      s.run_big[tid] = (e1 - s.run_pos[tid] >= BIG_RUN) ? 1 : 0;
    }
    __syncwarp();
    // ---- duplicates (S10).  A listed word is a candidate when a slot below its own holds its tag (or when the second
    // level is involved).  Rare: then every word looks at its own bucket exactly, every entry of a pixel that appears
    // twice is made to name the lowest word, and the other words become DUPLICATE before anybody looks up.
    {
      nd = nd < ECAP ? nd : ECAP;
      for (uint32_t i0 = 0u; i0 < nd; i0 += 32u) {
        if (i0 + lane < nd) {
          const uint32_t e = dl[i0 + lane], k = (e >> 11) & 7u, tag = e >> 14;
          cand |= k >= 4u || entries_of(s.ent[e & (NBK - 1u)], (tag - 1u) << 11) >= 2u;
        }
      }
    }
    if (!ordered && __syncthreads_or(cand)) {  // (words in read-out order are all different)
#pragma unroll
      for (int j = 0; j < NJ; ++j) {
        const uint32_t kj = key[j];
        if (kj == NOKEY) continue;
        const uint32_t h = hash_of(kj), b = bucket_of(h);
        const uint4 x = s.ent[b];
        uint32_t nm = entries_of(x, tag_word(h));
        if (x.w != FREE) nm += matches_B(s, b, want_of(h));
        if (nm >= 2u && resolve_dup(s, b, h, tid + NT * j, (kj >> K_SLOT) & 15u)) { key[j] = kj | K_DUP; s.label[tid + NT * j] = MARK; }
      }
      __syncthreads();
    }
    const bool long_item = R * 96u < len;  // long runs on average (PU200's inner modules): the other union
    // ---- Forward neighbours (S13): E (r, c+1), SW (r+1, c-1), S (r+1, c), SE (r+1, c+1); col 416..511 and row 160..255
    // never occur, so no bounds checks.  When S is live, SW and SE are joined to it by their own E edges; when E is
    // live, SE is E's S neighbour; when E, S and SE are all live, S is reached through E - SE - S (E's own S edge, or by
    // the same argument further along the row, and S's E edge).  Every lane looks up (a word that is no live pixel drops what it finds), the edges
    // go to the warp's list, and the list is united with all lanes busy.
    {
      uint32_t* const el = s.edge[warp];
#pragma unroll 1  // the largest loop body stays rolled (measured: unrolling it changes nothing)
      for (int j = 0; j < NJ; ++j) {
        uint32_t ne = 0u;
        {
          const uint32_t kj = key[0];
          const bool live = k_live(kj);
          const uint32_t p = tid + NT * j;
          const uint32_t h = hash_of(kj);
          const uint32_t hn[4] = {h + D_E, h + D_S, h + D_SW, h + D_SE};
          uint32_t nb[4];
          lookup4(s, hn, nb);
          const uint32_t nE = nb[0], nS = nb[1], nSW = nb[2], nSE = nb[3];  // >= 1024: no live pixel there
          const uint32_t t1 = nS < 1024u ? nS : nSW;
          const bool f0 = live && nE < 1024u, f1 = live && t1 < 1024u && (nS | nE | nSE) >= 1024u, f2 = live && nS >= 1024u && nE >= 1024u && nSE < 1024u;
          const uint32_t m0 = __ballot_sync(FULL, f0), m1 = __ballot_sync(FULL, f1), m2 = __ballot_sync(FULL, f2);
          if (f0) el[ne + __popc(m0 & lt_mask)] = p | (nE << 16);
          ne += __popc(m0);
          if (f1) el[ne + __popc(m1 & lt_mask)] = p | (t1 << 16);
          ne += __popc(m1);
          if (f2) el[ne + __popc(m2 & lt_mask)] = p | (nSE << 16);
          ne += __popc(m2);
        }
        __syncwarp();
        for (uint32_t i0 = 0u; i0 < ne; i0 += 32u) {  // warp-uniform trip count: the lanes reconverge every iteration
          if (i0 + lane < ne) {
            const uint32_t e = el[i0 + lane];
            if (long_item) unite_roots(s.label, e & 0xFFFFu, e >> 16); else hook(s.label, e & 0xFFFFu, e >> 16);
          }
          __syncwarp();
        }
        ROT4(key);
      }
    }
    __syncthreads();
    // ================================================================== P3: roots; sums
    // One pointer-jumping step first (a label only ever moves to an ancestor, so concurrent walkers stay correct).
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
      const uint32_t p = tid + NT * j;
      const uint32_t l = s.label[p];
      if (l < TILE_WORDS) { const uint32_t ll = s.label[l]; if (ll != l) s.label[p] = ll; }
    }
    __syncwarp();
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
      const uint32_t p = tid + NT * j, kj = key[0], e = cr[0] & 0xFFFFu;
      const bool live = k_live(kj);
      uint32_t r = live ? s.label[p] : 0u;
      bool done = !live;
      while (!done) { const uint32_t n = s.label[r]; done = n == r; r = n; }  // single exit: the warp reconverges
      cr[0] = e | ((live ? r : NONE) << 16);
      const bool is_root = live && r == p;
      if (is_root) {  // a root starts its accumulators with its own pixel (the hash is dead: nobody looks up any more)
        const uint32_t big = s.run_big[k_run(kj)];
        s.sum.qn[p] = big ? e : (e | (1u << 24));  // below BIG_RUN words a cluster has at most 255 pixels and Q < 2^24
        s.sum.sx[p] = e * (kj & 511u);
        s.sum.sy[p] = e * ((kj >> 9) & 255u);
        s.sum.npx[p] = 1u;
      }
      const uint32_t bal = __ballot_sync(FULL, is_root);
      if (lane == 0) s.rootb[j * NWARP + warp] = bal;
      ROT4(key); ROT4(cr);
    }
    __syncthreads();
    // every warp scans the 32 words of the root bitmap for itself: lane l holds word l and the roots before it
    const uint32_t rt_bits = s.rootb[lane];
    uint32_t rt_pre = __popc(rt_bits);
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t o = __shfl_up_sync(FULL, rt_pre, d);
      if (lane >= (uint32_t)d) rt_pre += o;
    }
    const uint32_t n_roots = __shfl_sync(FULL, rt_pre, 31);
    rt_pre -= __popc(rt_bits);
    auto roots_before = [&](uint32_t pos) {  // roots among the words before pos (all lanes call it together)
      const uint32_t wi = pos >> 5;
      const uint32_t r = __shfl_sync(FULL, rt_pre, wi) + __popc(__shfl_sync(FULL, rt_bits, wi) & ((1u << (pos & 31u)) - 1u));
      return pos >= 1024u ? n_roots : r;
    };
    uint16_t* const rlist = reinterpret_cast<uint16_t*>(s.edge);  // the roots in word order (the edge lists are dead)
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
      const uint32_t p = tid + NT * j, kj = key[0], e = cr[0] & 0xFFFFu, r = cr[0] >> 16;
      const uint32_t di = __shfl_sync(FULL, rt_pre, j * NWARP + warp) + __popc(__shfl_sync(FULL, rt_bits, j * NWARP + warp) & lt_mask);
      if (r == p) rlist[di] = (uint16_t)p;
      if (r != NONE && r != p) {
        const uint32_t big = s.run_big[k_run(kj)];
        atomicAdd(&s.sum.qn[r], big ? e : (e | (1u << 24)));
        atomicAdd(&s.sum.sx[r], e * (kj & 511u));
        atomicAdd(&s.sum.sy[r], e * ((kj >> 9) & 255u));
        if (big) atomicAdd(&s.sum.npx[r], 1u);
      }
      ROT4(key); ROT4(cr);
    }
    __syncthreads();
    // ================================================================== P4: cut, renumber, temp records -- one root per thread
    // root i of the list: word, run, charge, pixels
    auto load_root = [&](uint32_t i, uint32_t& p, uint32_t& run, uint32_t& Q, uint32_t& np) {
      p = rlist[i];
      run = s.pre[p >> 5] + __popc(s.bits[p >> 5] & ((2u << (p & 31u)) - 1u)) - 1u;
      const uint32_t big = s.run_big[run], a = s.sum.qn[p];
      Q = big ? a : (a & 0xFFFFFFu); np = big ? s.sum.npx[p] : (a >> 24);
    };
    uint32_t p_0 = 0u, run_0 = 0u, Q_0 = 0u, np_0 = 0u;  // the root of the first round stays in registers for the second loop
    for (uint32_t i0 = 0u; i0 < n_roots; i0 += NT) {  // block-uniform trip count (one round unless the item is all single pixels)
      const uint32_t i = i0 + tid;
      bool sv = false;
      if (i < n_roots) {
        uint32_t p, run, Q, np;
        load_root(i, p, run, Q, np);
        if (i0 == 0u) { p_0 = p; run_0 = run; Q_0 = Q; np_0 = np; }
        sv = (int32_t)Q >= c.cut;  // S9: equality keeps (Q < 2^31)
        if (Q > Q_SAFE) rbad[run] = 1;  // 32-bit weighted sums may have wrapped
      }
      const uint32_t bal = __ballot_sync(FULL, sv);
      if (lane == 0) s.survb[i >> 5] = bal;  // the words beyond the roots stay 0 (P0)
    }
    __syncthreads();
    // survivors in root order: lane l holds word l of the bitmap and the survivors before it
    const uint32_t sv_bits = s.survb[lane];
    uint32_t sv_pre = __popc(sv_bits);
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t o = __shfl_up_sync(FULL, sv_pre, d);
      if (lane >= (uint32_t)d) sv_pre += o;
    }
    const uint32_t sv_total = __shfl_sync(FULL, sv_pre, 31);
    sv_pre -= __popc(sv_bits);
    auto surv_before_root = [&](uint32_t d) {  // survivors among the roots before root d (all lanes call it together)
      const uint32_t wi = d >> 5;
      const uint32_t r = __shfl_sync(FULL, sv_pre, wi) + __popc(__shfl_sync(FULL, sv_bits, wi) & ((1u << (d & 31u)) - 1u));
      return d >= 1024u ? sv_total : r;
    };
    auto rank_before = [&](uint32_t pos) { return surv_before_root(roots_before(pos)); };  // survivors among the words before pos
    const uint32_t wbase = s.wbase;
    for (uint32_t i0 = 0u; i0 < n_roots; i0 += NT) {
      const uint32_t i = i0 + tid;
      const bool valid = i < n_roots;
      uint32_t p = p_0, run = run_0, Q = Q_0, np = np_0;
      if (valid && i0 != 0u) load_root(i, p, run, Q, np);
      const uint32_t rank = surv_before_root(i), base = rank_before(valid ? (uint32_t)s.run_pos[run] : 0u);
      if (valid) {
        uint32_t id = NO_ID;
        if ((int32_t)Q >= c.cut) {
          id = rank - base;
          const float fq = (float)Q;  // S18: exact integer sums, one rounding each + a 2-ulp division (within 1e-5)
          put_temp(c, wbase + rank, g0 + p - ebase, np, Q, __fdividef((float)s.sum.sx[p], fq), __fdividef((float)s.sum.sy[p], fq));
        }
        lid[p] = (uint16_t)id;
      }
    }
    __syncthreads();
    // ================================================================== P5: final status and clus, run outputs, counters
    uint32_t cntA = 0u, cntB = 0u, cntP = 0u;  // dup | below << 16 ; ok | cut << 16 ; roots
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
      const uint32_t kj = key[0], rt = cr[0] >> 16;
      ROT4(key); ROT4(cr);
      if (kj == NOKEY) continue;
      if (rbad[k_run(kj)]) continue;
      const uint32_t p = tid + NT * j;
      uint32_t so; int32_t cl = -1;
      if (kj & K_DUP) { so = ST_DUP; cntA += 1u; }
      else if (kj & K_BELOW) { so = ST_BELOW; cntA += 0x10000u; }
      else {
        const uint32_t id = lid[rt];
        if (id != NO_ID) { so = ST_OK; cl = (int32_t)id; cntB += 1u; } else { so = ST_CUT; cntB += 0x10000u; }
        cntP += rt == p ? 1u : 0u;
      }
      __stcs(c.d_status + g0 + p, (uint8_t)so); __stcs(c.d_clus + g0 + p, cl);
    }
    __syncwarp();
    if (warp * 32u < R) {  // the warps that hold a run each in some lane
      const bool has = tid < R;
      const uint32_t p0 = has ? (uint32_t)s.run_pos[tid] : 0u, p1 = (has && tid + 1u < R) ? (uint32_t)s.run_pos[tid + 1u] : len;
      const uint32_t b0 = rank_before(p0), b1 = rank_before(p1);  // all lanes shuffle together
      if (has) {
        const uint32_t m = s.run_mod[tid];
        if (rbad[tid]) push_run(c, c.ovf_list, CTL_OVF_COUNT, er, m);
        else {
          const size_t mo = (size_t)er * c.M + m;
          c.n_clus[mo] = b1 - b0; c.t_base[mo] = wbase + b0;
        }
      }
    }
    {
      const uint32_t a = __reduce_add_sync(FULL, cntA), bb = __reduce_add_sync(FULL, cntB), pp = __reduce_add_sync(FULL, cntP);
      if (lane == 0) {
        uint32_t* ec = c.ev_cnt + (size_t)er * EC_STRIDE;
        if (a & 0xFFFFu) atomicAdd(ec + EC_DUP, a & 0xFFFFu);
        if (a >> 16) atomicAdd(ec + EC_BELOW, a >> 16);
        if (bb & 0xFFFFu) atomicAdd(ec + EC_OK, bb & 0xFFFFu);
        if (bb >> 16) atomicAdd(ec + EC_CUT, bb >> 16);
        if (pp) atomicAdd(ec + EC_PRECUT, pp);
      }
    }
  }
}

}  // namespace

cudaError_t configure_tile_kernel() {
  return cudaFuncSetAttribute(tile_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(TileSmem));
}

void launch_tile(const Chunk& c, int n_sm, cudaStream_t stream) {
  launch_chained(true, tile_kernel, n_sm * BLOCKS_PER_SM, NT, sizeof(TileSmem), stream, c);
}

}  // namespace pix
