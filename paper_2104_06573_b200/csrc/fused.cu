// fused.cu -- the fused warp kernel of the Clusters path ("unpacks them, calibrates the individual
// pixels, and clusters the pixels on each detector module"): a1 decode (S1-S6), a2 calibrate (S7-S9),
// a3 module boundaries (S11, S12), a4 findClus (S10, S13) and a5 sums / charge cut / renumber / temp records
// (S9, S14, S18) in one pass over the raw words.  SURVEY 8f NEXT-3.
//
// The word stream is cut into chunks of 128 words.  A warp takes a ticket of consecutive chunks and walks it with a
// two-chunk ring in shared memory: while the window of chunk i is clustered, chunk i+1 is already decoded (four
// consecutive words per lane: one 128-bit load, 128-bit / 64-bit stores), so
//   - the "previous decodable word" that decides whether a word starts a module run is carried in registers from
//     chunk to chunk (a look-back into memory happens once per ticket, bounded by the start of the event; every
//     event's last run is closed by segfill_kernel),
//   - the look-ahead a window needs (a run belongs to the warp whose chunk holds its first word; the last run of a
//     chunk may end in the next chunk) is the next chunk's own decode, done once,
//   - the raw words of the chunk after that are already in flight (loaded one iteration ahead),
//   - per-event counters live in registers and are flushed when the ticket ends or the event changes.
// The decode stages every word in its final form: position | run (counted inside the chunk) | below-threshold |
// run start.  Per window (the runs that start in chunk i, up to the first run start of chunk i+1; at most 256
// slots, numbered from the window's first word so that the rounds of 32 are full):
//   B  clear the position hash; insert every digi keyed by (run, row, col); equal keys keep the lowest digi (S10)
//   D  forward-neighbour lookups (one branch for the four) -> dense edge list -> unions (lock-free
//      hook-and-descend, pix_device.cuh), two pointer-jumping rounds
//   E  every live digi adds charge | 1 << 24, charge*col, charge*row into its root's accumulators; dense root list
//   F  one root per lane: Q >= cut survives, numbered per run (ballot/popc); temp records into the window's stretch
//      of the temp area
//   G  final status and clus of the window's digis, counters (undecodable words are finished by the decode)
// Warps never wait for each other (no block barrier); all tables are per-warp shared memory.  Runs that do not fit
// the window, chunks with more than RC runs, hash buckets that overflow and charge sums that could overflow 32 bits go
// to the block-per-run kernel (findrun.cu).  Measured: the kernel is bound by instruction issue and, with 50 KB of
// code walked once per window, by instruction fetch: unrolling any of its loops makes it slower.
// Nothing here is shared with oracle/.
#include "pix_common.cuh"
#include "pix_device.cuh"

namespace pix {

namespace {

constexpr int WPB = 4;                    // warps per block (they share nothing but the block)
constexpr int FT = WPB * 32;
constexpr int BLOCKS_PER_SM = 7;          // 8000 B of shared memory per warp, 72 registers per thread
constexpr uint32_t HC = CHUNK_WORDS;      // words of a chunk (rounds 0-3 of a window)
constexpr uint32_t MAXT = 256;            // window: home chunk + up to 4 rounds of the next chunk
constexpr uint32_t RC = 62;               // runs a window can own
constexpr uint32_t ECAP = 256;            // edge list; flushed (united) when a round might not fit
constexpr uint32_t GMAX = 32;             // chunks per ticket, at most
constexpr uint32_t NOKEY = 0xFFFFFFFFu, FULL = 0xFFFFFFFFu;
constexpr uint32_t MARK_DUP = 0xFFFFFFFEu, MARK_BELOW = 0xFFFFFFFDu;  // label of a digi that is not live
constexpr uint32_t Q_SAFE = 0xFFFFFFFFu / 415u;  // sum(e*col), sum(e*row) fit 32 bits while sum(e) <= Q_SAFE
constexpr uint32_t NO_ID = 0xFFFFu;
using PH = BucketHash<23, 8, 8>;          // key: run (6 bits) | row (8) | col (9); 256 buckets of 4; digi = window slot
constexpr uint32_t WTAB = PH::SLOTS;

// Staged word (ring entry), written by the decode in its final form: pos | run | below | start, where run is the
// word's run counted inside its own chunk (0: it continues a run begun in an earlier chunk; RC+1: too many runs).
// As the head of the next window's... previous window such a word joins that window's last run (phase B writes the run
// back).  Neighbour keys are key+1 (col+1) and key+512-1, +512, +512+1 (row+1): col 416..511 and row 160..255 never
// occur, so no bounds checks (S13).
constexpr uint32_t SK_NONE = 0xFFFFFFFFu;   // no such word (outside the launch group)
constexpr uint32_t SK_BAD = 0xFFFFFF00u;    // >= SK_BAD: undecodable word, status in the low byte
constexpr uint32_t SK_POS = 0x1FFFFu;       // row << 9 | col
constexpr uint32_t SK_RUN_SHIFT = 17, SK_KEY = 0x7FFFFFu;  // run in bits 17-22; hash key = sk & SK_KEY
constexpr uint32_t SK_BELOW = 1u << 23, SK_START = 1u << 24;
static_assert(RC + 1u < 64u && MAXT <= 256u && 3u * MAXT + MAXT / 4u <= WTAB, "run field, slot field; sums + root list fit the hash memory");

struct __align__(16) WarpSmem {
  uint32_t tab[WTAB];      // position hash, EMPTY-filled.  After phase D: qn = tab, sx = tab + 256, sy = tab + 512, root list
  uint32_t label[MAXT];    // union-find parent of window slot t, or MARK_*
  uint32_t skey[MAXT];     // ring of two chunks: staged words (lane-private while staged: slot t belongs to lane t & 31)
  uint16_t chg[MAXT];      // ring: charges
  uint16_t edge[ECAP];     // a | b << 8; after the unions: local id of a root, or NO_ID
  uint32_t run_key[RC + 2];     // event_rel << 16 | module
  uint16_t run_base[RC + 2];    // clusters of the window that survive the cut before the run's first
  uint16_t run_cnt[RC + 2];     // clusters of the run that survive the cut
  uint8_t run_bad[RC + 2];      // the run is left to the warp-per-run kernel
};
static_assert(sizeof(WarpSmem) % 16 == 0, "per-warp slices stay 16-byte aligned");

struct Dec {          // what the decode of a chunk leaves in (warp-uniform) registers for its turn as home chunk
  uint32_t R;         // runs that start in the chunk
  uint32_t fs, ls;    // slot of the first / last run start (fs = HC: none)
  uint32_t ebase0;    // global index of word 0 of the event of the chunk's first word
  uint32_t er0;       // that event
  bool one_event;     // all 128 words exist and belong to event er0
};

// rare: event of word g (a FED / event boundary inside the chunk whose first word lies in segment sg0)
__device__ __noinline__ uint32_t event_of(const Chunk& c, uint32_t S, uint32_t sg0, uint32_t g) {
  uint32_t sg = sg0;
  while (sg + 1u < S && c.segB[sg + 1u] <= g) ++sg;
  return div_F(c, sg);
}

__global__ void __launch_bounds__(FT, BLOCKS_PER_SM) fused_kernel(const __grid_constant__ Chunk c) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  WarpSmem& s = reinterpret_cast<WarpSmem*>(smem_raw)[warp];
  const uint32_t F = c.F, S = (c.e1 - c.e0) * F;
  const uint32_t* __restrict__ segB = c.segB;
  const uint32_t gBeg = segB[0], gEnd = segB[S];
  if (gBeg >= gEnd) return;
  const uint32_t T0 = gBeg & ~(HC - 1u);
  const uint32_t n_chunks = (gEnd - T0 + HC - 1u) / HC;
  const uint32_t lt_mask = (1u << lane) - 1u, le_mask = lt_mask | (1u << lane);
  uint32_t* const qn = s.tab; uint32_t* const sx = s.tab + MAXT; uint32_t* const sy = s.tab + 2 * MAXT;
  uint8_t* const rlist = reinterpret_cast<uint8_t*>(s.tab + 3 * MAXT);  // roots in digi order (after phase D)
  uint16_t* const lid = s.edge;
  uint32_t G = n_chunks / (gridDim.x * WPB * 6u);  // about six tickets per warp
  G = G < 1u ? 1u : (G > GMAX ? GMAX : G);

  // per-event counters of the digis this lane has finished: dup | below << 16, ok | cut << 16, roots
  uint32_t acc_ev = NOKEY, accA = 0u, accB = 0u, accP = 0u;
  auto flush = [&]() {
    if (acc_ev != NOKEY) {
      const uint32_t a = __reduce_add_sync(FULL, accA), bb = __reduce_add_sync(FULL, accB), p = __reduce_add_sync(FULL, accP);
      if (lane == 0) {
        uint32_t* ec = c.ev_cnt + (size_t)acc_ev * EC_STRIDE;
        if (a & 0xFFFFu) atomicAdd(ec + EC_DUP, a & 0xFFFFu);
        if (a >> 16) atomicAdd(ec + EC_BELOW, a >> 16);
        if (bb & 0xFFFFu) atomicAdd(ec + EC_OK, bb & 0xFFFFu);
        if (bb >> 16) atomicAdd(ec + EC_CUT, bb >> 16);
        if (p) atomicAdd(ec + EC_PRECUT, p);
      }
    }
    accA = accB = accP = 0u;
  };

  while (true) {
    uint32_t ri = 0u;
    if (lane == 0) ri = atomicAdd(c.ctl + CTL_RANGE_TICKET, 1u);
    ri = __shfl_sync(FULL, ri, 0);
    const uint32_t c0 = ri * G;
    if (c0 >= n_chunks) break;
    const uint32_t c1 = c0 + G < n_chunks ? c0 + G : n_chunks;

    // ---- the last decodable word before the range, inside the event of the range's first word (an earlier event's
    // word never continues a run; segfill_kernel closes every event's last run)
    uint32_t carry_key = NOKEY, carry_g = 0u;
    {
      const uint32_t b = T0 + c0 * HC, gw = b < gBeg ? gBeg : b;
      const uint32_t sg0 = c.chunk_seg[c0], er = div_F(c, sg0), evb = segB[er * F];
      uint32_t g = gw;  // words [evb, g) are still to be searched, backwards
      while (g > evb) {
        const bool in = lane < g - evb;
        const uint32_t gi = g - 1u - lane;
        uint32_t key = NOKEY;
        if (in) {
          uint32_t sg = sg0;
          while (segB[sg] > gi) --sg;
          uint32_t m, r, cc;
          if (decode_word(c.cab, __ldg(c.words + gi), (sg - er * F) << 11, m, r, cc) == ST_OK) key = (er << 16) | m;
        }
        const uint32_t bal = __ballot_sync(FULL, key != NOKEY);
        if (bal) {
          const int src = __ffs(bal) - 1;
          carry_key = __shfl_sync(FULL, key, src);
          carry_g = g - 1u - (uint32_t)src;
          break;
        }
        g = (g - evb > 32u) ? g - 32u : evb;
      }
    }

    Dec cur, nxt;
    cur.R = 0u; cur.fs = HC; cur.ls = 0u; cur.ebase0 = 0u; cur.er0 = 0u; cur.one_event = false;
    uint32_t sgc = 0u;   // segment of the home chunk's first word
    uint4 wn = make_uint4(0u, 0u, 0u, 0u);  // the raw words of the chunk that is decoded next (loaded one iteration ahead)
    {
      const uint32_t g0 = T0 + c0 * HC + 4u * lane;
      if (g0 >= gBeg && g0 + 4u <= gEnd) wn = __ldg(reinterpret_cast<const uint4*>(c.words + g0));
      else {
        if (g0 >= gBeg && g0 < gEnd) wn.x = __ldg(c.words + g0);
        if (g0 + 1u >= gBeg && g0 + 1u < gEnd) wn.y = __ldg(c.words + g0 + 1u);
        if (g0 + 2u >= gBeg && g0 + 2u < gEnd) wn.z = __ldg(c.words + g0 + 2u);
        if (g0 + 3u >= gBeg && g0 + 3u < gEnd) wn.w = __ldg(c.words + g0 + 3u);
      }
    }

    for (uint32_t ci = c0;; ++ci) {
      const uint32_t hn = ((ci - c0) & 1u) * HC;  // ring half of chunk ci; chunk ci-1 sits in the other half
      // ================================================================== decode chunk ci (a1, a2, a3): four consecutive words per lane
      nxt.R = 0u; nxt.fs = HC; nxt.ls = 0u; nxt.ebase0 = 0u; nxt.er0 = 0u; nxt.one_event = false;
      uint32_t sgn = 0u;
      if (ci < n_chunks) {
        const bool owner = ci < c1;  // else: the look-ahead of the range's last window, nothing is written
        const uint32_t b = T0 + ci * HC, g0 = b + 4u * lane;
        const uint32_t sg0 = c.chunk_seg[ci];
        const uint32_t er0 = div_F(c, sg0), fed0 = sg0 - er0 * F;
        const uint32_t nextB0 = segB[sg0 + 1u], evend0 = segB[(er0 + 1u) * F], ebase0 = segB[er0 * F];
        const bool all_in = b >= gBeg && b + HC <= gEnd;
        const bool one_seg = all_in && b + HC <= nextB0;
        nxt.ebase0 = ebase0; nxt.er0 = er0; nxt.one_event = all_in && b + HC <= evend0;
        sgn = sg0;
        const uint32_t w[4] = {wn.x, wn.y, wn.z, wn.w};
        wn = make_uint4(0u, 0u, 0u, 0u);
        if (owner && ci + 1u < n_chunks) {  // the words of chunk ci + 1: in flight while this chunk is decoded and the window clustered
          const uint32_t h0 = g0 + HC;
          if (h0 + 4u <= gEnd) wn = __ldg(reinterpret_cast<const uint4*>(c.words + h0));
          else {
            if (h0 < gEnd) wn.x = __ldg(c.words + h0);
            if (h0 + 1u < gEnd) wn.y = __ldg(c.words + h0 + 1u);
            if (h0 + 2u < gEnd) wn.z = __ldg(c.words + h0 + 2u);
          }
        }
        uint32_t st[4], key[4], sk[4];
        uint32_t mod[4], row[4], col[4];
        int32_t chg[4];
        uint32_t exmask = 0u;  // words of the lane that exist
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const uint32_t g = g0 + j;
          const bool exists = all_in || (g >= gBeg && g < gEnd);
          exmask |= exists ? 1u << j : 0u;
          uint32_t er = er0, fed = fed0;
          if (!one_seg && exists) {  // rare: a FED / event boundary inside the chunk
            uint32_t sg = sg0;
            while (sg + 1u < S && segB[sg + 1u] <= g) ++sg;
            er = div_F(c, sg); fed = sg - er * F;
          }
          uint32_t m, r, cc;
          st[j] = decode_word(c.cab, w[j], fed << 11, m, r, cc);
          const bool ok = exists && st[j] == ST_OK;
          mod[j] = row[j] = col[j] = 0xFFFFu; chg[j] = 0; key[j] = NOKEY;
          if (ok) {
            mod[j] = m; row[j] = r; col[j] = cc;
            chg[j] = calibrate(c, w[j] & 255u, __ldg(c.gp + (m * (uint32_t)COLS + cc)));  // S8: one pair per (module, col)
            key[j] = (er << 16) | m;
          } else if (owner && exists) {
            atomicAdd(c.ev_cnt + (size_t)er * EC_STRIDE + (st[j] - ST_EMPTY), 1u);
          }
        }
        if (owner) {
          if (exmask == 15u) {
            *reinterpret_cast<ushort4*>(c.d_module + g0) = make_ushort4(mod[0], mod[1], mod[2], mod[3]);
            *reinterpret_cast<ushort4*>(c.d_row + g0) = make_ushort4(row[0], row[1], row[2], row[3]);
            *reinterpret_cast<ushort4*>(c.d_col + g0) = make_ushort4(col[0], col[1], col[2], col[3]);
            *reinterpret_cast<int4*>(c.d_charge + g0) = make_int4(chg[0], chg[1], chg[2], chg[3]);
          } else {
#pragma unroll
            for (int j = 0; j < 4; ++j) {
              if (!(exmask >> j & 1u)) continue;
              const uint32_t g = g0 + j;
              c.d_module[g] = (uint16_t)mod[j]; c.d_row[g] = (uint16_t)row[j]; c.d_col[g] = (uint16_t)col[j];
              c.d_charge[g] = chg[j];
            }
          }
          // undecodable words are finished here (status, clus = -1)
          const uint32_t badmask = (key[0] == NOKEY ? 1u : 0u) | (key[1] == NOKEY ? 2u : 0u) | (key[2] == NOKEY ? 4u : 0u) | (key[3] == NOKEY ? 8u : 0u);
          if (badmask & exmask) {
            if (badmask == 15u && exmask == 15u) {
              *reinterpret_cast<uchar4*>(c.d_status + g0) = make_uchar4(st[0], st[1], st[2], st[3]);
              *reinterpret_cast<int4*>(c.d_clus + g0) = make_int4(-1, -1, -1, -1);
            } else {
#pragma unroll
              for (int j = 0; j < 4; ++j)
                if ((badmask & exmask) >> j & 1u) { c.d_status[g0 + j] = (uint8_t)st[j]; c.d_clus[g0 + j] = -1; }
            }
          }
        }
        // a3: a word starts a run when its (event, module) differs from the previous decodable word's
        uint32_t tkey = NOKEY, tj = 0u;  // the lane's last decodable word
#pragma unroll
        for (int j = 0; j < 4; ++j) if (key[j] != NOKEY) { tkey = key[j]; tj = j; }
        const uint32_t has = __ballot_sync(FULL, tkey != NOKEY);
        const uint32_t below_l = has & lt_mask;
        const int src = below_l ? 31 - __clz(below_l) : 0;
        uint32_t pkey = __shfl_sync(FULL, tkey, src), pg = b + 4u * (uint32_t)src + __shfl_sync(FULL, tj, src);
        if (!below_l) { pkey = carry_key; pg = carry_g; }
        uint32_t startmask = 0u;
        uint32_t s_key = NOKEY, s_g = 0u, s_pkey = NOKEY, s_pg = 0u;  // the lane's first run start and its predecessor
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          if (key[j] == NOKEY) continue;
          if (key[j] != pkey) {
            if (!startmask) { s_key = key[j]; s_g = g0 + j; s_pkey = pkey; s_pg = pg; }
            startmask |= 1u << j;
          }
          pkey = key[j]; pg = g0 + j;
        }
        if (owner) {
          if (s_key != NOKEY) {  // one copy of the atomics for the usual case of at most one start per lane
            run_start(c, s_key, s_g);
            if (s_pkey != NOKEY) run_end(c, s_pkey, s_pg);
          }
          if (startmask & (startmask - 1u)) {  // rare: several runs start inside the lane's four words
            uint32_t pk = NOKEY, pgg = 0u;
            bool first = true;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
              if (key[j] == NOKEY) continue;
              if (startmask >> j & 1u) {
                if (!first) { run_start(c, key[j], g0 + j); run_end(c, pk, pgg); }
                first = false;
              }
              pk = key[j]; pgg = g0 + j;
            }
          }
        }
        if (has) {
          const int top = 31 - __clz(has);
          carry_key = __shfl_sync(FULL, tkey, top); carry_g = b + 4u * (uint32_t)top + __shfl_sync(FULL, tj, top);
        }
        // runs: the word's run counted inside the chunk; chunk totals
        const uint32_t anyst = __ballot_sync(FULL, startmask != 0u);
        uint32_t rbefore = __popc(startmask);  // inclusive scan over the lanes, then made exclusive
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
          const uint32_t o = __shfl_up_sync(FULL, rbefore, d);
          if (lane >= (uint32_t)d) rbefore += o;
        }
        nxt.R = __shfl_sync(FULL, rbefore, 31);
        rbefore -= __popc(startmask);
        if (anyst) {
          const int fl = __ffs(anyst) - 1, ll = 31 - __clz(anyst);
          nxt.fs = 4u * (uint32_t)fl + (uint32_t)__ffs(__shfl_sync(FULL, startmask, fl)) - 1u;
          nxt.ls = 4u * (uint32_t)ll + 31u - (uint32_t)__clz(__shfl_sync(FULL, startmask, ll));
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          uint32_t r = rbefore + __popc(startmask & ((2u << j) - 1u));
          r = r <= RC ? r : RC + 1u;
          sk[j] = key[j] != NOKEY ? ((row[j] << 9) | col[j] | (r << SK_RUN_SHIFT) | (chg[j] < c.thr ? SK_BELOW : 0u) | ((startmask >> j & 1u) ? SK_START : 0u))
                                  : ((exmask >> j & 1u) ? (SK_BAD | st[j]) : SK_NONE);
        }
        *reinterpret_cast<uint4*>(&s.skey[hn + 4u * lane]) = make_uint4(sk[0], sk[1], sk[2], sk[3]);
        *reinterpret_cast<ushort4*>(&s.chg[hn + 4u * lane]) = make_ushort4(chg[0], chg[1], chg[2], chg[3]);
      }
      __syncwarp();  // the staged chunk is visible to every lane

      // ================================================================== cluster the window of chunk ci - 1
      if (ci > c0) {
        const uint32_t hb = hn ^ HC;                 // ring half of the home chunk
        const uint32_t b = T0 + (ci - 1u) * HC;      // global index of the home chunk's word 0
        const uint32_t R = cur.R;
        uint32_t f_t = MAXT, e_t = 0u;               // window = chunk slots [f_t, e_t); empty when nothing is owned
        uint32_t Rown = R;                           // runs of the window (the last run may be left to findrun)
        if (R) {
          f_t = cur.fs;
          // end of the last run: the first run start of the next chunk, the end of the data, or "does not fit"
          if (nxt.fs < HC) {
            e_t = HC + nxt.fs;
          } else if (b + MAXT >= gEnd) {
            e_t = gEnd - b;
          } else {  // the last run does not end inside the next chunk: the warp-per-run kernel takes it
            e_t = cur.ls;
            if (lane == 0) {
              const uint32_t er = cur.one_event ? cur.er0 : event_of(c, S, sgc, b + e_t);
              push_run(c, c.mid_list, CTL_MID_COUNT, er, c.d_module[b + e_t]);
            }
            Rown = R - 1u;
            if (e_t == f_t) { f_t = MAXT; e_t = 0u; }  // it was the only run
          }
        }
        if (e_t > f_t) {
          // window slot t <-> chunk slot f_t + t <-> ring entry (hb + f_t + t) & 255 <-> word wb + t
          const uint32_t len = e_t - f_t, nk = (len + 31u) >> 5, pb = hb + f_t, wb = b + f_t;
          const uint32_t nhome = HC - f_t;  // window slots of the home chunk; the rest is the head of the next chunk
          // the window's stretch of the temp record area, one slot per digi: asked for now, needed in phase F
          uint32_t wbase_l = 0u;
          if (lane == 0) wbase_l = alloc_temp(c, len);
          // ============================================================== B: clear; run tables; insert
          {
            uint4* t4 = reinterpret_cast<uint4*>(s.tab);
            const uint4 e4 = make_uint4(PH::EMPTY, PH::EMPTY, PH::EMPTY, PH::EMPTY);
#pragma unroll
            for (int k = 0; k < (int)(WTAB / 4 / 32); ++k) t4[lane + 32 * k] = e4;
            if (lane < (RC + 2u) / 4u) reinterpret_cast<uint32_t*>(s.run_bad)[lane] = 0u;
            reinterpret_cast<uint32_t*>(s.run_cnt)[lane] = 0u;
          }
          __syncwarp();  // the cleared hash is visible
          if (Rown > RC && lane == 0) s.run_bad[RC + 1u] = 1;  // the runs beyond RC are all "run RC + 1"
          bool dup_seen = false;
          const uint32_t Rr = R <= RC ? R : RC + 1u;             // run of the slots of the next chunk
#pragma unroll 1
          for (uint32_t k = 0; k < nk; ++k) {
            const uint32_t t = 32u * k + lane, ph = (pb + t) & (MAXT - 1u);
            uint32_t sk = s.skey[ph];
            const bool dec = t < len && sk < SK_BAD;
            if (t >= nhome && dec) { sk |= Rr << SK_RUN_SHIFT; s.skey[ph] = sk; }  // the head of the next chunk: the rest of run R
            const uint32_t r = (sk >> SK_RUN_SHIFT) & 63u;
            if (dec && (sk & SK_START)) {
              const uint32_t er = cur.one_event ? cur.er0 : event_of(c, S, sgc, wb + t);
              const uint32_t m = c.d_module[wb + t];  // written by this warp when it decoded the chunk
              if (r <= RC) {
                s.run_key[r] = (er << 16) | m;
              } else {
                push_run(c, c.mid_list, CTL_MID_COUNT, er, m);  // too many runs: left to findrun
              }
            }
            const bool live = dec && !(sk & SK_BELOW) && r <= RC;
            s.label[t] = live ? t : MARK_BELOW;
            if (dec && r <= RC) {
              const uint32_t ins = PH::insert(s.tab, sk & SK_KEY, t, (sk & SK_BELOW) ? 1u : 0u);
              dup_seen |= ins == 1u;
              if (ins == 2u) s.run_bad[r] = 1;  // no room near the home bucket: findrun takes the run
            }
          }
          __syncwarp();  // hash, labels, run tables complete
          const uint32_t Rw = Rown < RC ? Rown : RC;  // runs of this window that are numbered here

          // ============================================================== D: duplicates; neighbours -> edges -> unions
          if (__any_sync(FULL, dup_seen)) {  // rare: some pixel appears twice; the digi not in the slot is a DUPLICATE (S10)
            for (uint32_t k = 0; k < nk; ++k) {
              const uint32_t t = 32u * k + lane, sk = s.skey[(pb + t) & (MAXT - 1u)];
              const bool dec = t < len && sk < SK_BAD && ((sk >> SK_RUN_SHIFT) & 63u) <= RC;
              if (dec && PH::digi(PH::find(s.tab, PH::mix(sk & SK_KEY))) != t) s.label[t] = MARK_DUP;
            }
            __syncwarp();
          }
          // Forward neighbours (S13): E (r, c+1), SW (r+1, c-1), S (r+1, c), SE (r+1, c+1).  When S is live, SW and SE
          // are joined to it by their own E edges, so d-S alone is enough; when E is live, SE is E's S neighbour.
          uint32_t ne = 0u;
#pragma unroll 1
          for (uint32_t k = 0; k <= nk; ++k) {
            if (k == nk || ne + 96u > ECAP) {  // the last round is done, or the next round's edges might not fit: unite what is listed
              __syncwarp();
              for (uint32_t i0 = 0u; i0 < ne; i0 += 32u) {  // warp-uniform trip count: the lanes reconverge every iteration
                if (i0 + lane < ne) {
                  const uint32_t e = s.edge[i0 + lane];
                  hook(s.label, e & 0xFFu, e >> 8);
                }
                __syncwarp();
              }
              ne = 0u;
              if (k == nk) break;
            }
            const uint32_t t = 32u * k + lane, sk = s.skey[(pb + t) & (MAXT - 1u)];
            const bool live = s.label[t] < MAXT;  // slots beyond the window and undecodable words carry MARK_BELOW
            bool f0 = false, f1 = false, f2 = false;
            uint32_t n0 = 0, n1 = 0, n2 = 0;
            if (live) {
              const uint32_t h = PH::mix(sk & SK_KEY);
              bool o0, o1, o2, o3;  // one branch for the four lookups: a full home bucket without a match is rare
              uint32_t eE = PH::find_home(s.tab, PH::step(h, 1u), o0), eS = PH::find_home(s.tab, PH::step(h, 512u), o1);
              uint32_t eSW = PH::find_home(s.tab, PH::step(h, 511u), o2), eSE = PH::find_home(s.tab, PH::step(h, 513u), o3);
              if (o0 | o1 | o2 | o3) {
                if (o0) eE = PH::find_slow(s.tab, PH::step(h, 1u));
                if (o1) eS = PH::find_slow(s.tab, PH::step(h, 512u));
                if (o2) eSW = PH::find_slow(s.tab, PH::step(h, 511u));
                if (o3) eSE = PH::find_slow(s.tab, PH::step(h, 513u));
              }
              const bool hS = PH::live(eS);
              f0 = PH::live(eE); n0 = PH::digi(eE);
              f1 = hS || PH::live(eSW); n1 = PH::digi(hS ? eS : eSW);
              f2 = !hS && !f0 && PH::live(eSE); n2 = PH::digi(eSE);  // with E live, SE is E's S: E joins it
            }
            const uint32_t m0 = __ballot_sync(FULL, f0), m1 = __ballot_sync(FULL, f1), m2 = __ballot_sync(FULL, f2);
            if (f0) s.edge[ne + __popc(m0 & lt_mask)] = (uint16_t)(t | (n0 << 8));
            ne += __popc(m0);
            if (f1) s.edge[ne + __popc(m1 & lt_mask)] = (uint16_t)(t | (n1 << 8));
            ne += __popc(m1);
            if (f2) s.edge[ne + __popc(m2 & lt_mask)] = (uint16_t)(t | (n2 << 8));
            ne += __popc(m2);
          }
#pragma unroll 1
          for (int pass = 0; pass < 2; ++pass) {  // two pointer-jumping rounds: the chains shrink 4x before the sums (measured: 0 -> 1 -> 2 rounds = 2.91 -> 2.78 -> 2.73 ms)
            for (uint32_t k = 0; k < nk; ++k) {
              const uint32_t t = 32u * k + lane;
              const uint32_t l = s.label[t];
              if (l < MAXT) { const uint32_t ll = s.label[l]; if (ll != l) s.label[t] = ll; }
            }
            __syncwarp();
          }

          // ============================================================== E: cluster sums (the hash is dead: qn / sx / sy / root list)
          {
            uint4* t4 = reinterpret_cast<uint4*>(s.tab);
            const uint4 z4 = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
            for (int k = 0; k < (int)(3 * MAXT / 4 / 32); ++k) t4[lane + 32 * k] = z4;
          }
          __syncwarp();
          uint32_t nr = 0u;  // roots so far
#pragma unroll 1
          for (uint32_t k = 0; k < nk; ++k) {
            const uint32_t t = 32u * k + lane;
            volatile uint32_t* L = s.label;
            uint32_t r = L[t];
            const bool live = r < MAXT;  // else MARK_*
            if (live) {
              while (true) { const uint32_t n = L[r]; if (n == r) break; r = n; }
              L[t] = r;  // flatten: r is the root, so other walkers through t stay correct
              const uint32_t ph = (pb + t) & (MAXT - 1u);
              const uint32_t sk = s.skey[ph], e = s.chg[ph];
              atomicAdd(&qn[r], e | (1u << 24));  // charge sum (< 2^24: 256 * 65535) | pixel count (256 wraps to 0)
              atomicAdd(&sx[r], e * (sk & 511u));
              atomicAdd(&sy[r], e * ((sk >> 9) & 255u));
            }
            const bool root = live && r == t;
            const uint32_t rm = __ballot_sync(FULL, root);
            if (root) rlist[nr + __popc(rm & lt_mask)] = (uint8_t)t;  // digi order
            nr += __popc(rm);
          }
          __syncwarp();

          // ============================================================== F: cut, renumber, temp records (one root per lane)
          uint32_t wbase_w = 0u;
          {
            uint32_t cnt = 0u;                   // surviving roots before this iteration
            uint32_t run_c = 0u, base_c = 0u;    // the run of the last root so far and the survivors before that run
            const uint32_t wbase = __shfl_sync(FULL, wbase_l, 0);
            wbase_w = wbase;
#pragma unroll 1
            for (uint32_t i0 = 0u; i0 < nr; i0 += 32u) {
              const bool valid = i0 + lane < nr;
              uint32_t t = 0u, r = 0u, Q = 0u, np = 0u;
              if (valid) {
                t = rlist[i0 + lane];
                r = (s.skey[(pb + t) & (MAXT - 1u)] >> SK_RUN_SHIFT) & 63u;
                const uint32_t v = qn[t];
                Q = v & 0xFFFFFFu; np = v >> 24;
                if (np == 0u) np = 256u;
                if (Q > Q_SAFE) s.run_bad[r] = 1;  // 32-bit weighted sums may have wrapped
              }
              const bool surv = valid && (int32_t)Q >= c.cut;  // S9: equality keeps
              const uint32_t sm = __ballot_sync(FULL, surv);
              const uint32_t rank = cnt + __popc(sm & lt_mask);
              // runs are contiguous in digi order: the first lane of this lane's run in this iteration
              const uint32_t rprev = __shfl_up_sync(FULL, r, 1);
              const uint32_t bnd = __ballot_sync(FULL, valid && (lane == 0u || r != rprev));
              const uint32_t fl = 31u - (uint32_t)__clz(bnd & le_mask);  // bit 0 of bnd is set: lane 0 is valid
              uint32_t base = cnt + __popc(sm & ((1u << fl) - 1u));
              if (fl == 0u && r == run_c) base = base_c;  // the run began in an earlier iteration
              if (valid) {
                uint32_t id = NO_ID;
                if (surv) {
                  id = rank - base;
                  // S18: exact integer sums, one rounding each + a 2-ulp division (within 1e-5)
                  const float fq = (float)Q;
                  const uint32_t ifirst = wb + t - (cur.one_event ? cur.ebase0 : segB[(s.run_key[r] >> 16) * F]);  // event-relative index
                  put_temp(c, wbase + rank, ifirst, np, Q, __fdividef((float)sx[t], fq), __fdividef((float)sy[t], fq));
                }
                lid[t] = (uint16_t)id;
                // the last root of the run in this iteration leaves the run's count so far
                const bool lastofrun = lane == 31u || i0 + lane + 1u == nr || ((bnd >> (lane + 1u)) & 1u);
                if (lastofrun) { s.run_cnt[r] = (uint16_t)(rank + (surv ? 1u : 0u) - base); s.run_base[r] = (uint16_t)base; }
              }
              const uint32_t lastl = 31u - (uint32_t)__clz(__ballot_sync(FULL, valid));
              run_c = __shfl_sync(FULL, r, lastl); base_c = __shfl_sync(FULL, base, lastl);
              cnt += __popc(sm);
            }
          }
          __syncwarp();  // run_cnt, run_bad, local ids final
          for (uint32_t r = 1u + lane; r <= Rw; r += 32u) {
            const uint32_t key = s.run_key[r];
            if (s.run_bad[r]) push_run(c, c.mid_list, CTL_MID_COUNT, key >> 16, key & 0xFFFFu);
            else {
              const uint32_t mo = (key >> 16) * c.M + (key & 0xFFFFu);
              c.n_clus[mo] = s.run_cnt[r]; c.t_base[mo] = wbase_w + s.run_base[r];
            }
          }

          // ============================================================== G: final status and clus, counters
          uint32_t cntA = 0u, cntB = 0u, n_pre = 0u;  // dup | below << 16 ; ok | cut << 16 ; roots
#pragma unroll 1
          for (uint32_t k = 0; k < nk; ++k) {
            const uint32_t t = 32u * k + lane, sk = s.skey[(pb + t) & (MAXT - 1u)];
            if (t < len && sk < SK_BAD && !s.run_bad[(sk >> SK_RUN_SHIFT) & 63u]) {
              const uint32_t lab = s.label[t];
              uint32_t so; int32_t cl = -1;
              if (lab == MARK_DUP) { so = ST_DUP; cntA += 1u; }
              else if (lab == MARK_BELOW) { so = ST_BELOW; cntA += 0x10000u; }
              else {
                const uint32_t id = lid[lab];
                if (id != NO_ID) { so = ST_OK; cl = (int32_t)id; cntB += 1u; } else { so = ST_CUT; cntB += 0x10000u; }
                n_pre += lab == t ? 1u : 0u;
              }
              c.d_status[wb + t] = (uint8_t)so; c.d_clus[wb + t] = cl;
              if (!cur.one_event) {  // rare: an event boundary inside the chunk; every digi counts for its own event
                uint32_t* ec = c.ev_cnt + (size_t)(s.run_key[(sk >> SK_RUN_SHIFT) & 63u] >> 16) * EC_STRIDE;
                atomicAdd(ec + (so == ST_DUP ? EC_DUP : (so == ST_BELOW ? EC_BELOW : (so == ST_OK ? EC_OK : EC_CUT))), 1u);
                if (lab == t) atomicAdd(ec + EC_PRECUT, 1u);
              }
            }
          }
          if (cur.one_event) {
            if (cur.er0 != acc_ev) { flush(); acc_ev = cur.er0; }
            accA += cntA; accB += cntB; accP += n_pre;
          }
          __syncwarp();  // shared state is rewritten by the next window
        }
      }
      if (ci >= c1) break;
      cur = nxt; sgc = sgn;
    }
    flush();
    acc_ev = NOKEY;
  }
}

}  // namespace

cudaError_t configure_fused_kernel() {
  return cudaFuncSetAttribute(fused_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(WPB * sizeof(WarpSmem)));
}

void launch_fused(const Chunk& c, uint32_t words_bound, int n_sm, cudaStream_t stream) {
  uint64_t nb = ((uint64_t)words_bound + 2 * HC + WPB * HC - 1) / (WPB * HC);
  if (nb < 1) nb = 1;
  if (nb > (uint64_t)n_sm * BLOCKS_PER_SM) nb = (uint64_t)n_sm * BLOCKS_PER_SM;
  fused_kernel<<<(int)nb, FT, WPB * sizeof(WarpSmem), stream>>>(c);
}

}  // namespace pix
