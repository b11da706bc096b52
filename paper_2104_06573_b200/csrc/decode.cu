// decode.cu -- init, and the streaming decode kernel: a1 decode (S1-S6), a2 calibrate (S7-S9) and a3
// module boundaries (S11, S12) of the path PAPER.md:31 describes ("unpacks them, calibrates the individual
// pixels, and clusters the pixels on each detector module").
//
// One warp per 128 consecutive words, 4 per lane (one 128-bit load, 128-bit / 64-bit stores).  The warp
//   - reads the (event, FED) segment of its first word (segfill_kernel) and looks back for the last decodable
//     word before the chunk
//   - decodes + calibrates, stores module / row / col / charge, and finishes the undecodable words
//     (status, clus = -1, per-event error counters)
//   - finds run starts (a decodable word whose (event, module) differs from the previous decodable word's)
//     with a ballot/shuffle scan, updates module_first / module_end (a3), and writes one start bit per word
//     for the cluster kernel (findclus.cu)
// Nothing here is shared with oracle/.
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
// chunk_seg[ci] = segment (event, FED) of the first word of 128-word chunk ci (its first word inside the launch
// group).  One thread per segment writes the chunks that start inside it.
__global__ void __launch_bounds__(256) segfill_kernel(const __grid_constant__ Chunk c) {
  const uint32_t S = (c.e1 - c.e0) * c.F;
  const uint32_t gBeg = c.segB[0], gEnd = c.segB[S];
  if (gBeg >= gEnd) return;
  const uint32_t T0 = gBeg & ~(CHUNK_WORDS - 1u);
  for (uint32_t sgi = blockIdx.x * blockDim.x + threadIdx.x; sgi < S; sgi += gridDim.x * blockDim.x) {
    const uint32_t lo = c.segB[sgi], hi = c.segB[sgi + 1u];
    if (lo >= hi) continue;
    const uint32_t c_lo = lo == gBeg ? 0u : (lo - T0 + CHUNK_WORDS - 1u) / CHUNK_WORDS;
    const uint32_t c_hi = (hi - T0 + CHUNK_WORDS - 1u) / CHUNK_WORDS;  // exclusive
    for (uint32_t ci = c_lo; ci < c_hi; ++ci) c.chunk_seg[ci] = sgi;
  }
}

// sg / F (F is a power of two in both detector configurations: a shift)
__device__ __forceinline__ uint32_t div_F(const Chunk& c, uint32_t sg) { return c.F_shift != 0xFFFFFFFFu ? sg >> c.F_shift : sg / c.F; }

// ------------------------------------------------------------------ the streaming decode kernel
constexpr int DT = 256;

__global__ void __launch_bounds__(DT) decode_kernel(const __grid_constant__ Chunk c) {
  const uint32_t F = c.F, S = (c.e1 - c.e0) * F;
  const uint32_t* __restrict__ segB = c.segB;
  const uint32_t gBeg = segB[0], gEnd = segB[S];
  if (gBeg >= gEnd) return;
  const uint32_t T0 = gBeg & ~(CHUNK_WORDS - 1u);
  const uint32_t n_chunks = (gEnd - T0 + CHUNK_WORDS - 1u) / CHUNK_WORDS;
  const uint32_t lane = threadIdx.x & 31u;
  const uint32_t lt_mask = (1u << lane) - 1u;
  constexpr uint32_t FULL = 0xFFFFFFFFu;

  for (uint32_t ci = (blockIdx.x * DT + threadIdx.x) >> 5; ci < n_chunks; ci += (gridDim.x * DT) >> 5) {
    const uint32_t b = T0 + ci * CHUNK_WORDS, g0 = b + lane * 4u;
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
    // ---- segment (event, FED) of the chunk's first word; look-back for the last decodable word before it
    const uint32_t gw = b < gBeg ? gBeg : b;  // b < gEnd by the chunk count
    const uint32_t sg0 = c.chunk_seg[ci];  // filled by segfill_kernel
    const uint32_t nextB0 = segB[sg0 + 1u];
    const bool allfull = __all_sync(FULL, full);
    uint32_t ckey = NOKEY, cg = 0u;
    if (gw > gBeg) {
      // common case, warp-uniform: the word just before the chunk is decodable
      uint32_t g = gw;  // words [gBeg, g) are still to be searched, backwards
      {
        const uint32_t gi = gw - 1u;
        uint32_t sg = sg0;
        while (segB[sg] > gi) --sg;  // segB[0] = gBeg <= gi
        const uint32_t er = div_F(c, sg), fed = sg - er * F;
        uint32_t m, r, cc;
        if (decode_word(c.cab, __ldg(c.words + gi), fed << 11, m, r, cc) == ST_OK) { ckey = (er << 16) | m; cg = gi; g = gBeg; }
        else g = gi;
      }
      while (g > gBeg) {  // rare: undecodable words before the chunk, 32 at a time
        const bool in = lane < g - gBeg;
        const uint32_t gi = g - 1u - lane;
        uint32_t key = NOKEY;
        if (in) {
          uint32_t sg = sg0;
          while (segB[sg] > gi) --sg;
          const uint32_t er = div_F(c, sg), fed = sg - er * F;
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
    // ---- a1 + a2
    uint32_t st[4], key[4];
    uint32_t tkey = NOKEY, tg = 0u;
    {
      uint32_t mod[4], row[4], col[4];
      int32_t chg[4];
      uint32_t inmask = 0u;
      uint32_t sg = sg0, nextB = nextB0;
      if (b + CHUNK_WORDS > nextB0 && any) {  // warp-uniform test; rare: a FED / event boundary inside the chunk
        const uint32_t gf = g0 < gBeg ? gBeg : g0;
        while (sg + 1u < S && segB[sg + 1u] <= gf) ++sg;
        nextB = segB[sg + 1u];
      }
      uint32_t er = div_F(c, sg), fed = sg - er * F;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const uint32_t g = g0 + j;
        st[j] = 0xFFu; key[j] = NOKEY; mod[j] = row[j] = col[j] = 0xFFFFu; chg[j] = 0;
        if (!allfull && (!any || g < gBeg || g >= gEnd)) continue;
        inmask |= 1u << j;
        if (g >= nextB) {  // rare: the thread's words straddle a FED / event boundary
          while (sg + 1u < S && segB[sg + 1u] <= g) ++sg;
          er = div_F(c, sg); fed = sg - er * F; nextB = segB[sg + 1u];
        }
        uint32_t m, r, cc;
        st[j] = decode_word(c.cab, w[j], fed << 11, m, r, cc);
        if (st[j] == ST_OK) {
          mod[j] = m; row[j] = r; col[j] = cc;
          const float2 gp = __ldg(c.gp + (m * (uint32_t)COLS + cc));  // S8: one pair per (module, col)
          chg[j] = calibrate(c, w[j] & 255u, gp);
          key[j] = (er << 16) | m;
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
        if (st[0] != ST_OK && st[1] != ST_OK && st[2] != ST_OK && st[3] != ST_OK) {  // undecodable: finished here
          *reinterpret_cast<uchar4*>(c.d_status + g0) = make_uchar4(st[0], st[1], st[2], st[3]);
          *reinterpret_cast<int4*>(c.d_clus + g0) = make_int4(-1, -1, -1, -1);
          inmask = 0u;
        }
      } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          if (!(inmask >> j & 1u)) continue;
          const uint32_t g = g0 + j;
          c.d_module[g] = (uint16_t)mod[j]; c.d_row[g] = (uint16_t)row[j]; c.d_col[g] = (uint16_t)col[j];
          c.d_charge[g] = chg[j];
        }
      }
#pragma unroll
      for (int j = 0; j < 4; ++j)
        if ((inmask >> j & 1u) && st[j] != ST_OK) { c.d_status[g0 + j] = (uint8_t)st[j]; c.d_clus[g0 + j] = -1; }
    }
    // ---- a3: previous decodable word of every thread (warp-shuffle last-valid scan + the look-back carry)
    const uint32_t has = __ballot_sync(FULL, tkey != NOKEY);
    const uint32_t below_l = has & lt_mask;
    const int src = below_l ? 31 - __clz(below_l) : 0;
    uint32_t pkey = __shfl_sync(FULL, tkey, src), pg = __shfl_sync(FULL, tg, src);
    if (!below_l) { pkey = ckey; pg = cg; }
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
    if (s_key != NOKEY) {  // one copy of the atomics for the usual case of at most one start per lane
      run_start(c, s_key, s_g);
      if (s_pkey != NOKEY) run_end(c, s_pkey, s_pg);
    }
    if (startmask & (startmask - 1u)) {  // rare: several runs start inside the lane's four words
      uint32_t pk = NOKEY, pgg = 0u;
      bool first = true;
#pragma unroll 1
      for (int j = 0; j < 4; ++j) {
        if (key[j] == NOKEY) continue;
        if (startmask >> j & 1u) {
          if (!first) { run_start(c, key[j], g0 + j); run_end(c, pk, pgg); }
          first = false;
        }
        pk = key[j]; pgg = g0 + j;
      }
    }
    if (ci == n_chunks - 1u) {  // the chunk's last run ends at the last decodable word
      const int top = has ? 31 - __clz(has) : 0;
      uint32_t lk = __shfl_sync(FULL, tkey, top), lg = __shfl_sync(FULL, tg, top);
      if (!has) { lk = ckey; lg = cg; }
      if (lane == 0 && lk != NOKEY) run_end(c, lk, lg);
    }
    // ---- one start bit per word: lanes 8q .. 8q+7 assemble mask word q of the chunk
    uint32_t v = startmask << (4u * (lane & 7u));
    v |= __shfl_xor_sync(FULL, v, 1); v |= __shfl_xor_sync(FULL, v, 2); v |= __shfl_xor_sync(FULL, v, 4);
    if ((lane & 7u) == 0u) c.startbits[ci * 4u + (lane >> 3)] = v;
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
  segfill_kernel<<<grid_for(Ec * c.F, 256, n_sm * 8), 256, 0, stream>>>(c);
}

void launch_decode(const Chunk& c, uint32_t words_bound, int n_sm, cudaStream_t stream) {
  decode_kernel<<<grid_for(words_bound + CHUNK_WORDS, (DT / 32) * CHUNK_WORDS, n_sm * 32), DT, 0, stream>>>(c);
}

}  // namespace pix
