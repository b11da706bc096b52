// unpack.cu -- init, unpack+calibrate+run-boundaries, classify.
//
// a1 decode (S1-S6), a2 calibrate (S7-S9), a3 module boundaries (S11, S12) of the path
// PAPER.md:31 describes ("unpacks them, calibrates the individual pixels ... on each detector module").
#include "pix_common.cuh"

namespace pix {

namespace {

constexpr int UNPACK_THREADS = 256;
constexpr int UNPACK_WARPS = UNPACK_THREADS / 32;
constexpr uint32_t TILE = UNPACK_THREADS * 4;  // one 128-bit load of 4 words per thread
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
  if (tid < 16) c.ctl[tid] = 0;
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
  for (uint32_t t = tid; t < nmod; t += nth) { mf[t] = NO_INDEX; me[t] = 0u; }
}

// ------------------------------------------------------------------ decode / calibrate
// S1-S6.  Returns the status; module/row/col are defined only for ST_OK.
__device__ __forceinline__ uint32_t decode_word(const uint32_t* __restrict__ cab, uint32_t w, uint32_t fed,
                                                uint32_t& module, uint32_t& row, uint32_t& col) {
  if (w == 0u) return ST_EMPTY;
  const uint32_t link = w >> 26, roc = (w >> 21) & 31u, dcol = (w >> 16) & 31u, pxid = (w >> 8) & 255u;
  const uint32_t e = __ldg(cab + ((fed * 64u + link) * 32u + roc));
  if (!(e & 1u)) return ST_ERR_LINK;
  if (!(e & 2u)) return ST_ERR_ROC;
  if (dcol >= 26u) return ST_ERR_DCOL;
  if (pxid >= 160u) return ST_ERR_PXID;
  const uint32_t rr = pxid >> 1, cc = 2u * dcol + (pxid & 1u);
  module = (e >> 2) & 0xFFFFu;
  row = ((e >> 21) & 1u) * ROC_ROWS + ((e & (1u << 22)) ? (ROC_ROWS - 1 - rr) : rr);
  col = ((e >> 18) & 7u) * ROC_COLS + ((e & (1u << 23)) ? (ROC_COLS - 1 - cc) : cc);
  return ST_OK;
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

__device__ __forceinline__ void run_start(const Chunk& c, uint32_t key, uint32_t g) {
  const uint32_t er = key >> 16, m = key & 0xFFFFu;
  const uint32_t i = g - c.segB[er * c.F];
  const uint32_t old = atomicMin(c.module_first + ((size_t)(c.e0 + er) * c.M + m), i);
  if (old != NO_INDEX) atomicOr(c.ev_cnt + (size_t)er * EC_STRIDE + EC_FLAGS, FLAG_NONCONTIGUOUS);  // S11
}
__device__ __forceinline__ void run_end(const Chunk& c, uint32_t key, uint32_t g) {
  const uint32_t er = key >> 16, m = key & 0xFFFFu;
  atomicMax(c.module_end + ((size_t)(c.e0 + er) * c.M + m), g - c.segB[er * c.F] + 1u);
}

// ------------------------------------------------------------------ unpack
// Grid-stride over tiles of 1024 words of the chunk's global word range.  Per thread: one 128-bit load,
// decode + calibrate 4 words, 64/128/32-bit stores per output array.  Run boundaries: a word starts a run
// iff the previous decodable word of the chunk has another (event, module) key; found with a ballot/shuffle
// "last valid" scan inside the warp, a per-warp carry through shared memory, and a look-back into the raw
// words across the tile boundary.
__global__ void __launch_bounds__(UNPACK_THREADS) unpack_kernel(const __grid_constant__ Chunk c) {
  __shared__ uint32_t s_seg;
  __shared__ uint2 s_carry;
  __shared__ uint2 s_warp_last[UNPACK_WARPS];
  const uint32_t Ec = c.e1 - c.e0, S = Ec * c.F;
  const uint32_t* __restrict__ segB = c.segB;
  const uint32_t gBeg = segB[0], gEnd = segB[S];
  if (gBeg >= gEnd) return;
  const uint32_t T0 = gBeg & ~3u;
  const uint32_t n_tiles = (gEnd - T0 + TILE - 1u) / TILE;
  const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;

  for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const uint32_t tBeg = T0 + tile * TILE;
    const uint32_t tFirst = tBeg < gBeg ? gBeg : tBeg;  // first word of the tile that belongs to the chunk
    // ---- warp 0: segment of the tile's first word, and look-back for the last decodable word before it
    if (warp == 0) {
      const uint32_t s0 = warp_find_segment(segB, S, tFirst, lane);
      uint2 carry = make_uint2(NOKEY, 0u);
      uint32_t g = tFirst;  // words [gBeg, g) are still to be searched, backwards
      while (g > gBeg) {
        const bool in = lane < g - gBeg;
        const uint32_t gi = g - 1u - lane;
        uint32_t key = NOKEY;
        if (in) {
          uint32_t s = s0;
          while (segB[s] > gi) --s;  // segB[0] = gBeg <= gi
          const uint32_t er = s / c.F, fed = s - er * c.F;
          uint32_t m, r, cc;
          if (decode_word(c.cab, c.words[gi], fed, m, r, cc) == ST_OK) key = (er << 16) | m;
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
      if (lane == 0) { s_seg = s0; s_carry = carry; }
    }
    __syncthreads();

    // ---- load, decode, calibrate
    const uint32_t g0 = tBeg + threadIdx.x * 4u;
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
    uint32_t st[4], mod[4], row[4], col[4], key[4];
    int32_t chg[4];
    uint32_t tkey = NOKEY, tg = 0u;
    if (any) {
      uint32_t s = s_seg;
      const uint32_t gf = g0 < gBeg ? gBeg : g0;
      while (s + 1u < S && segB[s + 1u] <= gf) ++s;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const uint32_t g = g0 + j;
        st[j] = 0xFFu; key[j] = NOKEY; mod[j] = row[j] = col[j] = 0xFFFFu; chg[j] = 0;
        if (g < gBeg || g >= gEnd) continue;
        while (s + 1u < S && segB[s + 1u] <= g) ++s;
        const uint32_t er = s / c.F, fed = s - er * c.F;
        uint32_t m, r, cc;
        st[j] = decode_word(c.cab, w[j], fed, m, r, cc);
        if (st[j] == ST_OK) {
          mod[j] = m; row[j] = r; col[j] = cc;
          const float2 gp = __ldg(c.gp + ((size_t)m * COLS + cc));  // S8: one pair per (module, col)
          chg[j] = calibrate(c, w[j] & 255u, gp);
          if (chg[j] < c.thr) st[j] = ST_BELOW;                       // S9
          key[j] = (er << 16) | m;
          tkey = key[j]; tg = g;
        } else {
          c.d_clus[g] = -1;                                            // S21; decodable words get clus in cluster
          atomicAdd(c.ev_cnt + (size_t)er * EC_STRIDE + (st[j] - ST_EMPTY), 1u);
        }
      }
      // ---- stores
      if (full) {
        *reinterpret_cast<ushort4*>(c.d_module + g0) = make_ushort4(mod[0], mod[1], mod[2], mod[3]);
        *reinterpret_cast<ushort4*>(c.d_row + g0) = make_ushort4(row[0], row[1], row[2], row[3]);
        *reinterpret_cast<ushort4*>(c.d_col + g0) = make_ushort4(col[0], col[1], col[2], col[3]);
        *reinterpret_cast<int4*>(c.d_charge + g0) = make_int4(chg[0], chg[1], chg[2], chg[3]);
        *reinterpret_cast<uchar4*>(c.d_status + g0) = make_uchar4(st[0], st[1], st[2], st[3]);
      } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const uint32_t g = g0 + j;
          if (g < gBeg || g >= gEnd) continue;
          c.d_module[g] = (uint16_t)mod[j]; c.d_row[g] = (uint16_t)row[j]; c.d_col[g] = (uint16_t)col[j];
          c.d_charge[g] = chg[j]; c.d_status[g] = (uint8_t)st[j];
        }
      }
    } else {
#pragma unroll
      for (int j = 0; j < 4; ++j) key[j] = NOKEY;
    }

    // ---- a3: previous decodable word of every thread (warp-shuffle last-valid scan + carries)
    const uint32_t has = __ballot_sync(0xFFFFFFFFu, tkey != NOKEY);
    const uint32_t below = has & ((1u << lane) - 1u);
    const int src = below ? 31 - __clz(below) : 0;
    uint32_t pkey = __shfl_sync(0xFFFFFFFFu, tkey, src);
    uint32_t pg = __shfl_sync(0xFFFFFFFFu, tg, src);
    {  // the warp's last decodable word: highest set lane of `has`
      const int top = has ? 31 - __clz(has) : 0;
      const uint32_t lk = __shfl_sync(0xFFFFFFFFu, tkey, top), lg = __shfl_sync(0xFFFFFFFFu, tg, top);
      if (lane == 0) s_warp_last[warp] = has ? make_uint2(lk, lg) : make_uint2(NOKEY, 0u);
    }
    __syncthreads();
    if (!below) {  // nothing decodable earlier in this warp: take the nearest earlier warp, else the look-back
      uint2 cin = s_carry;
      for (int wq = (int)warp - 1; wq >= 0; --wq) {
        const uint2 v = s_warp_last[wq];
        if (v.x != NOKEY) { cin = v; break; }
      }
      pkey = cin.x; pg = cin.y;
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      if (key[j] == NOKEY) continue;
      if (key[j] != pkey) {
        run_start(c, key[j], g0 + j);
        if (pkey != NOKEY) run_end(c, pkey, pg);
      }
      pkey = key[j]; pg = g0 + j;
    }
    // the chunk's last decodable word ends the last run
    if (tile == n_tiles - 1u && threadIdx.x == 0) {
      uint2 last = s_carry;
      for (int wq = UNPACK_WARPS - 1; wq >= 0; --wq) {
        const uint2 v = s_warp_last[wq];
        if (v.x != NOKEY) { last = v; break; }
      }
      if (last.x != NOKEY) run_end(c, last.x, last.y);
    }
    __syncthreads();  // shared carries are rewritten by the next tile
  }
}

// ------------------------------------------------------------------ classify
// One thread per (event, module): absent-module fix-up (S12: absent -> 0,0), zero counts, and the task
// lists of the four size classes (warp-aggregated append).
__global__ void __launch_bounds__(256) classify_kernel(const __grid_constant__ Chunk c) {
  const uint32_t Ec = c.e1 - c.e0, n_tasks = Ec * c.M;
  const uint32_t lane = threadIdx.x & 31u;
  const uint32_t n_rounded = (n_tasks + 31u) & ~31u;
  for (uint32_t t = blockIdx.x * blockDim.x + threadIdx.x; t < n_rounded; t += gridDim.x * blockDim.x) {
    int tier = -1;
    if (t < n_tasks) {
      const uint32_t er = t / c.M, m = t - er * c.M;
      const size_t o = (size_t)(c.e0 + er) * c.M + m;
      uint32_t first = c.module_first[o], end = c.module_end[o];
      const uint32_t nw = c.segB[(er + 1u) * c.F] - c.segB[er * c.F];
      const uint32_t flags = c.ev_cnt[(size_t)er * EC_STRIDE + EC_FLAGS];
      const bool present = first != NO_INDEX && first < end && end <= nw;
      if (first == NO_INDEX) c.module_first[o] = 0u;
      c.n_clus[t] = 0u;
#pragma unroll
      for (int k = 0; k < MC_STRIDE; ++k) c.mod_cnt[(size_t)t * MC_STRIDE + k] = 0u;
      if (present && !(flags & FLAG_NONCONTIGUOUS)) {
        const uint32_t n = end - first;
        tier = n <= TIER_WARP_MAX ? 0 : (n <= TIER_SMALL_MAX ? 1 : (n <= TIER_LARGE_MAX ? 2 : 3));
      }
    }
#pragma unroll
    for (int q = 0; q < N_TIERS; ++q) {
      const uint32_t mask = __ballot_sync(0xFFFFFFFFu, tier == q);
      if (!mask) continue;
      uint32_t base = 0;
      if (lane == (uint32_t)(__ffs(mask) - 1)) base = atomicAdd(c.ctl + q, (uint32_t)__popc(mask));
      base = __shfl_sync(0xFFFFFFFFu, base, __ffs(mask) - 1);
      if (tier == q) c.lists[(size_t)q * c.list_stride + base + __popc(mask & ((1u << lane) - 1u))] = t;
    }
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

void launch_unpack(const Chunk& c, uint32_t words_bound, int n_sm, cudaStream_t stream) {
  unpack_kernel<<<grid_for(words_bound + 3u, TILE, n_sm * 8), UNPACK_THREADS, 0, stream>>>(c);
}

void launch_classify(const Chunk& c, int n_sm, cudaStream_t stream) {
  const uint32_t Ec = c.e1 - c.e0;
  classify_kernel<<<grid_for(Ec * c.M, 256, n_sm * 8), 256, 0, stream>>>(c);
}

}  // namespace pix
