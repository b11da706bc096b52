// decode.cu -- the two set-up kernels of a launch group: init (segment table, range sentinels, zeroed counters) and
// segfill (segment of every 128-word chunk; end of every event's last module run, a3 of the path PAPER.md:31
// describes).  The decode itself (a1, a2) lives in the tile kernel (tile.cu).  Nothing here is shared with oracle/.
#include "pix_common.cuh"
#include "pix_device.cuh"

namespace pix {

namespace {

// ------------------------------------------------------------------ init
// One warp per event of the chunk builds the clamped, monotone segment table
//   segB[e_rel*F + f] = global word index where FED f of event e starts,  segB[Ec*F] = end of chunk.
// Offsets are clamped into [lo, hi] (lo = start of chunk, hi = min(n_total, lo + cap_words)) so that
// whatever the caller's offset arrays hold, every index derived later stays inside the buffers.
// Other threads initialise the per-(event,module) range sentinels and zero the counters.
__global__ void __launch_bounds__(256) init_kernel(const __grid_constant__ Chunk c, uint32_t n_total) {
  chain_begin();
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
    const uint32_t flags = (re > hi || rb > hi || re < rb || rb < lo || re - rb > c.max_wpe) ? FLAG_TOO_LARGE : 0u;
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
  for (uint32_t t = tid; t < nmod; t += nth) { mf[t] = NO_INDEX; me[t] = 0u; c.n_clus[t] = 0u; c.n_runs[t] = 0u; }
}

// chunk_seg[ci] = event << 16 | FED of the first word of 128-word chunk ci (its first word inside the launch
// group).  One thread per segment writes the chunks that start inside it.  One warp per event closes the event's
// last run: module_end of the module of the event's last decodable word (the runs kernel closes a run when it
// sees the next run start of the same event, and never looks back beyond the start of an event).
__global__ void __launch_bounds__(256) segfill_kernel(const __grid_constant__ Chunk c) {
  chain_begin();
  const uint32_t F = c.F, Ec = c.e1 - c.e0, S = Ec * F;
  const uint32_t gBeg = c.segB[0], gEnd = c.segB[S];
  if (gBeg >= gEnd) return;
  const uint32_t T0 = gBeg & ~(CHUNK_WORDS - 1u);
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
  for (uint32_t sgi = tid; sgi < S; sgi += nth) {
    const uint32_t lo = c.segB[sgi], hi = c.segB[sgi + 1u];
    if (lo >= hi) continue;
    const uint32_t c_lo = lo == gBeg ? 0u : (lo - T0 + CHUNK_WORDS - 1u) / CHUNK_WORDS;
    const uint32_t c_hi = (hi - T0 + CHUNK_WORDS - 1u) / CHUNK_WORDS;  // exclusive
    const uint32_t er = div_F(c, sgi), packed = (er << 16) | (sgi - er * F);  // F, Ec <= 65535 (pix_create)
    for (uint32_t ci = c_lo; ci < c_hi; ++ci) c.chunk_seg[ci] = packed;
  }
  const uint32_t lane = threadIdx.x & 31u;
  for (uint32_t er = tid >> 5; er < Ec; er += nth >> 5) {
    const uint32_t evb = c.segB[er * F];
    uint32_t g = c.segB[(er + 1u) * F];  // words [evb, g) are still to be searched, backwards, 32 at a time
    while (g > evb) {
      const bool in = lane < g - evb;
      const uint32_t gi = g - 1u - lane;
      uint32_t m = 0xFFFFFFFFu;
      if (in) {
        uint32_t sg = (er + 1u) * F - 1u;
        while (c.segB[sg] > gi) --sg;
        uint32_t mm, r, cc;
        if (decode_word(c.cab, __ldg(c.words + gi), (sg - er * F) << 11, mm, r, cc) == ST_OK) m = mm;
      }
      const uint32_t bal = __ballot_sync(0xFFFFFFFFu, m != 0xFFFFFFFFu);
      if (bal) {
        const int src = __ffs(bal) - 1;
        if ((int)lane == src) run_end(c, (er << 16) | m, gi);
        break;
      }
      g = (g - evb > 32u) ? g - 32u : evb;
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
  launch_chained(true, init_kernel, grid_for(Ec * c.M, 256, n_sm * 8), 256, 0, stream, c, n_total);
  launch_chained(true, segfill_kernel, grid_for(Ec * (c.F > 32u ? c.F : 32u), 256, n_sm * 8), 256, 0, stream, c);
}

}  // namespace pix
