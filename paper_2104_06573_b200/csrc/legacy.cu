// legacy.cu -- legacy digi format and FED error-word list (PAPER.md:31 names "optional modules ...
// to convert the SoA to legacy data formats" and leaves them out of its measurements; the format is this build's own,
// DESIGN.md readings S29-S31).
//
// One block per event walks the event's words in tiles of 256: pdigi = row | col << 11 | adc << 22 and the module's
// raw detector id for a decodable word (0, 0 otherwise), coalesced stores; words with an ERR_* status are appended
// to the event's error list in word order (ballot + a prefix over the warps of the tile), the true count goes to
// n_errors.  Not part of the timed step.  Nothing here is shared with oracle/.
#include "../../include/pixclus.h"
#include "pix_common.cuh"

namespace pix {

namespace {

constexpr int LG_THREADS = 256;

__global__ void __launch_bounds__(LG_THREADS) legacy_kernel(uint32_t n_events, uint32_t F, uint32_t M, uint32_t n_total,
                                                            const uint32_t* __restrict__ words, const uint32_t* __restrict__ ev_off,
                                                            const uint32_t* __restrict__ fed_off, pix_digis d,
                                                            const uint32_t* __restrict__ raw_id_of, uint32_t cap, pix_legacy o) {
  __shared__ uint32_t s_warp[LG_THREADS / 32];
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  for (uint32_t e = blockIdx.x; e < n_events; e += gridDim.x) {
    uint32_t b = ev_off[e], en = ev_off[e + 1];
    en = en < n_total ? en : n_total; b = b < en ? b : en;
    const uint32_t* fo = fed_off ? fed_off + (size_t)e * (F + 1) : nullptr;
    uint32_t n_err = 0u;  // errors before this tile (block-uniform)
    for (uint32_t i0 = b; i0 < en; i0 += LG_THREADS) {
      const uint32_t g = i0 + tid;
      uint32_t st = 0xFFu, w = 0u;
      if (g < en) {
        st = d.status[g]; w = words[g];
        const bool dec = st <= ST_DUP;
        const uint32_t m = dec ? (uint32_t)d.module[g] : 0u;
        o.pdigi[g] = dec ? ((uint32_t)d.row[g] | ((uint32_t)d.col[g] << 11) | ((w & 255u) << 22)) : 0u;  // S29
        o.raw_id[g] = (dec && m < M) ? raw_id_of[m] : 0u;                                                   // S30
      }
      const bool err = st >= ST_ERR_LINK && st <= ST_ERR_PXID;  // S31: padding words are not errors
      const uint32_t bal = __ballot_sync(0xFFFFFFFFu, err);
      __syncthreads();  // the previous tile is done with s_warp
      if (lane == 0) s_warp[warp] = __popc(bal);
      __syncthreads();
      uint32_t before = 0u, total = 0u;
#pragma unroll
      for (int q = 0; q < LG_THREADS / 32; ++q) { const uint32_t v = s_warp[q]; before += q < (int)warp ? v : 0u; total += v; }
      if (err) {
        const uint32_t k = n_err + before + __popc(bal & ((1u << lane) - 1u));
        if (k < cap) {
          const size_t at = (size_t)e * cap + k;
          uint32_t fed = 0u;
          if (fo) {  // the FED block of word g - b: the last f with fed_off[f] <= index
            const uint32_t idx = g - b;
            uint32_t lo = 0u, hi = F - 1u;
            while (lo < hi) { const uint32_t mid = (lo + hi + 1u) >> 1; if (fo[mid] <= idx) lo = mid; else hi = mid - 1u; }
            fed = lo;
          }
          o.err_word[at] = w; o.err_fed[at] = (uint16_t)fed; o.err_type[at] = (uint8_t)st;
        }
      }
      n_err += total;
    }
    if (tid == 0) o.n_errors[e] = n_err;
  }
}

}  // namespace

void launch_legacy(uint32_t n_events, uint32_t F, uint32_t M, uint32_t n_total, const uint32_t* words, const uint32_t* ev_off,
                   const uint32_t* fed_off, const pix_digis& d, const uint32_t* raw_id_of, uint32_t cap, const pix_legacy& o,
                   int n_sm, cudaStream_t stream) {
  uint32_t nb = n_events < (uint32_t)n_sm * 8u ? n_events : (uint32_t)n_sm * 8u;
  legacy_kernel<<<nb, LG_THREADS, 0, stream>>>(n_events, F, M, n_total, words, ev_off, fed_off, d, raw_id_of, cap, o);
}

}  // namespace pix
