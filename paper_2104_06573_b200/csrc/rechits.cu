// rechits.cu -- RecHits-lite ("The RecHits module estimates the 3D position of each
// cluster forming hits"; module-local part only, readings S25-S28).
//
// One thread per emitted cluster record.  The cluster's digis lie in its module's run [module_first, module_end)
// and carry the cluster's local id in clus, so the thread scans the run for its id and takes the bounding box;
// neighbouring threads hold clusters of the same module and read the same addresses (broadcast).  No atomics, no
// workspace.  Nothing here is shared with oracle/.
#include "../../include/pixclus.h"
#include "pix_common.cuh"

namespace pix {

namespace {

constexpr int RH_THREADS = 128;

__global__ void __launch_bounds__(RH_THREADS) rechits_kernel(uint32_t M, uint32_t cap_ev, const uint32_t* __restrict__ ev_off,
                                                             pix_digis d, pix_clusters k, pix_hits h) {
  const uint32_t e = blockIdx.y;
  const uint32_t n_emit = k.summary[(size_t)e * 16 + PIX_SUM_N_CLUSTERS_EMITTED];
  const uint32_t* cms = k.clus_module_start + (size_t)e * (M + 1);
  const size_t base = ev_off[e];
  for (uint32_t g = blockIdx.x * RH_THREADS + threadIdx.x; g < n_emit; g += gridDim.x * RH_THREADS) {
    const size_t o = (size_t)e * cap_ev + g;
    const uint32_t m = k.module[o];
    const int32_t local = (int32_t)(g - cms[m]);
    const uint32_t first = k.module_first[(size_t)e * M + m], end = k.module_end[(size_t)e * M + m];
    uint32_t r0 = 0xFFFFu, r1 = 0u, c0 = 0xFFFFu, c1 = 0u;
    for (uint32_t i = first; i < end; ++i) {
      if (d.clus[base + i] != local) continue;  // clus >= 0 only for digis of surviving clusters
      const uint32_t r = d.row[base + i], c = d.col[base + i];
      r0 = r < r0 ? r : r0; r1 = r > r1 ? r : r1; c0 = c < c0 ? c : c0; c1 = c > c1 ? c : c1;
    }
    h.min_row[o] = (uint16_t)r0; h.max_row[o] = (uint16_t)r1; h.min_col[o] = (uint16_t)c0; h.max_col[o] = (uint16_t)c1;
    // S27: three separately rounded binary32 operations per coordinate
    h.x_local[o] = __fmul_rn(__fsub_rn(__fadd_rn(k.y_row[o], 0.5f), 80.0f), 0.0100f);
    h.y_local[o] = __fmul_rn(__fsub_rn(__fadd_rn(k.x_col[o], 0.5f), 208.0f), 0.0150f);
    uint32_t f = 0u;
    if (r0 == 0u || r1 == (uint32_t)ROWS - 1u || c0 == 0u || c1 == (uint32_t)COLS - 1u) f |= PIX_HIT_ON_EDGE;
    if ((r0 < (uint32_t)ROC_ROWS && r1 >= (uint32_t)ROC_ROWS) || c0 / (uint32_t)ROC_COLS != c1 / (uint32_t)ROC_COLS) f |= PIX_HIT_SPANS_ROC;
    if (k.n_pix[o] == 1u) f |= PIX_HIT_SINGLE_PIXEL;
    h.flags[o] = (uint8_t)f;
  }
}

}  // namespace

void launch_rechits(uint32_t n_events, uint32_t M, uint32_t cap_ev, const uint32_t* ev_off, const pix_digis& d,
                    const pix_clusters& k, const pix_hits& h, cudaStream_t stream) {
  uint32_t nb = (cap_ev + RH_THREADS - 1) / RH_THREADS;
  if (nb > 256u) nb = 256u;
  // events in slabs of 65535 (grid.y limit)
  for (uint32_t e0 = 0; e0 < n_events; e0 += 65535u) {
    const uint32_t ne = n_events - e0 < 65535u ? n_events - e0 : 65535u;
    pix_digis dd = d; pix_clusters kk = k; pix_hits hh = h;
    kk.module += (size_t)e0 * cap_ev; kk.first_digi += (size_t)e0 * cap_ev; kk.n_pix += (size_t)e0 * cap_ev;
    kk.charge += (size_t)e0 * cap_ev; kk.x_col += (size_t)e0 * cap_ev; kk.y_row += (size_t)e0 * cap_ev;
    kk.module_first += (size_t)e0 * M; kk.module_end += (size_t)e0 * M; kk.clus_module_start += (size_t)e0 * (M + 1);
    kk.summary += (size_t)e0 * 16;
    hh.x_local += (size_t)e0 * cap_ev; hh.y_local += (size_t)e0 * cap_ev; hh.min_row += (size_t)e0 * cap_ev;
    hh.max_row += (size_t)e0 * cap_ev; hh.min_col += (size_t)e0 * cap_ev; hh.max_col += (size_t)e0 * cap_ev;
    hh.flags += (size_t)e0 * cap_ev;
    rechits_kernel<<<dim3(nb, ne), RH_THREADS, 0, stream>>>(M, cap_ev, ev_off + e0, dd, kk, hh);
  }
}

}  // namespace pix
