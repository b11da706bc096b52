// finalize.cu -- a6 cluster offsets (Fig. 3, lines 76-81: moduleStart[i+1] = min(maxHitsInModule(),
// cluStart[i]), followed by the prefix sum the figure leaves implicit, S19), the scatter of the temp
// cluster records to their final place clus_module_start[module] + local id (S14), and the summary (S20).
//
// Two kernels.  offsets: one block per event computes the event's M-entry scan (warp-shuffle scan), writes the
// offsets and the summary, and appends the event's record slices (SLICE records each, with the modules of the first
// and the last record) to a work list.  scatter: a persistent grid takes slices from the list; a block stages the
// offsets of the slice's modules in shared memory and copies its records, one thread per output record, module found
// by binary search among those offsets.
#include "pix_common.cuh"
#include "pix_device.cuh"

namespace pix {

namespace {

constexpr int FIN_THREADS = 256;

__device__ __forceinline__ uint32_t warp_inclusive_scan(uint32_t v, uint32_t lane) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, v, d);
    if (lane >= (uint32_t)d) v += t;
  }
  return v;
}

constexpr uint32_t SLICE = 1024;  // records per scatter work item

__global__ void __launch_bounds__(FIN_THREADS) offsets_kernel(const __grid_constant__ Chunk c) {
  chain_begin();
  extern __shared__ uint32_t s_start[];  // [M+1]
  __shared__ uint32_t s_warp[FIN_THREADS / 32];
  __shared__ uint32_t s_red[8];
  const uint32_t er = blockIdx.x, e = c.e0 + er, M = c.M;
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const uint32_t* n_clus_raw = c.n_clus + (size_t)er * M;
  // S11: a module with two or more runs makes the event NONCONTIGUOUS; clustering is not defined for such an event
  bool split = false;
  for (uint32_t m = tid; m < M; m += FIN_THREADS) split |= c.n_runs[(size_t)er * M + m] >= 2u;
  const bool skip = __syncthreads_or(split);
  const uint32_t flags = c.ev_cnt[(size_t)er * EC_STRIDE + EC_FLAGS] | (skip ? FLAG_NONCONTIGUOUS : 0u);
  auto n_clus = [&](uint32_t m) { return n_clus_raw[m]; };

  // ---- Fig. 3 clamp + exclusive prefix sum over the M modules
  const uint32_t ipt = (M + FIN_THREADS - 1) / FIN_THREADS;
  const uint32_t m0 = tid * ipt, m1 = (m0 + ipt < M) ? m0 + ipt : M;
  uint32_t local = 0;
  for (uint32_t m = m0; m < m1; ++m) {
    const uint32_t n = skip ? 0u : n_clus(m);
    local += n < c.cap_mod ? n : c.cap_mod;
  }
  const uint32_t incl = warp_inclusive_scan(local, lane);
  if (lane == 31) s_warp[warp] = incl;
  if (tid < 8) s_red[tid] = 0u;
  __syncthreads();
  uint32_t base = incl - local;
  for (uint32_t w = 0; w < warp; ++w) base += s_warp[w];
  for (uint32_t m = m0; m < m1; ++m) {
    s_start[m] = base;
    const uint32_t n = skip ? 0u : n_clus(m);
    base += n < c.cap_mod ? n : c.cap_mod;
  }
  if (m0 < M && m1 == M) s_start[M] = base;
  __syncthreads();
  const uint32_t total = s_start[M];
  const uint32_t n_emit = total < c.cap_ev ? total : c.cap_ev;
  const uint32_t ebase = c.segB[er * c.F];
  const uint32_t n_words = c.segB[(er + 1u) * c.F] - ebase;

  // ---- an event whose modules are not contiguous is not clustered (S11): every decodable word is BELOW_THRESHOLD or
  // CUT with clus = -1, whatever the cluster kernels did or did not do with its runs
  uint32_t fix_below = 0u, fix_cut = 0u;
  if (skip) {
    for (uint32_t i = tid; i < n_words; i += FIN_THREADS) {
      const size_t g = (size_t)ebase + i;
      c.d_clus[g] = -1;
      if (c.d_row[g] != 0xFFFFu) {
        const bool below = c.d_charge[g] < c.thr;
        c.d_status[g] = below ? ST_BELOW : ST_CUT;
        fix_below += below ? 1u : 0u; fix_cut += below ? 0u : 1u;
      }
    }
  }
  // ---- offsets + summary + work items
  uint32_t* cms = c.clus_module_start + (size_t)e * (M + 1);
  for (uint32_t m = tid; m <= M; m += FIN_THREADS) cms[m] = s_start[m];
  uint32_t acc[4] = {0, 0, fix_below, fix_cut};  // modules present, clusters surviving the cut, S11 counts
  for (uint32_t m = tid; m < M; m += FIN_THREADS) {
    const bool present = c.module_end[(size_t)e * M + m] > 0u;
    if (!present) c.module_first[(size_t)e * M + m] = 0u;  // S12: absent -> 0,0 (init left the atomicMin sentinel)
    acc[0] += present ? 1u : 0u;
    acc[1] += skip ? 0u : n_clus(m);
  }
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const uint32_t v = __reduce_add_sync(0xFFFFFFFFu, acc[k]);
    if (lane == 0 && v) atomicAdd(s_red + k, v);
  }
  __syncthreads();
  if (tid == 0) {
    const uint32_t* ec = c.ev_cnt + (size_t)er * EC_STRIDE;
    uint32_t* s = c.summary + (size_t)e * 16;
    const uint32_t bad = ec[EC_EMPTY] + ec[EC_ERR_LINK] + ec[EC_ERR_ROC] + ec[EC_ERR_DCOL] + ec[EC_ERR_PXID];
    s[0] = n_words; s[1] = n_words - bad; s[2] = ec[EC_EMPTY];
    s[3] = ec[EC_ERR_LINK]; s[4] = ec[EC_ERR_ROC]; s[5] = ec[EC_ERR_DCOL]; s[6] = ec[EC_ERR_PXID];
    s[7] = skip ? 0u : ec[EC_DUP]; s[8] = skip ? s_red[2] : ec[EC_BELOW]; s[9] = skip ? 0u : ec[EC_OK];
    s[10] = skip ? s_red[3] : ec[EC_CUT];
    s[11] = s_red[0]; s[12] = skip ? 0u : ec[EC_PRECUT]; s[13] = s_red[1]; s[14] = n_emit;
    s[15] = flags | (total > c.cap_ev ? FLAG_CAPACITY : 0u);
  }
  // work items of the scatter: slices of SLICE records, each with the modules its first and last record belong to
  const uint32_t nsl = (n_emit + SLICE - 1u) / SLICE;
  if (tid == 0 && nsl) s_red[4] = atomicAdd(c.ctl + CTL_SLICE_COUNT, nsl);
  __syncthreads();
  auto module_of = [&](uint32_t g) {  // last m with s_start[m] <= g
    uint32_t lo = 0, hi = M;
    while (lo < hi) {
      const uint32_t mid = (lo + hi + 1u) >> 1;
      if (s_start[mid] <= g) lo = mid; else hi = mid - 1u;
    }
    return lo;
  };
  for (uint32_t q = tid; q < nsl; q += FIN_THREADS) {
    const uint32_t g_first = q * SLICE, g_last = (g_first + SLICE < n_emit ? g_first + SLICE : n_emit) - 1u;
    const uint32_t at = s_red[4] + q;
    c.slice_list[2u * at] = (er << 16) | q;  // cap_ev <= 2^26 records (pix_create)
    c.slice_list[2u * at + 1u] = module_of(g_first) | (module_of(g_last) << 16);  // (module ids stay below 16384)
  }
}

// ---- records: output record g of the event <- temp record (run first + local id)
__global__ void __launch_bounds__(FIN_THREADS) scatter_kernel(const __grid_constant__ Chunk c) {
  chain_begin();
  extern __shared__ uint32_t s_start[];  // [M+1]
  const uint32_t M = c.M, tid = threadIdx.x;
  const uint32_t count = c.ctl[CTL_SLICE_COUNT];
  for (uint32_t it = blockIdx.x; it < count; it += gridDim.x) {
    const uint32_t item = c.slice_list[2u * it], mods = c.slice_list[2u * it + 1u];
    const uint32_t er = item >> 16, e = c.e0 + er, g0 = (item & 0xFFFFu) * SLICE;
    const uint32_t m_first = mods & 0xFFFFu, m_last = mods >> 16;  // the slice's records lie in these modules
    const uint32_t* cms = c.clus_module_start + (size_t)e * (M + 1);
    __syncthreads();  // the previous item is done with s_start
    for (uint32_t m = m_first + tid; m <= m_last + 1u; m += FIN_THREADS) s_start[m] = cms[m];
    const uint32_t total = cms[M];
    __syncthreads();
    const uint32_t n_emit = total < c.cap_ev ? total : c.cap_ev;
    const uint32_t* tbase = c.t_base + (size_t)er * M;
#pragma unroll
    for (uint32_t j = 0; j < SLICE / FIN_THREADS; ++j) {
      const uint32_t g = g0 + j * FIN_THREADS + tid;
      if (g >= n_emit) continue;
      uint32_t lo = m_first, hi = m_last;  // last m with s_start[m] <= g
      while (lo < hi) {
        const uint32_t mid = (lo + hi + 1u) >> 1;
        if (s_start[mid] <= g) lo = mid; else hi = mid - 1u;
      }
      const uint32_t src = tbase[lo] + (g - s_start[lo]);
      const size_t o = (size_t)e * c.cap_ev + g;
      c.c_module[o] = (uint16_t)lo;
      const uint4 a = c.t_a[src];
      const float y = c.t_y[src];
      c.c_first[o] = a.x; c.c_npix[o] = a.y; c.c_charge[o] = a.z; c.c_x[o] = __uint_as_float(a.w); c.c_y[o] = y;
    }
  }
}

}  // namespace

cudaError_t configure_finalize_kernel() {
  cudaError_t e = cudaFuncSetAttribute(offsets_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(scatter_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
}

void launch_finalize(const Chunk& c, int n_sm, cudaStream_t stream) {
  const uint32_t Ec = c.e1 - c.e0;
  const size_t smem = (size_t)(c.M + 1) * sizeof(uint32_t);
  launch_chained(true, offsets_kernel, Ec, FIN_THREADS, smem, stream, c);
  launch_chained(false, scatter_kernel, n_sm * 8, FIN_THREADS, smem, stream, c);
}

}  // namespace pix
