// pix_common.cuh -- shared declarations of the CUDA Clusters path (sm_100a only).
//
// The path (section 2): "unpacks [the raw data], calibrates the individual pixels, and
// clusters the pixels on each detector module", plus the per-module offset table of PAPER.md Fig. 3
// (lines 76-81).  Readings S1..S24 of DESIGN.md fix what the paper leaves open.
//
// Kernel chain for one chunk of events:
//   init      -> segment table, range sentinels, zeroed counters
//   unpack    -> a1 decode + a2 calibrate + a3 run boundaries (ballot/shuffle last-valid scan)
//   classify  -> per (event, module) task: absent-module fix-up, size class lists
//   cluster   -> a4 findClus (position hash + min-index union-find) fused with a5 (sums, cut, renumber)
//                in four size classes: warp / small block / large block (all shared memory) / global
//   finalize  -> a6 clamp + prefix scan (Fig. 3), record scatter, summary
// Nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace pix {

constexpr int ROWS = 160, COLS = 416, ROC_ROWS = 80, ROC_COLS = 52;
constexpr uint32_t NPOS = ROWS * COLS;  // 66560 < 2^17

// status codes (S6)
enum : uint8_t { ST_OK = 0, ST_CUT = 1, ST_BELOW = 2, ST_DUP = 3, ST_EMPTY = 4, ST_ERR_LINK = 5, ST_ERR_ROC = 6,
                 ST_ERR_DCOL = 7, ST_ERR_PXID = 8 };

constexpr uint32_t FLAG_NONCONTIGUOUS = 1u, FLAG_CAPACITY = 2u, FLAG_TOO_LARGE = 4u;
constexpr uint32_t NO_INDEX = 0xFFFFFFFFu;

// size classes of the cluster step, by run length n = module_end - module_first
constexpr int N_TIERS = 4;
constexpr uint32_t TIER_WARP_MAX = 128;    // one warp per module, <= 4 digis per lane
constexpr uint32_t TIER_SMALL_MAX = 768;   // 128-thread block, shared memory
constexpr uint32_t TIER_LARGE_MAX = 4096;  // 512-thread block, shared memory
                                           // beyond: 512-thread block, tables in global workspace

// per-event counters produced by unpack (the rest of the summary comes from per-module counts)
enum { EC_EMPTY = 0, EC_ERR_LINK, EC_ERR_ROC, EC_ERR_DCOL, EC_ERR_PXID, EC_FLAGS, EC_STRIDE = 8 };
// per-(event,module) counts produced by cluster
enum { MC_PRECUT = 0, MC_DUP, MC_BELOW, MC_OK, MC_CUT, MC_STRIDE = 5 };

// Everything a kernel needs for one chunk of events [e0, e1).  Passed by value (__grid_constant__).
struct Chunk {
  // ---- input (device)
  const uint32_t* words;    // all events concatenated
  const uint32_t* ev_off;   // [E+1] or nullptr for the single-event call (offsets 0, n_single)
  const uint32_t* fed_off;  // [E*(F+1)] event-relative, or nullptr iff F == 1
  uint32_t n_single;
  uint32_t e0, e1;          // event range of this chunk
  uint32_t F, M;
  // ---- tables (device, owned by the handle)
  const uint32_t* cab;      // [F*64*32]
  const float2* gp;         // [M*416] (gain, pedestal) interleaved
  // ---- parameters
  float vcal_gain, vcal_offset, max_e_f;
  int32_t thr, cut;
  uint32_t cap_mod, cap_ev; // max_clusters_per_module, max_clusters_per_event
  uint32_t cap_words;       // word capacity of the chunk workspace
  // ---- digi outputs, indexed by global word index
  uint16_t* d_module; uint16_t* d_row; uint16_t* d_col; int32_t* d_charge; int32_t* d_clus; uint8_t* d_status;
  // ---- cluster outputs; per-event strides cap_ev, M, M, M+1, 16 (event index absolute)
  uint16_t* c_module; uint32_t* c_first; uint32_t* c_npix; uint32_t* c_charge; float* c_x; float* c_y;
  uint32_t* module_first; uint32_t* module_end; uint32_t* clus_module_start; uint32_t* summary;
  // ---- workspace (device, owned by the handle), indexed by chunk-relative event / word
  uint32_t* segB;           // [(e1-e0)*F + 1] global word index where segment (event, fed) starts
  uint32_t* ev_cnt;         // [(e1-e0)*EC_STRIDE]
  uint32_t* ctl;            // [16]: 0..3 list counts, 4..7 tickets, 8 chunk skip flag
  uint32_t* lists;          // [N_TIERS][(e1-e0)*M] task ids (event_rel*M + module)
  uint32_t list_stride;
  uint32_t* n_clus;         // [(e1-e0)*M] clusters surviving the cut, per module
  uint32_t* mod_cnt;        // [(e1-e0)*M*MC_STRIDE]
  // temp cluster records, indexed by chunk-relative word index (run first + local id)
  uint32_t* t_first; uint32_t* t_npix; uint32_t* t_charge; float* t_x; float* t_y;
  // global-tier scratch, indexed by chunk-relative word index
  unsigned long long* g_hash;  // [2*cap_words]
  uint32_t* g_pos; uint32_t* g_q; uint32_t* g_npix; unsigned long long* g_sx; unsigned long long* g_sy;
};

__device__ __forceinline__ uint32_t ev_offset(const Chunk& c, uint32_t e) {
  return c.ev_off ? c.ev_off[e] : (e ? c.n_single : 0u);
}

// launchers (host), one per kernel family; all asynchronous on `stream`
void launch_init(const Chunk& c, uint32_t n_total, int n_sm, cudaStream_t stream);
void launch_unpack(const Chunk& c, uint32_t words_bound, int n_sm, cudaStream_t stream);
void launch_classify(const Chunk& c, int n_sm, cudaStream_t stream);
// ev (optional): 4 events, recorded after each of the four class kernels (global, large, small, warp)
void launch_cluster(const Chunk& c, uint32_t words_bound, int n_sm, cudaStream_t stream, cudaEvent_t* ev = nullptr);
void launch_finalize(const Chunk& c, int n_sm, cudaStream_t stream);
cudaError_t configure_cluster_kernels();
cudaError_t configure_finalize_kernel();
constexpr uint32_t MAX_MODULES = 16383;  // finalize keeps the M+1 offsets of an event in shared memory
constexpr int LAUNCHES_PER_CHUNK = 8;  // init, unpack, classify, cluster x4, finalize

}  // namespace pix
