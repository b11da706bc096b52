// pix_common.cuh -- shared declarations of the CUDA Clusters path (sm_100a only).
//
// The path (section 2): "unpacks [the raw data], calibrates the individual pixels, and
// clusters the pixels on each detector module", plus the per-module offset table of PAPER.md Fig. 3
// (lines 76-81).  Readings S1..S24 of DESIGN.md fix what the paper leaves open.
//
// Kernel chain for one chunk of events:
//   init      -> segment table, range sentinels, zeroed counters; segfill -> segment of every 128-word chunk,
//                end of every event's last run
//   runs      -> a3 run boundaries: one start bit per word, module_first / module_end, run counts (runs.cu)
//   pack      -> work items: stretches of at most 1024 words holding whole module runs (runs.cu)
//   tile      -> a1 decode + a2 calibrate + a4 findClus + a5 sums/cut/renumber, one block per item (tile.cu)
//   overflow  -> a4 + a5 for the runs the tile kernel could not take (longer than a tile, pathological
//                charge sums, hash overflow): generic block-per-run kernel, tables in global workspace (cluster.cu)
//   offsets   -> a6 clamp + prefix scan (Fig. 3), summary, scatter work list
//   scatter   -> cluster records to their final place
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
constexpr uint32_t CHUNK_WORDS = 128;  // words per warp in decode and findclus; chunk ci starts at (gBeg & ~127) + 128 ci

// per-event counters (integer atomics only), one row of EC_STRIDE per event of the chunk
enum { EC_EMPTY = 0, EC_ERR_LINK, EC_ERR_ROC, EC_ERR_DCOL, EC_ERR_PXID, EC_FLAGS, EC_DUP, EC_BELOW, EC_OK, EC_CUT,
       EC_PRECUT, EC_PUSHED /* runs the event has put on the task lists (at most M) */, EC_STRIDE = 16 };
// ctl words
enum { CTL_OVF_COUNT = 0, CTL_OVF_TICKET = 1, CTL_SLICE_COUNT = 2, CTL_TEMP_COUNT = 8, CTL_ITEM_COUNT = 9, CTL_ITEM_NEXT = 10, CTL_WORDS = 16 };
// work items of the tile kernel (runs.cu packs them, tile.cu takes them): x = global index of the first word,
// y = words | flags << 16, z = event (launch-group relative) | FED of the first word << 16
#ifndef PIX_TILE_WORDS
#define PIX_TILE_WORDS 1024
#endif
constexpr uint32_t TILE_WORDS = PIX_TILE_WORDS, ITEM_WIN = TILE_WORDS - 32, ITEM_WIN2 = 224, ITEM_RUNS = 255;
constexpr uint32_t ITEM_DECODE_ONLY = 1u, ITEM_LONG_HEAD = 2u;

// Cabling table as the kernels read it (built once in pix_create from pix_cabling_map.entry, reading S3):
//   x = module | bad << 16 | scol << 24     bad: 0, ST_ERR_LINK or ST_ERR_ROC; scol = +1 / -1 (int8)
//   y = row0 | col0 << 8 | srow << 24       row0 = rocy*80 + (flip_r ? 79 : 0), col0 = rocx*52 + (flip_c ? 51 : 0)
// so that row = row0 + srow * (pxid >> 1), col = col0 + scol * (2*dcol + (pxid & 1)).
typedef uint2 CabEntry;


// Everything a kernel needs for one chunk of events [e0, e1).  Passed by value (__grid_constant__).
struct Chunk {
  // ---- input (device)
  const uint32_t* words;    // all events concatenated
  const uint32_t* ev_off;   // [E+1] or nullptr for the single-event call (offsets 0, n_single)
  const uint32_t* fed_off;  // [E*(F+1)] event-relative, or nullptr iff F == 1
  uint32_t n_single;
  uint32_t e0, e1;          // event range of this chunk
  uint32_t F, M;
  uint32_t F_shift;         // log2(F) when F is a power of two, else 0xFFFFFFFF
  // ---- tables (device, owned by the handle)
  const CabEntry* cab;      // [F*64*32]
  const float2* gp;         // [M*416] (gain, pedestal) interleaved
  // ---- parameters
  float vcal_gain, vcal_offset, max_e_f;
  int32_t thr, cut;
  uint32_t cap_mod, cap_ev; // max_clusters_per_module, max_clusters_per_event
  uint32_t cap_words;       // word capacity of the chunk workspace
  uint32_t max_wpe;         // max_words_per_event (longer events are flagged)
  // ---- digi outputs, indexed by global word index
  uint16_t* d_module; uint16_t* d_row; uint16_t* d_col; int32_t* d_charge; int32_t* d_clus; uint8_t* d_status;
  // ---- cluster outputs; per-event strides cap_ev, M, M, M+1, 16 (event index absolute)
  uint16_t* c_module; uint32_t* c_first; uint32_t* c_npix; uint32_t* c_charge; float* c_x; float* c_y;
  uint32_t* module_first; uint32_t* module_end; uint32_t* clus_module_start; uint32_t* summary;
  // ---- workspace (device, owned by the handle), indexed by chunk-relative event / word
  uint32_t* segB;           // [(e1-e0)*F + 1] global word index where segment (event, fed) starts
  uint32_t* ev_cnt;         // [(e1-e0)*EC_STRIDE]
  uint32_t* ctl;            // [CTL_WORDS]
  uint32_t* ovf_list;       // [(e1-e0)*M] task ids (event_rel*M + module) left to the overflow kernel
  uint32_t list_cap;        // (e1-e0)*M: every event lists at most M runs (push_run)
  uint32_t* chunk_seg;      // [cap_words/128 + 2] event_rel << 16 | fed of the chunk's first word
  uint32_t* slice_list;     // [2 * (cap_words/1024 + (e1-e0))] scatter work items: event_rel << 16 | slice, first | last << 16 module
  uint32_t* sbits;          // [cap_words/32 + 64] run-start bits, bit (g - T0) (runs.cu)
  uint8_t* cbad;            // [cap_words/128 + 2] per 128-word chunk: 0 when every word is decodable and the words of a
                            // run ascend strictly in (link, roc, dcol, pxid), the detector's read-out order (runs.cu)
  uint32_t geom_unique;     // 1 when no two valid cabling entries name the same ROC position of a module
  uint4* items;             // [item_cap] work items of the tile kernel
  uint32_t item_cap;
  uint32_t* n_clus;         // [(e1-e0)*M] clusters surviving the cut, per module
  uint32_t* n_runs;         // [(e1-e0)*M] runs of the module (more than one: the event is NONCONTIGUOUS, S11)
  // temp cluster records: every window / run takes a stretch of the area (alloc_temp) and leaves its start in t_base,
  // so the records are dense in memory whatever the words-per-cluster ratio; 16 + 4 bytes per record.
  // Capacity 2 x cap_words: a window allots one slot per root (<= its digis), a run that is redone by a later
  // kernel (32-bit sums at risk) is allotted once more, by the kernel that finishes it.
  uint4* t_a;               // [2*cap_words] first_digi, n_pix, charge, x_col bits
  float* t_y;               // [2*cap_words]
  uint32_t* t_base;         // [(e1-e0)*M] index of the module's first temp record (local id 0)
  // overflow-kernel scratch, indexed by chunk-relative word index
  unsigned long long* g_hash;  // [2*cap_words]
  uint32_t* g_pos; uint32_t* g_q; uint32_t* g_npix; unsigned long long* g_sx; unsigned long long* g_sy;
};

__device__ __forceinline__ uint32_t ev_offset(const Chunk& c, uint32_t e) {
  return c.ev_off ? c.ev_off[e] : (e ? c.n_single : 0u);
}
__device__ __forceinline__ uint32_t alloc_temp(const Chunk& c, uint32_t count) { return atomicAdd(c.ctl + CTL_TEMP_COUNT, count); }
__device__ __forceinline__ void put_temp(const Chunk& c, uint32_t i, uint32_t first, uint32_t npix, uint32_t charge, float x, float y) {
  c.t_a[i] = make_uint4(first, npix, charge, __float_as_uint(x)); c.t_y[i] = y;
}

// The kernels of a launch group are chained by programmatic dependent launch: each one lets its successor's blocks
// be placed as soon as all of its own blocks have started, and each one waits for its predecessor to finish (and its
// writes to be visible) before it touches memory.  That hides the launch and ramp-up latency between the eight
// kernels (one event per call: 74 -> 66 us); the order of the work is that of the stream.  Two launches stay plain
// (`chained` false), measured: the overflow kernel and the scatter, whose early blocks cost the large batch 0.5-4 %.
__device__ __forceinline__ void chain_begin() {
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}
template <typename... KArgs, typename... Args>
inline void launch_chained(bool chained, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = chained ? 1 : 0;
  cudaLaunchKernelEx(&cfg, kernel, args...);
}

// launchers (host), one per kernel; all asynchronous on `stream`
void launch_init(const Chunk& c, uint32_t n_total, int n_sm, cudaStream_t stream);
void launch_runs(const Chunk& c, uint32_t words_bound, int n_sm, cudaStream_t stream);
void launch_tile(const Chunk& c, int n_sm, cudaStream_t stream);
cudaError_t configure_tile_kernel();

void launch_overflow(const Chunk& c, int n_sm, cudaStream_t stream);
void launch_finalize(const Chunk& c, int n_sm, cudaStream_t stream);
cudaError_t configure_finalize_kernel();
cudaError_t configure_overflow_kernel();
constexpr uint32_t MAX_MODULES = 16383;  // finalize keeps the M+1 offsets of an event in shared memory
constexpr int LAUNCHES_PER_CHUNK = 8;    // init, segfill, runs, pack, tile, overflow, offsets, scatter

}  // namespace pix
