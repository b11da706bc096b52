/* pixclus.h -- C ABI of libpixclus.so: the pixel "Clusters" hot path on one B200 (sm_100a).
 *
 * The path (section 2): the Clusters module "transfers the raw data to the GPU,
 * unpacks them, calibrates the individual pixels, and clusters the pixels on each detector
 * module"; plus the per-module offset table of PAPER.md Fig. 3 (lines 76-81):
 * moduleStart[i+1] = min(maxHitsInModule(), cluStart[i]).  Everything the paper leaves open is
 * fixed by the numbered readings S1..S24 in DESIGN.md (after BASELINE.json north_star/configs).
 *
 * Conventions
 *  - pix_create/pix_clone/pix_destroy take HOST pointers.  pix_process and pix_process_batch take
 *    DEVICE pointers only (caller-owned, e.g. torch tensors) and a CUDA stream; they never
 *    allocate, free, synchronise or copy to the host, so they are legal during stream capture.
 *    pix_process_batch_host takes HOST pointers and does the copies itself (synchronous; internally the
 *    input copy, the kernels and the output copy of consecutive groups of events overlap on three streams;
 *    pass pinned host memory for the overlap to take effect).
 *  - The library owns device copies of the two tables and a workspace, all allocated in
 *    pix_create / pix_clone (a memory pool gave 4.5x; here nothing allocates per event).
 *  - One in-flight call per handle; use pix_clone to get one handle per stream.
 *  - Return value 0 = PIX_OK, negative = error (nothing was launched unless PIX_ERR_CUDA).
 *    Bad DATA is not an API error: invalid words, duplicates, capacity overflow and non-contiguous
 *    modules are reported in status[] and summary[], in device memory.
 *  - Every element of every output array in [0,n_words), [0,M), [0,M+1), [0,16) and
 *    [0,n_clusters_emitted) is written on every call (the first access to all device
 *    memory is a write; no buffer needs pre-initialisation).  Cluster-record elements at and
 *    beyond n_clusters_emitted are left untouched.
 */
#ifndef PIXCLUS_H
#define PIXCLUS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PIX_OK 0
#define PIX_ERR_INVALID_ARG (-1)
#define PIX_ERR_CAPACITY (-2)  /* n_words / n_events beyond the create-time capacity */
#define PIX_ERR_CUDA (-3)      /* CUDA runtime error; text via pix_last_error */
#define PIX_ERR_ALLOC (-4)

/* Module geometry (reading S3): 2 x 8 read-out chips of 80 rows x 52 columns. */
#define PIX_ROWS 160
#define PIX_COLS 416

/* digi status codes (reading S6); exactly one per word, first failing check wins */
#define PIX_ST_OK 0              /* in a surviving cluster */
#define PIX_ST_CUT 1             /* its cluster failed the charge cut */
#define PIX_ST_BELOW_THRESHOLD 2 /* charge < pixel_threshold_e */
#define PIX_ST_DUPLICATE 3       /* an earlier word of the event has the same (module,row,col) (S10) */
#define PIX_ST_EMPTY 4           /* all-zero padding word (S5) */
#define PIX_ST_ERR_LINK 5        /* link not mapped in this FED (S4) */
#define PIX_ST_ERR_ROC 6         /* roc id unused on this link (S4) */
#define PIX_ST_ERR_DCOL 7        /* dcol >= 26 */
#define PIX_ST_ERR_PXID 8        /* pxid >= 160 */

/* summary[] indices (reading S20) */
enum {
  PIX_SUM_N_WORDS = 0, PIX_SUM_N_DECODED, PIX_SUM_N_EMPTY, PIX_SUM_N_ERR_LINK, PIX_SUM_N_ERR_ROC,
  PIX_SUM_N_ERR_DCOL, PIX_SUM_N_ERR_PXID, PIX_SUM_N_DUPLICATE, PIX_SUM_N_BELOW_THRESHOLD, PIX_SUM_N_OK_DIGIS,
  PIX_SUM_N_CUT_DIGIS, PIX_SUM_N_MODULES_PRESENT, PIX_SUM_N_CLUSTERS_PRECUT, PIX_SUM_N_CLUSTERS,
  PIX_SUM_N_CLUSTERS_EMITTED, PIX_SUM_FLAGS
};
#define PIX_FLAG_NONCONTIGUOUS 1u             /* some module's words form more than one run (S11): the event is not clustered.
                                                 Every decodable word gets status BELOW_THRESHOLD or CUT and clus = -1, the
                                                 counters follow (no duplicates, no OK digis, no clusters); decode fields,
                                                 module_first / module_end and n_modules_present are as for any event */
#define PIX_FLAG_CLUSTER_CAPACITY_OVERFLOW 2u /* more clusters than max_clusters_per_event; the rest are dropped */
#define PIX_FLAG_EVENT_TOO_LARGE 4u           /* batch only: the event is longer than max_words_per_event, its offsets are not
                                                 ascending, or it reaches beyond the word capacity of its launch group
                                                 (chunk_events x max_words_per_event words counted from the group's first
                                                 word).  The words inside the capacity are processed as usual -- a long
                                                 event that fits its group is complete -- and the outputs of the words beyond
                                                 it are NOT written (the one exception to "every element is written").
                                                 A batch whose events all respect max_words_per_event never raises it. */

typedef struct pix_handle pix_handle;

/* Raw word (reading S1), host-endian uint32, fields MSB->LSB:
 *   link 6b (w>>26) | roc 5b ((w>>21)&31) | dcol 5b ((w>>16)&31) | pxid 8b ((w>>8)&255) | adc 8b (w&255).
 * Raw data are grouped by front-end driver (FED): fed_offsets[F+1] gives each FED's contiguous
 * word block; the cabling key is (fed, link, roc) (reading S2). */

typedef struct {          /* host memory, copied during pix_create */
  uint32_t n_feds;        /* F >= 1 */
  uint32_t n_modules;     /* M, 1..65534 (0xFFFF is the invalid module id) */
  const uint32_t* entry;  /* [F*64*32], index (fed*64+link)*32+roc.  Packing (reading S3):
                             bit0 link_mapped (replicated in all 32 entries of a mapped link),
                             bit1 roc_valid, bits2-17 module, bits18-20 rocx (0..7), bit21 rocy,
                             bit22 flip_r, bit23 flip_c.  0 = unmapped link.
                             ROC-local rr = pxid>>1, cc = 2*dcol + (pxid&1);
                             row = rocy*80 + (flip_r ? 79-rr : rr); col = rocx*52 + (flip_c ? 51-cc : cc). */
} pix_cabling_map;

typedef struct {          /* host memory, copied during pix_create */
  uint32_t n_modules;     /* must equal the cabling map's */
  const float* gain;      /* [M*416], index module*416+col (reading S8: one pair per module column) */
  const float* pedestal;  /* [M*416] */
} pix_gain_table;

/* Calibration (reading S7), four separately rounded binary32 RN operations, no FMA:
 *   f1 = (float)adc - pedestal; f2 = f1*gain; f3 = f2*vcal_gain; f4 = f3 + vcal_offset;
 *   e  = !(f4 >= 0) ? 0 : (int32)trunc(min(f4, (float)max_electrons)). */
typedef struct {
  float vcal_gain, vcal_offset;     /* defaults 47.0f, -60.0f */
  int32_t pixel_threshold_e;        /* pixel kept iff e >= this; must be >= 1 (BASELINE cfg0: 1000) */
  int32_t cluster_charge_cut_e;     /* cluster kept iff sum(e) >= this (BASELINE cfg0: 4000) */
  int32_t max_electrons;            /* clamp, 1..65535 so that cluster charge fits uint32 (default 64000) */
  uint32_t max_clusters_per_module; /* the paper's maxHitsInModule() (value omitted there); 0xFFFFFFFF = none */
  uint32_t max_words_per_event;     /* capacity: longest event accepted */
  uint32_t max_clusters_per_event;  /* capacity (and per-event stride) of the cluster record arrays */
  uint32_t max_events_per_batch;    /* capacity of pix_process_batch (>= 1) */
  uint32_t chunk_events;            /* events per internal launch group of pix_process_batch; 0 = library default */
} pix_params;

/* Digis, SoA, 15 B/word; digi i <-> word i (never compacted).  Batch: indexed by global word index.
 * Undecodable words: module=row=col=0xFFFF, charge=0.  Decodable but rejected: true fields.  All
 * non-OK: clus = -1.  clus is module-local, 0..k_m-1, ordered by the cluster's first digi index (S14). */
typedef struct {
  uint16_t* module; uint16_t* row; uint16_t* col; int32_t* charge; int32_t* clus; uint8_t* status;
} pix_digis;

/* Cluster records, SoA, 22 B/cluster, plus per-module arrays and the summary.  Record index =
 * clus_module_start[module] + clus.  Batch: per-event strides max_clusters_per_event, M, M, M+1, 16.
 * first_digi is the event-relative index of the cluster's lowest-index digi.  x_col / y_row are the
 * charge-weighted mean col / row (reading S18). */
typedef struct {
  uint16_t* module; uint32_t* first_digi; uint32_t* n_pix; uint32_t* charge; float* x_col; float* y_row;
  uint32_t* module_first; uint32_t* module_end; /* [M]: index range of the module's decodable words; absent -> 0,0 (S12) */
  uint32_t* clus_module_start;                  /* [M+1]: [0]=0, [m+1]=[m]+min(max_clusters_per_module, n_clus[m]) (Fig. 3) */
  uint32_t* summary;                            /* [16] */
} pix_clusters;

/* Allocates device tables + workspace.  All pointers host.  *out is set only on success. */
int pix_create(const pix_cabling_map* cabling, const pix_gain_table* gains, const pix_params* params, pix_handle** out);

/* New handle with its own workspace over the same (shared, read-only) device tables. */
int pix_clone(const pix_handle* src, pix_handle** out);

int pix_destroy(pix_handle* h);

/* One event.  raw_words [n_words] and fed_offsets [F+1] (ascending, [0]=0, [F]=n_words; NULL iff F==1)
 * are DEVICE pointers; n_words may be 0.  Asynchronous on cuda_stream (a cudaStream_t; NULL = default). */
int pix_process(pix_handle* h, void* cuda_stream, const uint32_t* raw_words, const uint32_t* fed_offsets,
                uint32_t n_words, const pix_digis* out_digis, const pix_clusters* out_clusters);

/* n_events independent events in one call.  raw_words: all events concatenated [n_words_total];
 * event_word_offsets [n_events+1] (ascending, [0]=0, [n_events]=n_words_total); fed_offsets
 * [n_events*(F+1)] event-relative (NULL iff F==1).  All DEVICE pointers. */
int pix_process_batch(pix_handle* h, void* cuda_stream, uint32_t n_events, const uint32_t* raw_words,
                      uint32_t n_words_total, const uint32_t* event_word_offsets, const uint32_t* fed_offsets,
                      const pix_digis* out_digis, const pix_clusters* out_clusters);

/* Same as pix_process_batch but every pointer is a HOST pointer (pinned memory recommended): copies the
 * inputs to library-owned device staging, runs the path, copies every non-NULL output array back and
 * synchronises cuda_stream before returning (on an error too: nothing is in flight when the call returns).
 * Any output array pointer may be NULL: that array is not copied (e.g. all digi arrays NULL: clusters only).
 * Cluster records travel as rows of max(n_clusters_emitted) over the events of a launch group, so record
 * elements at and beyond an event's n_clusters_emitted are UNSPECIFIED after this call (not "untouched").
 * Staging is allocated on first use (sized by the capacities). */
int pix_process_batch_host(pix_handle* h, void* cuda_stream, uint32_t n_events, const uint32_t* raw_words,
                           uint32_t n_words_total, const uint32_t* event_word_offsets, const uint32_t* fed_offsets,
                           const pix_digis* out_digis, const pix_clusters* out_clusters);

/* RecHits-lite ("The RecHits module estimates the 3D position of each cluster
 * forming hits" -- only the module-local part: the detector geometry conditions are not available).
 * Readings S25-S28 of DESIGN.md.  One hit per emitted cluster record, same index and same per-event stride
 * (max_clusters_per_event): the per-module offsets of the hits are clus_module_start, which is what the
 * paper's fillHitsModuleStart (Fig. 3) fills.
 *   x_local, y_local  cm, origin at the module centre: x = (y_row + 0.5 - 80) * 0.0100, y = (x_col + 0.5 - 208) * 0.0150
 *                     (binary32, three separately rounded operations each)
 *   min_row .. max_col bounding box over the cluster's digis
 *   flags             bit0 ON_EDGE (box touches row 0 / 159 or col 0 / 415), bit1 SPANS_ROC (box crosses the row
 *                     79|80 boundary or a multiple-of-52 column boundary), bit2 SINGLE_PIXEL
 * All pointers DEVICE.  Inputs are the outputs of pix_process_batch on the same handle / sizes (n_events events,
 * event_word_offsets as given there).  Never allocates or synchronises; elements at and beyond an event's
 * n_clusters_emitted are left untouched. */
typedef struct {
  float* x_local; float* y_local; uint16_t* min_row; uint16_t* max_row; uint16_t* min_col; uint16_t* max_col; uint8_t* flags;
} pix_hits;
#define PIX_HIT_ON_EDGE 1u
#define PIX_HIT_SPANS_ROC 2u
#define PIX_HIT_SINGLE_PIXEL 4u
int pix_rechits(pix_handle* h, void* cuda_stream, uint32_t n_events, const uint32_t* event_word_offsets,
                const pix_digis* digis, const pix_clusters* clusters, const pix_hits* out_hits);

/* Legacy digi format and FED error words ("optional modules ... to convert the SoA to
 * legacy data formats", which the paper leaves out; the format is this build's own, readings S29-S31 of DESIGN.md).
 * Per word i (batch: global word index):
 *   pdigi[i]  = row | col << 11 | adc << 22 for a decodable word (status OK / CUT / BELOW_THRESHOLD / DUPLICATE; adc = the
 *               raw word's low byte), 0 otherwise                                                              (S29)
 *   raw_id[i] = module_raw_id[module] for a decodable word, 0 otherwise                                        (S30)
 * Error list of event e, at stride max_errors_per_event: every word with status ERR_LINK / ERR_ROC / ERR_DCOL / ERR_PXID
 * (padding words are not errors), in word order: the raw word, the FED block it sits in, the status code; n_errors[e]
 * is the true count, the list holds the first max_errors_per_event of them (S31).
 * All pointers DEVICE; raw_words, event_word_offsets and fed_offsets as given to pix_process_batch, digis its output;
 * module_raw_id [M].  Never allocates or synchronises; list elements beyond n_errors[e] are left untouched. */
typedef struct {
  uint32_t* pdigi; uint32_t* raw_id;                         /* [n_words_total] */
  uint32_t* err_word; uint16_t* err_fed; uint8_t* err_type;  /* [n_events * max_errors_per_event] */
  uint32_t* n_errors;                                        /* [n_events] */
} pix_legacy;
int pix_legacy_format(pix_handle* h, void* cuda_stream, uint32_t n_events, const uint32_t* raw_words, uint32_t n_words_total,
                      const uint32_t* event_word_offsets, const uint32_t* fed_offsets, const pix_digis* digis,
                      const uint32_t* module_raw_id, uint32_t max_errors_per_event, const pix_legacy* out);

/* Number of CUDA kernels this handle has launched so far (for launch accounting). */
uint64_t pix_kernel_launches(const pix_handle* h);

/* Device->host bytes the last pix_process_batch_host call on this handle copied (for transfer accounting). */
uint64_t pix_host_bytes_out(const pix_handle* h);

/* Diagnostic: module runs the LAST internal chunk of the last call left to the overflow kernel (runs longer than the
 * warp kernels' windows, pathological charge sums).  Synchronises the device; not for the hot path. */
int pix_overflow_runs(pix_handle* h, uint32_t* out);

/* Optional per-kernel timing for benchmarks (not legal during stream capture).  While enabled, every chunk
 * records CUDA events between its kernels on the caller's stream.  pix_read_profile waits for them and adds up
 * the device time per kernel since the last read: ms_out[8] = {init, runs, tile, overflow, finalize, 0, 0, 0};
 * *n_chunks_out = chunks covered. */
int pix_set_profiling(pix_handle* h, int enable);
int pix_read_profile(pix_handle* h, float* ms_out, uint32_t* n_chunks_out);

/* Clustering of ONE module's decoded digis without any allocation (for callers that cannot call cudaMalloc: code under
 * CUDA graph capture, tight serving loops; pix_create allocates, so this entry point takes no handle).
 * "clusters the pixels on each detector module"; the same readings as pix_process (S9 threshold and charge cut, S10
 * first digi of a pixel wins, S13 8-connectivity, S14 clusters numbered by their lowest digi, S18 records), run by the
 * block-per-run kernel with its tables in a static device array of 1 MiB + 256 B (64 B per digi) that every GPU
 * holds from the moment it loads the library.
 *   n_digis <= PIX_NOALLOC_MAX_DIGIS, else PIX_ERR_CAPACITY (nothing is launched).
 *   row, col, charge [n_digis]  DEVICE, inputs (the digi arrays pix_process wrote for the module's words, in word
 *                    order): row < 160 and col < 416, or row == 0xFFFF for a word that is not a pixel.
 *   clus, status [n_digis]      DEVICE, outputs as in pix_digis; a word with row == 0xFFFF gets clus = -1 and its
 *                    status is left untouched.
 *   c_first_digi .. c_y_row [max_clusters]  DEVICE, outputs: the module's cluster records in local-id order
 *                    (first_digi = index into the module's digis); records at and beyond counts[1] are untouched.
 *   counts [8]       DEVICE, output: clusters surviving the cut, records emitted (min with max_clusters), clusters
 *                    before the cut, digis DUPLICATE / BELOW_THRESHOLD / OK / CUT, 0.
 * One 512-thread block on the caller's stream; asynchronous; calls no cudaMalloc / cudaFree or allocating routine.
 * Every call shares the static array (it keeps the last call's contents; the kernel clears what must start at zero),
 * so two calls that overlap on one GPU (two streams, two host threads) race: serialise them.
 * pix_noalloc_setup looks the array's device address up (cudaGetSymbolAddress) for the current device; call it once
 * per device, with that device current, before a region where even that is unwelcome (stream capture);
 * pix_cluster_module_noalloc does it itself on first use otherwise.  Errors: the codes above; the text comes from
 * pix_noalloc_last_error (per host thread, "" if the last call succeeded). */
#define PIX_NOALLOC_MAX_DIGIS 16384u
int pix_noalloc_setup(void);
int pix_cluster_module_noalloc(void* cuda_stream, uint32_t n_digis, const uint16_t* row, const uint16_t* col,
                               const int32_t* charge, int32_t pixel_threshold_e, int32_t cluster_charge_cut_e,
                               uint32_t max_clusters, int32_t* clus, uint8_t* status, uint32_t* c_first_digi,
                               uint32_t* c_n_pix, uint32_t* c_charge, float* c_x_col, float* c_y_row, uint32_t* counts);
const char* pix_noalloc_last_error(void);

/* Text of the last error on this handle ("" if none).  Valid until the next call on the handle. */
const char* pix_last_error(const pix_handle* h);

#ifdef __cplusplus
}
#endif
#endif /* PIXCLUS_H */
