// api.cu -- the C ABI of libpixclus.so (include/pixclus.h).  Host code only: argument checks, device tables,
// workspace, the per-chunk launch sequence.  No step of the path runs here; there is no CPU fallback.
#include <atomic>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/pixclus.h"
#include "pix_common.cuh"

namespace pix {
void launch_rechits(uint32_t n_events, uint32_t M, uint32_t cap_ev, const uint32_t* ev_off, const pix_digis& d,
                    const pix_clusters& k, const pix_hits& h, cudaStream_t stream);
void launch_legacy(uint32_t n_events, uint32_t F, uint32_t M, uint32_t n_total, const uint32_t* words, const uint32_t* ev_off,
                   const uint32_t* fed_off, const pix_digis& d, const uint32_t* raw_id_of, uint32_t cap, const pix_legacy& o,
                   int n_sm, cudaStream_t stream);
}

namespace {

struct SharedTables {  // read-only device tables shared by clones
  std::atomic<int> refs{1};
  pix::CabEntry* cab = nullptr;
  float2* gp = nullptr;
};

struct HostStage {  // device staging of pix_process_batch_host, allocated on first use
  bool ready = false;
  uint32_t *words = nullptr, *ev_off = nullptr, *fed_off = nullptr;
  uint16_t *d_module = nullptr, *d_row = nullptr, *d_col = nullptr; int32_t *d_charge = nullptr, *d_clus = nullptr;
  uint8_t* d_status = nullptr;
  uint16_t* c_module = nullptr; uint32_t *c_first = nullptr, *c_npix = nullptr, *c_charge = nullptr;
  float *c_x = nullptr, *c_y = nullptr;
  uint32_t *module_first = nullptr, *module_end = nullptr, *clus_module_start = nullptr, *summary = nullptr;
  std::vector<void*> allocs;
  cudaStream_t s_in = nullptr, s_out = nullptr;  // copy streams of the pipelined host path
  std::vector<cudaEvent_t> ev;                   // three per launch group: input landed, group computed, summaries landed
  uint32_t* h_summary = nullptr;                 // pinned host copy of the summaries (sizes the record copies)
};

}  // namespace

struct pix_handle {
  int device = 0, n_sm = 0;
  uint32_t F = 0, M = 0;
  pix_params p{};
  uint32_t chunk_events = 0, cap_words = 0;
  uint64_t cap_total = 0;
  SharedTables* tables = nullptr;
  void* ws = nullptr;  // one allocation, carved below
  pix::Chunk proto{};  // tables, params and workspace pointers filled once
  uint64_t launches = 0;
  uint64_t hs_d2h_bytes = 0;  // device->host bytes of the last pix_process_batch_host call
  std::string err;
  HostStage hs;
  bool profiling = false;
  std::vector<cudaEvent_t> prof_events;  // LAUNCHES_PER_CHUNK + 1 per chunk, in launch order
  size_t prof_used = 0;
};

namespace {

int fail(pix_handle* h, int code, const char* msg) {
  if (h) h->err = msg;
  return code;
}
int fail_cuda(pix_handle* h, cudaError_t e, const char* where) {
  if (h) h->err = std::string(where) + ": " + cudaGetErrorString(e);
  return PIX_ERR_CUDA;
}

size_t align_up(size_t v) { return (v + 255) & ~(size_t)255; }

// workspace layout; pass base == nullptr to get the size only
size_t carve_workspace(pix_handle* h, unsigned char* base) {
  size_t off = 0;
  auto take = [&](size_t bytes) { unsigned char* p = base ? base + off : nullptr; off += align_up(bytes); return p; };
  const size_t Ec = h->chunk_events, M = h->M, F = h->F, W = h->cap_words;
  pix::Chunk& c = h->proto;
  c.segB = (uint32_t*)take((Ec * F + 1) * 4);
  c.ev_cnt = (uint32_t*)take(Ec * pix::EC_STRIDE * 4);
  c.ctl = (uint32_t*)take(pix::CTL_WORDS * 4);
  c.ovf_list = (uint32_t*)take(Ec * M * 4);
  c.list_cap = (uint32_t)(Ec * M);
  c.slice_list = (uint32_t*)take((W / 1024 + Ec + 1) * 8);  // two words per slice
  c.chunk_seg = (uint32_t*)take((W / 128 + 2) * 4);
  c.sbits = (uint32_t*)take((W / 32 + 64) * 4);  // the tile kernel reads 33 words from an item's first bit on
  c.cbad = (uint8_t*)take(W / 128 + 2);
  c.item_cap = (uint32_t)(W / 64 + 16 * Ec + 64);  // runs.cu: at most W_e / 112 + 2 items per piece of an event, 8 pieces
  c.items = (uint4*)take((size_t)c.item_cap * sizeof(uint4));
  c.n_clus = (uint32_t*)take(Ec * M * 4);
  c.n_runs = (uint32_t*)take(Ec * M * 4);
  c.t_a = (uint4*)take(2 * W * sizeof(uint4));
  c.t_y = (float*)take(2 * W * sizeof(float));
  c.t_base = (uint32_t*)take(Ec * M * 4);
  c.g_hash = (unsigned long long*)take(W * 16);
  c.g_pos = (uint32_t*)take(W * 4); c.g_q = (uint32_t*)take(W * 4); c.g_npix = (uint32_t*)take(W * 4);
  c.g_sx = (unsigned long long*)take(W * 8); c.g_sy = (unsigned long long*)take(W * 8);
  return off;
}

int make_workspace(pix_handle* h) {
  const size_t bytes = carve_workspace(h, nullptr);
  cudaError_t e = cudaMalloc(&h->ws, bytes);
  if (e != cudaSuccess) { h->ws = nullptr; cudaGetLastError(); return PIX_ERR_ALLOC; }
  carve_workspace(h, (unsigned char*)h->ws);
  return PIX_OK;
}

void release_tables(SharedTables* t) {
  if (t && t->refs.fetch_sub(1) == 1) { cudaFree(t->cab); cudaFree(t->gp); delete t; }
}

bool aligned16(const void* p) { return ((uintptr_t)p & 15u) == 0; }

int check_outputs(pix_handle* h, const pix_digis* d, const pix_clusters* k) {
  if (!d || !k) return fail(h, PIX_ERR_INVALID_ARG, "out_digis / out_clusters is NULL");
  if (!d->module || !d->row || !d->col || !d->charge || !d->clus || !d->status)
    return fail(h, PIX_ERR_INVALID_ARG, "a digi output array is NULL");
  if (!k->module || !k->first_digi || !k->n_pix || !k->charge || !k->x_col || !k->y_row || !k->module_first ||
      !k->module_end || !k->clus_module_start || !k->summary)
    return fail(h, PIX_ERR_INVALID_ARG, "a cluster output array is NULL");
  if (!aligned16(d->module) || !aligned16(d->row) || !aligned16(d->col) || !aligned16(d->charge) ||
      !aligned16(d->clus) || !aligned16(d->status))
    return fail(h, PIX_ERR_INVALID_ARG, "digi output arrays must be 16-byte aligned");
  return PIX_OK;
}

void bind_outputs(pix::Chunk& c, const pix_digis* d, const pix_clusters* k) {
  c.d_module = d->module; c.d_row = d->row; c.d_col = d->col; c.d_charge = d->charge; c.d_clus = d->clus;
  c.d_status = d->status;
  c.c_module = k->module; c.c_first = k->first_digi; c.c_npix = k->n_pix; c.c_charge = k->charge;
  c.c_x = k->x_col; c.c_y = k->y_row;
  c.module_first = k->module_first; c.module_end = k->module_end; c.clus_module_start = k->clus_module_start;
  c.summary = k->summary;
}

// the launch sequence of one chunk
constexpr int PROF_EVENTS = 6;  // families: init, runs (runs + pack), tile, overflow, finalize (offsets + scatter)
int run_chunk(pix_handle* h, const pix::Chunk& c, uint32_t n_total, uint32_t words_bound, cudaStream_t s) {
  cudaEvent_t* ev = nullptr;
  if (h->profiling) {
    while (h->prof_events.size() < h->prof_used + PROF_EVENTS) {
      cudaEvent_t x;
      if (cudaEventCreate(&x) != cudaSuccess) return fail(h, PIX_ERR_ALLOC, "cudaEventCreate");
      h->prof_events.push_back(x);
    }
    ev = h->prof_events.data() + h->prof_used;
    h->prof_used += PROF_EVENTS;
    cudaEventRecord(ev[0], s);
  }
  pix::launch_init(c, n_total, h->n_sm, s);
  if (ev) cudaEventRecord(ev[1], s);
  pix::launch_runs(c, words_bound, h->n_sm, s);
  if (ev) cudaEventRecord(ev[2], s);
  pix::launch_tile(c, h->n_sm, s);
  if (ev) cudaEventRecord(ev[3], s);
  pix::launch_overflow(c, h->n_sm, s);
  if (ev) cudaEventRecord(ev[4], s);
  pix::launch_finalize(c, h->n_sm, s);
  if (ev) cudaEventRecord(ev[5], s);
  h->launches += pix::LAUNCHES_PER_CHUNK;
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail_cuda(h, e, "kernel launch");
  return PIX_OK;
}

}  // namespace

extern "C" {

int pix_create(const pix_cabling_map* cabling, const pix_gain_table* gains, const pix_params* params, pix_handle** out) {
  if (!cabling || !gains || !params || !out || !cabling->entry || !gains->gain || !gains->pedestal) return PIX_ERR_INVALID_ARG;
  const uint32_t F = cabling->n_feds, M = cabling->n_modules;
  if (F < 1 || F > 65535 || M < 1 || M > pix::MAX_MODULES || gains->n_modules != M) return PIX_ERR_INVALID_ARG;
  if (params->pixel_threshold_e < 1 || params->max_electrons < 1 || params->max_electrons > 65535) return PIX_ERR_INVALID_ARG;
  if (params->max_words_per_event < 1 || params->max_events_per_batch < 1 || params->max_clusters_per_event < 1 ||
      params->max_clusters_per_event > (1u << 26))
    return PIX_ERR_INVALID_ARG;
  for (size_t i = 0; i < (size_t)F * 64 * 32; ++i)  // every mapped entry must name a module of the gain table
    if ((cabling->entry[i] & 2u) && ((cabling->entry[i] >> 2) & 0xFFFFu) >= M) return PIX_ERR_INVALID_ARG;

  pix_handle* h = new (std::nothrow) pix_handle;
  if (!h) return PIX_ERR_ALLOC;
  h->F = F; h->M = M; h->p = *params;
  cudaError_t e = cudaGetDevice(&h->device);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&h->n_sm, cudaDevAttrMultiProcessorCount, h->device);
  if (e == cudaSuccess) e = pix::configure_tile_kernel();
  if (e == cudaSuccess) e = pix::configure_finalize_kernel();
  if (e == cudaSuccess) e = pix::configure_overflow_kernel();
  if (e != cudaSuccess) { delete h; cudaGetLastError(); return PIX_ERR_CUDA; }

  // chunking: events per internal launch group; default: up to 64 Mi words per group (the path is bound by
  // instruction issue, not by HBM, so few large launches beat L2-sized ones)
  uint64_t ce = params->chunk_events;
  if (ce == 0) { ce = (64u << 20) / params->max_words_per_event; if (ce < 1) ce = 1; }
  if (ce > params->max_events_per_batch) ce = params->max_events_per_batch;
  if (ce > 65535) ce = 65535;
  const uint64_t capw = ce * (uint64_t)params->max_words_per_event;
  if (capw > 0x7FFFFFFFull || ce * (uint64_t)M > 0x7FFFFFFFull) { delete h; return PIX_ERR_INVALID_ARG; }
  h->chunk_events = (uint32_t)ce; h->cap_words = (uint32_t)capw;
  h->cap_total = (uint64_t)params->max_words_per_event * params->max_events_per_batch;
  if (h->cap_total > 0xFFFFFFFFull) h->cap_total = 0xFFFFFFFFull;

  // tables: cabling as given; (gain, pedestal) interleaved so that a digi costs one 8-byte gather
  SharedTables* t = new (std::nothrow) SharedTables;
  if (!t) { delete h; return PIX_ERR_ALLOC; }
  h->tables = t;
  const size_t ncab = (size_t)F * 64 * 32, ngp = (size_t)M * PIX_COLS;
  std::vector<float2> gp(ngp);
  for (size_t i = 0; i < ngp; ++i) gp[i] = make_float2(gains->gain[i], gains->pedestal[i]);
  // cabling re-laid out so that a decode is one 8-byte gather and two multiply-adds (pix_common.cuh; reading S3)
  std::vector<pix::CabEntry> cab(ncab);
  // Words of a run that ascend strictly in (link, roc, dcol, pxid) are different pixels (the tile kernel then skips its
  // search for duplicates) unless two valid entries of the table name the same ROC position of a module.
  std::vector<unsigned char> roc_seen((size_t)M * 16, 0);
  bool geom_unique = true;
  for (size_t i = 0; i < ncab; ++i) {
    const uint32_t e = cabling->entry[i];
    const uint32_t bad = !(e & 1u) ? PIX_ST_ERR_LINK : (!(e & 2u) ? PIX_ST_ERR_ROC : 0u);
    const uint32_t rocx = (e >> 18) & 7u, rocy = (e >> 21) & 1u, flip_r = (e >> 22) & 1u, flip_c = (e >> 23) & 1u;
    if (!bad) {
      const size_t pos = (size_t)((e >> 2) & 0xFFFFu) * 16 + rocy * 8 + rocx;
      if (pos >= roc_seen.size() || roc_seen[pos]) geom_unique = false; else roc_seen[pos] = 1;
    }
    const uint32_t row0 = rocy * 80u + (flip_r ? 79u : 0u), col0 = rocx * 52u + (flip_c ? 51u : 0u);
    cab[i].x = ((e >> 2) & 0xFFFFu) | (bad << 16) | ((flip_c ? 0xFFu : 0x01u) << 24);
    cab[i].y = row0 | (col0 << 8) | ((flip_r ? 0xFFu : 0x01u) << 24);
  }
  bool ok = cudaMalloc(&t->cab, ncab * sizeof(pix::CabEntry)) == cudaSuccess && cudaMalloc(&t->gp, ngp * sizeof(float2)) == cudaSuccess;
  ok = ok && cudaMemcpy(t->cab, cab.data(), ncab * sizeof(pix::CabEntry), cudaMemcpyHostToDevice) == cudaSuccess;
  ok = ok && cudaMemcpy(t->gp, gp.data(), ngp * sizeof(float2), cudaMemcpyHostToDevice) == cudaSuccess;
  if (!ok) { cudaGetLastError(); release_tables(t); delete h; return PIX_ERR_ALLOC; }

  pix::Chunk& c = h->proto;
  c.F = F; c.M = M; c.cab = t->cab; c.gp = t->gp; c.geom_unique = geom_unique ? 1u : 0u;
  c.F_shift = 0xFFFFFFFFu;
  for (uint32_t sh = 0; sh < 17; ++sh) if ((1u << sh) == F) c.F_shift = sh;
  c.vcal_gain = params->vcal_gain; c.vcal_offset = params->vcal_offset; c.max_e_f = (float)params->max_electrons;
  c.thr = params->pixel_threshold_e; c.cut = params->cluster_charge_cut_e;
  c.cap_mod = params->max_clusters_per_module; c.cap_ev = params->max_clusters_per_event; c.cap_words = h->cap_words; c.max_wpe = params->max_words_per_event;
  if (make_workspace(h) != PIX_OK) { release_tables(t); delete h; return PIX_ERR_ALLOC; }
  *out = h;
  return PIX_OK;
}

int pix_clone(const pix_handle* src, pix_handle** out) {
  if (!src || !out) return PIX_ERR_INVALID_ARG;
  pix_handle* h = new (std::nothrow) pix_handle;
  if (!h) return PIX_ERR_ALLOC;
  h->device = src->device; h->n_sm = src->n_sm; h->F = src->F; h->M = src->M; h->p = src->p;
  h->chunk_events = src->chunk_events; h->cap_words = src->cap_words; h->cap_total = src->cap_total;
  h->tables = src->tables; h->tables->refs.fetch_add(1);
  h->proto = src->proto;
  if (make_workspace(h) != PIX_OK) { release_tables(h->tables); delete h; return PIX_ERR_ALLOC; }
  *out = h;
  return PIX_OK;
}

int pix_destroy(pix_handle* h) {
  if (!h) return PIX_ERR_INVALID_ARG;
  cudaFree(h->ws);
  for (void* p : h->hs.allocs) cudaFree(p);
  if (h->hs.h_summary) cudaFreeHost(h->hs.h_summary);
  for (cudaEvent_t x : h->hs.ev) cudaEventDestroy(x);
  if (h->hs.s_in) cudaStreamDestroy(h->hs.s_in);
  if (h->hs.s_out) cudaStreamDestroy(h->hs.s_out);
  for (cudaEvent_t x : h->prof_events) cudaEventDestroy(x);
  release_tables(h->tables);
  delete h;
  return PIX_OK;
}

int pix_process(pix_handle* h, void* cuda_stream, const uint32_t* raw_words, const uint32_t* fed_offsets,
                uint32_t n_words, const pix_digis* out_digis, const pix_clusters* out_clusters) {
  if (!h) return PIX_ERR_INVALID_ARG;
  h->err.clear();
  if (n_words > 0 && !raw_words) return fail(h, PIX_ERR_INVALID_ARG, "raw_words is NULL");
  if (!aligned16(raw_words)) return fail(h, PIX_ERR_INVALID_ARG, "raw_words must be 16-byte aligned");
  if (h->F > 1 && !fed_offsets) return fail(h, PIX_ERR_INVALID_ARG, "fed_offsets is NULL but n_feds > 1");
  if (int rc = check_outputs(h, out_digis, out_clusters)) return rc;
  if (n_words > h->p.max_words_per_event || n_words > h->cap_words) return fail(h, PIX_ERR_CAPACITY, "n_words > max_words_per_event");
  pix::Chunk c = h->proto;
  c.words = raw_words; c.ev_off = nullptr; c.fed_off = h->F > 1 ? fed_offsets : nullptr; c.n_single = n_words;
  c.e0 = 0; c.e1 = 1;
  bind_outputs(c, out_digis, out_clusters);
  return run_chunk(h, c, n_words, n_words, (cudaStream_t)cuda_stream);
}

int pix_process_batch(pix_handle* h, void* cuda_stream, uint32_t n_events, const uint32_t* raw_words,
                      uint32_t n_words_total, const uint32_t* event_word_offsets, const uint32_t* fed_offsets,
                      const pix_digis* out_digis, const pix_clusters* out_clusters) {
  if (!h) return PIX_ERR_INVALID_ARG;
  h->err.clear();
  if (n_events == 0) return PIX_OK;
  if (!event_word_offsets) return fail(h, PIX_ERR_INVALID_ARG, "event_word_offsets is NULL");
  if (n_words_total > 0 && !raw_words) return fail(h, PIX_ERR_INVALID_ARG, "raw_words is NULL");
  if (!aligned16(raw_words)) return fail(h, PIX_ERR_INVALID_ARG, "raw_words must be 16-byte aligned");
  if (h->F > 1 && !fed_offsets) return fail(h, PIX_ERR_INVALID_ARG, "fed_offsets is NULL but n_feds > 1");
  if (int rc = check_outputs(h, out_digis, out_clusters)) return rc;
  if (n_events > h->p.max_events_per_batch) return fail(h, PIX_ERR_CAPACITY, "n_events > max_events_per_batch");
  if ((uint64_t)n_words_total > h->cap_total) return fail(h, PIX_ERR_CAPACITY, "n_words_total > max_words_per_event * max_events_per_batch");
  pix::Chunk c = h->proto;
  c.words = raw_words; c.ev_off = event_word_offsets; c.fed_off = h->F > 1 ? fed_offsets : nullptr; c.n_single = 0;
  bind_outputs(c, out_digis, out_clusters);
  const uint32_t bound = n_words_total < h->cap_words ? n_words_total : h->cap_words;
  for (uint32_t e0 = 0; e0 < n_events; e0 += h->chunk_events) {
    c.e0 = e0; c.e1 = (n_events - e0 > h->chunk_events) ? e0 + h->chunk_events : n_events;
    if (int rc = run_chunk(h, c, n_words_total, bound, (cudaStream_t)cuda_stream)) return rc;
  }
  return PIX_OK;
}

int pix_process_batch_host(pix_handle* h, void* cuda_stream, uint32_t n_events, const uint32_t* raw_words,
                           uint32_t n_words_total, const uint32_t* event_word_offsets, const uint32_t* fed_offsets,
                           const pix_digis* od, const pix_clusters* oc) {
  if (!h) return PIX_ERR_INVALID_ARG;
  h->err.clear();
  if (n_events == 0) return PIX_OK;
  if (!event_word_offsets || !od || !oc) return fail(h, PIX_ERR_INVALID_ARG, "NULL argument");
  if (n_words_total > 0 && !raw_words) return fail(h, PIX_ERR_INVALID_ARG, "raw_words is NULL");
  if (h->F > 1 && !fed_offsets) return fail(h, PIX_ERR_INVALID_ARG, "fed_offsets is NULL but n_feds > 1");
  if (n_events > h->p.max_events_per_batch) return fail(h, PIX_ERR_CAPACITY, "n_events > max_events_per_batch");
  if ((uint64_t)n_words_total > h->cap_total) return fail(h, PIX_ERR_CAPACITY, "n_words_total > capacity");
  const bool want_rec = oc->module || oc->first_digi || oc->n_pix || oc->charge || oc->x_col || oc->y_row;
  HostStage& s = h->hs;
  const size_t E = h->p.max_events_per_batch, W = (size_t)h->cap_total, M = h->M, F = h->F, K = h->p.max_clusters_per_event;
  if (!s.ready) {
    bool ok = true;
    auto dev = [&](size_t bytes) -> void* {
      void* p = nullptr;
      if (!ok) return p;
      if (cudaMalloc(&p, bytes ? bytes : 16) != cudaSuccess) { ok = false; cudaGetLastError(); return (void*)nullptr; }
      cudaMemset(p, 0, bytes ? bytes : 16);  // record slots beyond n_clusters_emitted may be copied out: never uninitialised memory
      s.allocs.push_back(p);
      return p;
    };
    s.words = (uint32_t*)dev(W * 4 + 64); s.ev_off = (uint32_t*)dev((E + 1) * 4); s.fed_off = (uint32_t*)dev(E * (F + 1) * 4);
    s.d_module = (uint16_t*)dev(W * 2 + 64); s.d_row = (uint16_t*)dev(W * 2 + 64); s.d_col = (uint16_t*)dev(W * 2 + 64);
    s.d_charge = (int32_t*)dev(W * 4 + 64); s.d_clus = (int32_t*)dev(W * 4 + 64); s.d_status = (uint8_t*)dev(W + 64);
    s.c_module = (uint16_t*)dev(E * K * 2); s.c_first = (uint32_t*)dev(E * K * 4); s.c_npix = (uint32_t*)dev(E * K * 4);
    s.c_charge = (uint32_t*)dev(E * K * 4); s.c_x = (float*)dev(E * K * 4); s.c_y = (float*)dev(E * K * 4);
    s.module_first = (uint32_t*)dev(E * M * 4); s.module_end = (uint32_t*)dev(E * M * 4);
    s.clus_module_start = (uint32_t*)dev(E * (M + 1) * 4); s.summary = (uint32_t*)dev(E * 16 * 4);
    if (ok && cudaMallocHost(&s.h_summary, E * 16 * 4) != cudaSuccess) { ok = false; cudaGetLastError(); s.h_summary = nullptr; }
    if (!ok) { for (void* p : s.allocs) cudaFree(p); s.allocs.clear(); return fail(h, PIX_ERR_ALLOC, "staging allocation failed"); }
    s.ready = true;
  }
  // Pipeline over launch groups of events (the transfer is part of the module):
  // group g's input copy (stream s_in), its kernels (the caller's stream) and its output copy (stream s_out) overlap
  // with the neighbouring groups'.  The workspace is shared, so the kernels of the groups run in stream order.
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (!s.s_in) {
    if (cudaStreamCreateWithFlags(&s.s_in, cudaStreamNonBlocking) != cudaSuccess ||
        cudaStreamCreateWithFlags(&s.s_out, cudaStreamNonBlocking) != cudaSuccess) {
      cudaGetLastError(); s.s_in = s.s_out = nullptr;
      return fail(h, PIX_ERR_ALLOC, "stream creation failed");
    }
  }
  uint32_t ge = (n_events + 7u) / 8u;  // about eight groups per call
  if (ge < 1u) ge = 1u;
  if (ge > h->chunk_events) ge = h->chunk_events;
  const uint32_t n_groups = (n_events + ge - 1u) / ge;
  while (s.ev.size() < 3 * (size_t)n_groups + 1) {  // all events exist before the first copy is issued
    cudaEvent_t x;
    if (cudaEventCreateWithFlags(&x, cudaEventDisableTiming) != cudaSuccess) return fail(h, PIX_ERR_ALLOC, "cudaEventCreate");
    s.ev.push_back(x);
  }
  const size_t Ev = n_events;
  cudaError_t e = cudaSuccess;
  int rc = PIX_OK;
  auto h2d = [&](void* d, const void* src, size_t bytes) { if (e == cudaSuccess && bytes) e = cudaMemcpyAsync(d, src, bytes, cudaMemcpyHostToDevice, s.s_in); };
  auto d2h = [&](void* dst, const void* d, size_t bytes) { if (e == cudaSuccess && dst && bytes) e = cudaMemcpyAsync(dst, d, bytes, cudaMemcpyDeviceToHost, s.s_out); };
  // record arrays: rows of `width` elements (the most any event of the group emitted) at the per-event stride K
  auto d2h_rec = [&](void* dst, const void* d, size_t elem, size_t k0, size_t width, size_t rows) {
    if (e == cudaSuccess && dst && width && rows)
      e = cudaMemcpy2DAsync((char*)dst + k0 * elem, K * elem, (const char*)d + k0 * elem, K * elem, width * elem, rows, cudaMemcpyDeviceToHost, s.s_out);
  };
  // the record copies of group g, once its summaries have landed in h_summary
  auto records_of = [&](uint32_t g) {
    if (!want_rec || e != cudaSuccess) return;
    const uint32_t e0 = g * ge, e1 = (n_events - e0 > ge) ? e0 + ge : n_events;
    e = cudaEventSynchronize(s.ev[3 * g + 2]);
    if (e != cudaSuccess) return;
    size_t width = 0;
    for (uint32_t ev = e0; ev < e1; ++ev) { const size_t n = s.h_summary[(size_t)ev * 16 + PIX_SUM_N_CLUSTERS_EMITTED]; width = n > width ? n : width; }
    if (width > K) width = K;
    const size_t k0 = (size_t)e0 * K, ne = e1 - e0;
    d2h_rec(oc->module, s.c_module, 2, k0, width, ne); d2h_rec(oc->first_digi, s.c_first, 4, k0, width, ne);
    d2h_rec(oc->n_pix, s.c_npix, 4, k0, width, ne); d2h_rec(oc->charge, s.c_charge, 4, k0, width, ne);
    d2h_rec(oc->x_col, s.c_x, 4, k0, width, ne); d2h_rec(oc->y_row, s.c_y, 4, k0, width, ne);
    h->hs_d2h_bytes += width * ne * ((oc->module ? 2 : 0) + (oc->first_digi ? 4 : 0) + (oc->n_pix ? 4 : 0) + (oc->charge ? 4 : 0) + (oc->x_col ? 4 : 0) + (oc->y_row ? 4 : 0));
  };
  h->hs_d2h_bytes = 0;
  // the copy streams start after whatever the caller's stream holds so far
  if (e == cudaSuccess) e = cudaEventRecord(s.ev[3 * n_groups], st);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(s.s_in, s.ev[3 * n_groups], 0);
  h2d(s.ev_off, event_word_offsets, (Ev + 1) * 4);
  if (F > 1) h2d(s.fed_off, fed_offsets, Ev * (F + 1) * 4);
  pix_digis dd{s.d_module, s.d_row, s.d_col, s.d_charge, s.d_clus, s.d_status};
  pix_clusters dc{s.c_module, s.c_first, s.c_npix, s.c_charge, s.c_x, s.c_y, s.module_first, s.module_end, s.clus_module_start, s.summary};
  pix::Chunk c = h->proto;
  c.words = s.words; c.ev_off = s.ev_off; c.fed_off = F > 1 ? s.fed_off : nullptr; c.n_single = 0;
  bind_outputs(c, &dd, &dc);
  uint32_t g = 0;
  for (; g < n_groups && e == cudaSuccess && rc == PIX_OK; ++g) {
    const uint32_t e0 = g * ge, e1 = (n_events - e0 > ge) ? e0 + ge : n_events;
    // host-side view of the group's word range, clamped like the device does
    size_t w0 = event_word_offsets[e0], w1 = event_word_offsets[e1];
    if (w1 > n_words_total) w1 = n_words_total;
    if (w0 > w1) w0 = w1;
    h2d(s.words + w0, raw_words + w0, (w1 - w0) * 4);
    if (e == cudaSuccess) e = cudaEventRecord(s.ev[3 * g], s.s_in);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(st, s.ev[3 * g], 0);
    if (e != cudaSuccess) break;
    c.e0 = e0; c.e1 = e1;
    size_t bound = w1 - w0;
    if (bound > h->cap_words) bound = h->cap_words;
    rc = run_chunk(h, c, n_words_total, (uint32_t)bound, st);
    if (rc != PIX_OK) break;
    if (e == cudaSuccess) e = cudaEventRecord(s.ev[3 * g + 1], st);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(s.s_out, s.ev[3 * g + 1], 0);
    const size_t nw = w1 - w0, ne = e1 - e0;
    // the summaries first: the record copies are sized by n_clusters_emitted
    if (e == cudaSuccess) e = cudaMemcpyAsync(s.h_summary + (size_t)e0 * 16, s.summary + (size_t)e0 * 16, ne * 64, cudaMemcpyDeviceToHost, s.s_out);
    if (e == cudaSuccess) e = cudaEventRecord(s.ev[3 * g + 2], s.s_out);
    d2h(od->module ? od->module + w0 : nullptr, s.d_module + w0, nw * 2); d2h(od->row ? od->row + w0 : nullptr, s.d_row + w0, nw * 2);
    d2h(od->col ? od->col + w0 : nullptr, s.d_col + w0, nw * 2); d2h(od->charge ? od->charge + w0 : nullptr, s.d_charge + w0, nw * 4);
    d2h(od->clus ? od->clus + w0 : nullptr, s.d_clus + w0, nw * 4); d2h(od->status ? od->status + w0 : nullptr, s.d_status + w0, nw);
    d2h(oc->module_first ? oc->module_first + (size_t)e0 * M : nullptr, s.module_first + (size_t)e0 * M, ne * M * 4);
    d2h(oc->module_end ? oc->module_end + (size_t)e0 * M : nullptr, s.module_end + (size_t)e0 * M, ne * M * 4);
    d2h(oc->clus_module_start ? oc->clus_module_start + (size_t)e0 * (M + 1) : nullptr, s.clus_module_start + (size_t)e0 * (M + 1), ne * (M + 1) * 4);
    h->hs_d2h_bytes += nw * ((od->module ? 2 : 0) + (od->row ? 2 : 0) + (od->col ? 2 : 0) + (od->charge ? 4 : 0) + (od->clus ? 4 : 0) + (od->status ? 1 : 0)) +
                       ne * ((oc->module_first ? M * 4 : 0) + (oc->module_end ? M * 4 : 0) + (oc->clus_module_start ? (M + 1) * 4 : 0) + 64);
    if (g > 0) records_of(g - 1);  // the previous group's summaries have had a whole group's time to land
  }
  if (e == cudaSuccess && rc == PIX_OK && g == n_groups) records_of(n_groups - 1);
  // every exit waits for what has been issued: the copies write the caller's buffers and read its input
  const cudaError_t e1 = cudaStreamSynchronize(s.s_in), e2 = cudaStreamSynchronize(st), e3 = cudaStreamSynchronize(s.s_out);
  if (rc != PIX_OK) return rc;
  if (e == cudaSuccess) e = e1 != cudaSuccess ? e1 : (e2 != cudaSuccess ? e2 : e3);
  if (e != cudaSuccess) { cudaGetLastError(); return fail_cuda(h, e, "pix_process_batch_host"); }
  if (oc->summary) std::memcpy(oc->summary, s.h_summary, Ev * 64);
  return PIX_OK;
}

uint64_t pix_host_bytes_out(const pix_handle* h) { return h ? h->hs_d2h_bytes : 0; }

int pix_rechits(pix_handle* h, void* cuda_stream, uint32_t n_events, const uint32_t* event_word_offsets,
                const pix_digis* digis, const pix_clusters* clusters, const pix_hits* out_hits) {
  if (!h) return PIX_ERR_INVALID_ARG;
  h->err.clear();
  if (n_events == 0) return PIX_OK;
  if (!event_word_offsets || !out_hits) return fail(h, PIX_ERR_INVALID_ARG, "NULL argument");
  if (int rc = check_outputs(h, digis, clusters)) return rc;
  if (!out_hits->x_local || !out_hits->y_local || !out_hits->min_row || !out_hits->max_row || !out_hits->min_col ||
      !out_hits->max_col || !out_hits->flags)
    return fail(h, PIX_ERR_INVALID_ARG, "a hit output array is NULL");
  if (n_events > h->p.max_events_per_batch) return fail(h, PIX_ERR_CAPACITY, "n_events > max_events_per_batch");
  pix::launch_rechits(n_events, h->M, h->p.max_clusters_per_event, event_word_offsets, *digis, *clusters, *out_hits,
                      (cudaStream_t)cuda_stream);
  h->launches += (n_events + 65534u) / 65535u;
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail_cuda(h, e, "kernel launch");
  return PIX_OK;
}

int pix_legacy_format(pix_handle* h, void* cuda_stream, uint32_t n_events, const uint32_t* raw_words, uint32_t n_words_total,
                      const uint32_t* event_word_offsets, const uint32_t* fed_offsets, const pix_digis* digis,
                      const uint32_t* module_raw_id, uint32_t max_errors_per_event, const pix_legacy* out) {
  if (!h) return PIX_ERR_INVALID_ARG;
  h->err.clear();
  if (n_events == 0) return PIX_OK;
  if (!event_word_offsets || !digis || !module_raw_id || !out) return fail(h, PIX_ERR_INVALID_ARG, "NULL argument");
  if (n_words_total > 0 && !raw_words) return fail(h, PIX_ERR_INVALID_ARG, "raw_words is NULL");
  if (h->F > 1 && !fed_offsets) return fail(h, PIX_ERR_INVALID_ARG, "fed_offsets is NULL but n_feds > 1");
  if (!digis->module || !digis->row || !digis->col || !digis->status) return fail(h, PIX_ERR_INVALID_ARG, "a digi input array is NULL");
  if (!out->pdigi || !out->raw_id || !out->n_errors || (max_errors_per_event && (!out->err_word || !out->err_fed || !out->err_type)))
    return fail(h, PIX_ERR_INVALID_ARG, "a legacy output array is NULL");
  if (n_events > h->p.max_events_per_batch) return fail(h, PIX_ERR_CAPACITY, "n_events > max_events_per_batch");
  pix::launch_legacy(n_events, h->F, h->M, n_words_total, raw_words, event_word_offsets, h->F > 1 ? fed_offsets : nullptr, *digis,
                     module_raw_id, max_errors_per_event, *out, h->n_sm, (cudaStream_t)cuda_stream);
  h->launches += 1;
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail_cuda(h, e, "kernel launch");
  return PIX_OK;
}

int pix_set_profiling(pix_handle* h, int enable) {
  if (!h) return PIX_ERR_INVALID_ARG;
  h->profiling = enable != 0;
  h->prof_used = 0;
  return PIX_OK;
}

int pix_read_profile(pix_handle* h, float* ms_out, uint32_t* n_chunks_out) {
  if (!h || !ms_out) return PIX_ERR_INVALID_ARG;
  for (int k = 0; k < 8; ++k) ms_out[k] = 0.0f;
  const size_t nch = h->prof_used / PROF_EVENTS;
  for (size_t q = 0; q < nch; ++q) {
    cudaEvent_t* ev = h->prof_events.data() + q * PROF_EVENTS;
    cudaError_t e = cudaEventSynchronize(ev[PROF_EVENTS - 1]);
    for (int k = 0; k < PROF_EVENTS - 1 && e == cudaSuccess; ++k) {
      float ms = 0.0f;
      e = cudaEventElapsedTime(&ms, ev[k], ev[k + 1]);
      ms_out[k] += ms;
    }
    if (e != cudaSuccess) return fail_cuda(h, e, "pix_read_profile");
  }
  if (n_chunks_out) *n_chunks_out = (uint32_t)nch;
  h->prof_used = 0;
  return PIX_OK;
}

uint64_t pix_kernel_launches(const pix_handle* h) { return h ? h->launches : 0; }

int pix_overflow_runs(pix_handle* h, uint32_t* out) {
  if (!h || !out) return PIX_ERR_INVALID_ARG;
  cudaError_t e = cudaDeviceSynchronize();
  if (e == cudaSuccess) e = cudaMemcpy(out, h->proto.ctl + pix::CTL_OVF_COUNT, 4, cudaMemcpyDeviceToHost);
  if (e != cudaSuccess) return fail_cuda(h, e, "pix_overflow_runs");
  return PIX_OK;
}

const char* pix_last_error(const pix_handle* h) { return h ? h->err.c_str() : "invalid handle"; }

}  // extern "C"
