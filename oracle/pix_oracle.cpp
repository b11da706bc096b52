// pix_oracle.cpp -- ORACLE for the pixel "Clusters" hot path.  TEST INFRASTRUCTURE ONLY.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// call this.  It shares no code with the CUDA path (paper_2104_06573_b200/csrc) and neither
// imports the other.  Plain, slow, single-threaded; compiled with g++ -O2 -ffp-contract=off.
//
// What it computes (section 2: the Clusters module "unpacks [the raw data],
// calibrates the individual pixels, and clusters the pixels on each detector module"; PAPER.md
// Fig. 3, lines 76-81: moduleStart[i+1] = min(maxHitsInModule(), cluStart[i])), in the order
// O1..O8 of DESIGN.md section 3.  Everything the paper leaves open (bit layout, calibration
// formula, 8-connectivity, duplicate rule, canonical ids, charge cut) follows the numbered
// readings S1..S24 in DESIGN.md, which restate BASELINE.json's north_star and configs.
//
// Nature of the result: connected components have a plain definition, so O5 is that definition
// written out as BFS flood fill (no union-find, no blocking, no reordering).
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): scipy.ndimage.label as an independent
// 8-connectivity routine; O(n^2) brute force on tiny modules; closed forms (full module,
// checkerboard, lattice, stripes, diagonal, no-wrap pair); the address bijection; step-by-step
// numpy.float32 calibration over all 256 ADC values; charge conservation and the structural
// invariants; metamorphic permutations; the generator's injected-error tallies.
// RecHits-lite (pixo_rechits, readings S25-S28): closed forms on hand-built clusters and a numpy group-by
// recomputation (tests/test_oracle_rechits.py).
// Legacy format (pixo_legacy, readings S29-S31): a hand-computed packed word, an independent numpy unpacking and
// error-list recomputation, the generator's injected-error tallies, the capacity clamp (tests/test_oracle_legacy.py).
// PARITY UNPINNED against paper-printed values: the paper prints no worked example, count or
// intermediate value for this path.
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

constexpr int ROWS = 160, COLS = 416, ROC_ROWS = 80, ROC_COLS = 52;
constexpr uint16_t INVALID16 = 0xFFFF;

// status codes, reading S6
enum : uint8_t { ST_OK = 0, ST_CUT = 1, ST_BELOW = 2, ST_DUP = 3, ST_EMPTY = 4, ST_ERR_LINK = 5, ST_ERR_ROC = 6,
                 ST_ERR_DCOL = 7, ST_ERR_PXID = 8 };

struct Decoded { uint8_t status; uint16_t module, row, col; uint8_t adc; };

}  // namespace

extern "C" {

struct pixo_params {
  float vcal_gain, vcal_offset;
  int32_t pixel_threshold_e, cluster_charge_cut_e, max_electrons;
  uint32_t max_clusters_per_module;  // the paper's maxHitsInModule() (value omitted; reading S16)
  uint32_t max_clusters_per_event;   // capacity of the cluster record arrays
};

// O1 (readings S1-S6): one raw word -> status + (module,row,col,adc).  fed = index of the FED
// block the word sits in.  Returns the status; outputs are defined only when it returns ST_OK.
int pixo_decode_word(uint32_t w, uint32_t fed, const uint32_t* cabling, uint16_t* module, uint16_t* row,
                     uint16_t* col, uint8_t* adc) {
  if (w == 0) return ST_EMPTY;                       // S5: padding
  uint32_t link = w >> 26;                           // S1: fields listed MSB -> LSB
  uint32_t roc = (w >> 21) & 31u;
  uint32_t dcol = (w >> 16) & 31u;
  uint32_t pxid = (w >> 8) & 255u;
  uint32_t e = cabling[(fed * 64u + link) * 32u + roc];
  if (!(e & 1u)) return ST_ERR_LINK;                 // S4: link not mapped
  if (!(e & 2u)) return ST_ERR_ROC;                  // S4: roc id unused on this link
  if (dcol >= 26u) return ST_ERR_DCOL;               // S3: 26 double columns
  if (pxid >= 160u) return ST_ERR_PXID;              // S3: 160 pixels per double column
  uint32_t rocx = (e >> 18) & 7u, rocy = (e >> 21) & 1u, flip_r = (e >> 22) & 1u, flip_c = (e >> 23) & 1u;
  uint32_t rr = pxid >> 1;                           // S3: ROC-local row
  uint32_t cc = 2u * dcol + (pxid & 1u);             //     ROC-local column
  *module = (uint16_t)((e >> 2) & 0xFFFFu);
  *row = (uint16_t)(rocy * ROC_ROWS + (flip_r ? (ROC_ROWS - 1 - rr) : rr));
  *col = (uint16_t)(rocx * ROC_COLS + (flip_c ? (ROC_COLS - 1 - cc) : cc));
  *adc = (uint8_t)(w & 255u);
  return ST_OK;
}

// O2 (reading S7): ADC -> electrons.  Four separately rounded binary32 operations in this order,
// no FMA contraction (-ffp-contract=off and the volatile temporaries keep them apart), then
// NaN/negative -> 0, clamp, truncate.
int32_t pixo_calibrate(uint8_t adc, float gain, float pedestal, const pixo_params* p) {
  volatile float f1 = (float)adc - pedestal;
  volatile float f2 = f1 * gain;
  volatile float f3 = f2 * p->vcal_gain;
  volatile float f4 = f3 + p->vcal_offset;
  float v = f4;
  if (!(v >= 0.0f)) return 0;
  float cap = (float)p->max_electrons;
  if (v > cap) v = cap;
  return (int32_t)v;  // truncation toward zero; v is within int32 range after the clamp
}

// The whole path for ONE event, host pointers.  Output arrays: digis [n_words]; cluster records
// [max_clusters_per_event]; module_first/module_end [M]; clus_module_start [M+1]; summary [16].
// Returns 0, or -1 on invalid arguments.
int pixo_process(uint32_t n_feds, uint32_t n_modules, const uint32_t* cabling, const float* gain,
                 const float* pedestal, const pixo_params* p, const uint32_t* words, const uint32_t* fed_offsets,
                 uint32_t n_words, uint16_t* d_module, uint16_t* d_row, uint16_t* d_col, int32_t* d_charge,
                 int32_t* d_clus, uint8_t* d_status, uint16_t* c_module, uint32_t* c_first_digi, uint32_t* c_n_pix,
                 uint32_t* c_charge, float* c_x_col, float* c_y_row, uint32_t* module_first, uint32_t* module_end,
                 uint32_t* clus_module_start, uint32_t* summary) {
  if (!cabling || !gain || !pedestal || !p || n_modules == 0 || n_modules > 65534 || n_feds == 0) return -1;
  if (n_feds > 1 && !fed_offsets) return -1;
  const uint32_t M = n_modules;
  uint32_t n_empty = 0, n_err[4] = {0, 0, 0, 0}, n_decoded = 0;

  // ---- O1 decode + O2 calibrate, per word in index order
  uint32_t fed = 0;
  for (uint32_t i = 0; i < n_words; ++i) {
    if (fed_offsets) while (fed + 1 < n_feds && i >= fed_offsets[fed + 1]) ++fed;  // S2: FED block of word i
    uint16_t m = 0, r = 0, c = 0; uint8_t adc = 0;
    int st = pixo_decode_word(words[i], fed, cabling, &m, &r, &c, &adc);
    d_clus[i] = -1;
    if (st != ST_OK) {                               // S21: undecodable -> all-ones fields, zero charge
      d_module[i] = d_row[i] = d_col[i] = INVALID16; d_charge[i] = 0; d_status[i] = (uint8_t)st;
      if (st == ST_EMPTY) ++n_empty; else ++n_err[st - ST_ERR_LINK];
      continue;
    }
    ++n_decoded;
    d_module[i] = m; d_row[i] = r; d_col[i] = c;
    size_t gi = (size_t)m * COLS + c;               // S8: one (gain, pedestal) pair per (module, col)
    int32_t e = pixo_calibrate(adc, gain[gi], pedestal[gi], p);
    d_charge[i] = e;
    d_status[i] = (e < p->pixel_threshold_e) ? ST_BELOW : ST_OK;  // S9: kept iff e >= threshold
  }

  // ---- O3 module ranges and runs (S11, S12)
  std::vector<uint32_t> n_runs(M, 0);
  for (uint32_t m = 0; m < M; ++m) { module_first[m] = 0; module_end[m] = 0; }
  {
    std::vector<uint8_t> seen(M, 0);
    uint32_t prev = 0xFFFFFFFFu;
    for (uint32_t i = 0; i < n_words; ++i) {
      if (d_module[i] == INVALID16) continue;        // undecodable words are transparent
      uint32_t m = d_module[i];
      if (!seen[m]) { seen[m] = 1; module_first[m] = i; }
      module_end[m] = i + 1;
      if (m != prev) { ++n_runs[m]; prev = m; }
    }
  }
  uint32_t n_modules_present = 0, flags = 0;
  for (uint32_t m = 0; m < M; ++m) {
    if (n_runs[m] > 0) ++n_modules_present;
    if (n_runs[m] > 1) flags |= 1u;                  // NONCONTIGUOUS
  }

  // digis of each module in increasing index order
  std::vector<uint32_t> bucket_start(M + 1, 0), bucket(n_decoded);
  for (uint32_t i = 0; i < n_words; ++i) if (d_module[i] != INVALID16) ++bucket_start[d_module[i] + 1];
  for (uint32_t m = 0; m < M; ++m) bucket_start[m + 1] += bucket_start[m];
  {
    std::vector<uint32_t> cur(bucket_start.begin(), bucket_start.end() - 1);
    for (uint32_t i = 0; i < n_words; ++i) if (d_module[i] != INVALID16) bucket[cur[d_module[i]]++] = i;
  }

  struct Rec { uint32_t first_digi, n_pix, charge; float x, y; };
  std::vector<std::vector<Rec>> recs(M);
  std::vector<int32_t> owner((size_t)ROWS * COLS, -1);  // dense grid of one module, -1 = free
  std::vector<uint32_t> queue, members;
  uint32_t n_dup = 0, n_below = 0, n_ok = 0, n_cut = 0, n_precut = 0, n_postcut = 0;

  for (uint32_t m = 0; m < M; ++m) {
    const uint32_t* idx = bucket.data() + bucket_start[m];
    const uint32_t nm = bucket_start[m + 1] - bucket_start[m];
    // ---- O4 duplicates (S10): first index wins, whatever the charges
    for (uint32_t k = 0; k < nm; ++k) {
      uint32_t i = idx[k];
      int32_t& o = owner[(size_t)d_row[i] * COLS + d_col[i]];
      if (o >= 0) d_status[i] = ST_DUP; else o = (int32_t)i;
    }
    // ---- O5 flood fill (S13), seeds in increasing index => components found in first-digi order
    // d_clus: -1 = unlabelled.  A provisional value -2 marks "visited, in the current component".
    uint32_t local = 0;
    for (uint32_t k = 0; k < nm; ++k) {
      uint32_t seed = idx[k];
      if (d_status[seed] != ST_OK || d_clus[seed] != -1) continue;
      queue.clear(); members.clear();
      queue.push_back(seed); d_clus[seed] = -2;
      for (size_t head = 0; head < queue.size(); ++head) {
        uint32_t i = queue[head];
        members.push_back(i);
        int r = d_row[i], c = d_col[i];
        for (int dr = -1; dr <= 1; ++dr)
          for (int dc = -1; dc <= 1; ++dc) {
            if (dr == 0 && dc == 0) continue;
            int rr = r + dr, cc = c + dc;
            if (rr < 0 || rr >= ROWS || cc < 0 || cc >= COLS) continue;   // no wrap, no other module
            int32_t j = owner[(size_t)rr * COLS + cc];
            if (j < 0) continue;
            if (d_status[j] != ST_OK || d_clus[j] != -1) continue;        // owner below threshold, or already taken
            d_clus[j] = -2; queue.push_back((uint32_t)j);
          }
      }
      // ---- O6 charge cut + renumber (S9, S14)
      ++n_precut;
      int64_t Q = 0, sx = 0, sy = 0;
      for (uint32_t i : members) { Q += d_charge[i]; sx += (int64_t)d_charge[i] * d_col[i]; sy += (int64_t)d_charge[i] * d_row[i]; }
      if (Q >= (int64_t)p->cluster_charge_cut_e) {
        for (uint32_t i : members) d_clus[i] = (int32_t)local;
        n_ok += (uint32_t)members.size();
        // ---- O7 record (S18): charge-weighted centroid, int64 sums -> double -> float
        Rec rec;
        rec.first_digi = seed; rec.n_pix = (uint32_t)members.size(); rec.charge = (uint32_t)Q;
        rec.x = (float)((double)sx / (double)Q); rec.y = (float)((double)sy / (double)Q);
        recs[m].push_back(rec);
        ++local; ++n_postcut;
      } else {
        for (uint32_t i : members) { d_clus[i] = -1; d_status[i] = ST_CUT; }
        n_cut += (uint32_t)members.size();
      }
    }
    for (uint32_t k = 0; k < nm; ++k) {
      uint32_t i = idx[k];
      if (d_status[i] == ST_DUP) ++n_dup;
      if (d_status[i] == ST_BELOW) ++n_below;
      owner[(size_t)d_row[i] * COLS + d_col[i]] = -1;   // sparse clear
    }
  }

  // ---- O8 offsets: Fig. 3's clamp followed by the running sum the paper leaves implicit (S19)
  clus_module_start[0] = 0;
  for (uint32_t m = 0; m < M; ++m) {
    uint32_t cnt = (uint32_t)recs[m].size();
    if (cnt > p->max_clusters_per_module) cnt = p->max_clusters_per_module;
    clus_module_start[m + 1] = clus_module_start[m] + cnt;
  }
  uint32_t n_emitted = clus_module_start[M];
  if (n_emitted > p->max_clusters_per_event) { n_emitted = p->max_clusters_per_event; flags |= 2u; }  // CLUSTER_CAPACITY_OVERFLOW
  for (uint32_t m = 0; m < M; ++m) {
    uint32_t cnt = clus_module_start[m + 1] - clus_module_start[m];
    for (uint32_t l = 0; l < cnt; ++l) {
      uint32_t g = clus_module_start[m] + l;
      if (g >= p->max_clusters_per_event) break;
      const Rec& rec = recs[m][l];
      c_module[g] = (uint16_t)m; c_first_digi[g] = rec.first_digi; c_n_pix[g] = rec.n_pix; c_charge[g] = rec.charge;
      c_x_col[g] = rec.x; c_y_row[g] = rec.y;
    }
  }

  // summary (S20)
  summary[0] = n_words; summary[1] = n_decoded; summary[2] = n_empty;
  summary[3] = n_err[0]; summary[4] = n_err[1]; summary[5] = n_err[2]; summary[6] = n_err[3];
  summary[7] = n_dup; summary[8] = n_below; summary[9] = n_ok; summary[10] = n_cut;
  summary[11] = n_modules_present; summary[12] = n_precut; summary[13] = n_postcut; summary[14] = n_emitted;
  summary[15] = flags;
  return 0;
}

// ---- RecHits-lite ("The RecHits module estimates the 3D position of each
// cluster forming hits"; only the module-local part is computable here: geometry conditions are missing).
// Readings S25-S28 of DESIGN.md: one hit per emitted cluster record, same index (the offsets are Fig. 3's
// fillHitsModuleStart); bounding box over the cluster's OK digis; local position in cm from the
// charge-weighted centroid with the module centre as origin and pitches 0.0100 cm (rows) x 0.0150 cm (columns),
// three separately rounded binary32 operations per coordinate; flags ON_EDGE | SPANS_ROC << 1 | SINGLE_PIXEL << 2.
// Inputs are one event's outputs of pixo_process.  Plain loops, no shared code with the CUDA path.
int pixo_rechits(uint32_t n_words, uint32_t M, const uint16_t* d_module, const uint16_t* d_row, const uint16_t* d_col,
                 const int32_t* d_clus, const uint8_t* d_status, const uint32_t* clus_module_start, uint32_t n_emitted,
                 const uint32_t* c_n_pix, const float* c_x_col, const float* c_y_row,
                 float* h_x_local, float* h_y_local, uint16_t* h_min_row, uint16_t* h_max_row, uint16_t* h_min_col,
                 uint16_t* h_max_col, uint8_t* h_flags) {
  for (uint32_t g = 0; g < n_emitted; ++g) { h_min_row[g] = 0xFFFF; h_max_row[g] = 0; h_min_col[g] = 0xFFFF; h_max_col[g] = 0; }
  for (uint32_t i = 0; i < n_words; ++i) {
    if (d_status[i] != ST_OK || d_clus[i] < 0) continue;
    const uint32_t m = d_module[i];
    if (m >= M) return 1;
    const uint32_t l = (uint32_t)d_clus[i];
    if (l >= clus_module_start[m + 1] - clus_module_start[m]) continue;  // beyond the per-module clamp: no record
    const uint32_t g = clus_module_start[m] + l;
    if (g >= n_emitted) continue;                                        // beyond the event capacity: no record
    if (d_row[i] < h_min_row[g]) h_min_row[g] = d_row[i];
    if (d_row[i] > h_max_row[g]) h_max_row[g] = d_row[i];
    if (d_col[i] < h_min_col[g]) h_min_col[g] = d_col[i];
    if (d_col[i] > h_max_col[g]) h_max_col[g] = d_col[i];
  }
  for (uint32_t g = 0; g < n_emitted; ++g) {
    volatile float fx = c_y_row[g] + 0.5f; fx = fx - 80.0f; fx = fx * 0.0100f;    // S27: local x runs along the rows
    volatile float fy = c_x_col[g] + 0.5f; fy = fy - 208.0f; fy = fy * 0.0150f;   //      local y along the columns
    h_x_local[g] = fx; h_y_local[g] = fy;
    uint8_t f = 0;
    if (h_min_row[g] == 0 || h_max_row[g] == ROWS - 1 || h_min_col[g] == 0 || h_max_col[g] == COLS - 1) f |= 1;  // ON_EDGE
    if ((h_min_row[g] < ROC_ROWS && h_max_row[g] >= ROC_ROWS) || h_min_col[g] / ROC_COLS != h_max_col[g] / ROC_COLS) f |= 2;  // SPANS_ROC
    if (c_n_pix[g] == 1) f |= 4;                                                                                   // SINGLE_PIXEL
    h_flags[g] = f;
  }
  return 0;
}

// ---- Legacy digi format and FED error words (PAPER.md:31 names "optional modules ... to convert
// the SoA to legacy data formats" and leaves them out; nothing about the format is in the paper).
// Readings S29-S31 of DESIGN.md.  Per word i of one event:
//   pdigi[i]  = row | col << 11 | adc << 22 for a decodable word (adc = the raw word's low byte), 0 otherwise      (S29)
//   raw_id[i] = module_raw_id[module] for a decodable word, 0 otherwise                                            (S30)
// Error list (S31): every word whose status is ERR_LINK / ERR_ROC / ERR_DCOL / ERR_PXID (padding words are not
// errors), in word order: the raw word, the FED block it sits in, the status code.  *n_errors is the true count;
// the list holds the first max_errors of them.
int pixo_legacy(uint32_t n_words, uint32_t n_feds, const uint32_t* words, const uint32_t* fed_offsets,
                const uint16_t* d_module, const uint16_t* d_row, const uint16_t* d_col, const uint8_t* d_status,
                const uint32_t* module_raw_id, uint32_t n_modules, uint32_t max_errors,
                uint32_t* pdigi, uint32_t* raw_id, uint32_t* err_word, uint16_t* err_fed, uint8_t* err_type, uint32_t* n_errors) {
  uint32_t ne = 0, fed = 0;
  for (uint32_t i = 0; i < n_words; ++i) {
    if (fed_offsets) while (fed + 1 < n_feds && i >= fed_offsets[fed + 1]) ++fed;
    const uint8_t st = d_status[i];
    if (st <= ST_DUP) {  // decodable: OK, CUT, BELOW_THRESHOLD, DUPLICATE
      if (d_module[i] >= n_modules) return 1;
      pdigi[i] = (uint32_t)d_row[i] | ((uint32_t)d_col[i] << 11) | ((words[i] & 255u) << 22);
      raw_id[i] = module_raw_id[d_module[i]];
    } else {
      pdigi[i] = 0; raw_id[i] = 0;
      if (st >= ST_ERR_LINK) {
        if (ne < max_errors) { err_word[ne] = words[i]; err_fed[ne] = (uint16_t)fed; err_type[ne] = st; }
        ++ne;
      }
    }
  }
  *n_errors = ne;
  return 0;
}

}  // extern "C"
