// cluster.cu -- the overflow kernel: a4 findClus fused with a5 (cluster sums, charge cut, renumber, temp records)
// for the module runs the tile kernel (tile.cu) could not take: runs longer than a tile (1024 words), items whose
// position hash overflowed, charge sums beyond 32 bits.  One block per run, tables in the global workspace, 64-bit sums.
//
// "clusters the pixels on each detector module".  The connectivity rule, the duplicate rule,
// the canonical numbering and the charge cut are DESIGN.md readings S9, S10, S13, S14, S18.
//
// One task = one (event, module) run [first, end) of digis.  Per task:
//   0  clear the position hash (2n slots)
//   1  stage (position, charge) of every digi; insert decodable digis into the hash keyed by
//      row*416+col; equal keys keep the MIN digi index (S10: first index wins)
//   2  a digi that is not the owner of its position is a DUPLICATE
//   3  every live digi (owner, charge >= threshold) looks up its 4 forward neighbours
//      (r,c+1) (r+1,c-1) (r+1,c) (r+1,c+1) and unites with live owners: representatives with pointer jumping, the
//      larger root hooked under the smaller by compare-and-swap (unite_roots, pix_device.cuh) => the root is the
//      component's min digi index
//   4  flatten labels; add charge, pixel count and charge-weighted col/row into the root's accumulators (the 64-bit
//      sums in shared memory as two 32-bit halves: add_weighted)
//   5  roots in digi order: Q >= cut survives and takes the next local id (ballot/popc scan); the root
//      writes the temp record at (run first + id)
//   6  per digi: final status and clus; per task: counts
// The digi fields (row, col, charge) are read back from the output arrays the decode kernel has written.
#include <cstdio>
#include <mutex>

#include "../../include/pixclus.h"
#include "pix_common.cuh"
#include "pix_device.cuh"

namespace pix {

namespace {

constexpr uint32_t LIVE = 0x80000000u, KEYMASK = 0x0001FFFFu, NOPOS = 0xFFFFFFFFu;
constexpr uint32_t HASH_MUL = 0x9E3779B1u;  // linear-probing table of 2n slots (sized per run, unlike the bucket hash)

// ------------------------------------------------------------------ hash slots
template <typename SlotT> struct SlotOps;
template <> struct SlotOps<uint32_t> {  // key 17 bits | index 15 bits  (n <= 32767)
  static constexpr uint32_t EMPTY = 0xFFFFFFFFu;
  static __device__ __forceinline__ uint32_t pack(uint32_t key, uint32_t k) { return (key << 15) | k; }
  static __device__ __forceinline__ uint32_t key(uint32_t v) { return v >> 15; }
  static __device__ __forceinline__ uint32_t idx(uint32_t v) { return v & 0x7FFFu; }
};
template <> struct SlotOps<unsigned long long> {
  static constexpr unsigned long long EMPTY = ~0ull;
  static __device__ __forceinline__ unsigned long long pack(uint32_t key, uint32_t k) {
    return ((unsigned long long)key << 32) | k;
  }
  static __device__ __forceinline__ uint32_t key(unsigned long long v) { return (uint32_t)(v >> 32); }
  static __device__ __forceinline__ uint32_t idx(unsigned long long v) { return (uint32_t)v; }
};

__device__ __forceinline__ uint32_t hash_slot(uint32_t key, uint32_t size) { return __umulhi(key * HASH_MUL, size); }

template <typename SlotT>
__device__ __forceinline__ void hash_insert(SlotT* tab, uint32_t size, uint32_t key, uint32_t k) {
  using O = SlotOps<SlotT>;
  const SlotT mine = O::pack(key, k);
  uint32_t s = hash_slot(key, size);
  while (true) {
    const SlotT old = atomicCAS(tab + s, O::EMPTY, mine);
    if (old == O::EMPTY) return;
    if (O::key(old) == key) { atomicMin(tab + s, mine); return; }  // same position: min index owns it (S10)
    if (++s == size) s = 0;
  }
}

// owner index of position `key`, or NO_INDEX
template <typename SlotT>
__device__ __forceinline__ uint32_t hash_find(const SlotT* tab, uint32_t size, uint32_t key) {
  using O = SlotOps<SlotT>;
  uint32_t s = hash_slot(key, size);
  while (true) {
    const SlotT v = tab[s];
    if (v == O::EMPTY) return NO_INDEX;
    if (O::key(v) == key) return O::idx(v);
    if (++s == size) s = 0;
  }
}

// ------------------------------------------------------------------ unions: unite_roots() of pix_device.cuh
// read-only walk to the root (step 4: own entries are being flattened concurrently, nobody else's may be written)
__device__ __forceinline__ uint32_t uf_root(const volatile uint32_t* L, uint32_t x) {
  uint32_t p = L[x];
  while (p != x) { x = p; p = L[x]; }
  return x;
}
// ------------------------------------------------------------------ groups
template <int THREADS>
struct BlockGroup {
  uint32_t* s_scan;  // [THREADS/32 + 1] shared scratch
  __device__ __forceinline__ uint32_t rank() const { return threadIdx.x; }
  __device__ __forceinline__ uint32_t size() const { return THREADS; }
  __device__ __forceinline__ void sync() const { __syncthreads(); }
  __device__ __forceinline__ uint32_t scan_flag(bool f, uint32_t& total) const {
    const uint32_t lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
    const uint32_t b = __ballot_sync(0xFFFFFFFFu, f);
    __syncthreads();  // previous use of s_scan is over
    if (lane == 0) s_scan[w] = __popc(b);
    __syncthreads();
    uint32_t base = 0, tot = 0;
#pragma unroll
    for (int q = 0; q < THREADS / 32; ++q) { const uint32_t v = s_scan[q]; if (q < (int)w) base += v; tot += v; }
    total = tot;
    return base + __popc(b & ((1u << lane) - 1u));
  }
  __device__ __forceinline__ uint32_t sum(uint32_t v) const {
    const uint32_t lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
    v = __reduce_add_sync(0xFFFFFFFFu, v);
    __syncthreads();
    if (lane == 0) s_scan[w] = v;
    __syncthreads();
    uint32_t tot = 0;
#pragma unroll
    for (int q = 0; q < THREADS / 32; ++q) tot += s_scan[q];
    return tot;
  }
};

// tables of one task
template <typename SlotT>
struct Tables {
  SlotT* tab;                 // [2n]
  uint32_t* pos;              // [n] key | LIVE, or NOPOS for undecodable words
  int32_t* chg;               // [n]
  uint32_t* label;            // [n]
  uint32_t* q;                // [n] charge sum of the root; after step 5: local id or NO_INDEX
  uint32_t* npix;             // [n]
  unsigned long long* sx;     // [n] sum charge*col
  unsigned long long* sy;     // [n] sum charge*row
};

// Charge-weighted sums (64 bits).  In shared memory a 64-bit atomicAdd is a compare-and-swap loop, and the hundreds of
// pixels of a long cluster all add to one root: there the two halves of the word take the low 16 bits and the rest of
// every addend (< 2^25) by 32-bit atomics, exact for up to 65536 addends.  In the global workspace: one 64-bit atomic.
template <bool SPLIT>
__device__ __forceinline__ void add_weighted(unsigned long long* a, uint32_t v) {
  if (SPLIT) {
    uint32_t* h = reinterpret_cast<uint32_t*>(a);
    atomicAdd(h, v & 0xFFFFu); atomicAdd(h + 1, v >> 16);
  } else {
    atomicAdd(a, (unsigned long long)v);
  }
}
template <bool SPLIT>
__device__ __forceinline__ unsigned long long weighted_sum(const unsigned long long* a) {
  if (SPLIT) {
    const uint32_t* h = reinterpret_cast<const uint32_t*>(a);
    return (unsigned long long)h[0] + ((unsigned long long)h[1] << 16);
  }
  return *a;
}

// ------------------------------------------------------------------ the task
template <typename G, typename SlotT, bool STAGE_CHARGE>
__device__ __forceinline__ void cluster_task(const Chunk& c, const G& g, const Tables<SlotT>& T, uint32_t task) {
  using O = SlotOps<SlotT>;
  const uint32_t er = task / c.M, m = task - er * c.M;
  const size_t mo = (size_t)(c.e0 + er) * c.M + m;
  const uint32_t first = c.module_first[mo], n = c.module_end[mo] - first;
  const uint32_t ebase = c.segB[er * c.F];           // global index of the event's word 0
  const size_t gb = (size_t)ebase + first;           // global index of the run's digi 0
  const uint32_t rb = ebase - c.segB[0] + first;     // chunk-relative index of the run's digi 0
  const uint32_t size = 2u * n;
  const uint32_t rk = g.rank(), gs = g.size();

  // 0: clear
  for (uint32_t s = rk; s < size; s += gs) T.tab[s] = O::EMPTY;
  g.sync();
  // 1: stage + insert
  for (uint32_t k = rk; k < n; k += gs) {
    const uint32_t row = c.d_row[gb + k], col = c.d_col[gb + k];
    const int32_t e = c.d_charge[gb + k];
    uint32_t p = NOPOS;
    if (row != 0xFFFFu) {
      const uint32_t key = row * COLS + col;
      p = key | (e >= c.thr ? LIVE : 0u);
      hash_insert(T.tab, size, key, k);
    }
    T.pos[k] = p;
    if (STAGE_CHARGE) T.chg[k] = e;
    T.label[k] = k; T.q[k] = 0u; T.npix[k] = 0u; T.sx[k] = 0ull; T.sy[k] = 0ull;
  }
  g.sync();
  // 2: duplicates
  uint32_t n_dup = 0, n_below = 0;
  for (uint32_t k = rk; k < n; k += gs) {
    const uint32_t p = T.pos[k];
    if (p == NOPOS) continue;
    if (hash_find(T.tab, size, p & KEYMASK) != k) { T.pos[k] = (p & KEYMASK) | 0x40000000u; ++n_dup; }  // not live
    else if (!(p & LIVE)) ++n_below;
  }
  g.sync();
  // 3: unions over forward neighbours (S13: max(|drow|,|dcol|) == 1, no wrap)
  for (uint32_t k = rk; k < n; k += gs) {
    const uint32_t p = T.pos[k];
    if (p == NOPOS || !(p & LIVE)) continue;
    const uint32_t key = p & KEYMASK;
    const uint32_t row = key / COLS, col = key - row * COLS;
    const bool right = col + 1u < COLS, left = col > 0u, down = row + 1u < ROWS;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const bool ok = q == 0 ? right : (q == 1 ? (down && left) : (q == 2 ? down : (down && right)));
      if (!ok) continue;
      const uint32_t nkey = q == 0 ? key + 1u : key + COLS + (uint32_t)(q - 2);
      const uint32_t j = hash_find(T.tab, size, nkey);
      if (j == NO_INDEX) continue;
      if (!(((volatile uint32_t*)T.pos)[j] & LIVE)) continue;
      unite_roots(T.label, k, j);  // (long clusters are why a run ends up here: not hook-and-descend)
    }
  }
  g.sync();
  // 4: flatten + accumulate
  for (uint32_t k = rk; k < n; k += gs) {
    const uint32_t p = T.pos[k];
    if (p == NOPOS || !(p & LIVE)) continue;
    const uint32_t r = uf_root(T.label, k);
    T.label[k] = r;
    const uint32_t key = p & KEYMASK;
    const uint32_t row = key / COLS, col = key - row * COLS;
    const uint32_t e = (uint32_t)(STAGE_CHARGE ? T.chg[k] : c.d_charge[gb + k]);
    atomicAdd(T.q + r, e);
    atomicAdd(T.npix + r, 1u);
    add_weighted<STAGE_CHARGE>(T.sx + r, e * col);
    add_weighted<STAGE_CHARGE>(T.sy + r, e * row);
  }
  g.sync();
  // 5: roots in digi order -> local ids (S14), temp records (S18) in a stretch of n slots of the temp area
  if (rk == 0) g.s_scan[0] = alloc_temp(c, n);
  g.sync();
  const uint32_t tbase = g.s_scan[0];
  uint32_t n_pre = 0, n_post = 0;
  for (uint32_t k0 = 0; k0 < n; k0 += gs) {
    const uint32_t k = k0 + rk;
    bool root = false, surv = false;
    uint32_t Q = 0;
    if (k < n) {
      const uint32_t p = T.pos[k];
      root = p != NOPOS && (p & LIVE) && T.label[k] == k;
      if (root) { Q = T.q[k]; surv = (long long)Q >= (long long)c.cut; }  // S9: equality keeps
    }
    uint32_t tot_pre, tot_post;
    (void)g.scan_flag(root, tot_pre);
    const uint32_t id = n_post + g.scan_flag(surv, tot_post);
    if (root) {
      if (surv) {
        put_temp(c, tbase + id, first + k, T.npix[k], Q, (float)((double)weighted_sum<STAGE_CHARGE>(T.sx + k) / (double)Q),
                 (float)((double)weighted_sum<STAGE_CHARGE>(T.sy + k) / (double)Q));
      }
      T.q[k] = surv ? id : NO_INDEX;
    }
    n_pre += tot_pre; n_post += tot_post;
  }
  g.sync();
  // 6: final status and clus of every decodable digi (undecodable ones were finished by the decode kernel)
  uint32_t n_ok = 0, n_cut = 0;
  for (uint32_t k = rk; k < n; k += gs) {
    const uint32_t p = T.pos[k];
    if (p == NOPOS) {
      if (!STAGE_CHARGE) c.d_clus[gb + k] = -1;  // the labels lived in clus: restore the -1 of an undecodable word
      continue;
    }
    int32_t clus = -1;
    uint8_t st;
    if (p & LIVE) {
      const uint32_t id = T.q[T.label[k]];
      if (id != NO_INDEX) { clus = (int32_t)id; st = ST_OK; ++n_ok; } else { st = ST_CUT; ++n_cut; }
    } else {
      st = (p & 0x40000000u) ? ST_DUP : ST_BELOW;
    }
    c.d_clus[gb + k] = clus;
    c.d_status[gb + k] = st;
  }
  n_dup = g.sum(n_dup); n_below = g.sum(n_below); n_ok = g.sum(n_ok); n_cut = g.sum(n_cut);
  if (rk == 0) {
    c.n_clus[task] = n_post; c.t_base[task] = tbase;
    uint32_t* ec = c.ev_cnt + (size_t)er * EC_STRIDE;
    atomicAdd(ec + EC_PRECUT, n_pre); atomicAdd(ec + EC_DUP, n_dup); atomicAdd(ec + EC_BELOW, n_below);
    atomicAdd(ec + EC_OK, n_ok); atomicAdd(ec + EC_CUT, n_cut);
  }
}

// ------------------------------------------------------------------ kernel
// One block per run, taken from a task list by ticket.  Runs of up to CAP digis keep all their tables in shared
// memory; longer ones go to the next list (a larger size of this kernel) or, in the last size, use the global
// workspace.  One size is in use: 512 threads / 2048 digis (88 KB).
constexpr size_t SMEM_PER_DIGI = 8 + 8 + 2 * 4 + 4 * 5;  // sx, sy, 2 hash slots, pos, chg, label, q, npix

__device__ __forceinline__ Tables<uint32_t> carve(unsigned char* base, uint32_t cap) {
  Tables<uint32_t> T;
  T.sx = reinterpret_cast<unsigned long long*>(base); base += (size_t)cap * 8;
  T.sy = reinterpret_cast<unsigned long long*>(base); base += (size_t)cap * 8;
  T.tab = reinterpret_cast<uint32_t*>(base); base += (size_t)cap * 2 * 4;
  T.pos = reinterpret_cast<uint32_t*>(base); base += (size_t)cap * 4;
  T.chg = reinterpret_cast<int32_t*>(base); base += (size_t)cap * 4;
  T.label = reinterpret_cast<uint32_t*>(base); base += (size_t)cap * 4;
  T.q = reinterpret_cast<uint32_t*>(base); base += (size_t)cap * 4;
  T.npix = reinterpret_cast<uint32_t*>(base);
  return T;
}

template <int THREADS, uint32_t CAP>
__global__ void __launch_bounds__(THREADS) block_kernel(const __grid_constant__ Chunk c, const uint32_t* __restrict__ in_list,
                                                        uint32_t ctl_count, uint32_t ctl_ticket, uint32_t* __restrict__ long_list,
                                                        uint32_t ctl_long) {
  chain_begin();
  extern __shared__ __align__(16) unsigned char ovf_smem[];
  __shared__ uint32_t s_scan[THREADS / 32 + 1];
  __shared__ uint32_t s_task;
  const BlockGroup<THREADS> g{s_scan};
  uint32_t count = c.ctl[ctl_count];
  count = count < c.list_cap ? count : c.list_cap;
  while (true) {
    __syncthreads();
    if (threadIdx.x == 0) s_task = atomicAdd(c.ctl + ctl_ticket, 1u);
    __syncthreads();
    const uint32_t t = s_task;
    if (t >= count) break;
    const uint32_t task = in_list[t];
    const uint32_t er = task / c.M, m = task - er * c.M;
    if (module_split(c, er, m)) continue;  // S11: the module has several runs; the event is not clustered
    const uint32_t first = c.module_first[(size_t)(c.e0 + er) * c.M + m];
    const uint32_t n = c.module_end[(size_t)(c.e0 + er) * c.M + m] - first;
    if (n <= CAP) {
      cluster_task<BlockGroup<THREADS>, uint32_t, true>(c, g, carve(ovf_smem, CAP), task);
      continue;
    }
    if (long_list) {  // too long for this size of the kernel: the next one takes it (a task moves down the lists once)
      if (threadIdx.x == 0) {
        const uint32_t i = atomicAdd(c.ctl + ctl_long, 1u);
        if (i < c.list_cap) long_list[i] = task;
      }
      continue;
    }
    const uint32_t ebase = c.segB[er * c.F];
    const uint32_t rb = ebase - c.segB[0] + first;
    Tables<unsigned long long> T;
    T.tab = c.g_hash + 2 * (size_t)rb;
    T.pos = c.g_pos + rb; T.chg = nullptr;
    T.label = reinterpret_cast<uint32_t*>(c.d_clus + (size_t)ebase + first);  // clus is written last, per digi
    T.q = c.g_q + rb; T.npix = c.g_npix + rb; T.sx = c.g_sx + rb; T.sy = c.g_sy + rb;
    cluster_task<BlockGroup<THREADS>, unsigned long long, false>(c, g, T, task);
  }
}

constexpr int T_B = 512;
constexpr uint32_t CAP_B = 2048;

}  // namespace

cudaError_t configure_overflow_kernel() {
  return cudaFuncSetAttribute(block_kernel<T_B, CAP_B>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(CAP_B * SMEM_PER_DIGI));
}

// the runs the tile kernel left: longer than 1024 digis, hash overflow, or with 64-bit charge sums
void launch_overflow(const Chunk& c, int n_sm, cudaStream_t stream) {
  launch_chained(false, block_kernel<T_B, CAP_B>, n_sm * 2, T_B, CAP_B * SMEM_PER_DIGI, stream, c, (const uint32_t*)c.ovf_list, (uint32_t)CTL_OVF_COUNT, (uint32_t)CTL_OVF_TICKET, (uint32_t*)nullptr, 0u);
}


// ------------------------------------------------------------------ the entry point that allocates nothing
// pix_cluster_module_noalloc (include/pixclus.h): the global-workspace path of the kernel above for ONE module's
// decoded digis, for callers that cannot call cudaMalloc (no handle: pix_create allocates).  Its tables live in a
// file-scope device array of fixed size, which every GPU that loads the library holds until the process exits:
//   header (256 B) + per digi 16 B hash + 4 B position + 4 B charge sum + 4 B pixel count + 8 + 8 B weighted sums
//   + 20 B temp record = 256 B + 64 B x PIX_NOALLOC_MAX_DIGIS (16384) = 1 MiB + 256 B.
// In host code the array's name is a host-side stand-in, not a device address: pix_noalloc_setup asks
// cudaGetSymbolAddress for the address once per device and the launch passes pointers made from it.
// Every call uses the same array: the kernel clears what has to start at zero, and calls that overlap on the GPU
// (two streams, two threads) race.
namespace {

constexpr uint32_t NA_MAX = PIX_NOALLOC_MAX_DIGIS;
constexpr size_t NA_HDR = 256, NA_BYTES = NA_HDR + (size_t)NA_MAX * 64;
static __device__ __align__(256) unsigned char g_noalloc_scratch[NA_BYTES];

// header words (uint32)
enum { NH_FIRST = 0, NH_END = 1, NH_SEG = 2 /* 2 words */, NH_NCLUS = 4, NH_TBASE = 5, NH_EVCNT = 16 /* 16 */, NH_CTL = 32 /* 16 */ };

struct NoallocOut {
  uint32_t* first_digi; uint32_t* n_pix; uint32_t* charge; float* x_col; float* y_row; uint32_t* counts;
};

__global__ void __launch_bounds__(T_B) noalloc_kernel(const __grid_constant__ Chunk c, uint32_t* hdr, uint32_t n,
                                                      uint32_t max_clusters, NoallocOut o) {
  __shared__ uint32_t s_scan[T_B / 32 + 1];
  const BlockGroup<T_B> g{s_scan};
  // the array keeps the last call's contents: the header (run bounds, counters) is written afresh, the tables are
  // cleared or overwritten by the task itself (steps 0 and 1)
  if (threadIdx.x < NA_HDR / 4) hdr[threadIdx.x] = (threadIdx.x == NH_END || threadIdx.x == NH_SEG + 1) ? n : 0u;
  __syncthreads();
  Tables<unsigned long long> T;
  T.tab = c.g_hash; T.pos = c.g_pos; T.chg = nullptr;
  T.label = reinterpret_cast<uint32_t*>(c.d_clus);  // clus is written last, per digi
  T.q = c.g_q; T.npix = c.g_npix; T.sx = c.g_sx; T.sy = c.g_sy;
  cluster_task<BlockGroup<T_B>, unsigned long long, false>(c, g, T, 0u);
  __syncthreads();
  const uint32_t total = hdr[NH_NCLUS], tb = hdr[NH_TBASE];
  const uint32_t emit = total < max_clusters ? total : max_clusters;
  for (uint32_t i = threadIdx.x; i < emit; i += T_B) {  // temp records (in local-id order) -> the caller's arrays
    const uint4 a = c.t_a[tb + i];
    o.first_digi[i] = a.x; o.n_pix[i] = a.y; o.charge[i] = a.z; o.x_col[i] = __uint_as_float(a.w); o.y_row[i] = c.t_y[tb + i];
  }
  if (threadIdx.x == 0) {
    const uint32_t* ec = hdr + NH_EVCNT;
    o.counts[0] = total; o.counts[1] = emit; o.counts[2] = ec[EC_PRECUT]; o.counts[3] = ec[EC_DUP];
    o.counts[4] = ec[EC_BELOW]; o.counts[5] = ec[EC_OK]; o.counts[6] = ec[EC_CUT]; o.counts[7] = 0u;
  }
}

constexpr int NA_MAX_DEVICES = 64;
std::mutex g_noalloc_mu;
unsigned char* g_noalloc_addr[NA_MAX_DEVICES];  // device address of g_noalloc_scratch, per device ordinal
thread_local char g_noalloc_err[192];

int noalloc_fail(int code, const char* fmt, unsigned long long a, unsigned long long b) {
  snprintf(g_noalloc_err, sizeof(g_noalloc_err), fmt, a, b);
  return code;
}
int noalloc_fail(int code, const char* msg) {
  snprintf(g_noalloc_err, sizeof(g_noalloc_err), "%s", msg);
  return code;
}

// the scratch array's address on the current device (looked up on first use, with that device current)
int noalloc_address(unsigned char** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return noalloc_fail(PIX_ERR_CUDA, cudaGetErrorString(e));
  if (dev < 0 || dev >= NA_MAX_DEVICES) return noalloc_fail(PIX_ERR_INVALID_ARG, "device ordinal %llu beyond %llu", (unsigned long long)dev, NA_MAX_DEVICES);
  std::lock_guard<std::mutex> lock(g_noalloc_mu);
  if (!g_noalloc_addr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    if (e != cudaSuccess || !p) { cudaGetLastError(); return noalloc_fail(PIX_ERR_CUDA, e != cudaSuccess ? cudaGetErrorString(e) : "cudaGetSymbolAddress returned NULL"); }
    g_noalloc_addr[dev] = static_cast<unsigned char*>(p);
  }
  *out = g_noalloc_addr[dev];
  return PIX_OK;
}

}  // namespace

}  // namespace pix

extern "C" {

int pix_noalloc_setup(void) {
  pix::g_noalloc_err[0] = 0;
  unsigned char* p = nullptr;
  return pix::noalloc_address(&p);
}

const char* pix_noalloc_last_error(void) { return pix::g_noalloc_err; }

int pix_cluster_module_noalloc(void* cuda_stream, uint32_t n_digis, const uint16_t* row, const uint16_t* col, const int32_t* charge,
                               int32_t pixel_threshold_e, int32_t cluster_charge_cut_e, uint32_t max_clusters, int32_t* clus,
                               uint8_t* status, uint32_t* c_first_digi, uint32_t* c_n_pix, uint32_t* c_charge, float* c_x_col,
                               float* c_y_row, uint32_t* counts) {
  using namespace pix;
  g_noalloc_err[0] = 0;
  if (n_digis > NA_MAX)
    return noalloc_fail(PIX_ERR_CAPACITY, "n_digis %llu is beyond PIX_NOALLOC_MAX_DIGIS = %llu (the static scratch array)", n_digis, NA_MAX);
  if (!counts || (n_digis && (!row || !col || !charge || !clus || !status)))
    return noalloc_fail(PIX_ERR_INVALID_ARG, "NULL argument");
  if (max_clusters && (!c_first_digi || !c_n_pix || !c_charge || !c_x_col || !c_y_row))
    return noalloc_fail(PIX_ERR_INVALID_ARG, "NULL record array with max_clusters > 0");
  unsigned char* base = nullptr;
  if (int rc = noalloc_address(&base)) return rc;
  // the task's view of the scratch array: one event, one module, one run [0, n_digis)
  uint32_t* hdr = reinterpret_cast<uint32_t*>(base);
  unsigned char* q = base + NA_HDR;
  Chunk c = {};
  c.e0 = 0; c.e1 = 1; c.F = 1; c.M = 1; c.F_shift = 0;
  c.thr = pixel_threshold_e; c.cut = cluster_charge_cut_e;
  c.d_row = const_cast<uint16_t*>(row); c.d_col = const_cast<uint16_t*>(col); c.d_charge = const_cast<int32_t*>(charge);  // read only
  c.d_clus = clus; c.d_status = status;
  c.module_first = hdr + NH_FIRST; c.module_end = hdr + NH_END; c.segB = hdr + NH_SEG;
  c.n_clus = hdr + NH_NCLUS; c.t_base = hdr + NH_TBASE; c.ev_cnt = hdr + NH_EVCNT; c.ctl = hdr + NH_CTL;
  c.g_hash = reinterpret_cast<unsigned long long*>(q); q += (size_t)NA_MAX * 16;
  c.t_a = reinterpret_cast<uint4*>(q); q += (size_t)NA_MAX * 16;
  c.g_sx = reinterpret_cast<unsigned long long*>(q); q += (size_t)NA_MAX * 8;
  c.g_sy = reinterpret_cast<unsigned long long*>(q); q += (size_t)NA_MAX * 8;
  c.g_pos = reinterpret_cast<uint32_t*>(q); q += (size_t)NA_MAX * 4;
  c.g_q = reinterpret_cast<uint32_t*>(q); q += (size_t)NA_MAX * 4;
  c.g_npix = reinterpret_cast<uint32_t*>(q); q += (size_t)NA_MAX * 4;
  c.t_y = reinterpret_cast<float*>(q); q += (size_t)NA_MAX * 4;
  NoallocOut o{c_first_digi, c_n_pix, c_charge, c_x_col, c_y_row, counts};
  noalloc_kernel<<<1, T_B, 0, (cudaStream_t)cuda_stream>>>(c, hdr, n_digis, max_clusters, o);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return noalloc_fail(PIX_ERR_CUDA, cudaGetErrorString(e));
  return PIX_OK;
}

}  // extern "C"
