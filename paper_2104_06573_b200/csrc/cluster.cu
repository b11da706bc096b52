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

}  // namespace pix
