// findrun.cu -- the block-per-run cluster kernel: a4 findClus (S10, S13) and a5 sums / charge cut /
// renumber / temp records (S9, S14, S18) for the module runs the fused kernel (fused.cu) could not take because
// they do not fit its 256-word window ("clusters the pixels on each detector module").
//
// One block per run, several warps sharing the run's tables (PU200-like events: 74 k such runs per 200 events, so
// the grid is full of blocks and the barriers between the phases are hidden by the other blocks of the SM).
// Two sizes: up to 512 words (4 warps, 15 KB of shared memory) and up to 1024 words (8 warps, 30 KB).  The phases
// are those of the fused kernel with a single run: stage + insert into the position hash (4 slots per bucket),
// duplicates, forward-neighbour lookups -> edge list -> hook-and-descend unions (one round of digis at a time),
// sums by shared atomics, cut + renumber in digi order through a survivor bitmap, temp records, final status /
// clus, counters.  Longer runs, runs whose hash bucket neighbourhood overflows and charge sums beyond 32 bits go
// on to the generic block kernel (cluster.cu).  Nothing here is shared with oracle/.
#include "pix_common.cuh"
#include "pix_device.cuh"

namespace pix {

namespace {

constexpr uint32_t EMPTY = 0xFFFFFFFFu, INVALID = 0xFFFFFFFFu;
constexpr uint32_t MARK_DUP = 0xFFFFFFFEu, MARK_BELOW = 0xFFFFFFFDu;
constexpr uint32_t Q_SAFE = 0xFFFFFFFFu / 415u;
constexpr uint32_t FL_DUP = 1u, FL_FULL = 2u, FL_WRAP = 4u;
// RM words per run.  Hash (pix_device.cuh): RM buckets of 4 slots; key: row (8) | col (9);
// slot: disp (2) | tag (17 - log2 RM) | digi (10) | below (1).
template <uint32_t RM> struct RK {
  static_assert(RM == 512 || RM == 1024, "run sizes");
  using PH = BucketHash<17, RM == 512 ? 9 : 10, 10>;
  static constexpr uint32_t RTAB = 4 * RM;
  static constexpr int NW = RM == 512 ? 4 : 8, NT = NW * 32;
  static constexpr uint32_t RECAP = 3 * NT;  // a round of NT digis lists at most three edges each
};

template <uint32_t RM>
struct __align__(16) RunSmem {
  uint32_t tab[4 * RM];   // position hash; after the lookups: q = tab, np = tab + RM, sx = tab + 2 RM, sy = tab + 3 RM
  uint32_t dkey[RM];      // row << 9 | col, INVALID for an undecodable word
  uint32_t label[RM];     // union-find parent, or MARK_*
  uint32_t edge[RK<RM>::RECAP];  // a | b << 16
  uint16_t chg[RM];       // charge; after the sums: local id of a root, or NO_ID
  uint32_t bits[RM / 32]; // roots that survive the cut, one bit per digi
  uint32_t wpre[RM / 32]; // survivors before each word of bits
  uint32_t ne[2];         // edges listed in this round / the next one
  uint32_t task, flags, n_surv, n_roots;
  uint32_t tbase, pad2[3];  // the run's stretch of the temp record area
  uint32_t cnt[4];        // dup, below, ok, cut
  uint32_t pad[2];
};

template <uint32_t RM>
__global__ void __launch_bounds__(RK<RM>::NT) findrun_kernel(const __grid_constant__ Chunk c, const uint32_t* __restrict__ in_list, uint32_t ctl_count,
                                                             uint32_t ctl_ticket, uint32_t* __restrict__ long_list, uint32_t ctl_long) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  RunSmem<RM>& s = *reinterpret_cast<RunSmem<RM>*>(smem_raw);
  using PH = typename RK<RM>::PH;
  constexpr uint32_t RTAB = RK<RM>::RTAB, NT = RK<RM>::NT;
  const uint32_t tid = threadIdx.x, lane = tid & 31u;
  const uint32_t lt_mask = (1u << lane) - 1u;
  constexpr uint32_t FULL = 0xFFFFFFFFu, NO_ID = 0xFFFFu;
  uint32_t* const q = s.tab; uint32_t* const np = s.tab + RM; uint32_t* const sx = s.tab + 2 * RM;
  uint32_t* const sy = s.tab + 3 * RM;
  uint16_t* const lid = s.chg;
  uint32_t count = c.ctl[ctl_count];
  count = count < c.list_cap ? count : c.list_cap;
  const uint32_t gBeg = c.segB[0];

  while (true) {
    __syncthreads();  // the previous run is done with the shared tables
    if (tid == 0) {
      s.task = atomicAdd(c.ctl + ctl_ticket, 1u);
      s.ne[0] = s.ne[1] = 0u; s.flags = 0u; s.n_surv = 0u; s.n_roots = 0u;
      s.cnt[0] = s.cnt[1] = s.cnt[2] = s.cnt[3] = 0u;
    }
    __syncthreads();
    const uint32_t ti = s.task;
    if (ti >= count) break;
    const uint32_t task = in_list[ti];
    const uint32_t er = task / c.M, m = task - er * c.M;
    if (module_split(c, er, m)) continue;  // S11: the module has several runs; the event is not clustered
    const size_t mo = (size_t)(c.e0 + er) * c.M + m;
    const uint32_t first = c.module_first[mo], n = c.module_end[mo] - first;
    if (n > RM) {  // too long for this size of the kernel: the next one takes it
      if (tid == 0) {
        const uint32_t i = atomicAdd(c.ctl + ctl_long, 1u);
        if (i < c.list_cap) long_list[i] = task;  // a task moves down the lists at most once: they never overflow
      }
      continue;
    }
    const uint32_t gb = c.segB[er * c.F] + first;  // global index of the run's digi 0
    const uint32_t nk = (n + NT - 1u) / NT;        // rounds of NT digis; nk * NT <= RM
    {
      uint4* t4 = reinterpret_cast<uint4*>(s.tab);
      const uint4 e4 = make_uint4(EMPTY, EMPTY, EMPTY, EMPTY);
      for (uint32_t i = tid; i < RTAB / 4; i += NT) t4[i] = e4;
      if (tid < RM / 32) s.bits[tid] = 0u;
    }
    __syncthreads();
    // ---- stage + insert
    bool dup_seen = false, full_seen = false;
#pragma unroll 1
    for (uint32_t k = 0; k < nk; ++k) {
      const uint32_t t = NT * k + tid;
      const bool in = t < n;
      const uint32_t row = in ? (uint32_t)c.d_row[gb + t] : 0xFFFFu, col = in ? (uint32_t)c.d_col[gb + t] : 0u;
      const int32_t e = in ? c.d_charge[gb + t] : 0;
      const bool dec = row != 0xFFFFu, below = e < c.thr;  // S9
      const uint32_t dk = dec ? ((row << 9) | col) : INVALID;
      s.dkey[t] = dk;
      s.label[t] = (dec && !below) ? t : MARK_BELOW;
      s.chg[t] = (uint16_t)e;
      if (dec) {
        const uint32_t ins = PH::insert(s.tab, dk, t, below ? 1u : 0u);
        dup_seen |= ins == 1u; full_seen |= ins == 2u;
      }
    }
    if (dup_seen) atomicOr(&s.flags, FL_DUP);
    if (full_seen) atomicOr(&s.flags, FL_FULL);
    __syncthreads();
    if (s.flags & FL_FULL) {  // no room near a home bucket (dense run): the generic block kernel takes it
      if (tid == 0) { const uint32_t i = atomicAdd(c.ctl + CTL_OVF_COUNT, 1u); if (i < c.list_cap) c.ovf_list[i] = task; }
      continue;
    }
    // ---- duplicates (S10): the digi that is not in the slot
    if (s.flags & FL_DUP) {
      for (uint32_t k = 0; k < nk; ++k) {
        const uint32_t t = NT * k + tid, key = s.dkey[t];
        if (key != INVALID && PH::digi(PH::find(s.tab, PH::mix(key))) != t) s.label[t] = MARK_DUP;
      }
      __syncthreads();
    }
    // ---- forward neighbours (S13) -> edges -> unions, one round of NT digis at a time
#pragma unroll 1
    for (uint32_t k = 0; k < nk; ++k) {
      const uint32_t t = NT * k + tid, key = s.dkey[t];
      const bool live = key != INVALID && s.label[t] < RM;
      bool f0 = false, f1 = false, f2 = false;
      uint32_t n0 = 0, n1 = 0, n2 = 0;
      if (live) {
        const uint32_t h = PH::mix(key);
        const uint32_t eE = PH::find(s.tab, PH::step(h, 1u)), eS = PH::find(s.tab, PH::step(h, 512u));
        const uint32_t eSW = PH::find(s.tab, PH::step(h, 511u)), eSE = PH::find(s.tab, PH::step(h, 513u));
        const bool hS = PH::live(eS);
        f0 = PH::live(eE); n0 = PH::digi(eE);
        f1 = hS || PH::live(eSW); n1 = PH::digi(hS ? eS : eSW);
        f2 = !hS && !f0 && PH::live(eSE); n2 = PH::digi(eSE);  // with E live, SE is E's S: E joins it
      }
      const uint32_t m0 = __ballot_sync(FULL, f0), m1 = __ballot_sync(FULL, f1), m2 = __ballot_sync(FULL, f2);
      const uint32_t c0 = __popc(m0), c1 = __popc(m1), c2 = __popc(m2);
      uint32_t base = 0u;
      if (lane == 0 && c0 + c1 + c2) base = atomicAdd(&s.ne[k & 1u], c0 + c1 + c2);  // the warp's slice of the edge list
      base = __shfl_sync(FULL, base, 0);
      if (f0) s.edge[base + __popc(m0 & lt_mask)] = t | (n0 << 16);
      if (f1) s.edge[base + c0 + __popc(m1 & lt_mask)] = t | (n1 << 16);
      if (f2) s.edge[base + c0 + c1 + __popc(m2 & lt_mask)] = t | (n2 << 16);
      __syncthreads();
      const uint32_t ne = s.ne[k & 1u];
      if (tid == 0) s.ne[(k + 1u) & 1u] = 0u;  // last read before this barrier, next used after the one below
      for (uint32_t i = tid; i < ne; i += NT) {
        const uint32_t e = s.edge[i];
        hook(s.label, e & 0xFFFFu, e >> 16);
      }
      __syncthreads();
    }
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {  // two pointer-jumping rounds: the chains shrink 4x before the sums
      for (uint32_t k = 0; k < nk; ++k) {
        const uint32_t t = NT * k + tid;
        const uint32_t l = s.label[t];
        if (l < RM) { const uint32_t ll = s.label[l]; if (ll != l) s.label[t] = ll; }
      }
      __syncthreads();
    }
    // ---- sums (the hash is dead, its memory becomes q / np / sx / sy)
    {
      uint4* t4 = reinterpret_cast<uint4*>(s.tab);
      const uint4 z4 = make_uint4(0u, 0u, 0u, 0u);
      for (uint32_t i = tid; i < RTAB / 4; i += NT) t4[i] = z4;
    }
    __syncthreads();
#pragma unroll 1
    for (uint32_t k = 0; k < nk; ++k) {
      const uint32_t t = NT * k + tid;
      volatile uint32_t* L = s.label;
      uint32_t r = L[t];
      if (r < RM) {  // live, else MARK_*
        while (true) { const uint32_t nx = L[r]; if (nx == r) break; r = nx; }
        L[t] = r;
        const uint32_t key = s.dkey[t], e = s.chg[t];
        atomicAdd(&q[r], e); atomicAdd(&np[r], 1u);
        atomicAdd(&sx[r], e * (key & 511u));
        atomicAdd(&sy[r], e * (key >> 9));
      }
    }
    __syncthreads();
    // ---- cut (S9: equality keeps): the roots that survive set their bit
    {
      uint32_t nroot = 0u;
      bool wrapped = false;
#pragma unroll 1
      for (uint32_t k = 0; k < nk; ++k) {
        const uint32_t t = NT * k + tid;
        const bool root = s.label[t] == t;  // MARK_* never equals t
        const uint32_t Q = root ? q[t] : 0u;
        wrapped |= Q > Q_SAFE;
        const bool surv = root && (long long)Q >= (long long)c.cut;
        const uint32_t sm = __ballot_sync(FULL, surv);
        if (lane == 0) s.bits[t >> 5] = sm;  // t >> 5 is the warp's own word of this round
        nroot += root ? 1u : 0u;
      }
      nroot = __reduce_add_sync(FULL, nroot);
      if (lane == 0 && nroot) atomicAdd(&s.n_roots, nroot);
      if (wrapped) atomicOr(&s.flags, FL_WRAP);
    }
    __syncthreads();
    if (tid < 32) {  // survivors before each word of the bitmap
      uint32_t tot = 0u;
      for (uint32_t w0 = 0; w0 < RM / 32; w0 += 32u) {
        const uint32_t v = w0 + lane < RM / 32 ? __popc(s.bits[w0 + lane]) : 0u;
        uint32_t inc = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
          const uint32_t o = __shfl_up_sync(FULL, inc, d);
          if (lane >= (uint32_t)d) inc += o;
        }
        if (w0 + lane < RM / 32) s.wpre[w0 + lane] = tot + inc - v;
        tot += __shfl_sync(FULL, inc, 31);
      }
      if (lane == 0) s.n_surv = tot;
    }
    __syncthreads();
    if (s.flags & FL_WRAP) {  // 32-bit weighted sums may have wrapped: the generic block kernel redoes the run
      if (tid == 0) { const uint32_t i = atomicAdd(c.ctl + CTL_OVF_COUNT, 1u); if (i < c.list_cap) c.ovf_list[i] = task; }
      continue;
    }
    if (tid == 0) s.tbase = alloc_temp(c, s.n_surv);  // after the check above: a run is allotted by the kernel that finishes it
    __syncthreads();
    // ---- renumber (S14: local id = rank among the surviving roots, in digi order), temp records (S18)
#pragma unroll 1
    for (uint32_t k = 0; k < nk; ++k) {
      const uint32_t t = NT * k + tid;
      if (s.label[t] == t) {
        uint32_t id = NO_ID;
        const uint32_t w = s.bits[t >> 5];
        if (w >> (t & 31u) & 1u) {
          id = s.wpre[t >> 5] + __popc(w & ((1u << (t & 31u)) - 1u));
          const uint32_t Q = q[t];
          const float fq = (float)Q;
          put_temp(c, s.tbase + id, first + t, np[t], Q, __fdividef((float)sx[t], fq), __fdividef((float)sy[t], fq));
        }
        lid[t] = (uint16_t)id;
      }
    }
    __syncthreads();
    // ---- final status and clus, counters
    uint32_t cntA = 0u, cntB = 0u;  // dup | below << 16 ; ok | cut << 16
#pragma unroll 1
    for (uint32_t k = 0; k < nk; ++k) {
      const uint32_t t = NT * k + tid, key = s.dkey[t];
      if (key == INVALID) continue;
      const uint32_t lab = s.label[t];
      uint32_t so; int32_t cl = -1;
      if (lab == MARK_DUP) { so = ST_DUP; cntA += 1u; }
      else if (lab == MARK_BELOW) { so = ST_BELOW; cntA += 0x10000u; }
      else {
        const uint32_t id = lid[lab];
        if (id != NO_ID) { so = ST_OK; cl = (int32_t)id; cntB += 1u; } else { so = ST_CUT; cntB += 0x10000u; }
      }
      c.d_status[gb + t] = (uint8_t)so; c.d_clus[gb + t] = cl;
    }
    const uint32_t a = __reduce_add_sync(FULL, cntA), bb = __reduce_add_sync(FULL, cntB);
    if (lane == 0) {
      if (a & 0xFFFFu) atomicAdd(&s.cnt[0], a & 0xFFFFu);
      if (a >> 16) atomicAdd(&s.cnt[1], a >> 16);
      if (bb & 0xFFFFu) atomicAdd(&s.cnt[2], bb & 0xFFFFu);
      if (bb >> 16) atomicAdd(&s.cnt[3], bb >> 16);
    }
    __syncthreads();
    if (tid == 0) {
      c.n_clus[task] = s.n_surv; c.t_base[task] = s.tbase;
      uint32_t* ec = c.ev_cnt + (size_t)er * EC_STRIDE;
      if (s.cnt[0]) atomicAdd(ec + EC_DUP, s.cnt[0]);
      if (s.cnt[1]) atomicAdd(ec + EC_BELOW, s.cnt[1]);
      if (s.cnt[2]) atomicAdd(ec + EC_OK, s.cnt[2]);
      if (s.cnt[3]) atomicAdd(ec + EC_CUT, s.cnt[3]);
      if (s.n_roots) atomicAdd(ec + EC_PRECUT, s.n_roots);
    }
  }
}

}  // namespace

cudaError_t configure_findrun_kernel() {
  cudaError_t e = cudaFuncSetAttribute(findrun_kernel<512>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(RunSmem<512>));
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(findrun_kernel<1024>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(RunSmem<1024>));
}

// runs of up to 512 words first (the fused kernel's list); what is longer goes to the 1024-word size, then to the
// generic block kernel
void launch_findrun(const Chunk& c, int n_sm, cudaStream_t stream) {
  findrun_kernel<512><<<n_sm * 14, RK<512>::NT, sizeof(RunSmem<512>), stream>>>(
      c, c.mid_list, CTL_MID_COUNT, CTL_MID_TICKET, c.big_list, CTL_BIG_COUNT);
  findrun_kernel<1024><<<n_sm * 7, RK<1024>::NT, sizeof(RunSmem<1024>), stream>>>(
      c, c.big_list, CTL_BIG_COUNT, CTL_BIG_TICKET, c.ovf_list, CTL_OVF_COUNT);
}

}  // namespace pix
