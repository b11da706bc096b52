// findrun.cu -- the warp-per-run cluster kernel: a4 findClus (S10, S13) and a5 sums / charge cut /
// renumber / temp records (S9, S14, S18) for the module runs the fused kernel (fused.cu) could not take
// because they do not fit its 256-word window ("clusters the pixels on each detector module").
//
// One warp per run, in two sizes: up to 512 words (15 KB of per-warp shared memory) and up to 1024 words (29 KB);
// the same phases as findclus.cu with a single run: stage + insert into the position hash (4 slots per bucket), duplicates,
// forward-neighbour lookups -> edge list (united whenever it fills) -> hook-and-descend unions, sums by
// shared atomics, dense root list, cut + renumber in digi order, temp records, final status / clus, counters.
// Longer runs, runs whose hash bucket neighbourhood overflows and charge sums beyond 32 bits go on to the block
// kernel (cluster.cu).  Nothing here is shared with oracle/.
#include "pix_common.cuh"
#include "pix_device.cuh"

namespace pix {

namespace {

constexpr uint32_t RECAP = 256;           // edge list entries
constexpr uint32_t EMPTY = 0xFFFFFFFFu, INVALID = 0xFFFFFFFFu;
constexpr uint32_t MARK_DUP = 0xFFFFFFFEu, MARK_BELOW = 0xFFFFFFFDu;
constexpr uint32_t Q_SAFE = 0xFFFFFFFFu / 415u;
// Two sizes of the kernel: RM = 512 words per run (15 KB of shared memory per warp, 2 warps per block) and
// RM = 1024 (29 KB, 1 warp per block).  Hash (pix_device.cuh): RM buckets of 4 slots; key: row (8) | col (9);
// slot: disp (2) | tag (17 - log2 RM) | digi (10) | below (1).
template <uint32_t RM> struct RK {
  static_assert(RM == 512 || RM == 1024, "run sizes");
  using PH = BucketHash<17, RM == 512 ? 9 : 10, 10>;
  static constexpr uint32_t RTAB = 4 * RM;
  static constexpr int WPB = RM == 512 ? 2 : 1;
};

template <uint32_t RM>
struct __align__(16) RunSmem {
  uint32_t tab[4 * RM];   // position hash; after the lookups: q = tab, np = tab + RM, sx = tab + 2 RM, sy = tab + 3 RM
  uint32_t dkey[RM];    // row << 9 | col, INVALID for an undecodable word
  uint32_t label[RM];   // union-find parent, or MARK_*
  uint32_t edge[RECAP];   // a | b << 16
  uint16_t chg[RM];     // charge; after the sums: local id of a root, or NO_ID
  uint16_t rlist[RM];   // roots in digi order
};

template <uint32_t RM>
__device__ __forceinline__ void unite_edges(RunSmem<RM>& s, uint32_t ne, uint32_t lane) {
  for (uint32_t i0 = 0u; i0 < ne; i0 += 32u) {  // warp-uniform trip count
    if (i0 + lane < ne) {
      const uint32_t e = s.edge[i0 + lane];
      hook(s.label, e & 0xFFFFu, e >> 16);
    }
    __syncwarp();
  }
}
template <uint32_t RM>
__global__ void __launch_bounds__(RK<RM>::WPB * 32) findrun_kernel(const __grid_constant__ Chunk c, const uint32_t* __restrict__ in_list, uint32_t ctl_count,
                                                                   uint32_t ctl_ticket, uint32_t* __restrict__ long_list, uint32_t ctl_long) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  RunSmem<RM>& s = reinterpret_cast<RunSmem<RM>*>(smem_raw)[warp];
  constexpr uint32_t RMAX = RM, RTAB = RK<RM>::RTAB;
  using PH = typename RK<RM>::PH;
  const uint32_t lt_mask = (1u << lane) - 1u;
  constexpr uint32_t FULL = 0xFFFFFFFFu, NO_ID = 0xFFFFu;
  uint32_t* const q = s.tab; uint32_t* const np = s.tab + RMAX; uint32_t* const sx = s.tab + 2 * RMAX;
  uint32_t* const sy = s.tab + 3 * RMAX;
  uint16_t* const lid = s.chg;
  uint32_t count = c.ctl[ctl_count];
  count = count < c.list_cap ? count : c.list_cap;
  const uint32_t gBeg = c.segB[0];

  while (true) {
    uint32_t ti = 0u;
    if (lane == 0) ti = atomicAdd(c.ctl + ctl_ticket, 1u);
    ti = __shfl_sync(FULL, ti, 0);
    if (ti >= count) break;
    const uint32_t task = in_list[ti];
    const uint32_t er = task / c.M, m = task - er * c.M;
    if (module_split(c, er, m)) continue;  // S11: the module has several runs; the event is not clustered
    const size_t mo = (size_t)(c.e0 + er) * c.M + m;
    const uint32_t first = c.module_first[mo], n = c.module_end[mo] - first;
    if (n > RMAX) {  // too long for this size of the kernel: the next one takes it
      if (lane == 0) {
        const uint32_t i = atomicAdd(c.ctl + ctl_long, 1u);
        if (i < c.list_cap) long_list[i] = task;  // a task moves down the lists at most once: they never overflow
      }
      continue;
    }
    const uint32_t gb = c.segB[er * c.F] + first;  // global index of the run's digi 0
    const uint32_t nk = (n + 31u) >> 5;
    {
      uint4* t4 = reinterpret_cast<uint4*>(s.tab);
      const uint4 e4 = make_uint4(EMPTY, EMPTY, EMPTY, EMPTY);
#pragma unroll
      for (int k = 0; k < (int)(RTAB / 4 / 32); ++k) t4[lane + 32 * k] = e4;
    }
    __syncwarp();
    // ---- stage + insert
    bool dup_seen = false, full_seen = false;
#pragma unroll 1
    for (uint32_t k = 0; k < nk; ++k) {
      const uint32_t t = 32u * k + lane;
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
    __syncwarp();
    if (__any_sync(FULL, full_seen)) {  // no room near a home bucket (dense run): the block kernel takes it
      if (lane == 0) { const uint32_t i = atomicAdd(c.ctl + CTL_OVF_COUNT, 1u); if (i < c.list_cap) c.ovf_list[i] = task; }
      continue;
    }
    // ---- duplicates (S10): the digi that is not in the slot
    if (__any_sync(FULL, dup_seen)) {
      for (uint32_t k = 0; k < nk; ++k) {
        const uint32_t t = 32u * k + lane, key = s.dkey[t];
        if (key != INVALID && PH::digi(PH::find(s.tab, PH::mix(key))) != t) s.label[t] = MARK_DUP;
      }
      __syncwarp();
    }
    // ---- forward neighbours (S13) -> edges -> unions
    uint32_t ne = 0u;
#pragma unroll 1
    for (uint32_t k = 0; k < nk; ++k) {
      const uint32_t t = 32u * k + lane, key = s.dkey[t];
      if (ne + 96u > RECAP) {  // the round's edges might not fit: unite what is listed (warp-uniform)
        __syncwarp();
        unite_edges(s, ne, lane);
        ne = 0u;
      }
      const bool live = key != INVALID && s.label[t] < RMAX;
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
      if (f0) s.edge[ne + __popc(m0 & lt_mask)] = t | (n0 << 16);
      ne += __popc(m0);
      if (f1) s.edge[ne + __popc(m1 & lt_mask)] = t | (n1 << 16);
      ne += __popc(m1);
      if (f2) s.edge[ne + __popc(m2 & lt_mask)] = t | (n2 << 16);
      ne += __popc(m2);
    }
    __syncwarp();
    unite_edges(s, ne, lane);
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {  // two pointer-jumping rounds: the chains shrink 4x before the sums
      for (uint32_t k = 0; k < nk; ++k) {
        const uint32_t t = 32u * k + lane;
        const uint32_t l = s.label[t];
        if (l < RMAX) { const uint32_t ll = s.label[l]; if (ll != l) s.label[t] = ll; }
      }
      __syncwarp();
    }
    __syncwarp();  // components complete; the hash is dead, its memory becomes q / np / sx / sy
    // ---- sums; dense list of the roots
    {
      uint4* t4 = reinterpret_cast<uint4*>(s.tab);
      const uint4 z4 = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
      for (int k = 0; k < (int)(RTAB / 4 / 32); ++k) t4[lane + 32 * k] = z4;
    }
    __syncwarp();
    uint32_t nr = 0u;
#pragma unroll 1
    for (uint32_t k = 0; k < nk; ++k) {
      const uint32_t t = 32u * k + lane;
      volatile uint32_t* L = s.label;
      uint32_t r = L[t];
      const bool live = r < RMAX;  // else MARK_*
      if (live) {
        while (true) { const uint32_t nx = L[r]; if (nx == r) break; r = nx; }
        L[t] = r;
        const uint32_t key = s.dkey[t], e = s.chg[t];
        atomicAdd(&q[r], e); atomicAdd(&np[r], 1u);
        atomicAdd(&sx[r], e * (key & 511u));
        atomicAdd(&sy[r], e * (key >> 9));
      }
      const bool root = live && r == t;
      const uint32_t rm = __ballot_sync(FULL, root);
      if (root) s.rlist[nr + __popc(rm & lt_mask)] = (uint16_t)t;  // digi order
      nr += __popc(rm);
    }
    __syncwarp();
    // ---- cut, renumber (S14: local id = rank among the surviving roots, in digi order), temp records (S18)
    uint32_t cnt = 0u;
    bool wrapped = false;
#pragma unroll 1
    for (uint32_t i0 = 0u; i0 < nr; i0 += 32u) {
      const bool valid = i0 + lane < nr;
      uint32_t t = 0u, Q = 0u;
      if (valid) { t = s.rlist[i0 + lane]; Q = q[t]; wrapped |= Q > Q_SAFE; }
      const bool surv = valid && (long long)Q >= (long long)c.cut;  // S9: equality keeps
      const uint32_t sm = __ballot_sync(FULL, surv);
      const uint32_t id = cnt + __popc(sm & lt_mask);
      if (valid) {
        if (surv) {
          const float fq = (float)Q;
          put_temp(c, (gb - gBeg) + id, first + t, np[t], Q, __fdividef((float)sx[t], fq), __fdividef((float)sy[t], fq));
        }
        lid[t] = surv ? (uint16_t)id : (uint16_t)NO_ID;
      }
      cnt += __popc(sm);
    }
    __syncwarp();
    if (__any_sync(FULL, wrapped)) {  // 32-bit weighted sums may have wrapped: the block kernel redoes the run
      if (lane == 0) { const uint32_t i = atomicAdd(c.ctl + CTL_OVF_COUNT, 1u); if (i < c.list_cap) c.ovf_list[i] = task; }
      continue;
    }
    // ---- final status and clus, counters
    uint32_t cntA = 0u, cntB = 0u;  // dup | below << 16 ; ok | cut << 16
#pragma unroll 1
    for (uint32_t k = 0; k < nk; ++k) {
      const uint32_t t = 32u * k + lane, key = s.dkey[t];
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
      c.n_clus[task] = cnt;
      uint32_t* ec = c.ev_cnt + (size_t)er * EC_STRIDE;
      if (a & 0xFFFFu) atomicAdd(ec + EC_DUP, a & 0xFFFFu);
      if (a >> 16) atomicAdd(ec + EC_BELOW, a >> 16);
      if (bb & 0xFFFFu) atomicAdd(ec + EC_OK, bb & 0xFFFFu);
      if (bb >> 16) atomicAdd(ec + EC_CUT, bb >> 16);
      if (nr) atomicAdd(ec + EC_PRECUT, nr);
    }
    __syncwarp();  // shared state is rewritten by the next run
  }
}

}  // namespace

cudaError_t configure_findrun_kernel() {
  cudaError_t e = cudaFuncSetAttribute(findrun_kernel<512>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)(RK<512>::WPB * sizeof(RunSmem<512>)));
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(findrun_kernel<1024>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)(RK<1024>::WPB * sizeof(RunSmem<1024>)));
}

// runs of up to 512 words first (findclus's list); what is longer goes to the 1024-word size, then to the block kernel
void launch_findrun(const Chunk& c, int n_sm, cudaStream_t stream) {
  findrun_kernel<512><<<n_sm * 7, RK<512>::WPB * 32, RK<512>::WPB * sizeof(RunSmem<512>), stream>>>(
      c, c.mid_list, CTL_MID_COUNT, CTL_MID_TICKET, c.big_list, CTL_BIG_COUNT);
  findrun_kernel<1024><<<n_sm * 7, RK<1024>::WPB * 32, RK<1024>::WPB * sizeof(RunSmem<1024>), stream>>>(
      c, c.big_list, CTL_BIG_COUNT, CTL_BIG_TICKET, c.ovf_list, CTL_OVF_COUNT);
}

}  // namespace pix
