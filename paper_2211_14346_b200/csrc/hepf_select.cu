// hepf_select.cu — hepf_select: ordered cut chain + stable stream compaction.
//
// Paper: a cut is `bool f(event)`, cuts are registered in order and an event is dropped at the first false
// (PAPER.md:96-102, :286-295); the survivors are the filtered output.  §4 (:136): "eighteen
// cuts, organised in a sequential way, as a computational pipeline".
//
// B200 mapping: the chain is HBM-bound (<= 180 B of columns per event, a handful of compares), so
//   K1 select_eval   : one thread = two adjacent events, every needed column read with 128-bit loads that are
//                      all issued before the first use (>= 20 independent 16-byte loads in flight per thread);
//                      cuts evaluated from registers; __ballot_sync -> two 32-bit survivor masks per warp
//                      (even/odd events) written to the workspace; per-block survivor count; cutflow by
//                      ballot/popc + one atomicAdd per cut per block.
//   K2 select_scatter: each block sums the counts of the blocks before it (<= 1184 values), then replays its
//                      range from the 1-bit-per-event masks (1/1440 of K1's traffic) and writes the ascending
//                      index list with popc-prefix offsets.  Deterministic, no atomics on the index cursor.
// Each block owns a contiguous range of 512-event tiles; the grid is one wave of resident blocks (occupancy query: 2 per SM at 111 registers).
#include <mutex>

#include "hepf_common.cuh"

namespace hepf {

constexpr int SEL_THREADS = 256;
constexpr int SEL_TILE = SEL_THREADS * 2;   // events per block iteration
constexpr int SEL_WARPS = SEL_THREADS / 32;

enum : uint32_t { NEED_LEP_PT = 1, NEED_LEP_ETA = 2, NEED_JET_PT = 4, NEED_JET_ETA = 8, NEED_MET = 16, NEED_MLL = 32 };

struct CutChain {
  int n;
  uint32_t need;
  int rec_cut;            // position of the recording cut (HEPF_CUT_MET_GT_RECORD), -1 = none
  double rec_default;     // value of the derived column for events that do not pass it
  hepf_cut_t c[HEPF_MAX_CUTS];
};

struct SelCols {
  const double *lep_pt, *lep_eta, *jet_pt, *jet_eta, *met, *mll;
  const uint32_t* flags;
  int64_t n, stride;
};

__device__ __forceinline__ double2 ld2(const double* p) { return __ldcs(reinterpret_cast<const double2*>(p)); }
__device__ __forceinline__ double pick(const double2& v, int k) { return k ? v.y : v.x; }

__global__ void __launch_bounds__(SEL_THREADS)
select_eval_kernel(SelCols ev, CutChain chain, int64_t n_tiles, int64_t tiles_per_block, uint2* __restrict__ masks,
                   uint32_t* __restrict__ block_count, unsigned long long* __restrict__ cutflow, double* __restrict__ derived) {
  __shared__ unsigned int s_cf[HEPF_MAX_CUTS];
  __shared__ unsigned int s_count;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid < HEPF_MAX_CUTS) s_cf[tid] = 0;
  if (tid == 0) s_count = 0;
  __syncthreads();
  const int64_t t0 = (int64_t)blockIdx.x * tiles_per_block;
  const int64_t t1 = min(t0 + tiles_per_block, n_tiles);
  unsigned int my_cf = 0, my_count = 0;   // lane c accumulates cut c; lane 0 accumulates survivors
  for (int64_t t = t0; t < t1; t++) {
    const int64_t i0 = t * SEL_TILE + 2 * tid;            // first of this thread's two events
    bool pass[2] = {false, false};
    int fail_at[2] = {0, 0};                              // number of cuts passed
    if (i0 < ev.n) {                                      // i0 + 1 <= stride - 1 is always readable (stride even)
      const uint2 fl = __ldcs(reinterpret_cast<const uint2*>(ev.flags + i0));
      double2 lpt[2], leta[2], jpt[HEPF_N_JET], jeta[HEPF_N_JET], met, mll;
      // ---- issue every load the chain needs before any use -----------------------------------------------
      if (chain.need & NEED_LEP_PT) { lpt[0] = ld2(ev.lep_pt + i0); lpt[1] = ld2(ev.lep_pt + ev.stride + i0); }
      if (chain.need & NEED_LEP_ETA) { leta[0] = ld2(ev.lep_eta + i0); leta[1] = ld2(ev.lep_eta + ev.stride + i0); }
      if (chain.need & NEED_JET_PT) {
#pragma unroll
        for (int s = 0; s < HEPF_N_JET; s++) jpt[s] = ld2(ev.jet_pt + s * ev.stride + i0);
      }
      if (chain.need & NEED_JET_ETA) {
#pragma unroll
        for (int s = 0; s < HEPF_N_JET; s++) jeta[s] = ld2(ev.jet_eta + s * ev.stride + i0);
      }
      if (chain.need & NEED_MET) met = ld2(ev.met + i0);
      if (chain.need & NEED_MLL) mll = ld2(ev.mll + i0);
      // ---- evaluate the chain from registers ------------------------------------------------------------------
#pragma unroll
      for (int k = 0; k < 2; k++) {
        const uint32_t f = k ? fl.y : fl.x;
        const int n_lep = f & 15u, n_jet = min(8u, (f >> 8) & 15u);
        bool alive = (i0 + k) < ev.n;
        int passed = 0;
        for (int c = 0; c < chain.n && alive; c++) {
          const hepf_cut_t cut = chain.c[c];
          bool ok = false;
          switch (cut.kind) {
            case HEPF_CUT_NLEP_EQ: ok = n_lep == (int)cut.n; break;
            case HEPF_CUT_LEP_OS: ok = ((f >> 4) & 1u) != ((f >> 5) & 1u); break;
            case HEPF_CUT_LEP_PT_GT: ok = pick(lpt[0], k) > cut.lo && pick(lpt[1], k) > cut.lo; break;
            case HEPF_CUT_LEP_ABSETA_LT: ok = fabs(pick(leta[0], k)) < cut.hi && fabs(pick(leta[1], k)) < cut.hi; break;
            case HEPF_CUT_NJET_GE:
            case HEPF_CUT_NBJET_GE: {
              const uint32_t tagmask = cut.kind == HEPF_CUT_NBJET_GE ? (f >> 16) : 0xffu;
              int cnt = 0;
#pragma unroll
              for (int s = 0; s < HEPF_N_JET; s++)
                cnt += (s < n_jet) && ((tagmask >> s) & 1u) && pick(jpt[s], k) > cut.lo && fabs(pick(jeta[s], k)) < cut.hi;
              ok = cnt >= (int)cut.n;
            } break;
            case HEPF_CUT_MET_GT:
            case HEPF_CUT_MET_GT_RECORD: ok = pick(met, k) > cut.lo; break;
            case HEPF_CUT_MLL_GT: ok = pick(mll, k) > cut.lo; break;
            case HEPF_CUT_MLL_OUTSIDE: ok = pick(mll, k) < cut.lo || pick(mll, k) > cut.hi; break;
            default: ok = false;
          }
          alive = ok;
          passed += ok;
        }
        pass[k] = alive;
        fail_at[k] = passed;
      }
      // the recording cut's side effect ("ETmis = met_met; ETmis *= 1.05"): one rounded multiplication
      // for the events that passed the chain up to and including it, the default value for all others
      if (derived) {
        const double sc = chain.c[chain.rec_cut].hi;
        const double d0 = fail_at[0] > chain.rec_cut ? __dmul_rn(met.x, sc) : chain.rec_default;
        const double d1 = fail_at[1] > chain.rec_cut ? __dmul_rn(met.y, sc) : chain.rec_default;
        if (i0 + 1 < ev.n) __stcs(reinterpret_cast<double2*>(derived + i0), make_double2(d0, d1));
        else derived[i0] = d0;
      }
    }
    // ---- warp compaction: survivor masks (even events, odd events) ---------------------------------------------
    const unsigned b0 = __ballot_sync(0xffffffffu, pass[0]), b1 = __ballot_sync(0xffffffffu, pass[1]);
    if (lane == 0) {
      masks[t * SEL_WARPS + warp] = make_uint2(b0, b1);
      my_count += __popc(b0) + __popc(b1);
    }
    if (cutflow) {
      for (int c = 0; c < chain.n; c++) {
        const unsigned m0 = __ballot_sync(0xffffffffu, fail_at[0] > c), m1 = __ballot_sync(0xffffffffu, fail_at[1] > c);
        if (lane == c) my_cf += __popc(m0) + __popc(m1);
      }
    }
  }
  if (lane == 0 && my_count) atomicAdd(&s_count, my_count);
  if (cutflow && lane < chain.n && my_cf) atomicAdd(&s_cf[lane], my_cf);
  __syncthreads();
  if (tid == 0) block_count[blockIdx.x] = s_count;
  if (cutflow && tid < chain.n && s_cf[tid]) atomicAdd(&cutflow[tid], (unsigned long long)s_cf[tid]);
}

__global__ void __launch_bounds__(SEL_THREADS)
select_scatter_kernel(int64_t n_tiles, int64_t tiles_per_block, const uint2* __restrict__ masks,
                      const uint32_t* __restrict__ block_count, uint32_t* __restrict__ out_idx,
                      int64_t* __restrict__ out_count) {
  __shared__ unsigned long long s_part[SEL_WARPS];
  __shared__ unsigned int s_wcount[SEL_WARPS];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  // exclusive offset of this block = sum of the counts of the blocks before it (grid <= ~1.2k blocks)
  unsigned long long part = 0;
  const int upto = (blockIdx.x == 0) ? gridDim.x : blockIdx.x;   // block 0 also produces the grand total
  for (int b = tid; b < upto; b += SEL_THREADS) part += block_count[b];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
  if (lane == 0) s_part[warp] = part;
  __syncthreads();
  unsigned long long base = 0;
#pragma unroll
  for (int w = 0; w < SEL_WARPS; w++) base += s_part[w];
  if (blockIdx.x == 0) {
    if (tid == 0) *out_count = (int64_t)base;
    base = 0;
  }
  const int64_t t0 = (int64_t)blockIdx.x * tiles_per_block;
  const int64_t t1 = min(t0 + tiles_per_block, n_tiles);
  for (int64_t t = t0; t < t1; t++) {
    const uint2 m = masks[t * SEL_WARPS + warp];
    const unsigned wc = __popc(m.x) + __popc(m.y);
    __syncthreads();                      // s_wcount of the previous tile fully consumed
    if (lane == 0) s_wcount[warp] = wc;
    __syncthreads();
    unsigned before = 0, total = 0;
#pragma unroll
    for (int w = 0; w < SEL_WARPS; w++) { const unsigned c = s_wcount[w]; before += (w < warp) ? c : 0; total += c; }
    const unsigned lt = (1u << lane) - 1u;
    const unsigned p0 = (m.x >> lane) & 1u, p1 = (m.y >> lane) & 1u;
    const unsigned long long pos = base + before + __popc(m.x & lt) + __popc(m.y & lt);
    const int64_t i0 = t * SEL_TILE + 2 * tid;
    if (p0) out_idx[pos] = (uint32_t)i0;
    if (p1) out_idx[pos + p0] = (uint32_t)(i0 + 1);
    base += total;
  }
}

// one cut on one event, columns read with scalar loads at the event's index: the form used where events are not
// contiguous (phase 2 of a planned chain works on a list) or where every cut is evaluated on its own (statistics)
__device__ __forceinline__ bool eval_cut_at(const SelCols& ev, const hepf_cut_t& cut, int64_t e, uint32_t f) {
  const int n_lep = f & 15u, n_jet = min(8u, (f >> 8) & 15u);
  switch (cut.kind) {
    case HEPF_CUT_NLEP_EQ: return n_lep == (int)cut.n;
    case HEPF_CUT_LEP_OS: return ((f >> 4) & 1u) != ((f >> 5) & 1u);
    case HEPF_CUT_LEP_PT_GT: return __ldg(ev.lep_pt + e) > cut.lo && __ldg(ev.lep_pt + ev.stride + e) > cut.lo;
    case HEPF_CUT_LEP_ABSETA_LT: return fabs(__ldg(ev.lep_eta + e)) < cut.hi && fabs(__ldg(ev.lep_eta + ev.stride + e)) < cut.hi;
    case HEPF_CUT_NJET_GE:
    case HEPF_CUT_NBJET_GE: {
      const uint32_t tagmask = cut.kind == HEPF_CUT_NBJET_GE ? (f >> 16) : 0xffu;
      int cnt = 0;
      for (int s = 0; s < n_jet; s++)
        cnt += ((tagmask >> s) & 1u) && __ldg(ev.jet_pt + s * ev.stride + e) > cut.lo && fabs(__ldg(ev.jet_eta + s * ev.stride + e)) < cut.hi;
      return cnt >= (int)cut.n;
    }
    case HEPF_CUT_MET_GT:
    case HEPF_CUT_MET_GT_RECORD: return __ldg(ev.met + e) > cut.lo;
    case HEPF_CUT_MLL_GT: return __ldg(ev.mll + e) > cut.lo;
    case HEPF_CUT_MLL_OUTSIDE: { const double m = __ldg(ev.mll + e); return m < cut.lo || m > cut.hi; }
    default: return false;
  }
}

// Phase 2 of a planned chain (NEXT-3): the sub-chain `chain` on the events of `list` (ascending survivors of phase 1, length
// *n_list on the device).  Same tile / mask layout as select_eval_kernel, positions are list positions; the scatter kernel
// below maps them back through the list.  Only the listed events' columns are touched, as sector-granular gathers; loading
// every jet slot up front instead of stopping at n_jet was measured slower (1.07 ms against 0.84 ms on cfg4): the gather is
// bound by the sectors it fetches, not by latency.
__global__ void __launch_bounds__(SEL_THREADS)
select_list_kernel(SelCols ev, CutChain chain, const uint32_t* __restrict__ list, const int64_t* __restrict__ n_list,
                   uint2* __restrict__ masks, uint32_t* __restrict__ block_count, unsigned long long* __restrict__ cutflow) {
  __shared__ unsigned int s_cf[HEPF_MAX_CUTS];
  __shared__ unsigned int s_count;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid < HEPF_MAX_CUTS) s_cf[tid] = 0;
  if (tid == 0) s_count = 0;
  __syncthreads();
  const int64_t n = *n_list, n_tiles = (n + SEL_TILE - 1) / SEL_TILE;
  const int64_t tiles_per_block = (n_tiles + gridDim.x - 1) / gridDim.x;   // contiguous, balanced over the ACTUAL list length
  const int64_t t0 = (int64_t)blockIdx.x * tiles_per_block;
  const int64_t t1 = min(t0 + tiles_per_block, n_tiles);
  unsigned int my_cf = 0, my_count = 0;
  for (int64_t t = t0; t < t1; t++) {
    const int64_t k0 = t * SEL_TILE + 2 * tid;
    bool pass[2] = {false, false};
    int fail_at[2] = {0, 0};
#pragma unroll
    for (int k = 0; k < 2; k++) {
      if (k0 + k < n) {
        const int64_t e = (int64_t)__ldg(list + k0 + k);
        const uint32_t f = __ldg(ev.flags + e);
        bool alive = true; int passed = 0;
        for (int c = 0; c < chain.n && alive; c++) { alive = eval_cut_at(ev, chain.c[c], e, f); passed += alive; }
        pass[k] = alive; fail_at[k] = passed;
      }
    }
    const unsigned b0 = __ballot_sync(0xffffffffu, pass[0]), b1 = __ballot_sync(0xffffffffu, pass[1]);
    if (lane == 0) { masks[t * SEL_WARPS + warp] = make_uint2(b0, b1); my_count += __popc(b0) + __popc(b1); }
    if (cutflow) {
      for (int c = 0; c < chain.n; c++) {
        const unsigned m0 = __ballot_sync(0xffffffffu, fail_at[0] > c), m1 = __ballot_sync(0xffffffffu, fail_at[1] > c);
        if (lane == c) my_cf += __popc(m0) + __popc(m1);
      }
    }
  }
  if (lane == 0 && my_count) atomicAdd(&s_count, my_count);
  if (cutflow && lane < chain.n && my_cf) atomicAdd(&s_cf[lane], my_cf);
  __syncthreads();
  if (tid == 0) block_count[blockIdx.x] = s_count;
  if (cutflow && tid < chain.n && s_cf[tid]) atomicAdd(&cutflow[tid], (unsigned long long)s_cf[tid]);
}

// select_scatter_kernel for a list whose length lives on the device: positions are list positions, the output is src[position]
__global__ void __launch_bounds__(SEL_THREADS)
select_scatter_list_kernel(const int64_t* __restrict__ n_list, const uint2* __restrict__ masks,
                           const uint32_t* __restrict__ block_count, uint32_t* __restrict__ out_idx,
                           int64_t* __restrict__ out_count, const uint32_t* __restrict__ src) {
  __shared__ unsigned long long s_part[SEL_WARPS];
  __shared__ unsigned int s_wcount[SEL_WARPS];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t n = *n_list, n_tiles = (n + SEL_TILE - 1) / SEL_TILE;
  const int64_t tiles_per_block = (n_tiles + gridDim.x - 1) / gridDim.x;
  unsigned long long part = 0;
  const int upto = (blockIdx.x == 0) ? gridDim.x : blockIdx.x;
  for (int b = tid; b < upto; b += SEL_THREADS) part += block_count[b];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
  if (lane == 0) s_part[warp] = part;
  __syncthreads();
  unsigned long long base = 0;
#pragma unroll
  for (int w = 0; w < SEL_WARPS; w++) base += s_part[w];
  if (blockIdx.x == 0) { if (tid == 0) *out_count = (int64_t)base; base = 0; }
  const int64_t t0 = (int64_t)blockIdx.x * tiles_per_block;
  const int64_t t1 = min(t0 + tiles_per_block, n_tiles);
  for (int64_t t = t0; t < t1; t++) {
    const uint2 m = masks[t * SEL_WARPS + warp];
    const unsigned wc = __popc(m.x) + __popc(m.y);
    __syncthreads();
    if (lane == 0) s_wcount[warp] = wc;
    __syncthreads();
    unsigned before = 0, total = 0;
#pragma unroll
    for (int w = 0; w < SEL_WARPS; w++) { const unsigned c = s_wcount[w]; before += (w < warp) ? c : 0; total += c; }
    const unsigned lt = (1u << lane) - 1u;
    const unsigned p0 = (m.x >> lane) & 1u, p1 = (m.y >> lane) & 1u;
    const unsigned long long pos = base + before + __popc(m.x & lt) + __popc(m.y & lt);
    const int64_t k0 = t * SEL_TILE + 2 * tid;
    if (p0) out_idx[pos] = src[k0];
    if (p1) out_idx[pos + p0] = src[k0 + 1];
    base += total;
  }
}

// Statistics for the planner (the framework measures each cut's filter ratio while it runs): every cut
// evaluated ON ITS OWN on the events of every `every`-th 512-event tile; out[c] = events that pass cut c, out[n_cuts] = events looked at.
__global__ void __launch_bounds__(SEL_THREADS)
cut_stats_kernel(SelCols ev, CutChain chain, int64_t n_tiles, int64_t every, unsigned long long* __restrict__ out) {
  __shared__ unsigned int s_c[HEPF_MAX_CUTS + 1];
  const int tid = threadIdx.x, lane = tid & 31;
  if (tid <= HEPF_MAX_CUTS) s_c[tid] = 0;
  __syncthreads();
  unsigned int mine = 0, seen = 0;   // lane c counts cut c, lane 0 also the events looked at
  for (int64_t t = (int64_t)blockIdx.x * every; t < n_tiles; t += (int64_t)gridDim.x * every) {
    for (int k = 0; k < 2; k++) {
      const int64_t e = t * SEL_TILE + k * SEL_THREADS + tid;
      const bool in = e < ev.n;
      const uint32_t f = in ? __ldg(ev.flags + e) : 0u;
      for (int c = 0; c < chain.n; c++) {
        const unsigned m = __ballot_sync(0xffffffffu, in && eval_cut_at(ev, chain.c[c], e, f));
        if (lane == c) mine += __popc(m);
      }
      const unsigned mi = __ballot_sync(0xffffffffu, in);
      if (lane == 0) seen += __popc(mi);
    }
  }
  if (lane < chain.n && mine) atomicAdd(&s_c[lane], mine);
  if (lane == 0 && seen) atomicAdd(&s_c[HEPF_MAX_CUTS], seen);
  __syncthreads();
  if (tid < chain.n && s_c[tid]) atomicAdd(&out[tid], (unsigned long long)s_c[tid]);
  if (tid == 0 && s_c[HEPF_MAX_CUTS]) atomicAdd(&out[chain.n], (unsigned long long)s_c[HEPF_MAX_CUTS]);
}

}  // namespace hepf

using namespace hepf;

// one wave: at most `slots` = SMs x resident blocks per SM blocks, each owning a contiguous range of tiles
static void sel_geometry(int64_t n_events, int slots, int64_t* n_tiles, int* grid, int64_t* tiles_per_block) {
  *n_tiles = (n_events + SEL_TILE - 1) / SEL_TILE;
  int64_t g = *n_tiles < (int64_t)slots ? *n_tiles : (int64_t)slots;
  if (g < 1) g = 1;
  *tiles_per_block = (*n_tiles + g - 1) / g;
  if (*tiles_per_block < 1) *tiles_per_block = 1;
  *grid = (int)((*n_tiles + *tiles_per_block - 1) / *tiles_per_block);
  if (*grid < 1) *grid = 1;
}

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

extern "C" size_t hepf_select_workspace_bytes(int64_t n_events) {
  if (n_events < 0) return 0;
  const int64_t n_tiles = (n_events + SEL_TILE - 1) / SEL_TILE;
  // masks: one uint2 per warp-tile; block counts: at most 8 blocks per SM, sized generously for 4096 blocks
  return align_up((size_t)(n_tiles + 1) * SEL_WARPS * sizeof(uint2), 256) + 4096 * sizeof(uint32_t);
}

// bytes of the column group(s) a set of NEED_* bits stands for, per event
static int need_bytes(uint32_t need) {
  return ((need & NEED_LEP_PT) ? 16 : 0) + ((need & NEED_LEP_ETA) ? 16 : 0) + ((need & NEED_JET_PT) ? 64 : 0) +
         ((need & NEED_JET_ETA) ? 64 : 0) + ((need & NEED_MET) ? 8 : 0) + ((need & NEED_MLL) ? 8 : 0);
}
static int cut_need(uint32_t kind, uint32_t* need) {
  switch (kind) {
    case HEPF_CUT_LEP_PT_GT: *need = NEED_LEP_PT; return HEPF_OK;
    case HEPF_CUT_LEP_ABSETA_LT: *need = NEED_LEP_ETA; return HEPF_OK;
    case HEPF_CUT_NJET_GE: case HEPF_CUT_NBJET_GE: *need = NEED_JET_PT | NEED_JET_ETA; return HEPF_OK;
    case HEPF_CUT_MET_GT: case HEPF_CUT_MET_GT_RECORD: *need = NEED_MET; return HEPF_OK;
    case HEPF_CUT_MLL_GT: case HEPF_CUT_MLL_OUTSIDE: *need = NEED_MLL; return HEPF_OK;
    case HEPF_CUT_NLEP_EQ: case HEPF_CUT_LEP_OS: *need = 0; return HEPF_OK;
    default: return HEPF_ERR_ARG;
  }
}
static int build_chain(const hepf_cut_t* host_cuts, int n_cuts, double derived_default, CutChain* chain) {
  chain->n = n_cuts; chain->need = 0; chain->rec_cut = -1; chain->rec_default = derived_default;
  for (int c = 0; c < n_cuts; c++) {
    chain->c[c] = host_cuts[c];
    uint32_t need = 0;
    if (cut_need(host_cuts[c].kind, &need) != HEPF_OK) {
      set_error("hepf_select: unknown cut kind %u at position %d", host_cuts[c].kind, c); return HEPF_ERR_ARG;
    }
    chain->need |= need;
    if (host_cuts[c].kind == HEPF_CUT_MET_GT_RECORD) {
      if (chain->rec_cut >= 0) { set_error("hepf_select: at most one recording cut per chain"); return HEPF_ERR_ARG; }
      chain->rec_cut = c;
    }
  }
  return HEPF_OK;
}

static int select_impl(const hepf_events_t* events, const hepf_cut_t* host_cuts, int n_cuts, uint32_t* out_idx,
                       int64_t* out_count, int64_t* out_cutflow, double* out_derived, double derived_default, void* ws,
                       size_t ws_bytes, cudaStream_t stream) {
  int rc = check_events(events);
  if (rc != HEPF_OK) return rc;
  if (n_cuts < 0 || n_cuts > HEPF_MAX_CUTS || (n_cuts > 0 && !host_cuts)) {
    set_error("hepf_select: n_cuts must be 0..%d with a non-NULL chain", HEPF_MAX_CUTS); return HEPF_ERR_ARG;
  }
  if (!out_count || !aligned(out_count, 8) || (events->n_events > 0 && (!out_idx || !aligned(out_idx, 4)))) {
    set_error("hepf_select: output pointer NULL or misaligned"); return HEPF_ERR_ARG;
  }
  if (out_cutflow && !aligned(out_cutflow, 8)) { set_error("hepf_select: out_cutflow misaligned"); return HEPF_ERR_ARG; }
  const int64_t n = events->n_events;
  if (ws_bytes < hepf_select_workspace_bytes(n) || !ws || !aligned(ws, 16)) {
    set_error("hepf_select: workspace too small or misaligned (%zu < %zu)", ws_bytes, hepf_select_workspace_bytes(n));
    return HEPF_ERR_CAPACITY;
  }
  CutChain chain{};
  rc = build_chain(host_cuts, n_cuts, derived_default, &chain);
  if (rc != HEPF_OK) return rc;
  if (out_derived && (chain.rec_cut < 0 || !aligned(out_derived, 16))) {
    set_error("hepf_select_record: out_derived needs a HEPF_CUT_MET_GT_RECORD cut in the chain and 16-byte alignment"); return HEPF_ERR_ARG;
  }
  if (out_cutflow && n_cuts > 0) HEPF_CUDA_TRY(cudaMemsetAsync(out_cutflow, 0, sizeof(int64_t) * n_cuts, stream));
  if (n == 0) { HEPF_CUDA_TRY(cudaMemsetAsync(out_count, 0, sizeof(int64_t), stream)); return HEPF_OK; }
  int dev = 0, sms = 148;
  HEPF_CUDA_TRY(cudaGetDevice(&dev));
  HEPF_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  int64_t n_tiles, tpb; int grid;
  static thread_local int resident = 0;   // blocks of select_eval_kernel that fit on one SM (register-limited)
  if (!resident) {
    HEPF_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&resident, select_eval_kernel, SEL_THREADS, 0));
    if (resident < 1) resident = 1;
  }
  sel_geometry(n, sms * resident, &n_tiles, &grid, &tpb);
  if (grid > 4096) { set_error("hepf_select: grid %d exceeds the workspace layout", grid); return HEPF_ERR_CAPACITY; }
  uint2* masks = reinterpret_cast<uint2*>(ws);
  uint32_t* block_count = reinterpret_cast<uint32_t*>(reinterpret_cast<char*>(ws) +
                                                      align_up((size_t)(n_tiles + 1) * SEL_WARPS * sizeof(uint2), 256));
  SelCols cols{events->lep_pt, events->lep_eta, events->jet_pt, events->jet_eta, events->met, events->mll,
               events->flags, n, events->stride};
  timing_mark(T_SEL0, stream);
  select_eval_kernel<<<grid, SEL_THREADS, 0, stream>>>(cols, chain, n_tiles, tpb, masks, block_count,
                                                       (n_cuts > 0) ? reinterpret_cast<unsigned long long*>(out_cutflow) : nullptr,
                                                       out_derived);
  count_launch();
  HEPF_CUDA_TRY(cudaGetLastError());
  timing_mark(T_SEL1, stream);
  select_scatter_kernel<<<grid, SEL_THREADS, 0, stream>>>(n_tiles, tpb, masks, block_count, out_idx, out_count);
  count_launch();
  timing_mark(T_SEL2, stream);
  HEPF_CUDA_TRY(cudaGetLastError());
  return HEPF_OK;
}

extern "C" int hepf_select(const hepf_events_t* events, const hepf_cut_t* host_cuts, int n_cuts, uint32_t* out_idx,
                           int64_t* out_count, int64_t* out_cutflow, void* ws, size_t ws_bytes, void* stream_) {
  return select_impl(events, host_cuts, n_cuts, out_idx, out_count, out_cutflow, nullptr, 0.0, ws, ws_bytes, (cudaStream_t)stream_);
}

extern "C" int hepf_select_record(const hepf_events_t* events, const hepf_cut_t* host_cuts, int n_cuts, uint32_t* out_idx,
                                  int64_t* out_count, int64_t* out_cutflow, double* out_derived, double derived_default,
                                  void* ws, size_t ws_bytes, void* stream_) {
  if (!out_derived) { set_error("hepf_select_record: out_derived is NULL"); return HEPF_ERR_ARG; }
  return select_impl(events, host_cuts, n_cuts, out_idx, out_count, out_cutflow, out_derived, derived_default, ws, ws_bytes,
                     (cudaStream_t)stream_);
}

// ---- hepf_select_static: the same path with its scratch in a file-scope device array (include/hepf.h) ----------------------
// In HOST code the name g_select_scratch is a host-side stand-in of the symbol, not a device address: what the kernels get is
// the address cudaGetSymbolAddress returns, looked up once per device with that device current.
constexpr size_t SELECT_STATIC_MASK_BYTES =
    ((size_t)((HEPF_SELECT_STATIC_MAX_EVENTS + SEL_TILE - 1) / SEL_TILE + 1) * SEL_WARPS * sizeof(uint2) + 255) / 256 * 256;
static_assert(SELECT_STATIC_MASK_BYTES + 4096 * sizeof(uint32_t) == HEPF_SELECT_STATIC_BYTES,
              "HEPF_SELECT_STATIC_BYTES must equal hepf_select_workspace_bytes(HEPF_SELECT_STATIC_MAX_EVENTS)");
static __device__ __align__(256) unsigned char g_select_scratch[HEPF_SELECT_STATIC_BYTES];

constexpr int SELECT_STATIC_MAX_DEVICES = 64;
static std::mutex g_select_scratch_lock;
static void* g_select_scratch_addr[SELECT_STATIC_MAX_DEVICES] = {};

static int select_static_scratch(void** addr) {
  int dev = -1;
  HEPF_CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= SELECT_STATIC_MAX_DEVICES) { set_error("hepf_select_static: device ordinal %d not supported", dev); return HEPF_ERR_ARG; }
  std::lock_guard<std::mutex> hold(g_select_scratch_lock);
  if (!g_select_scratch_addr[dev]) {
    void* p = nullptr;
    HEPF_CUDA_TRY(cudaGetSymbolAddress(&p, g_select_scratch));
    if (!p || !aligned(p, 256)) { set_error("hepf_select_static: bad address of the scratch array"); return HEPF_ERR_CUDA; }
    g_select_scratch_addr[dev] = p;
  }
  *addr = g_select_scratch_addr[dev];
  return HEPF_OK;
}

extern "C" int hepf_select_static(const hepf_events_t* events, const hepf_cut_t* host_cuts, int n_cuts, uint32_t* out_idx,
                                  int64_t* out_count, int64_t* out_cutflow, void* stream_) {
  int rc = check_events(events);
  if (rc != HEPF_OK) return rc;
  if (events->n_events > HEPF_SELECT_STATIC_MAX_EVENTS) {
    set_error("hepf_select_static: %lld events exceed the static scratch (at most %d events; use hepf_select with a workspace)",
              (long long)events->n_events, HEPF_SELECT_STATIC_MAX_EVENTS);
    return HEPF_ERR_CAPACITY;
  }
  void* scratch = nullptr;
  rc = select_static_scratch(&scratch);
  if (rc != HEPF_OK) return rc;
  return select_impl(events, host_cuts, n_cuts, out_idx, out_count, out_cutflow, nullptr, 0.0, scratch, HEPF_SELECT_STATIC_BYTES,
                     (cudaStream_t)stream_);
}

// ---- NEXT-3: the device analogue of the paper's cut-level scheduler (section 5.2) -----------------------
extern "C" size_t hepf_select_planned_workspace_bytes(int64_t n_events) {
  if (n_events < 0) return 0;
  return 2 * align_up(hepf_select_workspace_bytes(n_events), 256) + align_up((size_t)(n_events + 2) * sizeof(uint32_t), 256) + 256;
}

extern "C" int hepf_cut_stats(const hepf_events_t* events, const hepf_cut_t* host_cuts, int n_cuts, int64_t sample_every,
                              int64_t* out_pass, void* stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  int rc = check_events(events);
  if (rc != HEPF_OK) return rc;
  if (n_cuts < 0 || n_cuts > HEPF_MAX_CUTS || (n_cuts > 0 && !host_cuts) || sample_every < 1 || !out_pass || !aligned(out_pass, 8)) {
    set_error("hepf_cut_stats: need 0 <= n_cuts <= %d, sample_every >= 1 and an 8-byte aligned output", HEPF_MAX_CUTS); return HEPF_ERR_ARG;
  }
  CutChain chain{};
  rc = build_chain(host_cuts, n_cuts, 0.0, &chain);
  if (rc != HEPF_OK) return rc;
  HEPF_CUDA_TRY(cudaMemsetAsync(out_pass, 0, sizeof(int64_t) * (size_t)(n_cuts + 1), stream));
  const int64_t n = events->n_events;
  if (n == 0) return HEPF_OK;
  const int64_t n_tiles = (n + SEL_TILE - 1) / SEL_TILE, sampled = (n_tiles + sample_every - 1) / sample_every;
  int dev = 0, sms = 148;
  HEPF_CUDA_TRY(cudaGetDevice(&dev));
  HEPF_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int64_t cap = (int64_t)sms * 8;
  SelCols cols{events->lep_pt, events->lep_eta, events->jet_pt, events->jet_eta, events->met, events->mll, events->flags, n, events->stride};
  cut_stats_kernel<<<(unsigned)(sampled < cap ? sampled : cap), SEL_THREADS, 0, stream>>>(cols, chain, n_tiles, sample_every,
                                                                                      reinterpret_cast<unsigned long long*>(out_pass));
  count_launch();
  HEPF_CUDA_TRY(cudaGetLastError());
  return HEPF_OK;
}

// Expected cost per event in bytes of streamed HBM traffic.  One phase streams flags + every column
// group the chain names.  Two phases stream flags + the groups of phase 1; phase 2 then GATHERS, for the fraction p1 of the
// events that survive phase 1, flags and its groups.  A gather moves whole 64-byte DRAM atoms (eight neighbouring events of a
// column), so an atom is fetched if ANY of its eight events survives, 1 - (1 - p1)^8, and it runs at about 55 % of the
// streaming bandwidth (measured on B200, cfg4: profiles/r02e) — both factors are in the cost.  The survivor list is written
// and read once (8 p1).
constexpr double kGatherEfficiency = 0.55;
static double two_phase_bytes(uint32_t need1, uint32_t need2, double p1) {
  double q = 1.0 - p1; q *= q; q *= q; q *= q;                   // (1 - p1)^8
  return 4.0 + need_bytes(need1) + (1.0 - q) * (4.0 + need_bytes(need2)) / kGatherEfficiency + 8.0 * p1;
}

extern "C" int hepf_plan_chain(const hepf_cut_t* host_cuts, int n_cuts, const double* pass_frac, const uint32_t* dep_mask,
                               int* out_order, int* out_split, double* out_bytes_per_event) {
  if (n_cuts < 0 || n_cuts > HEPF_MAX_CUTS || (n_cuts > 0 && (!host_cuts || !pass_frac || !out_order)) || !out_split) {
    set_error("hepf_plan_chain: bad arguments"); return HEPF_ERR_ARG;
  }
  uint32_t need[HEPF_MAX_CUTS], all = 0;
  for (int c = 0; c < n_cuts; c++) {
    if (cut_need(host_cuts[c].kind, &need[c]) != HEPF_OK) { set_error("hepf_plan_chain: unknown cut kind %u", host_cuts[c].kind); return HEPF_ERR_ARG; }
    if (host_cuts[c].kind == HEPF_CUT_MET_GT_RECORD) { set_error("hepf_plan_chain: a recording cut cannot be reordered"); return HEPF_ERR_ARG; }
    if (!(pass_frac[c] >= 0.0 && pass_frac[c] <= 1.0)) { set_error("hepf_plan_chain: pass_frac[%d] outside [0, 1]", c); return HEPF_ERR_ARG; }
    all |= need[c];
  }
  const double one = 4.0 + need_bytes(all);
  const uint32_t full = n_cuts == 32 ? 0xffffffffu : ((1u << n_cuts) - 1u);
  double best = one; uint32_t best_set = 0;            // bit c of best_set: cut c runs in phase 1; 0 = one phase
  for (uint32_t G = 0; G < 64; G++) {                  // every subset of the six column groups
    if (G & ~all) continue;
    uint32_t S1 = 0;
    for (int c = 0; c < n_cuts; c++) if (!(need[c] & ~G)) S1 |= 1u << c;
    for (bool changed = true; changed;) {              // a cut whose prerequisite is left for phase 2 goes to phase 2 too
      changed = false;
      for (int c = 0; c < n_cuts; c++)
        if ((S1 >> c & 1u) && dep_mask && (dep_mask[c] & full & ~S1)) { S1 &= ~(1u << c); changed = true; }
    }
    if (S1 == 0 || S1 == full) continue;
    // pass fraction of phase 1: cuts that read the same columns are strongly correlated (two jet-count thresholds on the same
    // jets), so each such family counts once, with its SMALLEST pass fraction (an upper bound of the family's joint
    // fraction); different families are taken as independent
    uint32_t n1 = 0, n2 = 0, done = 0; double p1 = 1.0;
    for (int c = 0; c < n_cuts; c++) {
      if (!(S1 >> c & 1u)) { n2 |= need[c]; continue; }
      n1 |= need[c];
      if (done >> c & 1u) continue;
      double pm = pass_frac[c];
      for (int d = c + 1; d < n_cuts; d++)
        if ((S1 >> d & 1u) && need[d] == need[c]) { done |= 1u << d; if (pass_frac[d] < pm) pm = pass_frac[d]; }
      p1 *= pm;
    }
    const double cost = two_phase_bytes(n1, n2, p1);
    if (cost < best) { best = cost; best_set = S1; }
  }
  if (!(best < 0.9 * one)) { best = one; best_set = 0; }   // a second pair of launches must buy at least 10 %
  int k = 0, split = 0;
  if (best_set) {
    for (int c = 0; c < n_cuts; c++) if (best_set >> c & 1u) out_order[k++] = c;
    split = k;
  }
  for (int c = 0; c < n_cuts; c++) if (!(best_set >> c & 1u)) out_order[k++] = c;
  *out_split = best_set ? split : n_cuts;
  if (out_bytes_per_event) { out_bytes_per_event[0] = best; out_bytes_per_event[1] = one; }
  return HEPF_OK;
}

extern "C" int hepf_select_planned(const hepf_events_t* events, const hepf_cut_t* host_cuts, int n_cuts, const int* order, int split,
                                   uint32_t* out_idx, int64_t* out_count, int64_t* out_cutflow, void* ws, size_t ws_bytes,
                                   void* stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  int rc = check_events(events);
  if (rc != HEPF_OK) return rc;
  if (n_cuts < 0 || n_cuts > HEPF_MAX_CUTS || (n_cuts > 0 && (!host_cuts || !order)) || split < 0 || split > n_cuts) {
    set_error("hepf_select_planned: need 0 <= split <= n_cuts <= %d, a chain and an order", HEPF_MAX_CUTS); return HEPF_ERR_ARG;
  }
  hepf_cut_t cuts[HEPF_MAX_CUTS];
  uint32_t seen = 0;
  for (int k = 0; k < n_cuts; k++) {
    if (order[k] < 0 || order[k] >= n_cuts || (seen >> order[k] & 1u)) { set_error("hepf_select_planned: order is not a permutation"); return HEPF_ERR_ARG; }
    seen |= 1u << order[k];
    cuts[k] = host_cuts[order[k]];
    if (cuts[k].kind == HEPF_CUT_MET_GT_RECORD) { set_error("hepf_select_planned: a recording cut cannot be reordered"); return HEPF_ERR_ARG; }
  }
  const int64_t n = events->n_events;
  const size_t ws1 = align_up(hepf_select_workspace_bytes(n), 256);
  if (split == n_cuts || split == 0 || n == 0)          // one phase: the chain in the given order
    return select_impl(events, cuts, n_cuts, out_idx, out_count, out_cutflow, nullptr, 0.0, ws, ws_bytes, stream);
  if (!ws || !aligned(ws, 256) || ws_bytes < hepf_select_planned_workspace_bytes(n)) {
    set_error("hepf_select_planned: workspace too small or not 256-byte aligned (%zu < %zu)", ws_bytes, hepf_select_planned_workspace_bytes(n));
    return HEPF_ERR_CAPACITY;
  }
  if (!out_count || !aligned(out_count, 8) || !out_idx || !aligned(out_idx, 4) || (out_cutflow && !aligned(out_cutflow, 8))) {
    set_error("hepf_select_planned: output pointer NULL or misaligned"); return HEPF_ERR_ARG;
  }
  char* base = reinterpret_cast<char*>(ws);
  uint32_t* list1 = reinterpret_cast<uint32_t*>(base + 2 * ws1);
  int64_t* count1 = reinterpret_cast<int64_t*>(base + 2 * ws1 + align_up((size_t)(n + 2) * sizeof(uint32_t), 256));
  // phase 1: cuts [0, split) on every event -> list1 (cutflow entries [0, split))
  rc = select_impl(events, cuts, split, list1, count1, out_cutflow, nullptr, 0.0, base, ws1, stream);
  if (rc != HEPF_OK) return rc;
  // phase 2: cuts [split, n_cuts) on the listed events only
  CutChain chain2{};
  rc = build_chain(cuts + split, n_cuts - split, 0.0, &chain2);
  if (rc != HEPF_OK) return rc;
  if (out_cutflow) HEPF_CUDA_TRY(cudaMemsetAsync(out_cutflow + split, 0, sizeof(int64_t) * (size_t)(n_cuts - split), stream));
  int dev = 0, sms = 148;
  HEPF_CUDA_TRY(cudaGetDevice(&dev));
  HEPF_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  int64_t n_tiles, tpb; int grid;
  sel_geometry(n, sms * 4, &n_tiles, &grid, &tpb);     // grid sized for the capacity; the kernels split the ACTUAL list evenly
  uint2* masks2 = reinterpret_cast<uint2*>(base + ws1);
  uint32_t* block_count2 = reinterpret_cast<uint32_t*>(base + ws1 + align_up((size_t)(n_tiles + 1) * SEL_WARPS * sizeof(uint2), 256));
  SelCols cols{events->lep_pt, events->lep_eta, events->jet_pt, events->jet_eta, events->met, events->mll, events->flags, n, events->stride};
  select_list_kernel<<<grid, SEL_THREADS, 0, stream>>>(cols, chain2, list1, count1, masks2, block_count2,
                                                       out_cutflow ? reinterpret_cast<unsigned long long*>(out_cutflow + split) : nullptr);
  count_launch();
  HEPF_CUDA_TRY(cudaGetLastError());
  select_scatter_list_kernel<<<grid, SEL_THREADS, 0, stream>>>(count1, masks2, block_count2, out_idx, out_count, list1);
  count_launch();
  HEPF_CUDA_TRY(cudaGetLastError());
  return HEPF_OK;
}
