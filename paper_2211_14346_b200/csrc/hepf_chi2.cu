// hepf_chi2.cu — hepf_chi2_semilep: chi^2 reconstruction of semileptonic ttbar events (eq. 1).
//
// One thread per listed event (coalesced column reads: consecutive list entries are consecutive events), persistent threads in
// a grid-stride loop.  The chi^2 of a combination is a sum of a leptonic part that depends on (b_lep, p_z solution) and a
// hadronic part that depends on (b_had, q1, q2), so the minimum over the <= 4*3*6*2 combinations factorises: L[i] = min over
// solutions, H[j] = min over light-jet pairs, then min over the ordered pairs i != j of L[i] + H[j] — 8 + 24 mass evaluations
// instead of 144 (rounding is monotone, so the value is the same as the plain enumeration's; the argmin can differ from it only
// between exactly tied sums).  The candidate jets and the two tables sit in shared memory, a column per thread (cp.async
// staging, no local memory); masses use the branch-free sqrt/rcp of hepf_common.cuh (<= 1 ulp), the p_z quadratic keeps IEEE
// sqrt and division.  DESIGN.md section 6.6 has the measurements.
#include <math_constants.h>

#include "hepf_common.cuh"

namespace hepf {

constexpr int C2_THREADS = 128, C2_BLOCKS_PER_SM = 4;   // 40 KB of shared memory and <= 128 registers per thread (5 blocks spill: measured 4 % slower)

struct Chi2Cols {
  const double *lep_px, *lep_py, *lep_pz, *lep_e, *jet_px, *jet_py, *jet_pz, *jet_e, *met_x, *met_y;
  const uint32_t* flags;
  int64_t n, stride;
};
struct P4 { double x, y, z, e; };
__device__ __forceinline__ P4 add4(const P4& a, const P4& b) { return P4{a.x + b.x, a.y + b.y, a.z + b.z, a.e + b.e}; }
__device__ __forceinline__ double mass4(const P4& a) {
  const double m2 = a.e * a.e - (a.x * a.x + a.y * a.y + a.z * a.z);
  return sqrt_fast(m2 > 0.0 ? m2 : 0.0);
}

__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gmem_src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// MODE 0: semileptonic ttbar (2 tops, 2 W);  MODE 1: single top, t-channel (1 top, 1 W: the leptonic ones);  MODE 2: single
// top, Wt (2 W, and one top that is either the leptonic or the hadronic one) — PAPER.md:327.
template <int MODE>
__global__ void __launch_bounds__(C2_THREADS, C2_BLOCKS_PER_SM)
chi2_semilep_kernel(Chi2Cols ev, const uint32_t* __restrict__ idx, int64_t n_idx, hepf_chi2_params_t P,
                    hepf_chi2_t* __restrict__ out) {
  // Persistent threads, grid-stride over the list, software-pipelined: the event index is fetched two iterations ahead and the
  // flags one iteration ahead, so that of the three dependent memory latencies of an event (index -> flags -> jets) only the
  // last one — jets, lepton and MET, all issued together — is in front of the arithmetic.
  __shared__ double sj[2][4][4][C2_THREADS], sL[4][C2_THREADS], sH[4][C2_THREADS];
  const int tid = threadIdx.x;
  const int64_t step = (int64_t)gridDim.x * C2_THREADS;
  int64_t k = (int64_t)blockIdx.x * C2_THREADS + tid;
  if (k >= n_idx) return;
  int64_t e = (int64_t)__ldg(idx + k);
  int64_t e1 = (k + step < n_idx) ? (int64_t)__ldg(idx + k + step) : 0;
  // a list entry beyond the store is "not applicable" (status 2 | 8) and nothing is read for it: its flags word is taken as 0
  uint32_t f = ((uint64_t)e < (uint64_t)ev.n) ? __ldg(ev.flags + e) : 0u;
  for (;;) {
  const int64_t e2 = (k + 2 * step < n_idx) ? (int64_t)__ldg(idx + k + 2 * step) : 0;
  const uint32_t f1 = (k + step < n_idx && (uint64_t)e1 < (uint64_t)ev.n) ? __ldg(ev.flags + e1) : 0u;
  const bool in_range = (uint64_t)e < (uint64_t)ev.n;
  const int64_t er = in_range ? e : 0;
  // lepton and MET go out together with the jets' copies below
  P4 lep{0.0, 0.0, 0.0, 0.0};
  double nux = 0.0, nuy = 0.0;
  if (in_range) {
    lep = P4{__ldg(ev.lep_px + er), __ldg(ev.lep_py + er), __ldg(ev.lep_pz + er), __ldg(ev.lep_e + er)};
    nux = __ldg(ev.met_x + er); nuy = __ldg(ev.met_y + er);
  }
  const int n_lep = f & 15u, n_jet = min(8u, (f >> 8) & 15u);
  // Candidate jets (the first <= 4 tagged and <= 4 untagged slots) are compacted into shared memory, one column of the block's
  // array per thread, by asynchronous 8-byte copies (cp.async: no register in between, so all <= 32 copies of an event are in
  // flight together — as loads into registers the compiler serialised them slot by slot, one memory latency each); the
  // dynamically indexed reads of the combination loops are then conflict-free shared-memory loads instead of local memory.
  // A thread reads only the column it wrote: cp.async.wait_all orders its own copies, no barrier is needed.
  uint32_t btw = 0, ltw = 0;                                    // slot numbers, 4 bits each
  int nbt = 0, nlt = 0;
#pragma unroll
  for (int s = 0; s < 8; s++) {
    const bool tag = (f >> (16 + s)) & 1u;
    const int pos = tag ? nbt : nlt;
    if (s < n_jet && pos < 4) {
      const int64_t at = s * ev.stride + e;
      cp_async8(&sj[tag][pos][0][tid], ev.jet_px + at); cp_async8(&sj[tag][pos][1][tid], ev.jet_py + at);
      cp_async8(&sj[tag][pos][2][tid], ev.jet_pz + at); cp_async8(&sj[tag][pos][3][tid], ev.jet_e + at);
      if (tag) { btw |= (uint32_t)s << (4 * nbt); nbt++; } else { ltw |= (uint32_t)s << (4 * nlt); nlt++; }
    }
  }
  auto bt = [&](int i) { return (int)((btw >> (4 * i)) & 15u); };
  auto lt = [&](int i) { return (int)((ltw >> (4 * i)) & 15u); };
  auto bj = [&](int i) { return P4{sj[1][i][0][tid], sj[1][i][1][tid], sj[1][i][2][tid], sj[1][i][3][tid]}; };
  auto lj = [&](int i) { return P4{sj[0][i][0][tid], sj[0][i][1][tid], sj[0][i][2][tid], sj[0][i][3][tid]}; };
  hepf_chi2_t o;
  o.chi2 = o.nu_pz = o.m_top_lep = o.m_top_had = o.m_w_lep = o.m_w_had = CUDART_NAN;
  o.jet_b_lep = o.jet_b_had = o.jet_q1 = o.jet_q2 = o.solution = -1; o.n_comb = 0; o.status = in_range ? 2u : 10u; o.event = (uint32_t)e;
  if (n_lep == 1 && nbt >= (MODE == 0 ? 2 : 1) && (MODE == 1 || nlt >= 2)) {
    // ---- neutrino p_z from m(l nu) = m_W ---------------------------------------------------------------------------------
    const double ml2 = lep.e * lep.e - (lep.x * lep.x + lep.y * lep.y + lep.z * lep.z);
    const double mu = (P.m_w * P.m_w - ml2) / 2.0 + (lep.x * nux + lep.y * nuy);
    const double a = lep.e * lep.e - lep.z * lep.z, pt2 = nux * nux + nuy * nuy;
    const double disc = mu * mu * lep.z * lep.z - a * (lep.e * lep.e * pt2 - mu * mu);
    const double ist = rcp_fast(P.sigma_top), isw = rcp_fast(P.sigma_w);
    double pz[2]; int nsol;
    if (mu > 0.0 && disc >= 0.0) { const double sq = sqrt(disc); pz[0] = (mu * lep.z - sq) / a; pz[1] = (mu * lep.z + sq) / a; nsol = 2; }
    else { pz[0] = sqrt(pt2) * lep.z / sqrt(a); pz[1] = pz[0]; nsol = 1; }
    // The per-candidate minima L[i], H[j] are dynamically indexed: they sit beside the jets in shared memory (in registers they
    // would need every loop unrolled to its bound of 4 — measured 25 % slower — and with run-time bounds the compiler puts them
    // in local memory).  Their arguments are packed into two words; the winner's masses are evaluated again at the end.
    // ---- leptonic side: L[i] = min over solutions ---------------------------------------------------------------------------
    const P4 nu0{nux, nuy, pz[0], sqrt_fast(pt2 + pz[0] * pz[0])}, nu1{nux, nuy, pz[1], sqrt_fast(pt2 + pz[1] * pz[1])};
    const P4 wl0 = add4(lep, nu0), wl1 = add4(lep, nu1);
    const double Lmw0 = mass4(wl0), Lmw1 = mass4(wl1);
    const double tw0 = (Lmw0 - P.m_w) * isw, tw1 = (Lmw1 - P.m_w) * isw;
    cp_async_wait_all();                                            // the jets are needed from here on
    uint32_t Lsw = 0;                                               // bit i: the solution that gives L[i]
    for (int i = 0; i < nbt; i++) {
      const P4 b = bj(i);
      const double mt0 = mass4(add4(wl0, b)), t0 = (mt0 - P.m_top) * ist;
      double v = t0 * t0 + tw0 * tw0;
      if (nsol == 2) {
        const double mt1 = mass4(add4(wl1, b)), t1 = (mt1 - P.m_top) * ist, v1 = t1 * t1 + tw1 * tw1;
        if (v1 < v || !(v < CUDART_INF)) { if (v1 < CUDART_INF) { v = v1; Lsw |= 1u << i; } }
      }
      sL[i][tid] = v < CUDART_INF ? v : CUDART_INF;                 // NaN never wins (the plain enumeration's strict <)
    }
    auto lep_side = [&](int bi, int& sl, double& mt, double& mw, double& pzs) {   // the winner's payload, evaluated again
      sl = (int)((Lsw >> bi) & 1u);
      const P4 w = sl ? wl1 : wl0;
      mt = mass4(add4(w, bj(bi))); mw = sl ? Lmw1 : Lmw0; pzs = sl ? pz[1] : pz[0];
    };
    if (MODE == 1) {
      // ---- t-channel: the leptonic top and W only; argmin over (b, solution) -----------------------------------------------
      double best = CUDART_INF; int bi = -1;
      for (int i = 0; i < nbt; i++) { const double v = sL[i][tid]; if (v < best) { best = v; bi = i; } }
      o.n_comb = nbt * nsol;
      o.status = bi >= 0 ? 1u : 0u;
      if (bi >= 0) {
        int sl; lep_side(bi, sl, o.m_top_lep, o.m_w_lep, o.nu_pz);
        o.chi2 = best; o.jet_b_lep = bt(bi); o.solution = sl;
      }
    } else {
    // ---- hadronic side: H[j] = min over light-jet pairs ---------------------------------------------------------------------
    uint32_t Hqw = 0;                                               // 4 bits per j: qa | qb << 2
    for (int j = 0; j < nbt; j++) sH[j][tid] = CUDART_INF;
    double Wb = CUDART_INF, Wmw = 0.0; int Wq = 4;                   // MODE 2: the hadronic W alone, min over pairs
    for (int qa = 0; qa < nlt; qa++) for (int qb = qa + 1; qb < nlt; qb++) {
      const P4 wh = add4(lj(qa), lj(qb));
      const double mw = mass4(wh), t4 = (mw - P.m_w) * isw;
      if (MODE == 2 && t4 * t4 < Wb) { Wb = t4 * t4; Wq = qa | (qb << 2); Wmw = mw; }
      for (int j = 0; j < nbt; j++) {
        const double mt = mass4(add4(wh, bj(j))), t3 = (mt - P.m_top) * ist;
        const double v = t3 * t3 + t4 * t4;
        if (v < sH[j][tid]) { sH[j][tid] = v; Hqw = (Hqw & ~(15u << (4 * j))) | ((uint32_t)(qa | (qb << 2)) << (4 * j)); }
      }
    }
    auto had_side = [&](int bjx, int& qa, int& qb, double& mt, double& mw) {
      const int hq = (int)((Hqw >> (4 * bjx)) & 15u);
      qa = hq & 3; qb = hq >> 2;
      const P4 wh = add4(lj(qa), lj(qb));
      mw = mass4(wh); mt = mass4(add4(wh, bj(bjx)));
    };
    if (MODE == 0) {
    // ---- combine over the ordered pairs (b_lep, b_had) ----------------------------------------------------------------------
    double best = CUDART_INF; int bi = -1, bjx = -1;
    for (int i = 0; i < nbt; i++) {
      const double li = sL[i][tid];
      for (int j = 0; j < nbt; j++) {
        if (i == j) continue;
        const double v = li + sH[j][tid];
        if (v < best) { best = v; bi = i; bjx = j; }
      }
    }
    o.n_comb = nbt * (nbt - 1) * (nlt * (nlt - 1) / 2) * nsol;
    o.status = bi >= 0 ? 1u : 0u;
    if (bi >= 0) {
      int sl, qa, qb;
      lep_side(bi, sl, o.m_top_lep, o.m_w_lep, o.nu_pz); had_side(bjx, qa, qb, o.m_top_had, o.m_w_had);
      o.chi2 = best; o.jet_b_lep = bt(bi); o.jet_b_had = bt(bjx); o.jet_q1 = lt(qa); o.jet_q2 = lt(qb); o.solution = sl;
    }
    } else {
      // ---- Wt: hypothesis 0 = leptonic top, L[i] + (hadronic W term); hypothesis 1 = hadronic top, (leptonic W term) + H[j] --
      double bestA = CUDART_INF; int ai = -1;
      for (int i = 0; i < nbt; i++) { const double v = sL[i][tid] + Wb; if (v < bestA) { bestA = v; ai = i; } }
      double wl2 = CUDART_INF; int ws = 0;
      if (tw0 * tw0 < wl2) { wl2 = tw0 * tw0; ws = 0; }
      if (nsol == 2 && tw1 * tw1 < wl2) { wl2 = tw1 * tw1; ws = 1; }
      double bestB = CUDART_INF; int bjx = -1;
      for (int j = 0; j < nbt; j++) { const double v = wl2 + sH[j][tid]; if (v < bestB) { bestB = v; bjx = j; } }
      o.n_comb = 2 * nbt * (nlt * (nlt - 1) / 2) * nsol;
      if (ai >= 0 && !(bestB < bestA)) {              // ties go to the first hypothesis in enumeration order
        int sl; lep_side(ai, sl, o.m_top_lep, o.m_w_lep, o.nu_pz);
        o.status = 1u; o.chi2 = bestA; o.m_w_had = Wmw;
        o.jet_b_lep = bt(ai); o.jet_q1 = lt(Wq & 3); o.jet_q2 = lt(Wq >> 2); o.solution = sl;
      } else if (bjx >= 0) {
        int qa, qb; had_side(bjx, qa, qb, o.m_top_had, o.m_w_had);
        o.status = 1u; o.chi2 = bestB; o.nu_pz = ws ? pz[1] : pz[0]; o.m_w_lep = ws ? Lmw1 : Lmw0;
        o.jet_b_had = bt(bjx); o.jet_q1 = lt(qa); o.jet_q2 = lt(qb); o.solution = ws;
      } else {
        o.status = 0u;
      }
    }
    }
  }
  cp_async_wait_all();      // also for an event that was not applicable: its copies must not land on the next event's
  out[k] = o;
  k += step;
  if (k >= n_idx) break;
  e = e1; e1 = e2; f = f1;
  }
}

}  // namespace hepf

using namespace hepf;

static int chi2_launch(const hepf_events_t* events, const uint32_t* idx, int64_t n_idx, int mode,
                       const hepf_chi2_params_t* host_params, hepf_chi2_t* out, cudaStream_t stream) {
  int rc = check_events(events);
  if (rc != HEPF_OK) return rc;
  if (n_idx < 0 || mode < 0 || mode > 2) { set_error("hepf_chi2: n_idx < 0 or unknown mode"); return HEPF_ERR_ARG; }
  if (n_idx == 0) return HEPF_OK;
  if (!idx || !aligned(idx, 4) || !out || !aligned(out, 16)) { set_error("hepf_chi2: idx/out NULL or misaligned"); return HEPF_ERR_ARG; }
  hepf_chi2_params_t P{172.5, 80.4, 11.5, 7.5};
  if (host_params) P = *host_params;
  if (!(P.sigma_top > 0.0) || !(P.sigma_w > 0.0)) { set_error("hepf_chi2: widths must be positive"); return HEPF_ERR_ARG; }
  const Chi2Cols cols{events->lep_px, events->lep_py, events->lep_pz, events->lep_e, events->jet_px, events->jet_py,
                      events->jet_pz, events->jet_e, events->met_x, events->met_y, events->flags, events->n_events, events->stride};
  int dev = 0, sms = 148;
  HEPF_CUDA_TRY(cudaGetDevice(&dev));
  HEPF_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int64_t want = (n_idx + C2_THREADS - 1) / C2_THREADS, cap = (int64_t)sms * C2_BLOCKS_PER_SM;   // one resident wave
  const int64_t blocks = want < cap ? want : cap;
  if (mode == 0) chi2_semilep_kernel<0><<<(unsigned)blocks, C2_THREADS, 0, stream>>>(cols, idx, n_idx, P, out);
  else if (mode == 1) chi2_semilep_kernel<1><<<(unsigned)blocks, C2_THREADS, 0, stream>>>(cols, idx, n_idx, P, out);
  else chi2_semilep_kernel<2><<<(unsigned)blocks, C2_THREADS, 0, stream>>>(cols, idx, n_idx, P, out);
  count_launch();
  HEPF_CUDA_TRY(cudaGetLastError());
  return HEPF_OK;
}

extern "C" int hepf_chi2_semilep(const hepf_events_t* events, const uint32_t* idx, int64_t n_idx,
                                 const hepf_chi2_params_t* host_params, hepf_chi2_t* out, void* stream_) {
  return chi2_launch(events, idx, n_idx, 0, host_params, out, (cudaStream_t)stream_);
}

extern "C" int hepf_chi2_single_top(const hepf_events_t* events, const uint32_t* idx, int64_t n_idx, int mode,
                                    const hepf_chi2_params_t* host_params, hepf_chi2_t* out, void* stream_) {
  if (mode != 1 && mode != 2) { set_error("hepf_chi2_single_top: mode must be 1 (t-channel) or 2 (Wt)"); return HEPF_ERR_ARG; }
  return chi2_launch(events, idx, n_idx, mode, host_params, out, (cudaStream_t)stream_);
}
