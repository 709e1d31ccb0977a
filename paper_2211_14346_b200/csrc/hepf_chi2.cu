// hepf_chi2.cu — hepf_chi2_semilep: chi^2 reconstruction of semileptonic ttbar events (eq. 1).
//
// One thread per listed event (coalesced column reads: consecutive list entries are consecutive events).  The chi^2 of a
// combination is a sum of a leptonic part that depends on (b_lep, p_z solution) and a hadronic part that depends on
// (b_had, q1, q2), so the minimum over the <= 4*3*6*2 combinations factorises: L[i] = min over solutions, H[j] = min over
// light-jet pairs, then min over the ordered pairs i != j of L[i] + H[j] — 8 + 24 mass evaluations instead of 144 (rounding is
// monotone, so the value is the same as the plain enumeration's; the argmin can differ from it only between exactly tied
// sums).  FP64 with IEEE division and square root; a few hundred FP64 instructions and ~300 bytes per event: the kernel is
// short; masses use the branch-free sqrt/rcp of hepf_common.cuh (<= 1 ulp), the p_z quadratic keeps IEEE sqrt and division.
#include <math_constants.h>

#include "hepf_common.cuh"

namespace hepf {

constexpr int C2_THREADS = 128;

struct Chi2Cols {
  const double *lep_px, *lep_py, *lep_pz, *lep_e, *jet_px, *jet_py, *jet_pz, *jet_e, *met_x, *met_y;
  const uint32_t* flags;
  int64_t stride;
};
struct P4 { double x, y, z, e; };
__device__ __forceinline__ P4 add4(const P4& a, const P4& b) { return P4{a.x + b.x, a.y + b.y, a.z + b.z, a.e + b.e}; }
__device__ __forceinline__ double mass4(const P4& a) {
  const double m2 = a.e * a.e - (a.x * a.x + a.y * a.y + a.z * a.z);
  return sqrt_fast(m2 > 0.0 ? m2 : 0.0);
}

// MODE 0: semileptonic ttbar (2 tops, 2 W);  MODE 1: single top, t-channel (1 top, 1 W: the leptonic ones);  MODE 2: single
// top, Wt (2 W, and one top that is either the leptonic or the hadronic one) — PAPER.md:327.
template <int MODE>
__global__ void __launch_bounds__(C2_THREADS)
chi2_semilep_kernel(Chi2Cols ev, const uint32_t* __restrict__ idx, int64_t n_idx, hepf_chi2_params_t P,
                    hepf_chi2_t* __restrict__ out) {
  const int64_t k = (int64_t)blockIdx.x * C2_THREADS + threadIdx.x;
  if (k >= n_idx) return;
  const int64_t e = (int64_t)__ldg(idx + k);
  const uint32_t f = __ldg(ev.flags + e);
  const int n_lep = f & 15u, n_jet = min(8u, (f >> 8) & 15u);
  int bt[4], lt[4], nbt = 0, nlt = 0;
  for (int s = 0; s < n_jet; s++) {
    if ((f >> (16 + s)) & 1u) { if (nbt < 4) bt[nbt++] = s; }
    else { if (nlt < 4) lt[nlt++] = s; }
  }
  hepf_chi2_t o;
  o.chi2 = o.nu_pz = o.m_top_lep = o.m_top_had = o.m_w_lep = o.m_w_had = CUDART_NAN;
  o.jet_b_lep = o.jet_b_had = o.jet_q1 = o.jet_q2 = o.solution = -1; o.n_comb = 0; o.status = 2u; o.event = (uint32_t)e;
  if (n_lep == 1 && nbt >= (MODE == 0 ? 2 : 1) && (MODE == 1 || nlt >= 2)) {
    const P4 lep{__ldg(ev.lep_px + e), __ldg(ev.lep_py + e), __ldg(ev.lep_pz + e), __ldg(ev.lep_e + e)};
    const double nux = __ldg(ev.met_x + e), nuy = __ldg(ev.met_y + e);
    P4 bj[4], lj[4];
    for (int c = 0; c < nbt; c++) { const int64_t at = bt[c] * ev.stride + e; bj[c] = P4{__ldg(ev.jet_px + at), __ldg(ev.jet_py + at), __ldg(ev.jet_pz + at), __ldg(ev.jet_e + at)}; }
    for (int c = 0; c < nlt; c++) { const int64_t at = lt[c] * ev.stride + e; lj[c] = P4{__ldg(ev.jet_px + at), __ldg(ev.jet_py + at), __ldg(ev.jet_pz + at), __ldg(ev.jet_e + at)}; }
    // ---- neutrino p_z from m(l nu) = m_W ---------------------------------------------------------------------------------
    const double ml2 = lep.e * lep.e - (lep.x * lep.x + lep.y * lep.y + lep.z * lep.z);
    const double mu = (P.m_w * P.m_w - ml2) / 2.0 + (lep.x * nux + lep.y * nuy);
    const double a = lep.e * lep.e - lep.z * lep.z, pt2 = nux * nux + nuy * nuy;
    const double disc = mu * mu * lep.z * lep.z - a * (lep.e * lep.e * pt2 - mu * mu);
    const double ist = rcp_fast(P.sigma_top), isw = rcp_fast(P.sigma_w);
    double pz[2]; int nsol;
    if (mu > 0.0 && disc >= 0.0) { const double sq = sqrt(disc); pz[0] = (mu * lep.z - sq) / a; pz[1] = (mu * lep.z + sq) / a; nsol = 2; }
    else { pz[0] = sqrt(pt2) * lep.z / sqrt(a); pz[1] = pz[0]; nsol = 1; }
    // ---- leptonic side: L[i] = min over solutions ---------------------------------------------------------------------------
    double L[4], Lmt[4], Lmw[2]; int Ls[4];
    P4 wl[2];
    for (int s = 0; s < nsol; s++) {
      const P4 nu{nux, nuy, pz[s], sqrt_fast(pt2 + pz[s] * pz[s])};
      wl[s] = add4(lep, nu); Lmw[s] = mass4(wl[s]);
    }
    for (int i = 0; i < nbt; i++) {
      L[i] = CUDART_INF; Ls[i] = 0; Lmt[i] = 0.0;
      for (int s = 0; s < nsol; s++) {
        const double mt = mass4(add4(wl[s], bj[i]));
        const double t1 = (mt - P.m_top) * ist, t2 = (Lmw[s] - P.m_w) * isw;
        const double v = t1 * t1 + t2 * t2;
        if (v < L[i]) { L[i] = v; Ls[i] = s; Lmt[i] = mt; }
      }
    }
    if (MODE == 1) {
      // ---- t-channel: the leptonic top and W only; argmin over (b, solution) -----------------------------------------------
      double best = CUDART_INF; int bi = -1;
      for (int i = 0; i < nbt; i++) if (L[i] < best) { best = L[i]; bi = i; }
      o.n_comb = nbt * nsol;
      o.status = bi >= 0 ? 1u : 0u;
      if (bi >= 0) {
        o.chi2 = best; o.nu_pz = pz[Ls[bi]]; o.m_top_lep = Lmt[bi]; o.m_w_lep = Lmw[Ls[bi]];
        o.jet_b_lep = bt[bi]; o.solution = Ls[bi];
      }
    } else {
    // ---- hadronic side: H[j] = min over light-jet pairs ---------------------------------------------------------------------
    double H[4], Hmt[4], Hmw[4]; int Ha[4], Hb[4];
    for (int j = 0; j < nbt; j++) { H[j] = CUDART_INF; Ha[j] = 0; Hb[j] = 1; Hmt[j] = Hmw[j] = 0.0; }
    double Wb = CUDART_INF, Wmw = 0.0; int Wa = 0, Wq = 1;          // MODE 2: the hadronic W alone, min over pairs
    for (int qa = 0; qa < nlt; qa++) for (int qb = qa + 1; qb < nlt; qb++) {
      const P4 wh = add4(lj[qa], lj[qb]);
      const double mw = mass4(wh), t4 = (mw - P.m_w) * isw;
      if (MODE == 2 && t4 * t4 < Wb) { Wb = t4 * t4; Wa = qa; Wq = qb; Wmw = mw; }
      for (int j = 0; j < nbt; j++) {
        const double mt = mass4(add4(wh, bj[j])), t3 = (mt - P.m_top) * ist;
        const double v = t3 * t3 + t4 * t4;
        if (v < H[j]) { H[j] = v; Ha[j] = qa; Hb[j] = qb; Hmt[j] = mt; Hmw[j] = mw; }
      }
    }
    if (MODE == 0) {
    // ---- combine over the ordered pairs (b_lep, b_had) ----------------------------------------------------------------------
    double best = CUDART_INF; int bi = -1, bjx = -1;
    for (int i = 0; i < nbt; i++) for (int j = 0; j < nbt; j++) {
      if (i == j) continue;
      const double v = L[i] + H[j];
      if (v < best) { best = v; bi = i; bjx = j; }
    }
    o.n_comb = nbt * (nbt - 1) * (nlt * (nlt - 1) / 2) * nsol;
    o.status = bi >= 0 ? 1u : 0u;
    if (bi >= 0) {
      o.chi2 = best; o.nu_pz = pz[Ls[bi]]; o.m_top_lep = Lmt[bi]; o.m_w_lep = Lmw[Ls[bi]];
      o.m_top_had = Hmt[bjx]; o.m_w_had = Hmw[bjx];
      o.jet_b_lep = bt[bi]; o.jet_b_had = bt[bjx]; o.jet_q1 = lt[Ha[bjx]]; o.jet_q2 = lt[Hb[bjx]]; o.solution = Ls[bi];
    }
    } else {
      // ---- Wt: hypothesis 0 = leptonic top, L[i] + (hadronic W term); hypothesis 1 = hadronic top, (leptonic W term) + H[j] --
      double bestA = CUDART_INF; int ai = -1;
      for (int i = 0; i < nbt; i++) { const double v = L[i] + Wb; if (v < bestA) { bestA = v; ai = i; } }
      double wl2 = CUDART_INF; int ws = 0;
      for (int sidx = 0; sidx < nsol; sidx++) { const double t2 = (Lmw[sidx] - P.m_w) * isw; if (t2 * t2 < wl2) { wl2 = t2 * t2; ws = sidx; } }
      double bestB = CUDART_INF; int bjx = -1;
      for (int j = 0; j < nbt; j++) { const double v = wl2 + H[j]; if (v < bestB) { bestB = v; bjx = j; } }
      o.n_comb = 2 * nbt * (nlt * (nlt - 1) / 2) * nsol;
      if (ai >= 0 && !(bestB < bestA)) {              // ties go to the first hypothesis in enumeration order
        o.status = 1u; o.chi2 = bestA; o.nu_pz = pz[Ls[ai]]; o.m_top_lep = Lmt[ai]; o.m_w_lep = Lmw[Ls[ai]]; o.m_w_had = Wmw;
        o.jet_b_lep = bt[ai]; o.jet_q1 = lt[Wa]; o.jet_q2 = lt[Wq]; o.solution = Ls[ai];
      } else if (bjx >= 0) {
        o.status = 1u; o.chi2 = bestB; o.nu_pz = pz[ws]; o.m_top_had = Hmt[bjx]; o.m_w_lep = Lmw[ws]; o.m_w_had = Hmw[bjx];
        o.jet_b_had = bt[bjx]; o.jet_q1 = lt[Ha[bjx]]; o.jet_q2 = lt[Hb[bjx]]; o.solution = ws;
      } else {
        o.status = 0u;
      }
    }
    }
  }
  out[k] = o;
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
                      events->jet_pz, events->jet_e, events->met_x, events->met_y, events->flags, events->stride};
  const int64_t blocks = (n_idx + C2_THREADS - 1) / C2_THREADS;
  if (blocks > 0x7fffffffll) { set_error("hepf_chi2: too many blocks"); return HEPF_ERR_ARG; }
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
