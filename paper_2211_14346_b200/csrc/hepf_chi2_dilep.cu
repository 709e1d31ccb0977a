// hepf_chi2_dilep.cu — hepf_chi2_dilep: chi^2 reconstruction of DILEPTONIC ttbar events (eq. 1; the text breaks
// off at "splitting the E_T^miss between the two neutrinos and determine, using the mass constraints from the chi^2":
// DESIGN.md R15).
//
// Method: the neutrino's transverse momentum is scanned over a G x G grid around MET/2, the antineutrino takes the rest of
// the MET, each p_z follows from its W (two roots of m(l nu) = m_W, else the p_z of closest approach), and
//   chi^2 = T1(b, point, s1) + T2(bbar, point, s2),   T = ((m_blnu - m_t)/sigma_t)^2 + ((m_lnu - m_W)/sigma_W)^2,
// is minimised over ordered pairs of b-tagged jets, grid points and p_z solutions, first minimum in the order
// (b, bbar, gx, gy, s1, s2).
//
// B200 mapping: one WARP per event, the lanes stride over the G^2 grid points (1024 by default: 32 per lane), all data of
// the event in registers.  At a grid point the two legs are independent, so each leg's term is evaluated once per
// (candidate b, solution) — 2 x 8 top masses — and the <= 12 ordered pairs only add two numbers (rounding is monotone: the
// minimum is the plain enumeration's).  Lane-local best under the total order (chi^2, key), a warp-shuffle argmin, then
// lane 0 recomputes the winner's record.  FP64-pipe bound: ~0.5 k FP64 instructions per grid point and no memory traffic
// to speak of (one event in, 128 bytes out).  No tensor cores: nothing here is a contraction.
#include <math_constants.h>

#include "hepf_common.cuh"

namespace hepf {

constexpr int CD_WARPS = 4;   // warps (events) per block

struct DilepCols {
  const double *lep_px, *lep_py, *lep_pz, *lep_e, *jet_px, *jet_py, *jet_pz, *jet_e, *met_x, *met_y;
  const uint32_t* flags;
  int64_t n, stride;
};
struct Q4 { double x, y, z, e; };

__device__ __forceinline__ double mass_q(double e, double x, double y, double z) {
  const double m2 = e * e - (x * x + y * y + z * z);
  return sqrt_fast(m2 > 0.0 ? m2 : 0.0);
}

// p_z of a neutrino with transverse momentum (nux, nuy) from m(l nu) = m_W: the two roots, or the p_z that minimises m(l nu).
// IEEE division and square root, as in the semileptonic kernel.  hmw2ml = (m_W^2 - m_l^2)/2, a = E_l^2 - l_z^2.
__device__ __forceinline__ int nu_pz(const Q4& l, double hmw2ml, double a, double nux, double nuy, double (&pz)[2]) {
  const double mu = hmw2ml + (l.x * nux + l.y * nuy);
  const double pt2 = nux * nux + nuy * nuy;
  const double disc = mu * mu * l.z * l.z - a * (l.e * l.e * pt2 - mu * mu);
  if (mu > 0.0 && disc >= 0.0) {
    const double sq = sqrt(disc);
    pz[0] = (mu * l.z - sq) / a; pz[1] = (mu * l.z + sq) / a;
    return 2;
  }
  pz[0] = sqrt(pt2) * l.z / sqrt(a); pz[1] = pz[0];
  return 1;
}

// One leg at one grid point: for every candidate b the smaller of the (up to two) terms and which solution gave it.
struct LegMin { double v[4]; int s[4]; };
__device__ __forceinline__ LegMin leg_min(const Q4& l, const Q4* __restrict__ b, int nbt, int nsol, const double (&pz)[2], double nux, double nuy,
                                          double m_top, double m_w, double ist, double isw) {
  LegMin L;
#pragma unroll
  for (int c = 0; c < 4; c++) { L.v[c] = CUDART_INF; L.s[c] = 0; }
  const double pt2 = nux * nux + nuy * nuy;
#pragma unroll
  for (int s = 0; s < 2; s++) {
    if (s < nsol) {
      const double en = sqrt_fast(pt2 + pz[s] * pz[s]);
      const double wx = l.x + nux, wy = l.y + nuy, wz = l.z + pz[s], we = l.e + en;
      const double tw = (mass_q(we, wx, wy, wz) - m_w) * isw, tw2 = tw * tw;
#pragma unroll
      for (int c = 0; c < 4; c++) {
        if (c < nbt) {
          const double tt = (mass_q(we + b[c].e, wx + b[c].x, wy + b[c].y, wz + b[c].z) - m_top) * ist;
          const double v = tt * tt + tw2;
          if (v < L.v[c]) { L.v[c] = v; L.s[c] = s; }
        }
      }
    }
  }
  return L;
}

__device__ __forceinline__ double grid_u(int g, double gn) { return (double)(2 * g + 1) / gn - 1.0; }

__global__ void __launch_bounds__(32 * CD_WARPS, 6)   // 80 registers, 24 warps per SM: the dependent FP64 chains want the occupancy (164 registers unbounded: 11.3 ms; 96 registers / 20 warps: 9.5 ms; this: 9.2 ms)
chi2_dilep_kernel(DilepCols ev, const uint32_t* __restrict__ idx, int64_t n_idx, hepf_chi2_params_t P, double split_range,
                  int G, hepf_chi2_dilep_t* __restrict__ out) {
  const int lane = threadIdx.x & 31;
  const int64_t k = (int64_t)blockIdx.x * CD_WARPS + (threadIdx.x >> 5);
  if (k >= n_idx) return;
  const int64_t e = (int64_t)__ldg(idx + k);
  const bool in_range = (uint64_t)e < (uint64_t)ev.n;
  const uint32_t f = in_range ? __ldg(ev.flags + e) : 0u;
  const int n_lep = f & 15u, n_jet = min(8u, (f >> 8) & 15u);
  const bool q0 = (f >> 4) & 1u, q1 = (f >> 5) & 1u;
  int bt[4] = {0, 0, 0, 0}, nbt = 0;
  for (int s = 0; s < n_jet; s++) if (((f >> (16 + s)) & 1u) && nbt < 4) bt[nbt++] = s;
  hepf_chi2_dilep_t* o = out + k;
  if (n_lep != 2 || q0 == q1 || nbt < 2) {
    if (lane == 0) {
      const double n = CUDART_NAN;
      o->chi2 = o->m_top = o->m_antitop = o->m_wplus = o->m_wminus = n;
      o->nu[0] = o->nu[1] = o->nu[2] = o->nubar[0] = o->nubar[1] = o->nubar[2] = n;
      o->jet_b = o->jet_bbar = o->grid_x = o->grid_y = o->sol_nu = o->sol_nubar = -1; o->n_comb = 0;
      o->status = 2u | (in_range ? 0u : 8u); o->event = (uint32_t)e; o->pad_ = 0;
    }
    return;
  }
  const int lp = q0 ? 0 : 1, lm = 1 - lp;
  const Q4 lplus{__ldg(ev.lep_px + lp * ev.stride + e), __ldg(ev.lep_py + lp * ev.stride + e), __ldg(ev.lep_pz + lp * ev.stride + e), __ldg(ev.lep_e + lp * ev.stride + e)};
  const Q4 lminus{__ldg(ev.lep_px + lm * ev.stride + e), __ldg(ev.lep_py + lm * ev.stride + e), __ldg(ev.lep_pz + lm * ev.stride + e), __ldg(ev.lep_e + lm * ev.stride + e)};
  // The candidate b jets are the same for every lane of the warp: they sit in shared memory (broadcast reads in the scan),
  // not in 32 registers of every thread.
  __shared__ Q4 s_b[CD_WARPS][4];
  Q4* b = s_b[threadIdx.x >> 5];
  if (lane < 4) {
    const int slot = lane == 0 ? bt[0] : lane == 1 ? bt[1] : lane == 2 ? bt[2] : bt[3];
    const int64_t at = (int64_t)slot * ev.stride + e;
    b[lane] = lane < nbt ? Q4{__ldg(ev.jet_px + at), __ldg(ev.jet_py + at), __ldg(ev.jet_pz + at), __ldg(ev.jet_e + at)} : Q4{0.0, 0.0, 0.0, 0.0};
  }
  __syncwarp();
  const double Mx = __ldg(ev.met_x + e), My = __ldg(ev.met_y + e);
  const double ist = rcp_fast(P.sigma_top), isw = rcp_fast(P.sigma_w), gn = (double)G;
  const double ml2p = lplus.e * lplus.e - (lplus.x * lplus.x + lplus.y * lplus.y + lplus.z * lplus.z);
  const double ml2m = lminus.e * lminus.e - (lminus.x * lminus.x + lminus.y * lminus.y + lminus.z * lminus.z);
  const double hp = (P.m_w * P.m_w - ml2p) / 2.0, hm = (P.m_w * P.m_w - ml2m) / 2.0;
  const double ap = lplus.e * lplus.e - lplus.z * lplus.z, am = lminus.e * lminus.e - lminus.z * lminus.z;

  double best = CUDART_INF; uint32_t best_key = 0xffffffffu; int n_comb = 0;
#pragma unroll 1
  for (int p = lane; p < G * G; p += 32) {
    const int gx = p / G, gy = p - gx * G;
    const double nux = 0.5 * Mx + split_range * grid_u(gx, gn), nuy = 0.5 * My + split_range * grid_u(gy, gn);
    const double qx = Mx - nux, qy = My - nuy;
    double pz1[2], pz2[2];
    const int ns1 = nu_pz(lplus, hp, ap, nux, nuy, pz1), ns2 = nu_pz(lminus, hm, am, qx, qy, pz2);
    const LegMin L1 = leg_min(lplus, b, nbt, ns1, pz1, nux, nuy, P.m_top, P.m_w, ist, isw);
    const LegMin L2 = leg_min(lminus, b, nbt, ns2, pz2, qx, qy, P.m_top, P.m_w, ist, isw);
    n_comb += ns1 * ns2;
#pragma unroll
    for (int i = 0; i < 4; i++)
#pragma unroll
      for (int j = 0; j < 4; j++) {
        if (i != j && i < nbt && j < nbt) {
          const double v = L1.v[i] + L2.v[j];
          if (v <= best) {
            const uint32_t key = ((uint32_t)i << 16) | ((uint32_t)j << 14) | ((uint32_t)gx << 8) | ((uint32_t)gy << 2) |
                                 ((uint32_t)L1.s[i] << 1) | (uint32_t)L2.s[j];
            if (v < best || key < best_key) { best = v; best_key = key; }
          }
        }
      }
  }
#pragma unroll
  for (int s = 16; s > 0; s >>= 1) {
    const double ov = __shfl_xor_sync(0xffffffffu, best, s);
    const uint32_t ok = __shfl_xor_sync(0xffffffffu, best_key, s);
    n_comb += __shfl_xor_sync(0xffffffffu, n_comb, s);
    if (ov < best || (ov == best && ok < best_key)) { best = ov; best_key = ok; }
  }
  if (lane != 0) return;
  o->event = (uint32_t)e; o->pad_ = 0; o->n_comb = n_comb * nbt * (nbt - 1);
  if (!(best < CUDART_INF)) {           // every term NaN or infinite (garbage inputs): no solution
    const double n = CUDART_NAN;
    o->chi2 = o->m_top = o->m_antitop = o->m_wplus = o->m_wminus = n;
    o->nu[0] = o->nu[1] = o->nu[2] = o->nubar[0] = o->nubar[1] = o->nubar[2] = n;
    o->jet_b = o->jet_bbar = o->grid_x = o->grid_y = o->sol_nu = o->sol_nubar = -1; o->status = 0u;
    return;
  }
  // ---- the winner's record, recomputed from its key -----------------------------------------------------------------------
  const int i = (best_key >> 16) & 3, j = (best_key >> 14) & 3, gx = (best_key >> 8) & 63, gy = (best_key >> 2) & 63;
  const int s1 = (best_key >> 1) & 1, s2 = best_key & 1;
  const double nux = 0.5 * Mx + split_range * grid_u(gx, gn), nuy = 0.5 * My + split_range * grid_u(gy, gn);
  const double qx = Mx - nux, qy = My - nuy;
  double pz1[2], pz2[2];
  nu_pz(lplus, hp, ap, nux, nuy, pz1); nu_pz(lminus, hm, am, qx, qy, pz2);
  Q4 bi = b[0], bj = b[0];
#pragma unroll
  for (int c = 1; c < 4; c++) { if (c == i) bi = b[c]; if (c == j) bj = b[c]; }
  const double en = sqrt_fast(nux * nux + nuy * nuy + pz1[s1] * pz1[s1]), eb = sqrt_fast(qx * qx + qy * qy + pz2[s2] * pz2[s2]);
  o->chi2 = best;
  o->nu[0] = nux; o->nu[1] = nuy; o->nu[2] = pz1[s1]; o->nubar[0] = qx; o->nubar[1] = qy; o->nubar[2] = pz2[s2];
  o->m_wplus = mass_q(lplus.e + en, lplus.x + nux, lplus.y + nuy, lplus.z + pz1[s1]);
  o->m_top = mass_q(lplus.e + en + bi.e, lplus.x + nux + bi.x, lplus.y + nuy + bi.y, lplus.z + pz1[s1] + bi.z);
  o->m_wminus = mass_q(lminus.e + eb, lminus.x + qx, lminus.y + qy, lminus.z + pz2[s2]);
  o->m_antitop = mass_q(lminus.e + eb + bj.e, lminus.x + qx + bj.x, lminus.y + qy + bj.y, lminus.z + pz2[s2] + bj.z);
  int sb = bt[0], sbb = bt[0];
#pragma unroll
  for (int c = 1; c < 4; c++) { if (c == i) sb = bt[c]; if (c == j) sbb = bt[c]; }
  o->jet_b = sb; o->jet_bbar = sbb; o->grid_x = gx; o->grid_y = gy; o->sol_nu = s1; o->sol_nubar = s2;
  o->status = 1u;
}

}  // namespace hepf

using namespace hepf;

extern "C" int hepf_chi2_dilep(const hepf_events_t* events, const uint32_t* idx, int64_t n_idx, const hepf_chi2_params_t* host_params,
                               const hepf_split_t* host_split, hepf_chi2_dilep_t* out, void* stream_) {
  int rc = check_events(events);
  if (rc != HEPF_OK) return rc;
  if (n_idx < 0) { set_error("hepf_chi2_dilep: n_idx < 0"); return HEPF_ERR_ARG; }
  if (n_idx == 0) return HEPF_OK;
  if (!idx || !aligned(idx, 4) || !out || !aligned(out, 16)) { set_error("hepf_chi2_dilep: idx/out NULL or misaligned"); return HEPF_ERR_ARG; }
  hepf_chi2_params_t P{172.5, 80.4, 11.5, 7.5};
  if (host_params) P = *host_params;
  if (!(P.sigma_top > 0.0) || !(P.sigma_w > 0.0)) { set_error("hepf_chi2_dilep: widths must be positive"); return HEPF_ERR_ARG; }
  hepf_split_t S{160.0, 32, 0};
  if (host_split) S = *host_split;
  if (S.split_n < 1 || S.split_n > 64 || !(S.split_range >= 0.0)) {
    set_error("hepf_chi2_dilep: need 1 <= split_n <= 64 and split_range >= 0"); return HEPF_ERR_ARG;
  }
  const DilepCols cols{events->lep_px, events->lep_py, events->lep_pz, events->lep_e, events->jet_px, events->jet_py,
                       events->jet_pz, events->jet_e, events->met_x, events->met_y, events->flags, events->n_events, events->stride};
  const int64_t blocks = (n_idx + CD_WARPS - 1) / CD_WARPS;
  if (blocks > 0x7fffffffll) { set_error("hepf_chi2_dilep: too many blocks"); return HEPF_ERR_ARG; }
  chi2_dilep_kernel<<<(unsigned)blocks, 32 * CD_WARPS, 0, (cudaStream_t)stream_>>>(cols, idx, n_idx, P, S.split_range, S.split_n, out);
  count_launch();
  HEPF_CUDA_TRY(cudaGetLastError());
  return HEPF_OK;
}
