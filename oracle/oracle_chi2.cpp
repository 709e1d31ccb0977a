// oracle/oracle_chi2.cpp — CPU ORACLE (test infrastructure).  chi^2 kinematic reconstruction of semileptonic ttbar events.
//
// PAPER.md:323-329 (section 6.2, eq. 1): "for each possible jet and lepton combination, a chi^2 function was minimised to
// derive the four-momentum of the undetected neutrino(s) and reconstruct the top-quark(s) and W-boson(s) masses",
//   chi^2 = sum_k (m_jlnu - m_t)^2 / sigma_t^2 + sum_m (m_lnu - m_W)^2 / sigma_W^2,
// m_t = 172.5, m_W = 80.4, sigma_t = 11.5, sigma_W = 7.5 GeV; "the E_T^miss is assumed to be the transverse momentum of
// the undetected neutrino"; "for the semileptonic final states only the p_Z component of the neutrino four-momentum
// remains to be determined".  For ttbar there are two tops and two W bosons: the leptonic ones (b l nu, l nu) and, reading
// "m_jlnu" / "m_lnu" of the hadronic side as the three-jet and two-jet masses, the hadronic ones (b j j, j j).
// Readings (R14): the minimisation over p_z is done in closed form — p_z solves m(l nu) = m_W (two solutions);
// if no real solution exists the p_z that minimises m(l nu), hence the W term: p_z = pT(nu) l_z / sqrt(E_l^2 - l_z^2); combinations: ordered pair
// (b_lep, b_had) of b-tagged jets (first 4 tagged slots) x unordered pair of untagged jets (first 4 untagged slots);
// argmin in enumeration order (b_lep, b_had, (q1, q2), solution) with strict <.  Nothing is hoisted or reordered here.
#include <cmath>
#include <cstdint>
#include <limits>

#include "hepf_oracle.h"

namespace {
struct P4 { double x, y, z, e; };
double mass4(const P4& a) {
  double m2 = a.e * a.e - (a.x * a.x + a.y * a.y + a.z * a.z);
  return std::sqrt(m2 > 0.0 ? m2 : 0.0);
}
P4 add(const P4& a, const P4& b) { return P4{a.x + b.x, a.y + b.y, a.z + b.z, a.e + b.e}; }
}  // namespace

extern "C" void orc_default_chi2_params(orc_chi2_params_t* p) {
  p->m_top = 172.5; p->m_w = 80.4; p->sigma_top = 11.5; p->sigma_w = 7.5;
}

// p_z of the neutrino from m(l nu) = m_W; returns the number of solutions written (1 or 2), ascending by the sign of the root
extern "C" int orc_nu_pz(const double lep[4], double nux, double nuy, double m_w, double pz[2]) {
  const double ml2 = lep[3] * lep[3] - (lep[0] * lep[0] + lep[1] * lep[1] + lep[2] * lep[2]);
  const double mu = (m_w * m_w - ml2) / 2.0 + (lep[0] * nux + lep[1] * nuy);
  const double a = lep[3] * lep[3] - lep[2] * lep[2];
  const double pt2 = nux * nux + nuy * nuy;
  const double disc = mu * mu * lep[2] * lep[2] - a * (lep[3] * lep[3] * pt2 - mu * mu);
  if (mu > 0.0 && disc >= 0.0) {       // E_l E_nu - l_z p_z = mu has real solutions (mu <= 0 would make the squared
    const double sq = std::sqrt(disc);  // equation's roots spurious: the left-hand side is positive)
    pz[0] = (mu * lep[2] - sq) / a; pz[1] = (mu * lep[2] + sq) / a;
    return 2;
  }
  pz[0] = std::sqrt(pt2) * lep[2] / std::sqrt(a);   // m(l nu) > m_W for every p_z: the p_z that minimises it (the chi^2 term)
  return 1;
}

extern "C" int orc_chi2_semilep(const orc_events_t* ev, const uint32_t* idx, int64_t n_idx, const orc_chi2_params_t* params,
                                orc_chi2_t* out, double* out_second) {
  if (!ev || (n_idx > 0 && !idx) || n_idx < 0 || !out) return -1;
  orc_chi2_params_t P; if (params) P = *params; else orc_default_chi2_params(&P);
  const double NaN = std::numeric_limits<double>::quiet_NaN();
  const int64_t S = ev->stride;
  for (int64_t k = 0; k < n_idx; k++) {
    const uint32_t e = idx[k];
    orc_chi2_t& o = out[k];
    o.chi2 = o.nu_pz = o.m_top_lep = o.m_top_had = o.m_w_lep = o.m_w_had = NaN;
    o.jet_b_lep = o.jet_b_had = o.jet_q1 = o.jet_q2 = o.solution = -1; o.n_comb = 0; o.status = 0; o.event = e;
    if (out_second) out_second[k] = INFINITY;
    const uint32_t f = ev->flags[e];
    const int n_lep = (int)(f & 15u); int n_jet = (int)((f >> 8) & 15u); if (n_jet > 8) n_jet = 8;
    int bt[4], nbt = 0, lt[4], nlt = 0;
    for (int s = 0; s < n_jet; s++) {
      if ((f >> (16 + s)) & 1u) { if (nbt < 4) bt[nbt++] = s; }
      else { if (nlt < 4) lt[nlt++] = s; }
    }
    if (n_lep != 1 || nbt < 2 || nlt < 2) { o.status = 2; continue; }
    const P4 lep{ev->lep_px[e], ev->lep_py[e], ev->lep_pz[e], ev->lep_e[e]};
    const double la[4] = {lep.x, lep.y, lep.z, lep.e};
    const double nux = ev->met_x[e], nuy = ev->met_y[e];
    double pz[2]; const int nsol = orc_nu_pz(la, nux, nuy, P.m_w, pz);
    P4 jet[8];
    for (int s = 0; s < n_jet; s++) jet[s] = P4{ev->jet_px[s * S + e], ev->jet_py[s * S + e], ev->jet_pz[s * S + e], ev->jet_e[s * S + e]};
    double best = INFINITY, second = INFINITY;
    for (int i = 0; i < nbt; i++) for (int j = 0; j < nbt; j++) {
      if (i == j) continue;
      for (int a = 0; a < nlt; a++) for (int b = a + 1; b < nlt; b++) {
        const P4 whad = add(jet[lt[a]], jet[lt[b]]), thad = add(whad, jet[bt[j]]);
        const double mwh = mass4(whad), mth = mass4(thad);
        for (int s = 0; s < nsol; s++) {
          const P4 nu{nux, nuy, pz[s], std::sqrt(nux * nux + nuy * nuy + pz[s] * pz[s])};
          const P4 wlep = add(lep, nu), tlep = add(wlep, jet[bt[i]]);
          const double mwl = mass4(wlep), mtl = mass4(tlep);
          const double t1 = (mtl - P.m_top) / P.sigma_top, t2 = (mwl - P.m_w) / P.sigma_w;
          const double t3 = (mth - P.m_top) / P.sigma_top, t4 = (mwh - P.m_w) / P.sigma_w;
          const double chi2 = (t1 * t1 + t2 * t2) + (t3 * t3 + t4 * t4);
          o.n_comb++;
          if (chi2 < best) {
            second = best; best = chi2;
            o.chi2 = chi2; o.nu_pz = pz[s]; o.m_top_lep = mtl; o.m_top_had = mth; o.m_w_lep = mwl; o.m_w_had = mwh;
            o.jet_b_lep = bt[i]; o.jet_b_had = bt[j]; o.jet_q1 = lt[a]; o.jet_q2 = lt[b]; o.solution = s;
          } else if (chi2 < second) {
            second = chi2;
          }
        }
      }
    }
    o.status = (best < INFINITY) ? 1u : 0u;
    if (out_second) out_second[k] = second;
  }
  return 0;
}

// Single-top variants of eq. (1) ("in single top quark events from Wt associated production, only 1 top quark
// and 2 W-bosons should be reconstructed, while for the t-channel only 1, of each, should exist"), semileptonic final state
// (one lepton; the neutrino p_z from the W-mass quadratic as above).
//   mode 1, t-channel (k = 1, m = 1):  chi^2 = ((m_blnu - m_t)/sigma_t)^2 + ((m_lnu - m_W)/sigma_W)^2,
//           minimised over the b-tagged jet (first 4 tagged slots) and the p_z solution; needs one lepton and one b-tag.
//   mode 2, Wt (k = 1, m = 2): two W bosons (l nu and j j) and ONE top, which is either the leptonic one (b l nu, hypothesis 0)
//           or the hadronic one (b j j, hypothesis 1):
//           chi^2 = ((m_top - m_t)/sigma_t)^2 + ((m_lnu - m_W)/sigma_W)^2 + ((m_jj - m_W)/sigma_W)^2,
//           minimised over the hypothesis, the b-tagged jet, the pair of untagged jets (first 4 untagged slots) and the p_z
//           solution; needs one lepton, one b-tag and two untagged jets.
// Enumeration order (hypothesis, b, (q1, q2), solution), strict <.  Record: jet_b_lep = the b-jet if the top is leptonic else
// -1, jet_b_had likewise; m_top_lep / m_top_had NaN for the top that is not there; t-channel: no hadronic entries at all.
// The dileptonic chi^2 of eq. (1) is in oracle_chi2_dilep.cpp (PAPER.md:329 breaks off in the middle of its description: reading R15).
extern "C" int orc_chi2_single_top(const orc_events_t* ev, const uint32_t* idx, int64_t n_idx, int mode,
                                   const orc_chi2_params_t* params, orc_chi2_t* out, double* out_second) {
  if (!ev || (n_idx > 0 && !idx) || n_idx < 0 || !out || (mode != 1 && mode != 2)) return -1;
  orc_chi2_params_t P; if (params) P = *params; else orc_default_chi2_params(&P);
  const double NaN = std::numeric_limits<double>::quiet_NaN();
  const int64_t S = ev->stride;
  for (int64_t k = 0; k < n_idx; k++) {
    const uint32_t e = idx[k];
    orc_chi2_t& o = out[k];
    o.chi2 = o.nu_pz = o.m_top_lep = o.m_top_had = o.m_w_lep = o.m_w_had = NaN;
    o.jet_b_lep = o.jet_b_had = o.jet_q1 = o.jet_q2 = o.solution = -1; o.n_comb = 0; o.status = 0; o.event = e;
    if (out_second) out_second[k] = INFINITY;
    const uint32_t f = ev->flags[e];
    const int n_lep = (int)(f & 15u); int n_jet = (int)((f >> 8) & 15u); if (n_jet > 8) n_jet = 8;
    int bt[4], nbt = 0, lt[4], nlt = 0;
    for (int s = 0; s < n_jet; s++) {
      if ((f >> (16 + s)) & 1u) { if (nbt < 4) bt[nbt++] = s; }
      else { if (nlt < 4) lt[nlt++] = s; }
    }
    if (n_lep != 1 || nbt < 1 || (mode == 2 && nlt < 2)) { o.status = 2; continue; }
    const P4 lep{ev->lep_px[e], ev->lep_py[e], ev->lep_pz[e], ev->lep_e[e]};
    const double la[4] = {lep.x, lep.y, lep.z, lep.e};
    const double nux = ev->met_x[e], nuy = ev->met_y[e];
    double pz[2]; const int nsol = orc_nu_pz(la, nux, nuy, P.m_w, pz);
    P4 jet[8];
    for (int s = 0; s < n_jet; s++) jet[s] = P4{ev->jet_px[s * S + e], ev->jet_py[s * S + e], ev->jet_pz[s * S + e], ev->jet_e[s * S + e]};
    double best = INFINITY, second = INFINITY;
    auto consider = [&](double chi2, int hyp, int b, int q1, int q2, int s, double mtl, double mth, double mwl, double mwh) {
      o.n_comb++;
      if (chi2 < best) {
        second = best; best = chi2;
        o.chi2 = chi2; o.nu_pz = pz[s]; o.m_top_lep = mtl; o.m_top_had = mth; o.m_w_lep = mwl; o.m_w_had = mwh;
        o.jet_b_lep = hyp == 0 ? b : -1; o.jet_b_had = hyp == 1 ? b : -1; o.jet_q1 = q1; o.jet_q2 = q2; o.solution = s;
      } else if (chi2 < second) {
        second = chi2;
      }
    };
    if (mode == 1) {
      for (int i = 0; i < nbt; i++) for (int s = 0; s < nsol; s++) {
        const P4 nu{nux, nuy, pz[s], std::sqrt(nux * nux + nuy * nuy + pz[s] * pz[s])};
        const P4 wlep = add(lep, nu), tlep = add(wlep, jet[bt[i]]);
        const double mwl = mass4(wlep), mtl = mass4(tlep);
        const double t1 = (mtl - P.m_top) / P.sigma_top, t2 = (mwl - P.m_w) / P.sigma_w;
        consider(t1 * t1 + t2 * t2, 0, bt[i], -1, -1, s, mtl, NaN, mwl, NaN);
      }
    } else {
      for (int hyp = 0; hyp < 2; hyp++) for (int i = 0; i < nbt; i++)
        for (int a = 0; a < nlt; a++) for (int b = a + 1; b < nlt; b++) {
          const P4 whad = add(jet[lt[a]], jet[lt[b]]);
          const double mwh = mass4(whad), t4 = (mwh - P.m_w) / P.sigma_w;
          for (int s = 0; s < nsol; s++) {
            const P4 nu{nux, nuy, pz[s], std::sqrt(nux * nux + nuy * nuy + pz[s] * pz[s])};
            const P4 wlep = add(lep, nu);
            const double mwl = mass4(wlep), t2 = (mwl - P.m_w) / P.sigma_w;
            const double mt = hyp == 0 ? mass4(add(wlep, jet[bt[i]])) : mass4(add(whad, jet[bt[i]]));
            const double t1 = (mt - P.m_top) / P.sigma_top;
            consider((t1 * t1 + t2 * t2) + t4 * t4, hyp, bt[i], lt[a], lt[b], s, hyp == 0 ? mt : NaN, hyp == 1 ? mt : NaN, mwl, mwh);
          }
        }
    }
    o.status = (best < INFINITY) ? 1u : 0u;
    if (out_second) out_second[k] = second;
  }
  return 0;
}
