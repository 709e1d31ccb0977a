// oracle/oracle_chi2_dilep.cpp — CPU ORACLE (test infrastructure).  chi^2 kinematic reconstruction of DILEPTONIC ttbar events.
//
// PAPER.md:323-329 (section 6.2, eq. 1): chi^2 = sum_{k=1(2)} (m_jlnu - m_t)^2 / sigma_t^2 + sum_{m=1(2)} (m_lnu - m_W)^2 / sigma_W^2
// with m_t = 172.5, m_W = 80.4, sigma_t = 11.5, sigma_W = 7.5 GeV, minimised "for each possible jet and lepton combination";
// "the E_T^miss is assumed to be the transverse momentum of the undetected neutrino(s).  While for the semileptonic final
// states only the p_Z component of the neutrino four-momentum remains to be determined, for the dileptonic final states, two
// neutrinos must be fully reconstructed.  This implies, splitting the E_T^miss between the two neutrinos and determine, using
// the mass constraints from the chi^2" — and there the text breaks off.
//
// Reading (R15), written out step by step below with nothing hoisted or reordered:
//   1. ttbar: k = m = 2, one top and one W per lepton.  l+ goes with the b-jet, l- with the bbar-jet.
//   2. "Splitting the E_T^miss": the transverse momentum of the neutrino is scanned over a G x G grid centred on half the
//      measured MET vector M, nu_T = M/2 + R (u_gx, u_gy), u_g = (2 g + 1)/G - 1 (cell midpoints of [-1, 1]); the antineutrino
//      takes the rest, nubar_T = M - nu_T.  G = split_n (default 32), R = split_range (default 160 GeV).
//   3. "using the mass constraints": for each neutrino the p_z follows from its W exactly as in the semileptonic case
//      (orc_nu_pz: the two roots of m(l nu) = m_W, or the p_z that minimises m(l nu) when there is none).
//   4. The chi^2 of eq. (1) is evaluated for every ordered pair of b-tagged jets (first 4 tagged slots), every grid point and
//      every combination of the p_z solutions, as T1 + T2 with T1 = t_top^2 + t_W^2 of the l+ leg and T2 that of the l- leg;
//      the minimum wins, enumeration order (b, bbar, gx, gy, solution of nu, solution of nubar), strict <.
// Where the analytic dilepton solution exists (oracle_reco.cpp) chi^2 -> 0 at it as the grid is refined; where it does not,
// the scan returns the closest approach, which the exact solver cannot.
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

// one leg at one transverse neutrino momentum: for each p_z solution the neutrino, m(l nu), m(l nu b) and the leg's term
struct Leg { int nsol; double pz[2], mw[2], mt[2], term[2]; };
Leg leg_terms(const P4& lep, const P4& b, double nux, double nuy, const orc_chi2_params_t& P) {
  Leg L;
  const double la[4] = {lep.x, lep.y, lep.z, lep.e};
  L.nsol = orc_nu_pz(la, nux, nuy, P.m_w, L.pz);
  for (int s = 0; s < L.nsol; s++) {
    const P4 nu{nux, nuy, L.pz[s], std::sqrt(nux * nux + nuy * nuy + L.pz[s] * L.pz[s])};
    const P4 w = add(lep, nu), t = add(w, b);
    L.mw[s] = mass4(w); L.mt[s] = mass4(t);
    const double tt = (L.mt[s] - P.m_top) / P.sigma_top, tw = (L.mw[s] - P.m_w) / P.sigma_w;
    L.term[s] = tt * tt + tw * tw;
  }
  return L;
}
}  // namespace

extern "C" void orc_default_split(orc_split_t* s) { s->split_range = 160.0; s->split_n = 32; s->pad_ = 0; }

// chi^2 of one (l+ with jet slot sb, l- with jet slot sbbar) hypothesis at one split nu_T = (nux, nuy): out[2 s1 + s2] for the
// p_z solutions s1 of the neutrino and s2 of the antineutrino (NaN where a solution does not exist); returns nsol1 | nsol2 << 4.
extern "C" int orc_chi2_dilep_point(const orc_events_t* ev, uint32_t e, int sb, int sbbar, double nux, double nuy,
                                    const orc_chi2_params_t* params, double out[4], double pz_nu[2], double pz_nubar[2]) {
  orc_chi2_params_t P; if (params) P = *params; else orc_default_chi2_params(&P);
  const int64_t S = ev->stride;
  const uint32_t f = ev->flags[e];
  const int lp = ((f >> 4) & 1u) ? 0 : 1, lm = 1 - lp;     // l+ is the lepton whose charge bit is set
  const P4 lplus{ev->lep_px[lp * S + e], ev->lep_py[lp * S + e], ev->lep_pz[lp * S + e], ev->lep_e[lp * S + e]};
  const P4 lminus{ev->lep_px[lm * S + e], ev->lep_py[lm * S + e], ev->lep_pz[lm * S + e], ev->lep_e[lm * S + e]};
  const P4 b{ev->jet_px[sb * S + e], ev->jet_py[sb * S + e], ev->jet_pz[sb * S + e], ev->jet_e[sb * S + e]};
  const P4 bb{ev->jet_px[sbbar * S + e], ev->jet_py[sbbar * S + e], ev->jet_pz[sbbar * S + e], ev->jet_e[sbbar * S + e]};
  const double qx = ev->met_x[e] - nux, qy = ev->met_y[e] - nuy;
  const Leg L1 = leg_terms(lplus, b, nux, nuy, P), L2 = leg_terms(lminus, bb, qx, qy, P);
  const double NaN = std::numeric_limits<double>::quiet_NaN();
  for (int s1 = 0; s1 < 2; s1++) for (int s2 = 0; s2 < 2; s2++)
    out[2 * s1 + s2] = (s1 < L1.nsol && s2 < L2.nsol) ? L1.term[s1] + L2.term[s2] : NaN;
  for (int s = 0; s < 2; s++) { pz_nu[s] = s < L1.nsol ? L1.pz[s] : NaN; pz_nubar[s] = s < L2.nsol ? L2.pz[s] : NaN; }
  return L1.nsol | (L2.nsol << 4);
}

extern "C" int orc_chi2_dilep(const orc_events_t* ev, const uint32_t* idx, int64_t n_idx, const orc_chi2_params_t* params,
                              const orc_split_t* split, orc_chi2_dilep_t* out, double* out_second, int n_threads) {
  if (!ev || (n_idx > 0 && !idx) || n_idx < 0 || !out) return -1;
  orc_chi2_params_t P; if (params) P = *params; else orc_default_chi2_params(&P);
  orc_split_t G; if (split) G = *split; else orc_default_split(&G);
  if (G.split_n < 1 || G.split_n > 64 || !(G.split_range >= 0.0)) return -1;
  const double NaN = std::numeric_limits<double>::quiet_NaN();
  const int64_t S = ev->stride;
  const int n = G.split_n;
#pragma omp parallel for schedule(dynamic, 4) num_threads(n_threads > 1 ? n_threads : 1)   // whole events per thread: no arithmetic changes
  for (int64_t k = 0; k < n_idx; k++) {
    const uint32_t e = idx[k];
    orc_chi2_dilep_t& o = out[k];
    o.chi2 = o.m_top = o.m_antitop = o.m_wplus = o.m_wminus = NaN;
    for (int c = 0; c < 3; c++) o.nu[c] = o.nubar[c] = NaN;
    o.jet_b = o.jet_bbar = o.grid_x = o.grid_y = o.sol_nu = o.sol_nubar = -1; o.n_comb = 0; o.status = 0; o.event = e; o.pad_ = 0;
    if (out_second) out_second[k] = INFINITY;
    const uint32_t f = ev->flags[e];
    const int n_lep = (int)(f & 15u); int n_jet = (int)((f >> 8) & 15u); if (n_jet > 8) n_jet = 8;
    const bool q0 = (f >> 4) & 1u, q1 = (f >> 5) & 1u;
    int bt[4], nbt = 0;
    for (int s = 0; s < n_jet; s++) if (((f >> (16 + s)) & 1u) && nbt < 4) bt[nbt++] = s;
    if (n_lep != 2 || q0 == q1 || nbt < 2) { o.status = 2; continue; }
    const int lp = q0 ? 0 : 1, lm = 1 - lp;
    const P4 lplus{ev->lep_px[lp * S + e], ev->lep_py[lp * S + e], ev->lep_pz[lp * S + e], ev->lep_e[lp * S + e]};
    const P4 lminus{ev->lep_px[lm * S + e], ev->lep_py[lm * S + e], ev->lep_pz[lm * S + e], ev->lep_e[lm * S + e]};
    const double Mx = ev->met_x[e], My = ev->met_y[e];
    P4 jet[8];
    for (int s = 0; s < n_jet; s++) jet[s] = P4{ev->jet_px[s * S + e], ev->jet_py[s * S + e], ev->jet_pz[s * S + e], ev->jet_e[s * S + e]};
    double best = INFINITY, second = INFINITY;
    for (int i = 0; i < nbt; i++) for (int j = 0; j < nbt; j++) {
      if (i == j) continue;
      for (int gx = 0; gx < n; gx++) for (int gy = 0; gy < n; gy++) {
        const double ux = (double)(2 * gx + 1) / (double)n - 1.0, uy = (double)(2 * gy + 1) / (double)n - 1.0;
        const double nux = 0.5 * Mx + G.split_range * ux, nuy = 0.5 * My + G.split_range * uy;
        const double qx = Mx - nux, qy = My - nuy;
        const Leg L1 = leg_terms(lplus, jet[bt[i]], nux, nuy, P), L2 = leg_terms(lminus, jet[bt[j]], qx, qy, P);
        for (int s1 = 0; s1 < L1.nsol; s1++) for (int s2 = 0; s2 < L2.nsol; s2++) {
          const double chi2 = L1.term[s1] + L2.term[s2];
          o.n_comb++;
          if (chi2 < best) {
            second = best; best = chi2;
            o.chi2 = chi2;
            o.nu[0] = nux; o.nu[1] = nuy; o.nu[2] = L1.pz[s1]; o.nubar[0] = qx; o.nubar[1] = qy; o.nubar[2] = L2.pz[s2];
            o.m_top = L1.mt[s1]; o.m_wplus = L1.mw[s1]; o.m_antitop = L2.mt[s2]; o.m_wminus = L2.mw[s2];
            o.jet_b = bt[i]; o.jet_bbar = bt[j]; o.grid_x = gx; o.grid_y = gy; o.sol_nu = s1; o.sol_nubar = s2;
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
