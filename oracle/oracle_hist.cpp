// oracle/oracle_hist.cpp — CPU ORACLE (test infrastructure).  Histogram of a reconstructed quantity.
//
// PAPER.md:410-419 (App. 8.2): the analysis' finalize() writes histograms of reconstructed quantities; PAPER.md:278:
// variables are recorded per cut.  The definition (stated in include/hepf.h for the CUDA path and
// restated here independently): only records with status bit 0 are filled; t = (value - lo) * (nbins / (hi - lo)), each
// operation rounded once (compile with -ffp-contract=off); t < 0 -> underflow slot 0, t >= nbins -> overflow slot
// nbins + 1, else slot 1 + (int)t; NaN is not counted.  Fields: 0 m_top, 1 m_antitop, 2 m_wplus, 3 m_wminus, 4 m_higgs,
// 5 loglik, 6 pT(nu) = sqrt(px*px + py*py), 7 pT(nubar), 8 variation.
#include <cmath>
#include <cstdint>

#include "hepf_oracle.h"

static double field_of(const orc_best_t& b, int field) {
  switch (field) {
    case 0: return b.m_top;
    case 1: return b.m_antitop;
    case 2: return b.m_wplus;
    case 3: return b.m_wminus;
    case 4: return b.m_higgs;
    case 5: return b.loglik;
    case 6: return std::sqrt(b.nu[0] * b.nu[0] + b.nu[1] * b.nu[1]);
    case 7: return std::sqrt(b.nubar[0] * b.nubar[0] + b.nubar[1] * b.nubar[1]);
    default: return (double)b.variation;
  }
}

extern "C" int orc_histogram(const orc_best_t* best, int64_t n, int field, double lo, double hi, int32_t nbins,
                             uint64_t* out) {
  if (n < 0 || nbins < 1 || !(hi > lo) || field < 0 || field > 8 || !out) return -1;
  for (int i = 0; i < nbins + 2; i++) out[i] = 0;
  const double inv_w = (double)nbins / (hi - lo);
  for (int64_t k = 0; k < n; k++) {
    if (!(best[k].status & 1u)) continue;
    const double v = field_of(best[k], field);
    const double t = (v - lo) * inv_w;
    if (t != t) continue;
    if (t < 0.0) out[0]++;
    else if (t >= (double)nbins) out[nbins + 1]++;
    else out[1 + (int)t]++;
  }
  return 0;
}

// The same binning for a plain column of doubles, element k at values[k * stride]: the per-event variables a cut or the
// reconstruction wrote (ETmis, m_ttH, pT_ttH: PAPER.md:278-295, :410-442).  Every finite value is filled; NaN marks "no value".
extern "C" int orc_histogram_values(const double* values, int64_t stride, int64_t n, double lo, double hi, int32_t nbins,
                                    uint64_t* out) {
  if (n < 0 || nbins < 1 || !(hi > lo) || stride < 1 || !out || (n > 0 && !values)) return -1;
  for (int i = 0; i < nbins + 2; i++) out[i] = 0;
  const double inv_w = (double)nbins / (hi - lo);
  for (int64_t k = 0; k < n; k++) {
    const double t = (values[k * stride] - lo) * inv_w;
    if (t != t) continue;
    if (t < 0.0) out[0]++;
    else if (t >= (double)nbins) out[nbins + 1]++;
    else out[1 + (int)t]++;
  }
  return 0;
}
