// oracle/oracle_select.cpp — CPU ORACLE (test infrastructure).  O3: the ordered cut chain.
//
// PAPER.md:96-102 (§3): a cut is a boolean function of one event, cuts are registered in order and an event
// is dropped at the first `false`; PAPER.md:286-295 (§6.1 listing): thresholds are strict ("<= -> fail").
// The output of the chain is the list of surviving events (the paper's filtered output) and,
// optionally, the cutflow.  Cut kinds: SURVEY.md §8(c) O3.  The definition is the loop below and nothing else.
#include <cmath>
#include <cstdint>

#include "hepf_oracle.h"

static bool pass_cut(const orc_events_t* ev, int64_t i, const orc_cut_t& c) {
  const int64_t S = ev->stride;
  const uint32_t f = ev->flags[i];
  const int n_lep = (int)(f & 15u);
  int n_jet = (int)((f >> 8) & 15u);
  if (n_jet > 8) n_jet = 8;
  switch (c.kind) {
    case ORC_NLEP_EQ: return n_lep == (int)c.n;
    case ORC_LEP_OS: return ((f >> 4) & 1u) != ((f >> 5) & 1u);
    case ORC_LEP_PT_GT: return ev->lep_pt[0 * S + i] > c.lo && ev->lep_pt[1 * S + i] > c.lo;
    case ORC_LEP_ABSETA_LT:
      return std::fabs(ev->lep_eta[0 * S + i]) < c.hi && std::fabs(ev->lep_eta[1 * S + i]) < c.hi;
    case ORC_NJET_GE:
    case ORC_NBJET_GE: {
      int count = 0;
      for (int s = 0; s < n_jet; s++) {
        bool ok = ev->jet_pt[s * S + i] > c.lo && std::fabs(ev->jet_eta[s * S + i]) < c.hi;
        if (c.kind == ORC_NBJET_GE) ok = ok && ((f >> (16 + s)) & 1u);
        if (ok) count++;
      }
      return count >= (int)c.n;
    }
    case ORC_MET_GT: return ev->met[i] > c.lo;
    case ORC_MET_GT_RECORD: return ev->met[i] > c.lo;   // the side effect is in orc_select_record
    case ORC_MLL_GT: return ev->mll[i] > c.lo;
    case ORC_MLL_OUTSIDE: return ev->mll[i] < c.lo || ev->mll[i] > c.hi;
    default: return false;  // unknown kind: nothing passes
  }
}

extern "C" int orc_select(const orc_events_t* ev, const orc_cut_t* cuts, int n_cuts, uint32_t* out_idx,
                          int64_t* out_count, int64_t* out_cutflow) {
  if (!ev || n_cuts < 0 || n_cuts > 32 || (n_cuts > 0 && !cuts)) return -1;
  int64_t n = 0;
  if (out_cutflow) for (int c = 0; c < n_cuts; c++) out_cutflow[c] = 0;
  for (int64_t i = 0; i < ev->n_events; i++) {
    bool alive = true;
    for (int c = 0; c < n_cuts && alive; c++) {
      alive = pass_cut(ev, i, cuts[c]);
      if (alive && out_cutflow) out_cutflow[c]++;  // cutflow[c] = events that passed cuts 0..c
    }
    if (alive) { if (out_idx) out_idx[n] = (uint32_t)i; n++; }
  }
  if (out_count) *out_count = n;
  return 0;
}

// PAPER.md:278-295 (§6.1 listing): a cut may write a new per-event variable when it passes — the paper's example is the
// missing-E_T cut, "if (met_met <= 30000.) return false; else { ETmis = met_met; ETmis *= 1.05; return true; }" — and
// such a variable holds a default value "for levels where the information was not yet updated".
// ORC_MET_GT_RECORD is that cut: met > lo, and on passing derived[i] = met * hi (one rounded multiplication); an event
// that does not reach the cut, or fails it, keeps derived_default.  Everything else is orc_select.
extern "C" int orc_select_record(const orc_events_t* ev, const orc_cut_t* cuts, int n_cuts, uint32_t* out_idx,
                                 int64_t* out_count, int64_t* out_cutflow, double* out_derived, double derived_default) {
  if (!ev || n_cuts < 0 || n_cuts > 32 || (n_cuts > 0 && !cuts)) return -1;
  int64_t n = 0;
  if (out_cutflow) for (int c = 0; c < n_cuts; c++) out_cutflow[c] = 0;
  for (int64_t i = 0; i < ev->n_events; i++) {
    if (out_derived) out_derived[i] = derived_default;
    bool alive = true;
    for (int c = 0; c < n_cuts && alive; c++) {
      alive = pass_cut(ev, i, cuts[c]);
      if (alive && cuts[c].kind == ORC_MET_GT_RECORD && out_derived) out_derived[i] = ev->met[i] * cuts[c].hi;
      if (alive && out_cutflow) out_cutflow[c]++;
    }
    if (alive) { if (out_idx) out_idx[n] = (uint32_t)i; n++; }
  }
  if (out_count) *out_count = n;
  return 0;
}

// PAPER.md:194-196 (§5.2): the framework measures each cut's filter ratio (and execution time) to order the pipeline.  The
// filter ratio of a cut ON ITS OWN: out_pass[c] = events of the sample that pass cut c alone, out_pass[n_cuts] = sample size.
// The sample is every `sample_every`-th block of 512 consecutive events (blocks 0, sample_every, 2 sample_every, ...).
extern "C" int orc_cut_stats(const orc_events_t* ev, const orc_cut_t* cuts, int n_cuts, int64_t sample_every, int64_t* out_pass) {
  if (!ev || n_cuts < 0 || n_cuts > 32 || (n_cuts > 0 && !cuts) || sample_every < 1 || !out_pass) return -1;
  for (int c = 0; c <= n_cuts; c++) out_pass[c] = 0;
  for (int64_t i = 0; i < ev->n_events; i++) {
    if ((i / 512) % sample_every != 0) continue;
    out_pass[n_cuts]++;
    for (int c = 0; c < n_cuts; c++) if (pass_cut(ev, i, cuts[c])) out_pass[c]++;
  }
  return 0;
}
