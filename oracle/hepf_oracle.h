/*
 * oracle/hepf_oracle.h — CPU ORACLE (TEST INFRASTRUCTURE, NOT THE PRODUCT).
 *
 * Plain, slow, obviously-correct FP64 restatement of the ttH hot path of arXiv 2211.14346 (HEP-Frame),
 * §4 "ttH case study": ordered boolean cuts, then per
 * event x smearing variation x b-jet/lepton pairing the analytic dilepton neutrino reconstruction with
 * m_W = 80.4, m_t = 172.5 and the Higgs pair at 125 GeV, "highest probability" wins.
 * The paper gives no equations (they are in its ref. [27]); the step-by-step definition followed here is
 * SURVEY.md §8(c) O1-O4 with the readings R1-R13 listed in DESIGN.md.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may use this
 * library.  It shares no code, header, table or constant generator with the CUDA path under
 * paper_2211_14346_b200/csrc: the struct definitions below are this tree's own declarations.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"):
 *   O1 Philox4x32-10 ......... known-answer vectors (tests/golden/philox_kat.txt)
 *   O2 uniforms / normals .... six printed hex-float normals, slice consistency, moments,
 *                              det-log / det-sincos against libm within 4 ulp
 *   O3 select ................ hand-built threshold tables, numpy restatement, cutflow invariants
 *   O4 conic/quartic algebra . worked example (tests/golden/worked_example.txt), closure invariant,
 *                              truth recovery in closure mode, multi-start Newton brute force on the
 *                              raw mass constraints, dense-grid sign-change brute force on the quartic
 *   O4 score / argmax ........ prefix property in V, sigma_scale = 0, z-rotation invariance, slot permutation
 *   chi2 (semileptonic) ...... p_z against a dense scan of m(l nu), truth recovery in closure mode (chi2 = 0 at the true
 *                              combination), brute-force enumeration in numpy, permutation invariance
 *   chi2 (dileptonic) ........ chi2 = 0 at the generator's true neutrinos and pairing (closure mode) and at the roots of the
 *                              pinned dilepton solve (orc_solve_pairing); the grid argmin against a Python loop over
 *                              orc_chi2_dilep_point; 90-degree rotation about z maps the grid onto itself
 *   histogram ................ hand-built edge cases (lower edge in, upper edge overflow, NaN, unsolved), numpy restatement
 *   PARITY UNPINNED against the paper: the likelihood formula, sigma_H, lambda_nu, the resolution model
 *   and the 8-cut thresholds are definitions of this build (R3, R7, R10), not paper values.
 */
#ifndef HEPF_ORACLE_H
#define HEPF_ORACLE_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  int64_t n_events, stride, event_base;
  const double *lep_px, *lep_py, *lep_pz, *lep_e, *lep_pt, *lep_eta; /* [2][stride] */
  const double *jet_px, *jet_py, *jet_pz, *jet_e, *jet_pt, *jet_eta; /* [8][stride] */
  const double *met_x, *met_y, *met, *mll;                           /* [stride]    */
  const uint32_t* flags;
} orc_events_t;

typedef struct { uint32_t kind, n; double lo, hi; } orc_cut_t;
enum { ORC_NLEP_EQ = 1, ORC_LEP_OS, ORC_LEP_PT_GT, ORC_LEP_ABSETA_LT, ORC_NJET_GE, ORC_NBJET_GE, ORC_MET_GT,
       ORC_MLL_GT, ORC_MLL_OUTSIDE, ORC_MET_GT_RECORD };

typedef struct {
  double m_top, m_w, m_higgs, sigma_higgs, lambda_nu, lep_sigma, jet_stoch, jet_const, sigma_scale, s_min;
} orc_params_t;

typedef struct {
  double nu[3], nubar[3];
  double m_top, m_antitop, m_wplus, m_wminus, m_higgs, loglik;
  int32_t variation, jet_b, jet_bbar, jet_h1, jet_h2, root;
  uint32_t status, event;
} orc_best_t;

typedef struct {      /* per-event diagnostics the parity harness needs (R11) */
  double kappa;       /* eps * sum|h_i x^i| / |x P'(x)| of the winning root            */
  double loglik2;     /* best log-likelihood among all other candidates (-inf if none)  */
  int64_t n_cand;     /* candidates enumerated                                          */
  int32_t pairing, higgs_pair; /* a = i*n_b + j and h of the winner                     */
  double pz_terms, pzbar_terms; /* |c0|+|c1 x|+|c2 y| of the two p_z linear forms (R11b)  */
} orc_aux_t;

typedef struct {      /* one pairing solved in isolation (worked example, brute-force pins, R11 ii/iii) */
  int32_t n_roots, n_higgs;
  double g[4];        /* monic quartic x^4 + g3 x^3 + g2 x^2 + g1 x + g0: g[0]=g0 .. g[3]=g3 */
  double h[5];        /* raw resultant coefficients h0..h4                                    */
  double conic1[6], conic2[6]; /* a b c d e f; conic2 already shifted by MET'                 */
  double x[4], kappa[4], nterm[4];
  double nu[4][4], nubar[4][4];  /* px py pz E per root                                        */
  double hterm[6], mbb[6];
  double min_abs_p_rel; /* min over critical points of |P|/sum|h_i x^i| (near-tangency measure) */
  double pz_terms[4], pzbar_terms[4]; /* per root: |c0|+|c1 x|+|c2 y| of the two p_z linear forms */
} orc_pairing_t;

void orc_default_params(orc_params_t* p);

/* O1 */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* O2 */
double orc_det_log(double u);
void orc_det_sincos2pi(double u, double* s, double* c);
void orc_philox_normal(uint64_t seed, uint64_t counter, uint64_t n, double* out);
/* O3 */
int orc_select(const orc_events_t* ev, const orc_cut_t* cuts, int n_cuts, uint32_t* out_idx, int64_t* out_count,
               int64_t* out_cutflow);
/* a chain with a recording cut (ORC_MET_GT_RECORD): see oracle_select.cpp */
int orc_select_record(const orc_events_t* ev, const orc_cut_t* cuts, int n_cuts, uint32_t* out_idx, int64_t* out_count,
                      int64_t* out_cutflow, double* out_derived, double derived_default);
/* per-cut filter ratios on a sample (oracle_select.cpp) */
int orc_cut_stats(const orc_events_t* ev, const orc_cut_t* cuts, int n_cuts, int64_t sample_every, int64_t* out_pass);
/* O4: n_threads > 1 only distributes whole events over OpenMP threads; per-event arithmetic is unchanged */
int orc_reconstruct_tth(const orc_events_t* ev, const uint32_t* idx, int64_t n_idx, int32_t n_variations,
                        uint64_t seed, const orc_params_t* params, orc_best_t* out_best, orc_aux_t* out_aux,
                        int n_threads);
/* one pairing from explicit four-vectors (px,py,pz,E); jets_h = n_h remaining b candidates (<= 4) */
int orc_solve_pairing(const double lp[4], const double b[4], const double lm[4], const double bbar[4],
                      const double met[2], const double* jets_h, int n_h, const orc_params_t* params,
                      orc_pairing_t* out);
/* the (event, variation, pairing a) cell of orc_reconstruct_tth, re-evaluated on request */
int orc_eval_cell(const orc_events_t* ev, uint32_t e, int32_t v, int32_t a, uint64_t seed,
                  const orc_params_t* params, orc_pairing_t* out);
/* the root finder alone: real simple roots (ascending) of the monic quartic g0..g3 and its tangency measure */
int orc_quartic(const double g[4], double roots[4], double* min_abs_p_rel);
/* smeared objects of one (event, variation): scales[10], met'[2] */
int orc_smear(const orc_events_t* ev, uint32_t e, int32_t v, uint64_t seed, const orc_params_t* params,
              double scales[10], double metp[2]);

/* chi^2 reconstruction of semileptonic ttbar (eq. 1; oracle_chi2.cpp) */
typedef struct { double m_top, m_w, sigma_top, sigma_w; } orc_chi2_params_t;
typedef struct {
  double chi2, nu_pz, m_top_lep, m_top_had, m_w_lep, m_w_had;
  int32_t jet_b_lep, jet_b_had, jet_q1, jet_q2, solution, n_comb;
  uint32_t status, event;
} orc_chi2_t;   /* 80 bytes */
void orc_default_chi2_params(orc_chi2_params_t* p);
int orc_nu_pz(const double lep[4], double nux, double nuy, double m_w, double pz[2]);
int orc_chi2_semilep(const orc_events_t* ev, const uint32_t* idx, int64_t n_idx, const orc_chi2_params_t* params,
                     orc_chi2_t* out, double* out_second);
/* single-top variants of eq. (1): mode 1 = t-channel (1 top, 1 W), mode 2 = Wt (1 top, 2 W), semileptonic final state */
int orc_chi2_single_top(const orc_events_t* ev, const uint32_t* idx, int64_t n_idx, int mode, const orc_chi2_params_t* params,
                        orc_chi2_t* out, double* out_second);

/* chi^2 reconstruction of DILEPTONIC ttbar (oracle_chi2_dilep.cpp, reading R15 of DESIGN.md): the neutrino's
 * transverse momentum is scanned over a split_n x split_n grid of half-width split_range around MET/2, the antineutrino
 * takes the rest of the MET, each p_z follows from its W as in the semileptonic case */
typedef struct { double split_range; int32_t split_n, pad_; } orc_split_t;
typedef struct {
  double chi2, nu[3], nubar[3], m_top, m_antitop, m_wplus, m_wminus;
  int32_t jet_b, jet_bbar, grid_x, grid_y, sol_nu, sol_nubar, n_comb;
  uint32_t status, event; int32_t pad_;
} orc_chi2_dilep_t;   /* 128 bytes */
void orc_default_split(orc_split_t* s);
int orc_chi2_dilep_point(const orc_events_t* ev, uint32_t e, int sb, int sbbar, double nux, double nuy,
                         const orc_chi2_params_t* params, double out[4], double pz_nu[2], double pz_nubar[2]);
int orc_chi2_dilep(const orc_events_t* ev, const uint32_t* idx, int64_t n_idx, const orc_chi2_params_t* params,
                   const orc_split_t* split, orc_chi2_dilep_t* out, double* out_second, int n_threads);

/* histogram of a field of the records (oracle_hist.cpp; pin: numpy restatement + hand-built edge cases) */
int orc_histogram(const orc_best_t* best, int64_t n, int field, double lo, double hi, int32_t nbins, uint64_t* out);

/* invariant mass and transverse momentum of the reconstructed ttH system of each record (oracle_reco.cpp), out[2k], out[2k+1] */
int orc_tth_system(const orc_events_t* ev, const orc_best_t* best, int64_t n, uint64_t seed, const orc_params_t* params,
                   double* out);
/* histogram of a plain column of doubles with the rules of orc_histogram (NaN not counted, every value filled) */
int orc_histogram_values(const double* values, int64_t stride, int64_t n, double lo, double hi, int32_t nbins, uint64_t* out);

#ifdef __cplusplus
}
#endif
#endif
