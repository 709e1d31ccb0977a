/*
 * include/hepf.h — C ABI of libhepf: the ttH selection + kinematic-reconstruction hot path of
 * arXiv 2211.14346 (HEP-Frame, §4 "ttH case study") as hand-written CUDA for sm_100a (one B200 per process).
 *
 * Conventions (all entry points)
 *   - plain C types only; no exceptions cross the boundary.
 *   - "device" pointers are caller-owned device memory (e.g. torch tensors); "host" pointers are ordinary
 *     host memory read during the call.  The library never allocates or frees device memory: scratch space
 *     is a caller-provided workspace whose size the *_workspace_bytes functions return.
 *   - every device entry point only ENQUEUES work on `stream` (a cudaStream_t passed as void*; NULL = the
 *     legacy default stream) and returns; results are valid after the caller synchronises that stream.
 *     hepf_tth_host is the exception: it takes host buffers and returns after its results are on the host.
 *   - return value: HEPF_OK or a negative error code; hepf_last_error() gives a host string (thread-local)
 *     for the last failure.  On error nothing is guaranteed about the output buffers.
 *   - there is NO CPU fallback: without a CUDA device every compute entry point returns HEPF_ERR_CUDA.
 *   - units GeV; FP64 throughout ("dtype f64").
 */
#ifndef HEPF_H
#define HEPF_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define HEPF_OK 0
#define HEPF_ERR_ARG (-1)      /* null / misaligned pointer, negative size, n_cuts > 32, n_variations < 1, odd stride, n_variations > 2^21 */
#define HEPF_ERR_CAPACITY (-2) /* workspace or arena too small                                                    */
#define HEPF_ERR_CUDA (-3)     /* CUDA runtime / launch failure, or no device                                     */

#define HEPF_MAX_CUTS 32
#define HEPF_N_LEP 2
#define HEPF_N_JET 8
#define HEPF_MAX_B 6

/*
 * SoA event store: a VIEW of caller-owned columns (§3: all in-flight events are kept in
 * memory by the framework and are visible to every cut).  Column c of object slot s lives at
 * ptr[s * stride + event].  Leptons and jets are pT-ordered; unused slots hold zeros.
 *   stride      >= n_events, even (so that every slot row is 16-byte aligned); every pointer 16-byte aligned.
 *   event_base  global index of event 0 of this view: the smearing stream of event e is keyed by
 *               event_base + e, so results do not depend on how a sample is split into views / ranks.
 *   flags       bits 0-3 n_lep | bit 4 q(lep0) > 0 | bit 5 q(lep1) > 0 | bits 8-11 n_jet | bits 16-23 b-tag mask.
 */
typedef struct {
  int64_t n_events, stride, event_base;
  const double *lep_px, *lep_py, *lep_pz, *lep_e, *lep_pt, *lep_eta; /* [2][stride] */
  const double *jet_px, *jet_py, *jet_pz, *jet_e, *jet_pt, *jet_eta; /* [8][stride] */
  const double *met_x, *met_y, *met, *mll;                           /* [stride]    */
  const uint32_t* flags;                                             /* [stride]    */
} hepf_events_t;

/*
 * One cut of the ordered chain (`bool cut(event)`, registered in order, an event is dropped
 * at the first false; thresholds are strict — "met <= 30000 -> fail").  A comparison with a
 * NaN is false, so the event fails.  Jet counts look at slots 0 .. n_jet-1 only.
 */
typedef enum {
  HEPF_CUT_NLEP_EQ = 1,       /* n_lep == n                                            */
  HEPF_CUT_LEP_OS = 2,        /* lepton charge bits differ                             */
  HEPF_CUT_LEP_PT_GT = 3,     /* both leptons: pt > lo                                 */
  HEPF_CUT_LEP_ABSETA_LT = 4, /* both leptons: |eta| < hi                              */
  HEPF_CUT_NJET_GE = 5,       /* #jets with pt > lo and |eta| < hi  >= n               */
  HEPF_CUT_NBJET_GE = 6,      /* same, b-tagged jets only                              */
  HEPF_CUT_MET_GT = 7,        /* met > lo                                              */
  HEPF_CUT_MLL_GT = 8,        /* mll > lo                                              */
  HEPF_CUT_MLL_OUTSIDE = 9,   /* mll < lo or mll > hi                                  */
  HEPF_CUT_MET_GT_RECORD = 10 /* met > lo; on passing writes the derived variable met * hi (hepf_select_record) */
} hepf_cut_kind_t;
typedef struct { uint32_t kind; uint32_t n; double lo, hi; } hepf_cut_t;

/* Parameters of the reconstruction (NULL = defaults).  m_top, m_w, m_higgs: PAPER.md:138 (172.5, 80.4, 125).
 * lep_sigma 0.01: PAPER.md:145; jet resolution sigma/E = jet_stoch/sqrt(E) + jet_const (0.5, 0.03):
 * BASELINE.json configs[0].  sigma_higgs 15, lambda_nu 40, sigma_scale 1, s_min 0.1: definitions of this
 * build (readings R3-R7). */
typedef struct {
  double m_top, m_w, m_higgs, sigma_higgs, lambda_nu, lep_sigma, jet_stoch, jet_const, sigma_scale, s_min;
} hepf_tth_params_t;

/* Best solution of one event ("the one with highest probability is considered to be the correct
 * solution"; "only the highest probable solution was considered").  128 bytes.
 * status bits: 1 = has a solution; 2 = not applicable (n_lep != 2, same-sign, < 4 b candidates);
 *              4 = more than 6 b candidates, truncated to the 6 lowest slots;
 *              8 = idx[k] >= n_events (the entry is treated as not applicable: bits 2 and 8, NaN / -1 payload).
 * Without a solution the floating-point payload is NaN and the integer payload is -1 (the paper's "discards the
 * event if no solution was found"). */
typedef struct {
  double nu[3], nubar[3];                                        /* neutrino / antineutrino 3-momenta        */
  double m_top, m_antitop, m_wplus, m_wminus, m_higgs, loglik;   /* recomputed from the output four-vectors  */
  int32_t variation, jet_b, jet_bbar, jet_h1, jet_h2, root;      /* jet_* are jet slot indices; root = rank  */
  uint32_t status, event;                                        /* event = idx[k] (index inside the view)   */
} hepf_best_t;

/*
 * hepf_select — evaluate the cut chain, one thread per event, and compact the survivors (PAPER.md:96-102,
 * :122 filtered output, §4 :136 "eighteen cuts, organised in a sequential way").
 *   events       host pointer to a view of DEVICE columns.
 *   host_cuts    host array of n_cuts (0..32) cuts, applied in order.
 *   out_idx      device, capacity n_events: ascending indices of surviving events (stable compaction).
 *   out_count    device int64: number of survivors.
 *   out_cutflow  device int64[n_cuts] or NULL: cutflow[c] = events that passed cuts 0..c.
 *   ws           device workspace of at least hepf_select_workspace_bytes(n_events) bytes, 16-byte aligned.
 */
int hepf_select(const hepf_events_t* events, const hepf_cut_t* host_cuts, int n_cuts, uint32_t* out_idx,
                int64_t* out_count, int64_t* out_cutflow, void* ws, size_t ws_bytes, void* stream);
size_t hepf_select_workspace_bytes(int64_t n_events);
/*
 * hepf_select_record — hepf_select for a chain that holds one RECORDING cut (section 6.1: a cut may
 * write a new per-event variable when it passes; the paper's example is "if (met_met <= 30000.) return false; else
 * { ETmis = met_met; ETmis *= 1.05; return true; }").  HEPF_CUT_MET_GT_RECORD is that cut: it passes if met > lo and then
 * sets the derived variable of the event to met * hi (one IEEE multiplication).  Events that fail it, or an earlier cut, keep
 * `derived_default` ("for levels where the information was not yet updated, their default value is used").
 *   out_derived  device double[n_events], 16-byte aligned: the derived column (the paper's ETmis), one value per event.
 * In hepf_select the same cut kind only filters.  At most one recording cut per chain.
 */
int hepf_select_record(const hepf_events_t* events, const hepf_cut_t* host_cuts, int n_cuts, uint32_t* out_idx,
                       int64_t* out_count, int64_t* out_cutflow, double* out_derived, double derived_default, void* ws,
                       size_t ws_bytes, void* stream);

/*
 * The device analogue of the paper's cut-level scheduler (section 5.2: "HEP-Frame dynamically optimises
 * the ordering of the cuts during execution", from each cut's measured filter ratio and execution time, "respecting the
 * dependencies among cuts").  On the GPU a cut's cost is the bytes of the columns it reads, and the lever is not the order of
 * the compares but WHICH EVENTS' columns are fetched at all: a chain is split into two phases, phase 1 (cheap columns) over
 * every event, phase 2 (the rest) over phase 1's survivors only.
 *   hepf_cut_stats      measures: every cut on its own on the events of every `sample_every`-th tile of 512 events;
 *                       out_pass device int64[n_cuts + 1]: [c] = events that pass cut c, [n_cuts] = events looked at.
 *   hepf_plan_chain     decides (host only, no device): given the measured pass fractions and a dependency mask (bit k of
 *                       dep_mask[c] set = cut c must not run in an earlier phase than cut k; NULL = cuts commute), the phase-1 set
 *                       that minimises the expected bytes read per event,
 *                         4 + B(phase 1) + (1 - (1 - p1)^8) (4 + B(phase 2)) / 0.55 + 8 p1,   p1 = product over phase 1's cut families (cuts
 *                       reading the same columns count once, with their smallest pass fraction) of the pass fractions,
 *                       B = bytes of the column groups named.  Phase 2 gathers: it moves whole 64-byte DRAM atoms (eight events of
 *                       a column; fetched if any of them survives) at about 55 % of the streaming bandwidth (measured on B200).
 *                       One phase is kept unless two save at least 10 %.  out_order: a permutation of the cuts,
 *                       phase 1 first, user order inside a phase; out_split: cuts [0, split) of it form phase 1 (n_cuts = one
 *                       phase); out_bytes_per_event (or NULL): [0] planned, [1] one phase.
 *   hepf_select_planned executes a chain in that order with that split.  The survivor list is that of hepf_select (cuts are
 *                       pure predicates: the set does not depend on the order; the list stays ascending).  out_cutflow, if
 *                       given, is in EXECUTED order: [k] = events that passed the first k + 1 executed cuts.  A recording
 *                       cut cannot be planned.  ws >= hepf_select_planned_workspace_bytes(n_events), 256-byte aligned.
 */
int hepf_cut_stats(const hepf_events_t* events, const hepf_cut_t* host_cuts, int n_cuts, int64_t sample_every,
                   int64_t* out_pass, void* stream);
int hepf_plan_chain(const hepf_cut_t* host_cuts, int n_cuts, const double* pass_frac, const uint32_t* dep_mask, int* out_order,
                    int* out_split, double* out_bytes_per_event);
int hepf_select_planned(const hepf_events_t* events, const hepf_cut_t* host_cuts, int n_cuts, const int* order, int split,
                        uint32_t* out_idx, int64_t* out_count, int64_t* out_cutflow, void* ws, size_t ws_bytes, void* stream);
size_t hepf_select_planned_workspace_bytes(int64_t n_events);

/*
 * hepf_select_static — hepf_select (§4 :136) for callers that cannot allocate device memory
 * (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): same arguments, same kernels and
 * byte-identical results, but no workspace argument.  The per-warp pass masks and the per-block survivor counts live in
 * a file-scope device array of the library, HEPF_SELECT_STATIC_BYTES (about 0.5 MB) on EVERY GPU that loads the library,
 * held until the process exits.  The call allocates nothing: no cudaMalloc / cudaFree and no allocating library routine;
 * its first call on a device looks the array's device address up (cudaGetSymbolAddress, with that device current) and
 * caches it per device, so make one call per device before a capture starts.
 *   events->n_events <= HEPF_SELECT_STATIC_MAX_EVENTS, otherwise HEPF_ERR_CAPACITY (hepf_last_error says so) and nothing
 *   is launched.  Everything else — host/device placement, alignment, ownership, asynchrony on `stream` — as hepf_select.
 * The array is shared by every call on that GPU and keeps the last call's contents.  Nothing in it has to start at zero
 * (every word a call reads was written by the same call's select_eval_kernel), so it is not cleared; but two calls that
 * OVERLAP on the GPU (different streams, or threads, without an ordering between them) race on it and give wrong
 * survivor lists.  Calls on one stream, or ordered by events, are safe.
 */
#define HEPF_SELECT_STATIC_MAX_EVENTS 4194304 /* 2^22 events (BASELINE.json configs[1] has 4e6)                      */
#define HEPF_SELECT_STATIC_BYTES 540928       /* = hepf_select_workspace_bytes(HEPF_SELECT_STATIC_MAX_EVENTS)         */
int hepf_select_static(const hepf_events_t* events, const hepf_cut_t* host_cuts, int n_cuts, uint32_t* out_idx,
                       int64_t* out_count, int64_t* out_cutflow, void* stream);

/*
 * hepf_reconstruct_tth — for each listed event: for every smearing variation v < n_variations draw ten
 * standard normals from Philox4x32-10 keyed (seed; event_base+e, v, block) + Box-Muller, scale the two leptons
 * and the jets, propagate the change to the missing transverse momentum, and for every ordered pair of b-jet
 * candidates solve the dileptonic ttbar kinematics (two leg conics -> quartic; Ferrari closed form + Newton
 * polish, FP64), score every solution (Higgs pair mass term + neutrino pT term) and keep the best over
 * variations x pairings x Higgs pairs x roots (§4; definition: DESIGN.md "Method").
 *   idx          device uint32[n_idx]: events to reconstruct (normally hepf_select's out_idx); an entry >= n_events
 *                gets status 2 | 8 and no event data is read for it.
 *   n_idx        host value.
 *   host_params  host pointer or NULL.
 *   out_best     device hepf_best_t[n_idx], 16-byte aligned; out_best[k] belongs to idx[k].
 *   ws           device workspace >= hepf_reconstruct_workspace_bytes(n_idx, n_variations), 8-byte aligned: one
 *                8-byte winner key per listed event, written by the search kernels and read by the finalize kernel, two
 *                8-byte work counters, and 42 columns of n_idx doubles in which the search kernels leave the nominal
 *                objects of the events they reconstructed (344 bytes per listed event in all), so that the finalize
 *                kernel reads them coalesced instead of gathering them from the store again.
 */
int hepf_reconstruct_tth(const hepf_events_t* events, const uint32_t* idx, int64_t n_idx, int32_t n_variations,
                         uint64_t seed, const hepf_tth_params_t* host_params, hepf_best_t* out_best, void* ws,
                         size_t ws_bytes, void* stream);
size_t hepf_reconstruct_workspace_bytes(int64_t n_idx, int32_t n_variations);
/*
 * hepf_reconstruct_tth_n — the same operation with the LENGTH OF THE LIST IN DEVICE MEMORY, so that select ->
 * reconstruct needs no host round trip in the middle of the path (the reconstruction is the last cut of one
 * pipeline): the kernels read *n_idx_device (normally hepf_select's out_count) when they run, clamped to [0, n_idx_cap].
 *   n_idx_device device int64, 8-byte aligned;  n_idx_cap host value: capacity of idx / out_best (e.g. n_events);
 *   ws           >= hepf_reconstruct_workspace_bytes(n_idx_cap, n_variations).   Everything else as above; records
 *   beyond the device-side length are not written.
 */
int hepf_reconstruct_tth_n(const hepf_events_t* events, const uint32_t* idx, const int64_t* n_idx_device, int64_t n_idx_cap,
                           int32_t n_variations, uint64_t seed, const hepf_tth_params_t* host_params, hepf_best_t* out_best,
                           void* ws, size_t ws_bytes, void* stream);
void hepf_default_params(hepf_tth_params_t* host_params);

/*
 * hepf_philox_normal — out[i] = Z[counter + i], i < n, of the single infinite stream of standard normals
 * Z[g]: Philox block b = g >> 1 with counter words (b mod 2^32, b >> 32, 0, 0) and key (seed mod 2^32,
 * seed >> 32); (Z[2b], Z[2b+1]) = rho (cos, sin)(2 pi u2), rho = sqrt(-2 ln u1) (the exact
 * operation sequence, identical bits for any split of a range into calls or blocks).  The paper's PRNG
 * offload: §5.3.   out: device double[n], 8-byte aligned.
 */
int hepf_philox_normal(uint64_t seed, uint64_t counter, uint64_t n, double* out, void* stream);

/*
 * hepf_tth_host — the whole path from HOST buffers: copies the columns of `host_events` (a view of HOST
 * memory, pinned for full speed) to the device arena, runs hepf_select and hepf_reconstruct_tth and copies the
 * results back.  Large samples are cut into up to 10 chunks of consecutive events whose copies (two internal copy
 * streams) overlap the kernels of the neighbouring chunks; the results are byte-identical to the device entry points
 * on one view.  Synchronous: returns when host_out_* are filled.
 *   host_out_idx   host uint32[n_events] or NULL;  host_out_best  host hepf_best_t[n_events] (first n_sel used);
 *   host_out_count host int64;  host_out_cutflow host int64[n_cuts] or NULL.
 *   arena          device scratch >= hepf_tth_host_arena_bytes(n_events, n_variations), 256-byte aligned.
 */
int hepf_tth_host(const hepf_events_t* host_events, const hepf_cut_t* host_cuts, int n_cuts, int32_t n_variations,
                  uint64_t seed, const hepf_tth_params_t* host_params, uint32_t* host_out_idx,
                  hepf_best_t* host_out_best, int64_t* host_out_count, int64_t* host_out_cutflow, void* arena,
                  size_t arena_bytes, void* stream);
size_t hepf_tth_host_arena_bytes(int64_t n_events, int32_t n_variations);

/*
 * hepf_chi2_semilep — chi^2 kinematic reconstruction of semileptonic ttbar events (section 6.2, eq. 1;
 * SURVEY.md 8(f) NEXT-2):  chi^2 = ((m_blnu - m_t)/sigma_t)^2 + ((m_lnu - m_W)/sigma_W)^2 + ((m_bjj - m_t)/sigma_t)^2 +
 * ((m_jj - m_W)/sigma_W)^2, minimised over the combinations (b_lep, b_had: ordered pair of the first 4 b-tagged jet slots;
 * q1 < q2: pair of the first 4 untagged slots) and over the neutrino p_z: pT(nu) = MET, p_z solves m(l nu) = m_W (two
 * solutions, index 0 = smaller p_z) or, without a real solution, minimises m(l nu) (R14).  Argmin in the order
 * (b_lep, b_had, (q1, q2), solution), strict <.
 *   idx          device uint32[n_idx] events to reconstruct;  host_params NULL = (172.5, 80.4, 11.5, 7.5).
 *   out          device hepf_chi2_t[n_idx], 16-byte aligned.  status 1 = reconstructed, 2 = not applicable (n_lep != 1,
 *                fewer than 2 b-tagged or fewer than 2 untagged jets): NaN / -1 payload.  A list entry idx[k] >= n_events
 *                is not applicable with bit 8 set as well (status 10); nothing is read for it.
 */
typedef struct { double m_top, m_w, sigma_top, sigma_w; } hepf_chi2_params_t;
typedef struct {
  double chi2, nu_pz, m_top_lep, m_top_had, m_w_lep, m_w_had;
  int32_t jet_b_lep, jet_b_had, jet_q1, jet_q2, solution, n_comb;
  uint32_t status, event;
} hepf_chi2_t;   /* 80 bytes */
int hepf_chi2_semilep(const hepf_events_t* events, const uint32_t* idx, int64_t n_idx, const hepf_chi2_params_t* host_params,
                      hepf_chi2_t* out, void* stream);
/*
 * hepf_chi2_single_top — the single-top variants of eq. (1) ("in single top quark events from Wt associated
 * production, only 1 top quark and 2 W-bosons should be reconstructed, while for the t-channel only 1, of each, should
 * exist"), semileptonic final state, same neutrino p_z and same record as hepf_chi2_semilep:
 *   mode 1, t-channel: chi^2 = ((m_blnu - m_t)/sigma_t)^2 + ((m_lnu - m_W)/sigma_W)^2 over (b, p_z solution); needs one
 *           lepton and one b-tagged jet; the hadronic fields of the record stay NaN / -1.
 *   mode 2, Wt: chi^2 = ((m_top - m_t)/sigma_t)^2 + ((m_lnu - m_W)/sigma_W)^2 + ((m_jj - m_W)/sigma_W)^2, the one top being
 *           the leptonic (b l nu) or the hadronic (b j j) one; over (hypothesis, b, (q1, q2), p_z solution); needs one lepton,
 *           one b-tagged and two untagged jets; jet_b_lep / m_top_lep are set for a leptonic top, jet_b_had / m_top_had for a
 *           hadronic one, the other pair stays -1 / NaN.
 * The dileptonic chi^2 of eq. (1) is not built: the paper's description of it breaks off mid-sentence.
 */
int hepf_chi2_single_top(const hepf_events_t* events, const uint32_t* idx, int64_t n_idx, int mode,
                         const hepf_chi2_params_t* host_params, hepf_chi2_t* out, void* stream);

/*
 * hepf_chi2_dilep — the dileptonic ttbar case of eq. (1) ("for the dileptonic final states, two neutrinos
 * must be fully reconstructed.  This implies, splitting the E_T^miss between the two neutrinos and determine, using the mass
 * constraints from the chi^2" — the sentence breaks off there; R15 is the reading).  The neutrino's transverse
 * momentum is scanned over a split_n x split_n grid, nu_T = MET/2 + split_range (u_gx, u_gy) with u_g = (2 g + 1)/split_n - 1,
 * the antineutrino takes nubar_T = MET - nu_T; each p_z follows from its W as in hepf_chi2_semilep (two roots of m(l nu) = m_W,
 * else the p_z of closest approach); chi^2 = [t_top^2 + t_W^2](l+, nu, b) + [t_top^2 + t_W^2](l-, nubar, bbar) over ordered
 * pairs (b, bbar) of the first 4 b-tagged jet slots; first minimum in the order (b, bbar, gx, gy, solution of nu, of nubar).
 *   idx          device uint32[n_idx] event indices of the view (an index >= n_events gives status 2 | 8).
 *   host_params  HOST pointer or NULL (172.5, 80.4, 11.5, 7.5);  host_split  HOST pointer or NULL (160 GeV, 32).
 *   out          device hepf_chi2_dilep_t[n_idx], 16-byte aligned.  status 1 = reconstructed, 2 = not applicable (n_lep != 2,
 *                same-sign leptons or fewer than two b-tags), 0 = no finite chi^2 anywhere; NaN / -1 payload unless status 1.
 *                n_comb = number of (b, bbar, grid point, solutions) combinations evaluated.
 * Errors: HEPF_ERR_ARG for NULL / misaligned pointers, non-positive widths, split_n outside 1..64, split_range < 0.
 */
typedef struct { double split_range; int32_t split_n, pad_; } hepf_split_t;
typedef struct {
  double chi2, nu[3], nubar[3], m_top, m_antitop, m_wplus, m_wminus;
  int32_t jet_b, jet_bbar, grid_x, grid_y, sol_nu, sol_nubar, n_comb;
  uint32_t status, event; int32_t pad_;
} hepf_chi2_dilep_t;   /* 128 bytes */
int hepf_chi2_dilep(const hepf_events_t* events, const uint32_t* idx, int64_t n_idx, const hepf_chi2_params_t* host_params,
                    const hepf_split_t* host_split, hepf_chi2_dilep_t* out, void* stream);

/*
 * hepf_histogram — fixed-width histogram of one quantity of the reconstructed events, filled on the device
 * (App. 8.2: the user's finalize() writes histograms of reconstructed quantities; PAPER.md:278:
 * per-cut variable recording).  Only records with status bit 0 (has a solution) are filled.
 *   best    device hepf_best_t[n].
 *   field   HEPF_H_* below.  NU_PT / NUBAR_PT = sqrt(px*px + py*py), each operation rounded once (no contraction).
 *   bins    t = (value - lo) * (nbins / (hi - lo)), every operation rounded once; t < 0 -> out[0] (underflow),
 *           t >= nbins -> out[nbins + 1] (overflow), else out[1 + (int)t]; a NaN value is not counted.
 *   out     device uint64[nbins + 2], ZEROED by the call before filling; 1 <= nbins <= 4096, hi > lo.
 */
typedef enum {
  HEPF_H_M_TOP = 0, HEPF_H_M_ANTITOP = 1, HEPF_H_M_WPLUS = 2, HEPF_H_M_WMINUS = 3, HEPF_H_M_HIGGS = 4,
  HEPF_H_LOGLIK = 5, HEPF_H_NU_PT = 6, HEPF_H_NUBAR_PT = 7, HEPF_H_VARIATION = 8
} hepf_hist_field_t;
int hepf_histogram(const hepf_best_t* best, int64_t n, int field, double lo, double hi, int32_t nbins, uint64_t* out,
                   void* stream);

/*
 * hepf_tth_system — the two quantities the paper's example analysis histograms (App. 8.2 listing:
 * "TLorentzVector ttH = Top + Tbar + Higgs; mTTH = ttH.M(); ptTTH = ttH.Pt();"): invariant mass and transverse momentum of
 * the reconstructed ttH system of each record, i.e. of l+ + l- + nu + nubar + b + bbar + h1 + h2 with the smeared objects
 * of the record's variation and E_nu = |p_nu|; m = sqrt(max(E^2 - |p|^2, 0)), pT = sqrt(px^2 + py^2), every operation one
 * IEEE operation in that order.  The reconstruction being the last cut, these are per-event variables written by a cut
 * (PAPER.md:278).   best: device hepf_best_t[n] (hepf_reconstruct_tth's output on the same view, seed and parameters);
 * out: device double[2 n], 16-byte aligned: out[2k] = m_ttH, out[2k+1] = pT_ttH of record k; NaN for a record without solution.
 */
int hepf_tth_system(const hepf_events_t* events, const hepf_best_t* best, int64_t n, uint64_t seed,
                    const hepf_tth_params_t* host_params, double* out, void* stream);
/*
 * hepf_histogram_values — hepf_histogram's binning for a plain device column of doubles (a derived per-event variable:
 * hepf_select_record's ETmis column, hepf_tth_system's m_ttH or pT_ttH): element k is values[k * stride]; every value is
 * filled except NaN ("no value").   out: device uint64[nbins + 2], zeroed by the call.
 */
int hepf_histogram_values(const double* values, int64_t stride, int64_t n, double lo, double hi, int32_t nbins, uint64_t* out,
                          void* stream);

/* Kernel launches enqueued by this thread's calls since the last reset (bench.py's `gpu_launches`). */
int64_t hepf_launch_count(int reset);
/* FP64 FMA-chain micro-benchmark used to measure the FP64 roof on the box: enqueues one kernel that performs
 * `fma_per_thread` dependent-chain-of-8 DFMAs per thread over blocks x threads; writes a checksum to `sink`. */
int hepf_fp64_peak_probe(int blocks, int threads, int64_t fma_per_thread, double* sink, void* stream);

/* Per-kernel device timing for bench.py's roofline: when enabled (per host thread) the library records a CUDA event on
 * the call's stream before and after each of its kernels.  Slots: 0 select start | 1 after select_eval | 2 after
 * select_scatter | 3 reconstruct start | 4 after the n_b = 4 search kernel | 5 after the n_b = 5,6 search kernel |
 * 6 after the finalize kernel.  hepf_timing_ms waits for the `to` event and returns the elapsed milliseconds of the
 * LAST call that recorded both (negative if unavailable). */
int hepf_timing_enable(int on);
double hepf_timing_ms(int from_slot, int to_slot);

const char* hepf_last_error(void);
const char* hepf_version(void);

#ifdef __cplusplus
}
#endif
#endif
