/*
 * hepf_synth/gen.c — seeded synthetic dileptonic ttH event generator (INPUT DATA ONLY).
 *
 * This module produces the inputs that both the CUDA path and the CPU oracle consume.  It holds
 * none of the method's arithmetic: no Philox, no cut evaluation, no conics, no solver, no score.
 * Its random numbers come from its own counter-based SplitMix64 stream keyed by (seed, global event
 * index), mapped through libm (log/cos/sin/tan), so an event depends only on (seed, index) and never
 * on how a sample is split into calls, threads or ranks.
 *
 * Recipe: BASELINE.json configs[1..4] as made concrete in SURVEY.md §8(d) and DESIGN.md §"Inputs";
 * it stands in for the paper's private MadGraph5_aMC@NLO+Pythia+Delphes ttH sample
 * (§4), which is not available.
 *
 * Column layout written here (one contiguous block, `stride` doubles per row, 64 rows):
 *   row  0..11 : lep_px[2] lep_py[2] lep_pz[2] lep_e[2] lep_pt[2] lep_eta[2]
 *   row 12..59 : jet_px[8] jet_py[8] jet_pz[8] jet_e[8] jet_pt[8] jet_eta[8]
 *   row 60..63 : met_x met_y met mll
 * plus flags[stride] (uint32): bits 0-3 n_lep | 4 q(lep0)>0 | 5 q(lep1)>0 | 8-11 n_jet | 16-23 b-tag mask.
 * Truth side table (optional, 12 doubles per event, AoS): nu[3], nubar[3], slot(b), slot(bbar),
 *   slot(h1), slot(h2), is_signal, lepton slot of l+.
 */
#include <math.h>
#include <stdint.h>
#include <string.h>

#define NROW 64
#define NJ 8
#define PI 3.14159265358979323846

typedef struct {
  int64_t n_events;      /* events to write                                   */
  int64_t first_event;   /* global index of the first one (keys the RNG)      */
  int64_t stride;        /* doubles per column row (>= n_events)              */
  uint64_t seed;
  int32_t n_fake_b;      /* extra b-tagged fake jets per signal event (0 / 2) */
  int32_t closure;       /* 1: zero widths, no detector smearing, no extras   */
  double bkg_frac;       /* probability of a structure-less background event  */
  int32_t semilep;       /* 1: semileptonic ttbar events (1 lepton, 2 b + 2 light jets) for the chi2 path */
  int32_t pad_;
} hepf_gen_cfg_t;

typedef struct { uint64_t s; } rng_t;

static inline uint64_t mix64(uint64_t z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}
static inline void rng_init(rng_t* r, uint64_t seed, uint64_t event) {
  r->s = mix64(seed * 0x9E3779B97F4A7C15ULL + 0x632BE59BD9B4E019ULL) ^ mix64(event + 0x2545F4914F6CDD1DULL);
}
static inline double rng_u(rng_t* r) { /* (0,1) */
  r->s += 0x9E3779B97F4A7C15ULL;
  return ((double)(mix64(r->s) >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}
static inline double rng_exp(rng_t* r, double mean) { return -mean * log(rng_u(r)); }
static inline double rng_norm(rng_t* r) {
  double u1 = rng_u(r), u2 = rng_u(r);
  return sqrt(-2.0 * log(u1)) * cos(2.0 * PI * u2);
}
static inline double rng_bw(rng_t* r, double m, double gamma, double lo, double hi) {
  double v = m + 0.5 * gamma * tan(PI * (rng_u(r) - 0.5));
  return v < lo ? lo : (v > hi ? hi : v);
}
static inline int rng_poisson(rng_t* r, double lam) {
  double l = exp(-lam), p = 1.0;
  int k = 0;
  do { k++; p *= rng_u(r); } while (p > l && k < 64);
  return k - 1;
}

typedef struct { double x, y, z, e; } v4;

static inline v4 v4_ptetaphim(double pt, double eta, double phi, double m) {
  v4 v; v.x = pt * cos(phi); v.y = pt * sin(phi); v.z = pt * sinh(eta);
  v.e = sqrt(v.x * v.x + v.y * v.y + v.z * v.z + m * m); return v;
}
static inline v4 v4_scale(v4 a, double s) { v4 v = {a.x * s, a.y * s, a.z * s, a.e * s}; return v; }

/* boost `d` (given in the rest frame of `p`) into the frame where `p` is measured */
static inline v4 boost_from_rest(v4 d, v4 p) {
  double m2 = p.e * p.e - p.x * p.x - p.y * p.y - p.z * p.z;
  double m = sqrt(m2 > 0 ? m2 : 0);
  if (m <= 0) return d;
  double bx = p.x / p.e, by = p.y / p.e, bz = p.z / p.e;
  double b2 = bx * bx + by * by + bz * bz;
  double g = p.e / m;
  double bp = bx * d.x + by * d.y + bz * d.z;
  double k = (b2 > 0 ? (g - 1.0) * bp / b2 : 0.0) + g * d.e;
  v4 o = {d.x + k * bx, d.y + k * by, d.z + k * bz, g * (d.e + bp)};
  return o;
}

/* isotropic two-body decay parent(mass M, lab four-vector P) -> m1 + m2; both returned in the lab */
static inline void decay2(rng_t* r, v4 P, double M, double m1, double m2, v4* d1, v4* d2) {
  double s = (M * M - (m1 + m2) * (m1 + m2)) * (M * M - (m1 - m2) * (m1 - m2));
  double ps = s > 0 ? sqrt(s) / (2.0 * M) : 0.0;
  double ct = 2.0 * rng_u(r) - 1.0, st = sqrt(1.0 - ct * ct), ph = 2.0 * PI * rng_u(r);
  v4 a = {ps * st * cos(ph), ps * st * sin(ph), ps * ct, sqrt(ps * ps + m1 * m1)};
  v4 b = {-a.x, -a.y, -a.z, sqrt(ps * ps + m2 * m2)};
  *d1 = boost_from_rest(a, P);
  *d2 = boost_from_rest(b, P);
}

typedef struct { v4 p; int tag; int role; } jet_t; /* role: 0 b, 1 bbar, 2 h1, 3 h2, -1 other */

static inline double pt_of(v4 a) { return sqrt(a.x * a.x + a.y * a.y); }
static inline double eta_of(v4 a) { double pt = pt_of(a); return pt > 0 ? asinh(a.z / pt) : 0.0; }

static void write_event(const hepf_gen_cfg_t* c, double* cols, uint32_t* flags, double* truth, int64_t k,
                        int n_lep, const v4* lep, const int* lq, int n_jet, jet_t* jets, double mx, double my,
                        const double* tnu, const double* tnub, int is_signal) {
  const int64_t S = c->stride;
  /* sort jets by pT, descending (insertion sort, stable) */
  for (int a = 1; a < n_jet; a++) {
    jet_t t = jets[a]; double pt = pt_of(t.p); int b = a - 1;
    while (b >= 0 && pt_of(jets[b].p) < pt) { jets[b + 1] = jets[b]; b--; }
    jets[b + 1] = t;
  }
  int nl = n_lep < 2 ? n_lep : 2;
  int order[2] = {0, 1};
  if (nl == 2 && pt_of(lep[1]) > pt_of(lep[0])) { order[0] = 1; order[1] = 0; }
  uint32_t f = (uint32_t)(n_lep & 15) | ((uint32_t)(n_jet & 15) << 8);
  for (int s = 0; s < 2; s++) {
    v4 p = {0, 0, 0, 0};
    if (s < nl) { p = lep[order[s]]; if (lq[order[s]] > 0) f |= 1u << (4 + s); }
    cols[(0 + s) * S + k] = p.x; cols[(2 + s) * S + k] = p.y; cols[(4 + s) * S + k] = p.z;
    cols[(6 + s) * S + k] = p.e; cols[(8 + s) * S + k] = pt_of(p); cols[(10 + s) * S + k] = eta_of(p);
  }
  int slot_role[4] = {-1, -1, -1, -1};
  for (int s = 0; s < NJ; s++) {
    v4 p = {0, 0, 0, 0};
    if (s < n_jet) {
      p = jets[s].p;
      if (jets[s].tag) f |= 1u << (16 + s);
      if (jets[s].role >= 0) slot_role[jets[s].role] = s;
    }
    cols[(12 + s) * S + k] = p.x; cols[(20 + s) * S + k] = p.y; cols[(28 + s) * S + k] = p.z;
    cols[(36 + s) * S + k] = p.e; cols[(44 + s) * S + k] = pt_of(p); cols[(52 + s) * S + k] = eta_of(p);
  }
  cols[60 * S + k] = mx; cols[61 * S + k] = my; cols[62 * S + k] = sqrt(mx * mx + my * my);
  double mll = 0.0;
  if (nl == 2) {
    double e = lep[0].e + lep[1].e, x = lep[0].x + lep[1].x, y = lep[0].y + lep[1].y, z = lep[0].z + lep[1].z;
    double m2 = e * e - x * x - y * y - z * z; mll = m2 > 0 ? sqrt(m2) : 0.0;
  }
  cols[63 * S + k] = mll;
  flags[k] = f;
  if (truth) {
    double* t = truth + 12 * k;
    for (int i = 0; i < 3; i++) { t[i] = tnu[i]; t[3 + i] = tnub[i]; }
    for (int i = 0; i < 4; i++) t[6 + i] = (double)slot_role[i];
    t[10] = (double)is_signal;
    /* store slot of l+ (generated as lepton 0) */
    t[11] = (nl == 2) ? (double)(order[0] == 0 ? 0 : 1) : -1.0;
  }
}

static void gen_signal(const hepf_gen_cfg_t* c, rng_t* r, double* cols, uint32_t* flags, double* truth, int64_t k) {
  const double MB = 4.7, MH = 125.0;
  double mt, mtb, mwp, mwm;
  if (c->closure) { mt = mtb = 172.5; mwp = mwm = 80.4; }
  else {
    mt = rng_bw(r, 172.5, 1.4, 150.0, 195.0); mtb = rng_bw(r, 172.5, 1.4, 150.0, 195.0);
    mwp = rng_bw(r, 80.4, 2.1, 60.0, 100.0); mwm = rng_bw(r, 80.4, 2.1, 60.0, 100.0);
  }
  double M = mt + mtb + MH + rng_exp(r, 150.0);
  double mtt = mt + mtb + rng_u(r) * (M - MH - mt - mtb);
  double spt = rng_exp(r, 50.0), sphi = 2.0 * PI * rng_u(r), sy = 1.5 * rng_norm(r);
  double mT = sqrt(M * M + spt * spt);
  v4 S = {spt * cos(sphi), spt * sin(sphi), mT * sinh(sy), mT * cosh(sy)};
  v4 TT, H, t, tb, wp, b, wm, bb, lp, nu, lm, nub, h1, h2;
  decay2(r, S, M, mtt, MH, &TT, &H);
  decay2(r, TT, mtt, mt, mtb, &t, &tb);
  decay2(r, t, mt, mwp, MB, &wp, &b);
  decay2(r, wp, mwp, 0.0, 0.0, &lp, &nu);
  decay2(r, tb, mtb, mwm, MB, &wm, &bb);
  decay2(r, wm, mwm, 0.0, 0.0, &lm, &nub);
  decay2(r, H, MH, MB, MB, &h1, &h2);
  /* massless leptons: make E exactly |p| so that m_l^2 is rounding-level, as for a measured lepton */
  lp.e = sqrt(lp.x * lp.x + lp.y * lp.y + lp.z * lp.z);
  lm.e = sqrt(lm.x * lm.x + lm.y * lm.y + lm.z * lm.z);
  v4 lep[2] = {lp, lm}; int lq[2] = {+1, -1};
  jet_t jets[NJ]; int nj = 0;
  v4 bj[4] = {b, bb, h1, h2};
  for (int i = 0; i < 4; i++) { jets[nj].p = bj[i]; jets[nj].tag = 1; jets[nj].role = i; nj++; }
  double mx = nu.x + nub.x, my = nu.y + nub.y;
  if (!c->closure) {
    for (int i = 0; i < 2; i++) lep[i] = v4_scale(lep[i], 1.0 + 0.01 * rng_norm(r));
    for (int i = 0; i < 4; i++) {
      double s = 1.0 + (0.5 / sqrt(jets[i].p.e) + 0.03) * rng_norm(r);
      jets[i].p = v4_scale(jets[i].p, s < 0.1 ? 0.1 : s);
    }
    int nl = rng_poisson(r, 0.7); if (nl > 2) nl = 2;
    for (int i = 0; i < nl; i++) {
      double pt = rng_exp(r, 40.0), eta = 5.0 * rng_u(r) - 2.5, phi = 2.0 * PI * rng_u(r);
      jets[nj].p = v4_ptetaphim(pt, eta, phi, 0.0); jets[nj].tag = 0; jets[nj].role = -1; nj++;
    }
    for (int i = 0; i < c->n_fake_b && nj < NJ; i++) {
      double pt = rng_exp(r, 35.0), eta = 5.0 * rng_u(r) - 2.5, phi = 2.0 * PI * rng_u(r);
      jets[nj].p = v4_ptetaphim(pt, eta, phi, 0.0); jets[nj].tag = 1; jets[nj].role = -1; nj++;
    }
  }
  double tnu[3] = {nu.x, nu.y, nu.z}, tnub[3] = {nub.x, nub.y, nub.z};
  write_event(c, cols, flags, truth, k, 2, lep, lq, nj, jets, mx, my, tnu, tnub, 1);
}

/* Semileptonic ttbar (section 6.2): t -> W b, W -> l nu; tbar -> W bbar, W -> q qbar'.  One lepton,
 * two b-tagged and two untagged jets (+ 0-2 extra untagged light jets), MET = neutrino pT.  Truth: nu[3], nubar unused (0),
 * slots of b_lep, b_had, q1, q2. */
static void gen_semilep(const hepf_gen_cfg_t* c, rng_t* r, double* cols, uint32_t* flags, double* truth, int64_t k) {
  const double MB = 4.7;
  double mt, mtb, mwp, mwm;
  if (c->closure) { mt = mtb = 172.5; mwp = mwm = 80.4; }
  else {
    mt = rng_bw(r, 172.5, 1.4, 150.0, 195.0); mtb = rng_bw(r, 172.5, 1.4, 150.0, 195.0);
    mwp = rng_bw(r, 80.4, 2.1, 60.0, 100.0); mwm = rng_bw(r, 80.4, 2.1, 60.0, 100.0);
  }
  double M = mt + mtb + rng_exp(r, 120.0);
  double spt = rng_exp(r, 40.0), sphi = 2.0 * PI * rng_u(r), sy = 1.2 * rng_norm(r);
  double mT = sqrt(M * M + spt * spt);
  v4 S = {spt * cos(sphi), spt * sin(sphi), mT * sinh(sy), mT * cosh(sy)};
  v4 t, tb, wp, b, wm, bb, lp, nu, q1, q2;
  decay2(r, S, M, mt, mtb, &t, &tb);
  decay2(r, t, mt, mwp, MB, &wp, &b);
  decay2(r, wp, mwp, 0.0, 0.0, &lp, &nu);
  decay2(r, tb, mtb, mwm, MB, &wm, &bb);
  decay2(r, wm, mwm, 0.0, 0.0, &q1, &q2);
  lp.e = sqrt(lp.x * lp.x + lp.y * lp.y + lp.z * lp.z);
  v4 lep[2] = {lp, lp}; int lq[2] = {rng_u(r) < 0.5 ? +1 : -1, 0};
  jet_t jets[NJ]; int nj = 0;
  v4 bj[4] = {b, bb, q1, q2};
  for (int i = 0; i < 4; i++) { jets[nj].p = bj[i]; jets[nj].tag = i < 2; jets[nj].role = i; nj++; }
  double mx = nu.x, my = nu.y;
  if (!c->closure) {
    lep[0] = v4_scale(lep[0], 1.0 + 0.01 * rng_norm(r));
    for (int i = 0; i < 4; i++) {
      double s = 1.0 + (0.5 / sqrt(jets[i].p.e) + 0.03) * rng_norm(r);
      jets[i].p = v4_scale(jets[i].p, s < 0.1 ? 0.1 : s);
    }
    int nl = rng_poisson(r, 0.7); if (nl > 2) nl = 2;
    for (int i = 0; i < nl; i++) {
      double pt = rng_exp(r, 40.0), eta = 5.0 * rng_u(r) - 2.5, phi = 2.0 * PI * rng_u(r);
      jets[nj].p = v4_ptetaphim(pt, eta, phi, 0.0); jets[nj].tag = 0; jets[nj].role = -1; nj++;
    }
  }
  double tnu[3] = {nu.x, nu.y, nu.z}, z3[3] = {0, 0, 0};
  write_event(c, cols, flags, truth, k, 1, lep, lq, nj, jets, mx, my, tnu, z3, 1);
}

static void gen_background(const hepf_gen_cfg_t* c, rng_t* r, double* cols, uint32_t* flags, double* truth, int64_t k) {
  double u = rng_u(r);
  int n_lep = u < 0.2 ? 1 : (u < 0.9 ? 2 : 3);
  v4 lep[2]; int lq[2] = {0, 0};
  for (int i = 0; i < 2; i++) {
    double pt = rng_exp(r, 35.0), eta = 5.0 * rng_u(r) - 2.5, phi = 2.0 * PI * rng_u(r);
    lep[i] = v4_ptetaphim(pt, eta, phi, 0.0); lq[i] = rng_u(r) < 0.5 ? +1 : -1;
  }
  int nj = 2 + (int)(rng_u(r) * 7.0); if (nj > NJ) nj = NJ;
  jet_t jets[NJ];
  for (int i = 0; i < nj; i++) {
    double pt = rng_exp(r, 40.0), eta = 5.0 * rng_u(r) - 2.5, phi = 2.0 * PI * rng_u(r);
    jets[i].p = v4_ptetaphim(pt, eta, phi, 0.0); jets[i].tag = rng_u(r) < 0.3; jets[i].role = -1;
  }
  double met = rng_exp(r, 25.0), mphi = 2.0 * PI * rng_u(r);
  double z3[3] = {0, 0, 0};
  write_event(c, cols, flags, truth, k, n_lep, lep, lq, nj, jets, met * cos(mphi), met * sin(mphi), z3, z3, 0);
}

/* Fill events [0, n_events) of the given buffers; event k has global index first_event + k. */
int hepf_synth_generate(const hepf_gen_cfg_t* c, double* cols, uint32_t* flags, double* truth) {
  if (!c || !cols || !flags || c->n_events < 0 || c->stride < c->n_events) return -1;
#pragma omp parallel for schedule(static)
  for (int64_t k = 0; k < c->n_events; k++) {
    rng_t r; rng_init(&r, c->seed, (uint64_t)(c->first_event + k));
    if (c->semilep) gen_semilep(c, &r, cols, flags, truth, k);
    else if (c->bkg_frac > 0.0 && rng_u(&r) < c->bkg_frac) gen_background(c, &r, cols, flags, truth, k);
    else gen_signal(c, &r, cols, flags, truth, k);
  }
  return 0;
}
