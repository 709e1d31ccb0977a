// oracle/oracle_reco.cpp — CPU ORACLE (test infrastructure).  O4: smear -> conics -> quartic -> score -> argmax.
//
// PAPER.md:134-138 (§4): the two neutrino four-momenta follow from energy-momentum conservation plus
// m(l nu) = m_W = 80.4 and m(l nu b) = m_t = 172.5 on both legs ("quadratic forms", several solutions or
// none); every b-jet/lepton pairing is tried, two of the remaining b-jets should give m_bb = 125, the
// solution with the highest probability wins; an event with no solution is discarded.  PAPER.md:145:
// the measured energies and momenta are varied V times within the resolution and only the most probable
// solution is kept.  The equations (the paper defers them to its ref. [27]) and every reading of a silent
// point are SURVEY.md §8(c) O4 / DESIGN.md R1-R13.  Nothing is blocked, fused or reordered: enumeration order
// is (variation, pairing, Higgs pair, root) and a candidate replaces the incumbent only if strictly better.
//
// The root finder is deliberately NOT the closed form the CUDA path uses: nested bisection on the derivative
// chain P'' -> P' -> P, then two Newton steps.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

#include "hepf_oracle.h"

void orc_block_normals(const uint32_t ctr[4], const uint32_t key[2], double* z_even, double* z_odd);

extern "C" void orc_default_params(orc_params_t* p) {
  p->m_top = 172.5; p->m_w = 80.4; p->m_higgs = 125.0;
  p->sigma_higgs = 15.0; p->lambda_nu = 40.0;               // definitions of this build (R7)
  p->lep_sigma = 0.01;                                      // PAPER.md:145 "1%"
  p->jet_stoch = 0.5; p->jet_const = 0.03;                  // BASELINE.json configs[0]
  p->sigma_scale = 1.0; p->s_min = 0.1;                     // R4, R5
}

namespace {

struct V4 { double x, y, z, e; };
struct Conic { double a, b, c, d, e, f; };      // a x^2 + b x y + c y^2 + d x + e y + f = 0
struct Leg { Conic q; double c0, c1, c2; bool ok; };  // p_z = c0 + c1 p_x + c2 p_y

const double EPS = 0x1p-53;
const double NaN = std::numeric_limits<double>::quiet_NaN();

V4 scaled(const V4& p, double s) { return V4{s * p.x, s * p.y, s * p.z, s * p.e}; }
double mass(double e, double x, double y, double z) {
  double m2 = e * e - (x * x + y * y + z * z);
  return std::sqrt(m2 > 0.0 ? m2 : 0.0);
}

// Leg conic for (lepton l, b-jet b): O4 step 3.
Leg leg_conic(const V4& l, const V4& b, double mt, double mw) {
  Leg g{};
  double ml2 = l.e * l.e - (l.x * l.x + l.y * l.y + l.z * l.z);
  double mb2 = b.e * b.e - (b.x * b.x + b.y * b.y + b.z * b.z);
  double bl = b.e * l.e - (b.x * l.x + b.y * l.y + b.z * l.z);
  double A = (mw * mw - ml2) / 2.0;                       // E_l E - l.p = A
  double B = (mt * mt - mw * mw - mb2) / 2.0 - bl;        // E_b E - b.p = B
  double nx = b.e * l.x - l.e * b.x, ny = b.e * l.y - l.e * b.y, nz = b.e * l.z - l.e * b.z;
  double k = l.e * B - b.e * A;                           // n.p = k
  g.ok = std::fabs(nz) > 1e-12 * b.e * l.e;
  if (!g.ok) return g;
  g.c0 = k / nz; g.c1 = -nx / nz; g.c2 = -ny / nz;
  double d0 = (A + l.z * g.c0) / l.e, d1 = (l.x + l.z * g.c1) / l.e, d2 = (l.y + l.z * g.c2) / l.e;
  g.q.a = d1 * d1 - 1.0 - g.c1 * g.c1;
  g.q.b = 2.0 * (d1 * d2 - g.c1 * g.c2);
  g.q.c = d2 * d2 - 1.0 - g.c2 * g.c2;
  g.q.d = 2.0 * (d0 * d1 - g.c0 * g.c1);
  g.q.e = 2.0 * (d0 * d2 - g.c0 * g.c2);
  g.q.f = d0 * d0 - g.c0 * g.c0;
  return g;
}

// conic of leg 2 is in q = M - p; rewrite it in p.
Conic shifted(const Conic& q, double Mx, double My) {
  Conic s;
  s.a = q.a; s.b = q.b; s.c = q.c;
  s.d = -2.0 * q.a * Mx - q.b * My - q.d;
  s.e = -2.0 * q.c * My - q.b * Mx - q.e;
  s.f = q.a * Mx * Mx + q.b * Mx * My + q.c * My * My + q.d * Mx + q.e * My + q.f;
  return s;
}

struct Resultant { double p[3], q[2], r[4], h[5]; };

Resultant resultant(const Conic& k1, const Conic& k2) {
  Resultant R;
  R.p[0] = k1.c * k2.f - k2.c * k1.f; R.p[1] = k1.c * k2.d - k2.c * k1.d; R.p[2] = k1.c * k2.a - k2.c * k1.a;
  R.q[0] = k1.c * k2.e - k2.c * k1.e; R.q[1] = k1.c * k2.b - k2.c * k1.b;
  R.r[0] = k1.e * k2.f - k2.e * k1.f;
  R.r[1] = k1.e * k2.d + k1.b * k2.f - k2.e * k1.d - k2.b * k1.f;
  R.r[2] = k1.e * k2.a + k1.b * k2.d - k2.e * k1.a - k2.b * k1.d;
  R.r[3] = k1.b * k2.a - k2.b * k1.a;
  // P = D1^2 - D2 D3
  R.h[0] = R.p[0] * R.p[0] - R.q[0] * R.r[0];
  R.h[1] = 2.0 * R.p[0] * R.p[1] - (R.q[0] * R.r[1] + R.q[1] * R.r[0]);
  R.h[2] = 2.0 * R.p[0] * R.p[2] + R.p[1] * R.p[1] - (R.q[0] * R.r[2] + R.q[1] * R.r[1]);
  R.h[3] = 2.0 * R.p[1] * R.p[2] - (R.q[0] * R.r[3] + R.q[1] * R.r[2]);
  R.h[4] = R.p[2] * R.p[2] - R.q[1] * R.r[3];
  return R;
}

double poly(const double* c, int deg, double x) {   // c[0] + c[1] x + ...
  double v = c[deg];
  for (int i = deg - 1; i >= 0; i--) v = v * x + c[i];
  return v;
}

// bisection on [lo, hi] with f(lo) f(hi) < 0, to machine convergence
bool bisect(const double* c, int deg, double lo, double hi, double* root) {
  double flo = poly(c, deg, lo), fhi = poly(c, deg, hi);
  if (!(flo * fhi < 0.0)) return false;
  for (int it = 0; it < 200; it++) {
    double mid = 0.5 * (lo + hi);
    if (mid == lo || mid == hi) break;
    double fm = poly(c, deg, mid);
    if (fm == 0.0) { lo = hi = mid; break; }
    if ((fm < 0.0) == (flo < 0.0)) { lo = mid; flo = fm; } else { hi = mid; }
  }
  *root = 0.5 * (lo + hi);
  return true;
}

// real roots of a polynomial of degree `deg` given sorted real roots of its derivative, inside [-R, R]
int roots_between(const double* c, int deg, const double* crit, int n_crit, double R, double* out) {
  double edges[8]; int ne = 0;
  edges[ne++] = -R;
  for (int i = 0; i < n_crit; i++) edges[ne++] = crit[i];
  edges[ne++] = R;
  int n = 0;
  for (int i = 0; i + 1 < ne; i++) {
    double r;
    if (edges[i] < edges[i + 1] && bisect(c, deg, edges[i], edges[i + 1], &r)) out[n++] = r;
  }
  return n;
}

// all simple real roots of the monic quartic x^4 + g3 x^3 + g2 x^2 + g1 x + g0, ascending
int quartic_roots(const double g[4], double roots[4]) {
  double P[5] = {g[0], g[1], g[2], g[3], 1.0};
  double R = 1.0;
  for (int i = 0; i < 4; i++) R = std::max(R, 1.0 + std::fabs(g[i]));
  double P1[4] = {g[1], 2.0 * g[2], 3.0 * g[3], 4.0};
  double P2[3] = {2.0 * g[2], 6.0 * g[3], 12.0};
  double c2[2]; int n2 = 0;
  double disc = P2[1] * P2[1] - 4.0 * P2[2] * P2[0];
  if (disc > 0.0) {
    double sq = std::sqrt(disc);
    c2[0] = (-P2[1] - sq) / (2.0 * P2[2]); c2[1] = (-P2[1] + sq) / (2.0 * P2[2]); n2 = 2;
  }
  double c1[3]; int n1 = roots_between(P1, 3, c2, n2, R, c1);
  int n = roots_between(P, 4, c1, n1, R, roots);
  for (int i = 0; i < n; i++)
    for (int it = 0; it < 2; it++) {
      double f = poly(P, 4, roots[i]), d = poly(P1, 3, roots[i]);
      if (d != 0.0 && std::isfinite(f / d)) roots[i] = roots[i] - f / d;
    }
  for (int i = 1; i < n; i++)  // ascending (Newton may in principle reorder two close roots)
    for (int j = i; j > 0 && roots[j] < roots[j - 1]; j--) std::swap(roots[j], roots[j - 1]);
  return n;
}

// near-tangency measure (R11 iii): min over the critical points of P of |P| / sum |g_i x^i| (1 if P' has no
// real root inside the Cauchy bound)
double tangency_measure(const double g[4]) {
  double m = 1.0;
  double P1[4] = {g[1], 2.0 * g[2], 3.0 * g[3], 4.0}, P2[3] = {2.0 * g[2], 6.0 * g[3], 12.0};
  double Rb = 1.0; for (int i = 0; i < 4; i++) Rb = std::max(Rb, 1.0 + std::fabs(g[i]));
  double c2[2]; int n2 = 0; double disc = P2[1] * P2[1] - 4.0 * P2[2] * P2[0];
  if (disc > 0.0) { double sq = std::sqrt(disc); c2[0] = (-P2[1] - sq) / 24.0; c2[1] = (-P2[1] + sq) / 24.0; n2 = 2; }
  double c1[3]; int n1 = roots_between(P1, 3, c2, n2, Rb, c1);
  double Pm[5] = {g[0], g[1], g[2], g[3], 1.0};
  for (int i = 0; i < n1; i++) {
    double xx = c1[i], sum = 0.0, xp = 1.0;
    for (int j = 0; j <= 4; j++) { sum += std::fabs(Pm[j] * xp); xp *= xx; }
    double rel = std::fabs(poly(Pm, 4, xx)) / sum;
    if (rel < m) m = rel;
  }
  return m;
}

struct PairingSolution {
  int n_roots = 0;
  double x[4], y[4], kappa[4], nterm[4], sz[4], szb[4];   // sz: sum of |terms| of the p_z linear forms (R11b)
  V4 nu[4], nub[4];
  Resultant R; double g[4]; Conic k1, k2; double min_abs_p_rel = 1.0;
};

// Solve one pairing: l+ with b (leg 1), l- with bbar (leg 2), MET' = (Mx, My).
PairingSolution solve_pairing(const V4& lp, const V4& b, const V4& lm, const V4& bb, double Mx, double My,
                              const orc_params_t& P) {
  PairingSolution S;
  Leg g1 = leg_conic(lp, b, P.m_top, P.m_w), g2 = leg_conic(lm, bb, P.m_top, P.m_w);
  if (!g1.ok || !g2.ok) return S;
  S.k1 = g1.q; S.k2 = shifted(g2.q, Mx, My);
  S.R = resultant(S.k1, S.k2);
  const double* h = S.R.h;
  if (!(h[4] != 0.0) || !std::isfinite(h[4])) return S;
  for (int i = 0; i < 4; i++) { S.g[i] = h[i] / h[4]; if (!std::isfinite(S.g[i])) return S; }
  double roots[4];
  int n = quartic_roots(S.g, roots);
  S.min_abs_p_rel = tangency_measure(S.g);
  for (int r = 0; r < n; r++) {
    double x = roots[r];
    double D1 = S.R.p[0] + S.R.p[1] * x + S.R.p[2] * x * x;
    double D2 = S.R.q[0] + S.R.q[1] * x;
    // D2(x) = 0: both conics have the same two y at this x, i.e. x is a double root of P, which the method skips
    // (SURVEY.md 8(c) O4 "exact double roots are skipped"; R11c).  The quotient is then not finite.
    double y = -D1 / D2;
    if (!std::isfinite(y)) continue;
    // Two Newton steps on the pair of conics in (x, y) — the defining equations of the intersection.  The
    // quotient -D1/D2 cancels catastrophically when D2(x) is small, and north_star asks for 1e-9 (R11a).
    for (int it = 0; it < 2; it++) {
      const Conic &A = S.k1, &B = S.k2;
      double F1 = A.a * x * x + A.b * x * y + A.c * y * y + A.d * x + A.e * y + A.f;
      double F2 = B.a * x * x + B.b * x * y + B.c * y * y + B.d * x + B.e * y + B.f;
      double F1x = 2.0 * A.a * x + A.b * y + A.d, F1y = A.b * x + 2.0 * A.c * y + A.e;
      double F2x = 2.0 * B.a * x + B.b * y + B.d, F2y = B.b * x + 2.0 * B.c * y + B.e;
      double det = F1x * F2y - F1y * F2x;
      double dx = (F1 * F2y - F2 * F1y) / det, dy = (F1x * F2 - F2x * F1) / det;
      x = x - dx; y = y - dy;
    }
    // a singular Jacobian at the intersection means tangent conics, again a double root: skipped (R11c)
    if (!std::isfinite(x) || !std::isfinite(y)) continue;
    int i = S.n_roots;
    S.x[i] = x; S.y[i] = y;
    double pz = g1.c0 + g1.c1 * x + g1.c2 * y;
    double qx = Mx - x, qy = My - y, qz = g2.c0 + g2.c1 * qx + g2.c2 * qy;
    S.sz[i] = std::fabs(g1.c0) + std::fabs(g1.c1 * x) + std::fabs(g1.c2 * y);
    S.szb[i] = std::fabs(g2.c0) + std::fabs(g2.c1 * qx) + std::fabs(g2.c2 * qy);
    S.nu[i] = V4{x, y, pz, std::sqrt(x * x + y * y + pz * pz)};
    S.nub[i] = V4{qx, qy, qz, std::sqrt(qx * qx + qy * qy + qz * qz)};
    double ptn = std::sqrt(x * x + y * y), ptb = std::sqrt(qx * qx + qy * qy);
    S.nterm[i] = std::log(ptn * ptb) - (ptn + ptb) / P.lambda_nu;
    double sum = 0.0, xp = 1.0;
    for (int j = 0; j <= 4; j++) { sum += std::fabs(h[j] * xp); xp *= x; }
    double dP = h[1] + x * (2.0 * h[2] + x * (3.0 * h[3] + x * 4.0 * h[4]));
    S.kappa[i] = EPS * sum / std::fabs(x * dP);
    S.n_roots++;
  }
  return S;
}

double higgs_term(double mbb, const orc_params_t& P) {
  double t = (mbb - P.m_higgs) / P.sigma_higgs;
  return -0.5 * (t * t);
}

struct EventObjects {
  bool applicable; uint32_t status;
  int n_jet, lp_slot, lm_slot, n_b, cand[6];
  V4 lep[2], jet[8]; double met_x, met_y; uint64_t gidx;
};

EventObjects load_event(const orc_events_t* ev, uint32_t e) {
  EventObjects o{}; const int64_t S = ev->stride;
  uint32_t f = ev->flags[e];
  int n_lep = (int)(f & 15u);
  o.n_jet = std::min(8, (int)((f >> 8) & 15u));
  bool q0 = (f >> 4) & 1u, q1 = (f >> 5) & 1u;
  o.gidx = (uint64_t)(ev->event_base + (int64_t)e);
  for (int s = 0; s < 2; s++)
    o.lep[s] = V4{ev->lep_px[s * S + e], ev->lep_py[s * S + e], ev->lep_pz[s * S + e], ev->lep_e[s * S + e]};
  for (int s = 0; s < 8; s++)
    o.jet[s] = V4{ev->jet_px[s * S + e], ev->jet_py[s * S + e], ev->jet_pz[s * S + e], ev->jet_e[s * S + e]};
  o.met_x = ev->met_x[e]; o.met_y = ev->met_y[e];
  o.status = 0; o.n_b = 0;
  int n_tag = 0;
  for (int s = 0; s < o.n_jet; s++)
    if ((f >> (16 + s)) & 1u) { if (o.n_b < 6) o.cand[o.n_b++] = s; n_tag++; }
  if (n_tag > 6) o.status |= 4u;
  o.applicable = (n_lep == 2) && (q0 != q1) && (o.n_b >= 4);
  o.lp_slot = q0 ? 0 : 1; o.lm_slot = 1 - o.lp_slot;
  return o;
}

// O4 step 2: scales and MET' of one (event, variation)
void smear(const EventObjects& o, int32_t v, uint64_t seed, const orc_params_t& P, double s[10], double* Mx,
           double* My) {
  const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  double z[10];
  for (int blk = 0; blk < 5; blk++) {
    uint32_t ctr[4] = {(uint32_t)o.gidx, (uint32_t)(o.gidx >> 32), (uint32_t)v, 0x54544800u + (uint32_t)blk};
    orc_block_normals(ctr, key, &z[2 * blk], &z[2 * blk + 1]);
  }
  for (int t = 0; t < 10; t++) {
    double sigma = (t < 2) ? P.lep_sigma : P.jet_stoch / std::sqrt(o.jet[t - 2].e) + P.jet_const;
    double ks = P.sigma_scale * sigma;
    double sc = std::fma(ks, z[t], 1.0);
    s[t] = sc > P.s_min ? sc : P.s_min;       // max(s_min, .); NaN -> s_min
  }
  double dx = 0.0, dy = 0.0;
  for (int t = 0; t < 2 + o.n_jet; t++) {
    const V4& p = (t < 2) ? o.lep[t] : o.jet[t - 2];
    dx = dx + (s[t] - 1.0) * p.x; dy = dy + (s[t] - 1.0) * p.y;
  }
  *Mx = o.met_x - dx; *My = o.met_y - dy;
}

void fill_nan(orc_best_t* b) {
  for (int i = 0; i < 3; i++) { b->nu[i] = NaN; b->nubar[i] = NaN; }
  b->m_top = b->m_antitop = b->m_wplus = b->m_wminus = b->m_higgs = b->loglik = NaN;
  b->variation = b->jet_b = b->jet_bbar = b->jet_h1 = b->jet_h2 = b->root = -1;
}

void reconstruct_event(const orc_events_t* ev, uint32_t e, int32_t V, uint64_t seed, const orc_params_t& P,
                       orc_best_t* out, orc_aux_t* aux) {
  EventObjects o = load_event(ev, e);
  fill_nan(out); out->event = e; out->status = o.status;
  if (aux) { aux->kappa = NaN; aux->loglik2 = -INFINITY; aux->n_cand = 0; aux->pairing = aux->higgs_pair = -1; aux->pz_terms = aux->pzbar_terms = 0.0; }
  if (!o.applicable) { out->status |= 2u; return; }
  const int nb = o.n_b;
  double best = -INFINITY, second = -INFINITY; bool have = false; int64_t n_cand = 0;
  for (int32_t v = 0; v < V; v++) {
    double s[10], Mx, My; smear(o, v, seed, P, s, &Mx, &My);
    V4 lp = scaled(o.lep[o.lp_slot], s[o.lp_slot]), lm = scaled(o.lep[o.lm_slot], s[o.lm_slot]);
    V4 bj[6]; for (int c = 0; c < nb; c++) bj[c] = scaled(o.jet[o.cand[c]], s[2 + o.cand[c]]);
    for (int i = 0; i < nb; i++) for (int j = 0; j < nb; j++) {
      if (i == j) continue;
      const int a = i * nb + j;
      PairingSolution S = solve_pairing(lp, bj[i], lm, bj[j], Mx, My, P);
      if (S.n_roots == 0) continue;
      int h = 0;
      for (int k = 0; k < nb; k++) for (int l = k + 1; l < nb; l++) {
        if (k == i || k == j || l == i || l == j) continue;
        double mbb = mass(bj[k].e + bj[l].e, bj[k].x + bj[l].x, bj[k].y + bj[l].y, bj[k].z + bj[l].z);
        double ht = higgs_term(mbb, P);
        for (int r = 0; r < S.n_roots; r++) {
          double ll = ht + S.nterm[r];
          n_cand++;
          if (ll > best) {                      // strictly greater: ties keep the first in (v, a, h, r)
            if (have) second = std::max(second, best);
            best = ll; have = true;
            const V4 &nu = S.nu[r], &nb4 = S.nub[r];
            out->nu[0] = nu.x; out->nu[1] = nu.y; out->nu[2] = nu.z;
            out->nubar[0] = nb4.x; out->nubar[1] = nb4.y; out->nubar[2] = nb4.z;
            out->m_wplus = mass(lp.e + nu.e, lp.x + nu.x, lp.y + nu.y, lp.z + nu.z);
            out->m_top = mass(lp.e + nu.e + bj[i].e, lp.x + nu.x + bj[i].x, lp.y + nu.y + bj[i].y,
                              lp.z + nu.z + bj[i].z);
            out->m_wminus = mass(lm.e + nb4.e, lm.x + nb4.x, lm.y + nb4.y, lm.z + nb4.z);
            out->m_antitop = mass(lm.e + nb4.e + bj[j].e, lm.x + nb4.x + bj[j].x, lm.y + nb4.y + bj[j].y,
                                  lm.z + nb4.z + bj[j].z);
            out->m_higgs = mbb; out->loglik = ll;
            out->variation = v; out->jet_b = o.cand[i]; out->jet_bbar = o.cand[j];
            out->jet_h1 = o.cand[k]; out->jet_h2 = o.cand[l]; out->root = r;
            if (aux) { aux->kappa = S.kappa[r]; aux->pairing = a; aux->higgs_pair = h; aux->pz_terms = S.sz[r]; aux->pzbar_terms = S.szb[r]; }
          } else if (ll > second) {
            second = ll;
          }
        }
        h++;
      }
    }
  }
  if (have) out->status |= 1u;
  if (aux) { aux->loglik2 = second; aux->n_cand = n_cand; }
}

void export_pairing(const PairingSolution& S, orc_pairing_t* out) {
  std::memset(out, 0, sizeof(*out));
  out->n_roots = S.n_roots;
  for (int i = 0; i < 4; i++) out->g[i] = S.g[i];
  for (int i = 0; i < 5; i++) out->h[i] = S.R.h[i];
  const Conic* ks[2] = {&S.k1, &S.k2}; double* dst[2] = {out->conic1, out->conic2};
  for (int c = 0; c < 2; c++) {
    dst[c][0] = ks[c]->a; dst[c][1] = ks[c]->b; dst[c][2] = ks[c]->c;
    dst[c][3] = ks[c]->d; dst[c][4] = ks[c]->e; dst[c][5] = ks[c]->f;
  }
  for (int r = 0; r < S.n_roots; r++) {
    out->x[r] = S.x[r]; out->kappa[r] = S.kappa[r]; out->nterm[r] = S.nterm[r];
    out->pz_terms[r] = S.sz[r]; out->pzbar_terms[r] = S.szb[r];
    out->nu[r][0] = S.nu[r].x; out->nu[r][1] = S.nu[r].y; out->nu[r][2] = S.nu[r].z; out->nu[r][3] = S.nu[r].e;
    out->nubar[r][0] = S.nub[r].x; out->nubar[r][1] = S.nub[r].y; out->nubar[r][2] = S.nub[r].z;
    out->nubar[r][3] = S.nub[r].e;
  }
  out->min_abs_p_rel = S.min_abs_p_rel;
}

}  // namespace

extern "C" int orc_reconstruct_tth(const orc_events_t* ev, const uint32_t* idx, int64_t n_idx, int32_t V,
                                   uint64_t seed, const orc_params_t* params, orc_best_t* out_best,
                                   orc_aux_t* out_aux, int n_threads) {
  if (!ev || (n_idx > 0 && !idx) || n_idx < 0 || V <= 0 || !out_best) return -1;
  orc_params_t P; if (params) P = *params; else orc_default_params(&P);
  if (n_threads < 1) n_threads = 1;
#pragma omp parallel for schedule(dynamic, 16) num_threads(n_threads)
  for (int64_t k = 0; k < n_idx; k++)
    reconstruct_event(ev, idx[k], V, seed, P, &out_best[k], out_aux ? &out_aux[k] : nullptr);
  return 0;
}

extern "C" int orc_solve_pairing(const double lp[4], const double b[4], const double lm[4], const double bbar[4],
                                 const double met[2], const double* jets_h, int n_h, const orc_params_t* params,
                                 orc_pairing_t* out) {
  if (!out || n_h < 0 || n_h > 4) return -1;
  orc_params_t P; if (params) P = *params; else orc_default_params(&P);
  V4 l1{lp[0], lp[1], lp[2], lp[3]}, b1{b[0], b[1], b[2], b[3]}, l2{lm[0], lm[1], lm[2], lm[3]},
      b2{bbar[0], bbar[1], bbar[2], bbar[3]};
  PairingSolution S = solve_pairing(l1, b1, l2, b2, met[0], met[1], P);
  export_pairing(S, out);
  int h = 0;
  for (int k = 0; k < n_h; k++) for (int l = k + 1; l < n_h; l++) {
    const double *p = jets_h + 4 * k, *q = jets_h + 4 * l;
    out->mbb[h] = mass(p[3] + q[3], p[0] + q[0], p[1] + q[1], p[2] + q[2]);
    out->hterm[h] = higgs_term(out->mbb[h], P); h++;
  }
  out->n_higgs = h;
  return 0;
}

extern "C" int orc_quartic(const double g[4], double roots[4], double* min_abs_p_rel) {
  if (!g || !roots) return -1;
  if (min_abs_p_rel) *min_abs_p_rel = tangency_measure(g);
  return quartic_roots(g, roots);
}

extern "C" int orc_smear(const orc_events_t* ev, uint32_t e, int32_t v, uint64_t seed, const orc_params_t* params,
                         double scales[10], double metp[2]) {
  if (!ev || e >= (uint64_t)ev->n_events) return -1;
  orc_params_t P; if (params) P = *params; else orc_default_params(&P);
  EventObjects o = load_event(ev, e);
  smear(o, v, seed, P, scales, &metp[0], &metp[1]);
  return 0;
}

extern "C" int orc_eval_cell(const orc_events_t* ev, uint32_t e, int32_t v, int32_t a, uint64_t seed,
                             const orc_params_t* params, orc_pairing_t* out) {
  if (!ev || !out || e >= (uint64_t)ev->n_events) return -1;
  orc_params_t P; if (params) P = *params; else orc_default_params(&P);
  EventObjects o = load_event(ev, e);
  std::memset(out, 0, sizeof(*out));
  if (!o.applicable) return 1;
  const int nb = o.n_b, i = a / nb, j = a % nb;
  if (a < 0 || i >= nb || i == j) return -1;
  double s[10], Mx, My; smear(o, v, seed, P, s, &Mx, &My);
  V4 lp = scaled(o.lep[o.lp_slot], s[o.lp_slot]), lm = scaled(o.lep[o.lm_slot], s[o.lm_slot]);
  V4 bj[6] = {}; for (int c = 0; c < nb; c++) bj[c] = scaled(o.jet[o.cand[c]], s[2 + o.cand[c]]);
  PairingSolution S = solve_pairing(lp, bj[i], lm, bj[j], Mx, My, P);
  export_pairing(S, out);
  int h = 0;
  for (int k = 0; k < nb; k++) for (int l = k + 1; l < nb; l++) {
    if (k == i || k == j || l == i || l == j) continue;
    out->mbb[h] = mass(bj[k].e + bj[l].e, bj[k].x + bj[l].x, bj[k].y + bj[l].y, bj[k].z + bj[l].z);
    out->hterm[h] = higgs_term(out->mbb[h], P); h++;
  }
  out->n_higgs = h;
  return 0;
}

// PAPER.md:410-442 (App. 8.2 listing): "TLorentzVector ttH = Top + Tbar + Higgs; mTTH = ttH.M(); ptTTH = ttH.Pt();" — the
// invariant mass and the transverse momentum of the reconstructed ttH system, the two quantities the example analysis
// histograms.  For a record with a solution: the smeared objects of the record's variation (O4 step 2), the neutrinos with
// E = |p|, and the eight four-vectors added in the order l+, l-, nu, nubar, b, bbar, h1, h2; m = sqrt(max(E^2 - |p|^2, 0)),
// pT = sqrt(px^2 + py^2).  Without a solution both are NaN.  Every operation is one IEEE operation in the order written.
extern "C" int orc_tth_system(const orc_events_t* ev, const orc_best_t* best, int64_t n, uint64_t seed,
                              const orc_params_t* params, double* out) {
  if (!ev || n < 0 || (n > 0 && (!best || !out))) return -1;
  orc_params_t P; if (params) P = *params; else orc_default_params(&P);
  for (int64_t k = 0; k < n; k++) {
    const orc_best_t& b = best[k];
    out[2 * k] = out[2 * k + 1] = NaN;
    if (!(b.status & 1u) || b.event >= (uint64_t)ev->n_events) continue;
    EventObjects o = load_event(ev, b.event);
    double s[10], Mx, My; smear(o, b.variation, seed, P, s, &Mx, &My);
    auto jet = [&](int slot) { return scaled(o.jet[slot], s[2 + slot]); };
    V4 nu{b.nu[0], b.nu[1], b.nu[2], std::sqrt(b.nu[0] * b.nu[0] + b.nu[1] * b.nu[1] + b.nu[2] * b.nu[2])};
    V4 nb{b.nubar[0], b.nubar[1], b.nubar[2],
          std::sqrt(b.nubar[0] * b.nubar[0] + b.nubar[1] * b.nubar[1] + b.nubar[2] * b.nubar[2])};
    const V4 parts[8] = {scaled(o.lep[o.lp_slot], s[o.lp_slot]), scaled(o.lep[o.lm_slot], s[o.lm_slot]), nu, nb,
                         jet(b.jet_b), jet(b.jet_bbar), jet(b.jet_h1), jet(b.jet_h2)};
    V4 sum = parts[0];
    for (int i = 1; i < 8; i++) { sum.x = sum.x + parts[i].x; sum.y = sum.y + parts[i].y; sum.z = sum.z + parts[i].z; sum.e = sum.e + parts[i].e; }
    double m2 = sum.e * sum.e - (sum.x * sum.x + sum.y * sum.y + sum.z * sum.z);
    out[2 * k] = std::sqrt(m2 > 0.0 ? m2 : 0.0);
    out[2 * k + 1] = std::sqrt(sum.x * sum.x + sum.y * sum.y);
  }
  return 0;
}
