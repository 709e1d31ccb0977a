/*
 * tests/referee_q128.c — TEST-ONLY high-precision referee (IEEE binary128, ~34 digits) for the dilepton solve.
 *
 * Purpose (R11): when the CUDA path and the FP64 oracle disagree beyond the 1e-9 that
 * BASELINE.json:north_star states, somebody has to say which side is farther from the exact answer.  This file computes
 * the exact answer of DESIGN.md section 2 ("Method") for one (event, variation, pairing) cell in binary128:
 *   - the smearing of step 2 in FP64, bit for bit (a third, independent restatement of Philox4x32-10 + the operation
 *     sequences L / SC of SURVEY.md 8(c) O1-O2; "varied within the resolution"),
 *   - the two leg conics, the shift by MET', the resultant quartic of step 3 in binary128 (the mass
 *     constraints "have quadratic forms", "normally several" solutions),
 *   - ALL real roots by a derivative-chain bisection in binary128,
 *   - and then, independently of that algebra, a 4-dimensional Newton iteration in binary128 on the RAW constraints
 *     m(l+ nu) = m_W, m(l+ nu b) = m_t, m(l- nubar) = m_W, m(l- nubar bbar) = m_t, nu_T + nubar_T = MET'
 *      started from every root: the reported solutions satisfy the physics, not a derived formula.
 * It calls neither oracle/ nor paper_2211_14346_b200/csrc/ and shares no code with them; only tests/ uses it.
 *
 * Build: gcc -O2 -ffp-contract=off -fPIC -shared tests/referee_q128.c -o tests/libreferee.so -lquadmath -lm
 */
#include <math.h>
#include <quadmath.h>
#include <stdint.h>
#include <string.h>

typedef __float128 Q;

typedef struct {
  int64_t n_events, stride, event_base;
  const double *lep_px, *lep_py, *lep_pz, *lep_e, *lep_pt, *lep_eta;
  const double *jet_px, *jet_py, *jet_pz, *jet_e, *jet_pt, *jet_eta;
  const double *met_x, *met_y, *met, *mll;
  const uint32_t* flags;
} ref_events_t;

typedef struct {
  double m_top, m_w, m_higgs, sigma_higgs, lambda_nu, lep_sigma, jet_stoch, jet_const, sigma_scale, s_min;
} ref_params_t;

typedef struct {
  int32_t status;        /* 0 = solved (n_roots may be 0); 1 = event not applicable / bad pairing; 2 = degenerate (n_z guard, h4 = 0) */
  int32_t n_roots, n_higgs, n_crit;
  double lp[4], b[4], lm[4], bbar[4], met[2];   /* the smeared FP64 inputs of the cell (px, py, pz, E), MET'          */
  double h[5], g[4];                            /* exact resultant h0..h4 and monic g0..g3, rounded to double          */
  double x[4], y[4];                            /* roots ascending in x                                                */
  double nu[4][4], nubar[4][4];                 /* exact solutions (px, py, pz, E), rounded to double                  */
  double nterm[4];                              /* ln(pT pT') - (pT + pT') / lambda_nu                                 */
  double kappa[4];                              /* 2^-53 sum|h_i x^i| / |x P'(x)|                                      */
  double pz_terms[4], pzbar_terms[4];           /* |c0| + |c1 x| + |c2 y| of the two p_z linear forms                  */
  double newton_shift[4];                       /* relative distance between the conic-algebra point and the raw-constraint solution */
  double residual[4];                           /* max |raw constraint| / m_t^2 at the reported solution               */
  double crit_x[3], crit_rel[3];                /* critical points of P and |P| / sum|h_i x^i| there                   */
  double min_abs_p_rel;                         /* min of crit_rel (1 if none)                                         */
  double hterm[6], mbb[6];                      /* Higgs term and m_bb of the Higgs pairs of this pairing, in order    */
} ref_cell_t;

/* ------------------------------------------------------------------------------------------------------------------
 * FP64 smearing, bit for bit (DESIGN.md section 2 step 2)
 * ------------------------------------------------------------------------------------------------------------------ */
static void philox_4x32_10(uint32_t c[4], uint32_t ka, uint32_t kb) {
  /* key schedule first, then ten rounds: round r uses key + r * (Weyl constants) */
  uint32_t ks[10][2];
  for (int r = 0; r < 10; r++) { ks[r][0] = ka + (uint32_t)r * 0x9E3779B9u; ks[r][1] = kb + (uint32_t)r * 0xBB67AE85u; }
  for (int r = 0; r < 10; r++) {
    uint64_t a = (uint64_t)0xD2511F53u * c[0], d = (uint64_t)0xCD9E8D57u * c[2];
    uint32_t n0 = (uint32_t)(d >> 32) ^ c[1] ^ ks[r][0], n2 = (uint32_t)(a >> 32) ^ c[3] ^ ks[r][1];
    c[1] = (uint32_t)d; c[3] = (uint32_t)a; c[0] = n0; c[2] = n2;
  }
}

static double seq_L(double u) {          /* ln u, u in (0, 1], operation sequence L */
  int e; double m = frexp(u, &e);        /* u = m 2^e, m in [0.5, 1) */
  m *= 2.0; e -= 1;                      /* m in [1, 2) */
  if (m > 0x1.6a09e667f3bcdp+0) { m *= 0.5; e += 1; }
  double f = m - 1.0, s = f / (2.0 + f), z = s * s;
  double p = 2.0 / 19.0;
  for (int k = 8; k >= 1; k--) p = fma(p, z, 2.0 / (2.0 * k + 1.0));
  p *= z;
  double lm = fma(s, p, 2.0 * s), ed = (double)e;
  return fma(ed, 0x1.62e42fee00000p-1, fma(ed, 0x1.a39ef35793c76p-33, lm));
}

static void seq_SC(double u, double* sn, double* cs) {   /* (sin, cos)(2 pi u), u in [0, 1), operation sequence SC */
  double t = 4.0 * u, n = floor(t + 0.5), r = t - n;
  double th = fma(r, 0x1.921fb54442d18p+0, r * 0x1.1a62633145c07p-54), z = th * th;
  double fs = 355687428096000.0 /* 17! */, fc = 20922789888000.0 /* 16! */;
  double ps = 1.0 / fs, pc = 1.0 / fc;
  for (int k = 7; k >= 1; k--) {
    fs /= (double)((2 * k + 2) * (2 * k + 3)); fc /= (double)((2 * k + 1) * (2 * k + 2));   /* (2k+1)!, (2k)!: exact */
    ps = fma(ps, z, ((k & 1) ? -1.0 : 1.0) / fs);
    pc = fma(pc, z, ((k & 1) ? -1.0 : 1.0) / fc);
  }
  double s = fma(th * z, ps, th), c = fma(z, pc, 1.0);
  switch (((int)n) & 3) {
    case 0: *sn = s; *cs = c; break;
    case 1: *sn = c; *cs = -s; break;
    case 2: *sn = -s; *cs = -c; break;
    default: *sn = -c; *cs = s; break;
  }
}

typedef struct {
  int applicable, n_jet, n_b, lp_slot, cand[6];
  double lep[2][4], jet[8][4], met[2];
  uint64_t gidx;
} ref_event_t;

static void load_event(const ref_events_t* ev, uint32_t e, ref_event_t* o) {
  const int64_t S = ev->stride;
  const uint32_t f = ev->flags[e];
  memset(o, 0, sizeof(*o));
  o->n_jet = (int)((f >> 8) & 15u); if (o->n_jet > 8) o->n_jet = 8;
  for (int s = 0; s < 2; s++) {
    o->lep[s][0] = ev->lep_px[s * S + e]; o->lep[s][1] = ev->lep_py[s * S + e];
    o->lep[s][2] = ev->lep_pz[s * S + e]; o->lep[s][3] = ev->lep_e[s * S + e];
  }
  for (int s = 0; s < 8; s++) {
    o->jet[s][0] = ev->jet_px[s * S + e]; o->jet[s][1] = ev->jet_py[s * S + e];
    o->jet[s][2] = ev->jet_pz[s * S + e]; o->jet[s][3] = ev->jet_e[s * S + e];
  }
  o->met[0] = ev->met_x[e]; o->met[1] = ev->met_y[e];
  for (int s = 0; s < o->n_jet; s++)
    if (((f >> (16 + s)) & 1u) && o->n_b < 6) o->cand[o->n_b++] = s;
  const int q0 = (f >> 4) & 1u, q1 = (f >> 5) & 1u;
  o->applicable = ((f & 15u) == 2u) && (q0 != q1) && (o->n_b >= 4);
  o->lp_slot = q0 ? 0 : 1;
  o->gidx = (uint64_t)(ev->event_base + (int64_t)e);
}

static void smear(const ref_event_t* o, int32_t v, uint64_t seed, const ref_params_t* P, double s[10], double M[2]) {
  double z[10];
  for (uint32_t blk = 0; blk < 5; blk++) {
    uint32_t c[4] = {(uint32_t)o->gidx, (uint32_t)(o->gidx >> 32), (uint32_t)v, 0x54544800u + blk};
    philox_4x32_10(c, (uint32_t)seed, (uint32_t)(seed >> 32));
    uint64_t w0 = ((uint64_t)c[1] << 32) | c[0], w1 = ((uint64_t)c[3] << 32) | c[2];
    double u1 = (double)((w0 >> 11) + 1) * 0x1p-53, u2 = (double)(w1 >> 11) * 0x1p-53;
    double rho = sqrt(-2.0 * seq_L(u1)), sn, cs;
    seq_SC(u2, &sn, &cs);
    z[2 * blk] = rho * cs; z[2 * blk + 1] = rho * sn;
  }
  for (int t = 0; t < 10; t++) {
    double sigma = t < 2 ? P->lep_sigma : P->jet_stoch / sqrt(o->jet[t - 2][3]) + P->jet_const;
    double sc = fma(P->sigma_scale * sigma, z[t], 1.0);
    s[t] = sc > P->s_min ? sc : P->s_min;
  }
  double ax = 0.0, ay = 0.0;
  for (int t = 0; t < 2 + o->n_jet; t++) {
    const double* p = t < 2 ? o->lep[t] : o->jet[t - 2];
    ax = ax + (s[t] - 1.0) * p[0]; ay = ay + (s[t] - 1.0) * p[1];
  }
  M[0] = o->met[0] - ax; M[1] = o->met[1] - ay;
}

int ref_smear(const ref_events_t* ev, uint32_t e, int32_t v, uint64_t seed, const ref_params_t* P, double scales[10],
              double metp[2]) {
  if (!ev || e >= (uint64_t)ev->n_events) return -1;
  ref_event_t o; load_event(ev, e, &o);
  smear(&o, v, seed, P, scales, metp);
  return 0;
}

/* ------------------------------------------------------------------------------------------------------------------
 * binary128 algebra (DESIGN.md section 2 step 3)
 * ------------------------------------------------------------------------------------------------------------------ */
typedef struct { Q a, b, c, d, e, f; } conic_t;
typedef struct { conic_t k; Q c0, c1, c2; int ok; } leg_t;

static leg_t leg_conic(const double l[4], const double b[4], Q mt, Q mw) {
  leg_t g; memset(&g, 0, sizeof(g));
  Q lx = l[0], ly = l[1], lz = l[2], le = l[3], bx = b[0], by = b[1], bz = b[2], be = b[3];
  Q ml2 = le * le - (lx * lx + ly * ly + lz * lz), mb2 = be * be - (bx * bx + by * by + bz * bz);
  Q bl = be * le - (bx * lx + by * ly + bz * lz);
  Q A = (mw * mw - ml2) / 2, B = (mt * mt - mw * mw - mb2) / 2 - bl;
  Q nx = be * lx - le * bx, ny = be * ly - le * by, nz = be * lz - le * bz, k = le * B - be * A;
  g.ok = fabsq(nz) > 1e-12Q * be * le;
  if (!g.ok) return g;
  g.c0 = k / nz; g.c1 = -nx / nz; g.c2 = -ny / nz;
  Q d0 = (A + lz * g.c0) / le, d1 = (lx + lz * g.c1) / le, d2 = (ly + lz * g.c2) / le;
  g.k.a = d1 * d1 - 1 - g.c1 * g.c1; g.k.b = 2 * (d1 * d2 - g.c1 * g.c2); g.k.c = d2 * d2 - 1 - g.c2 * g.c2;
  g.k.d = 2 * (d0 * d1 - g.c0 * g.c1); g.k.e = 2 * (d0 * d2 - g.c0 * g.c2); g.k.f = d0 * d0 - g.c0 * g.c0;
  return g;
}

static Q polyv(const Q* c, int deg, Q x) { Q v = c[deg]; for (int i = deg - 1; i >= 0; i--) v = v * x + c[i]; return v; }

static int bisect(const Q* c, int deg, Q lo, Q hi, Q* root) {
  Q flo = polyv(c, deg, lo), fhi = polyv(c, deg, hi);
  if (flo == 0) { *root = lo; return 1; }
  if (!((flo < 0) != (fhi < 0)) || fhi == 0) return 0;
  for (int it = 0; it < 400; it++) {
    Q mid = (lo + hi) / 2;
    if (mid == lo || mid == hi) break;
    Q fm = polyv(c, deg, mid);
    if (fm == 0) { lo = hi = mid; break; }
    if ((fm < 0) == (flo < 0)) { lo = mid; flo = fm; } else hi = mid;
  }
  *root = (lo + hi) / 2;
  return 1;
}

static int roots_between(const Q* c, int deg, const Q* crit, int n_crit, Q R, Q* out) {
  Q edges[8]; int ne = 0, n = 0;
  edges[ne++] = -R;
  for (int i = 0; i < n_crit; i++) edges[ne++] = crit[i];
  edges[ne++] = R;
  for (int i = 0; i + 1 < ne; i++) {
    Q r;
    if (edges[i] < edges[i + 1] && bisect(c, deg, edges[i], edges[i + 1], &r)) out[n++] = r;
  }
  return n;
}

/* 4-D Newton on the raw constraints; u = (px, py, pz, qz).  Returns the number of iterations used, -1 on failure. */
typedef struct { Q l[4], b[4], lb[4], bb[4], Mx, My, mt2, mw2, ml2, mb2, mlb2, mbb2, lbl, lbb; } raw_t;

static void raw_setup(raw_t* R, const double lp[4], const double b[4], const double lm[4], const double bb[4], double Mx,
                      double My, double mt, double mw) {
  for (int i = 0; i < 4; i++) { R->l[i] = lp[i]; R->b[i] = b[i]; R->lb[i] = lm[i]; R->bb[i] = bb[i]; }
  R->Mx = Mx; R->My = My; R->mt2 = (Q)mt * mt; R->mw2 = (Q)mw * mw;
#define M2(v) ((v)[3] * (v)[3] - ((v)[0] * (v)[0] + (v)[1] * (v)[1] + (v)[2] * (v)[2]))
#define DOT4(u, v) ((u)[3] * (v)[3] - ((u)[0] * (v)[0] + (u)[1] * (v)[1] + (u)[2] * (v)[2]))
  R->ml2 = M2(R->l); R->mb2 = M2(R->b); R->mlb2 = M2(R->lb); R->mbb2 = M2(R->bb);
  R->lbl = DOT4(R->l, R->b); R->lbb = DOT4(R->lb, R->bb);
}

static void raw_eval(const raw_t* R, const Q u[4], Q F[4], Q J[4][4]) {
  Q px = u[0], py = u[1], pz = u[2], qx = R->Mx - px, qy = R->My - py, qz = u[3];
  Q E = sqrtq(px * px + py * py + pz * pz), Eq = sqrtq(qx * qx + qy * qy + qz * qz);
  /* (l + nu)^2 = m_W^2 ;  (l + nu + b)^2 = m_t^2, as invariant masses of the sums */
  F[0] = R->ml2 + 2 * (R->l[3] * E - (R->l[0] * px + R->l[1] * py + R->l[2] * pz)) - R->mw2;
  F[1] = R->ml2 + R->mb2 + 2 * R->lbl + 2 * ((R->l[3] + R->b[3]) * E - ((R->l[0] + R->b[0]) * px + (R->l[1] + R->b[1]) * py +
                                                                      (R->l[2] + R->b[2]) * pz)) - R->mt2;
  F[2] = R->mlb2 + 2 * (R->lb[3] * Eq - (R->lb[0] * qx + R->lb[1] * qy + R->lb[2] * qz)) - R->mw2;
  F[3] = R->mlb2 + R->mbb2 + 2 * R->lbb + 2 * ((R->lb[3] + R->bb[3]) * Eq - ((R->lb[0] + R->bb[0]) * qx +
                                               (R->lb[1] + R->bb[1]) * qy + (R->lb[2] + R->bb[2]) * qz)) - R->mt2;
  if (!J) return;
  Q s1 = R->l[3], s2 = R->l[3] + R->b[3], t1 = R->lb[3], t2 = R->lb[3] + R->bb[3];
  Q ux = px / E, uy = py / E, uz = pz / E, vx = qx / Eq, vy = qy / Eq, vz = qz / Eq;
  J[0][0] = 2 * (s1 * ux - R->l[0]); J[0][1] = 2 * (s1 * uy - R->l[1]); J[0][2] = 2 * (s1 * uz - R->l[2]); J[0][3] = 0;
  J[1][0] = 2 * (s2 * ux - (R->l[0] + R->b[0])); J[1][1] = 2 * (s2 * uy - (R->l[1] + R->b[1]));
  J[1][2] = 2 * (s2 * uz - (R->l[2] + R->b[2])); J[1][3] = 0;
  J[2][0] = -2 * (t1 * vx - R->lb[0]); J[2][1] = -2 * (t1 * vy - R->lb[1]); J[2][2] = 0; J[2][3] = 2 * (t1 * vz - R->lb[2]);
  J[3][0] = -2 * (t2 * vx - (R->lb[0] + R->bb[0])); J[3][1] = -2 * (t2 * vy - (R->lb[1] + R->bb[1])); J[3][2] = 0;
  J[3][3] = 2 * (t2 * vz - (R->lb[2] + R->bb[2]));
}

static int solve4(Q A[4][4], Q b[4], Q x[4]) {
  int p[4] = {0, 1, 2, 3};
  for (int c = 0; c < 4; c++) {
    int best = c;
    for (int r = c + 1; r < 4; r++) if (fabsq(A[p[r]][c]) > fabsq(A[p[best]][c])) best = r;
    int t = p[c]; p[c] = p[best]; p[best] = t;
    if (A[p[c]][c] == 0) return -1;
    for (int r = c + 1; r < 4; r++) {
      Q m = A[p[r]][c] / A[p[c]][c];
      for (int k = c; k < 4; k++) A[p[r]][k] -= m * A[p[c]][k];
      b[p[r]] -= m * b[p[c]];
    }
  }
  for (int c = 3; c >= 0; c--) {
    Q s = b[p[c]];
    for (int k = c + 1; k < 4; k++) s -= A[p[c]][k] * x[k];
    x[c] = s / A[p[c]][c];
  }
  return 0;
}

static int raw_newton(const raw_t* R, Q u[4]) {
  /* converged when a step no longer moves the point beyond binary128 rounding: either below 1e-28 relative, or (for an
   * ill-conditioned intersection, where rounding in the residuals limits the attainable step) below 1e-20 and no longer
   * shrinking.  Either way the point is exact to many more digits than the FP64 sides being refereed. */
  Q prev = -1;
  for (int it = 0; it < 80; it++) {
    Q F[4], J[4][4], d[4];
    raw_eval(R, u, F, J);
    if (solve4(J, F, d) != 0) return -1;
    Q mv = 0, sc = 0;
    for (int i = 0; i < 4; i++) {
      if (!finiteq(d[i])) return -1;
      u[i] -= d[i]; mv += fabsq(d[i]); sc += fabsq(u[i]);
    }
    if (mv <= 1e-28Q * sc) return it + 1;
    if (prev >= 0 && mv <= 1e-20Q * sc && mv >= prev / 4) return it + 1;
    prev = mv;
  }
  return -1;
}

static double raw_residual(const raw_t* R, const Q u[4]) {
  Q F[4], m = 0; raw_eval(R, u, F, 0);
  for (int i = 0; i < 4; i++) if (fabsq(F[i]) > m) m = fabsq(F[i]);
  return (double)(m / R->mt2);
}

static Q mass4(const Q a[4]) { Q m2 = a[3] * a[3] - (a[0] * a[0] + a[1] * a[1] + a[2] * a[2]); return sqrtq(m2 > 0 ? m2 : 0); }

/* solve the cell whose smeared inputs are in out->lp, b, lm, bbar, met */
static int solve_core(ref_cell_t* out, const ref_params_t* P) {
  const double* M = out->met;
  const Q mt = P->m_top, mw = P->m_w, Mx = M[0], My = M[1];
  leg_t g1 = leg_conic(out->lp, out->b, mt, mw), g2 = leg_conic(out->lm, out->bbar, mt, mw);
  if (!g1.ok || !g2.ok) { out->status = 2; return 0; }
  conic_t k1 = g1.k, q = g2.k, k2;
  k2.a = q.a; k2.b = q.b; k2.c = q.c;
  k2.d = -2 * q.a * Mx - q.b * My - q.d; k2.e = -2 * q.c * My - q.b * Mx - q.e;
  k2.f = q.a * Mx * Mx + q.b * Mx * My + q.c * My * My + q.d * Mx + q.e * My + q.f;
  Q p[3] = {k1.c * k2.f - k2.c * k1.f, k1.c * k2.d - k2.c * k1.d, k1.c * k2.a - k2.c * k1.a};
  Q d2[2] = {k1.c * k2.e - k2.c * k1.e, k1.c * k2.b - k2.c * k1.b};
  Q r[4] = {k1.e * k2.f - k2.e * k1.f, k1.e * k2.d + k1.b * k2.f - k2.e * k1.d - k2.b * k1.f,
            k1.e * k2.a + k1.b * k2.d - k2.e * k1.a - k2.b * k1.d, k1.b * k2.a - k2.b * k1.a};
  Q h[5] = {p[0] * p[0] - d2[0] * r[0], 2 * p[0] * p[1] - (d2[0] * r[1] + d2[1] * r[0]),
            2 * p[0] * p[2] + p[1] * p[1] - (d2[0] * r[2] + d2[1] * r[1]), 2 * p[1] * p[2] - (d2[0] * r[3] + d2[1] * r[2]),
            p[2] * p[2] - d2[1] * r[3]};
  if (h[4] == 0 || !finiteq(h[4])) { out->status = 2; return 0; }
  Q g[5]; for (int k = 0; k < 4; k++) g[k] = h[k] / h[4];
  g[4] = 1;
  for (int k = 0; k < 5; k++) out->h[k] = (double)h[k];
  for (int k = 0; k < 4; k++) out->g[k] = (double)g[k];
  /* derivative chain */
  Q R = 1; for (int k = 0; k < 4; k++) if (1 + fabsq(g[k]) > R) R = 1 + fabsq(g[k]);
  Q P1[4] = {g[1], 2 * g[2], 3 * g[3], 4}, P2[3] = {2 * g[2], 6 * g[3], 12};
  Q c2[2]; int n2 = 0;
  Q disc = P2[1] * P2[1] - 4 * P2[2] * P2[0];
  if (disc > 0) { Q sq = sqrtq(disc); c2[0] = (-P2[1] - sq) / 24; c2[1] = (-P2[1] + sq) / 24; n2 = 2; }
  Q c1[3]; int n1 = roots_between(P1, 3, c2, n2, R, c1);
  Q xr[4]; int n = roots_between(g, 4, c1, n1, R, xr);
  out->n_crit = n1;
  for (int k = 0; k < n1; k++) {
    Q sum = 0, xp = 1; for (int m = 0; m <= 4; m++) { sum += fabsq(g[m] * xp); xp *= c1[k]; }
    out->crit_x[k] = (double)c1[k]; out->crit_rel[k] = (double)(fabsq(polyv(g, 4, c1[k])) / sum);
    if (out->crit_rel[k] < out->min_abs_p_rel) out->min_abs_p_rel = out->crit_rel[k];
  }
  raw_t RW; raw_setup(&RW, out->lp, out->b, out->lm, out->bbar, M[0], M[1], P->m_top, P->m_w);
  int nr = 0;
  for (int k = 0; k < n; k++) {
    Q x = xr[k];
    for (int it = 0; it < 3; it++) { Q d = polyv(P1, 3, x); if (d != 0) x -= polyv(g, 4, x) / d; }
    Q D1 = p[0] + p[1] * x + p[2] * x * x, D2 = d2[0] + d2[1] * x;
    if (D2 == 0) continue;
    Q y = -D1 / D2;
    Q u[4] = {x, y, g1.c0 + g1.c1 * x + g1.c2 * y, g2.c0 + g2.c1 * (Mx - x) + g2.c2 * (My - y)};
    Q u0[4] = {u[0], u[1], u[2], u[3]};
    if (raw_newton(&RW, u) < 0) continue;
    Q mv = 0, sc = 0; for (int m = 0; m < 4; m++) { mv += fabsq(u[m] - u0[m]); sc += fabsq(u[m]); }
    Q px = u[0], py = u[1], pz = u[2], qx = Mx - px, qy = My - py, qz = u[3];
    Q En = sqrtq(px * px + py * py + pz * pz), Eb = sqrtq(qx * qx + qy * qy + qz * qz);
    Q ptn = sqrtq(px * px + py * py), ptb = sqrtq(qx * qx + qy * qy);
    out->x[nr] = (double)px; out->y[nr] = (double)py;
    out->nu[nr][0] = (double)px; out->nu[nr][1] = (double)py; out->nu[nr][2] = (double)pz; out->nu[nr][3] = (double)En;
    out->nubar[nr][0] = (double)qx; out->nubar[nr][1] = (double)qy; out->nubar[nr][2] = (double)qz; out->nubar[nr][3] = (double)Eb;
    out->nterm[nr] = (double)(logq(ptn * ptb) - (ptn + ptb) / (Q)P->lambda_nu);
    Q sum = 0, xp = 1; for (int m = 0; m <= 4; m++) { sum += fabsq(h[m] * xp); xp *= px; }
    Q dP = h[1] + px * (2 * h[2] + px * (3 * h[3] + px * 4 * h[4]));
    out->kappa[nr] = (double)(0x1p-53Q * sum / fabsq(px * dP));
    out->pz_terms[nr] = (double)(fabsq(g1.c0) + fabsq(g1.c1 * px) + fabsq(g1.c2 * py));
    out->pzbar_terms[nr] = (double)(fabsq(g2.c0) + fabsq(g2.c1 * qx) + fabsq(g2.c2 * qy));
    out->newton_shift[nr] = (double)(mv / sc);
    out->residual[nr] = raw_residual(&RW, u);
    nr++;
  }
  out->n_roots = nr;
  return 0;
}


/* the cell: everything about (event e, variation v, pairing a = i * n_b + j) */
int ref_cell(const ref_events_t* ev, uint32_t e, int32_t v, int32_t a, uint64_t seed, const ref_params_t* P, ref_cell_t* out) {
  if (!ev || !out || !P || e >= (uint64_t)ev->n_events) return -1;
  memset(out, 0, sizeof(*out));
  out->min_abs_p_rel = 1.0;
  ref_event_t o; load_event(ev, e, &o);
  if (!o.applicable) { out->status = 1; return 0; }
  const int nb = o.n_b, i = a / nb, j = a % nb;
  if (a < 0 || i >= nb || i == j) { out->status = 1; return 0; }
  double s[10], M[2]; smear(&o, v, seed, P, s, M);
  const int lps = o.lp_slot, lms = 1 - o.lp_slot;
  double jets[6][4];
  for (int k = 0; k < 4; k++) {
    out->lp[k] = s[lps] * o.lep[lps][k]; out->lm[k] = s[lms] * o.lep[lms][k];
    for (int c = 0; c < nb; c++) jets[c][k] = s[2 + o.cand[c]] * o.jet[o.cand[c]][k];
  }
  memcpy(out->b, jets[i], sizeof(out->b)); memcpy(out->bbar, jets[j], sizeof(out->bbar));
  out->met[0] = M[0]; out->met[1] = M[1];
  /* Higgs pairs: candidates not in {i, j}, k < l lexicographic */
  for (int k = 0; k < nb; k++) for (int l = k + 1; l < nb; l++) {
    if (k == i || k == j || l == i || l == j) continue;
    Q sum[4]; for (int c = 0; c < 4; c++) sum[c] = (Q)jets[k][c] + (Q)jets[l][c];
    /* the definition adds the two smeared jets in FP64 before taking the mass; the sum of two doubles is what is squared */
    Q mbb = mass4(sum), t = (mbb - (Q)P->m_higgs) / (Q)P->sigma_higgs;
    out->mbb[out->n_higgs] = (double)mbb; out->hterm[out->n_higgs] = (double)(-t * t / 2); out->n_higgs++;
  }
  return solve_core(out, P);
}

/* 4-D Newton in binary128 from a caller-supplied FP64 point (a record of either side): which exact solution does it
 * belong to, and how far from it is it?  out7 = nu(px, py, pz), nubar(px, py, pz), neutrino term.  Returns iterations, -1. */
int ref_polish(const ref_events_t* ev, uint32_t e, int32_t v, int32_t a, uint64_t seed, const ref_params_t* P,
               const double nu[3], double nubar_z, double out7[7]) {
  ref_cell_t c;   /* only for the smeared inputs */
  if (!ev || !P || e >= (uint64_t)ev->n_events) return -1;
  ref_event_t o; load_event(ev, e, &o);
  if (!o.applicable) return -1;
  const int nb = o.n_b, i = a / nb, j = a % nb;
  if (a < 0 || i >= nb || i == j) return -1;
  double s[10], M[2]; smear(&o, v, seed, P, s, M);
  const int lps = o.lp_slot, lms = 1 - o.lp_slot;
  for (int k = 0; k < 4; k++) {
    c.lp[k] = s[lps] * o.lep[lps][k]; c.lm[k] = s[lms] * o.lep[lms][k];
    c.b[k] = s[2 + o.cand[i]] * o.jet[o.cand[i]][k]; c.bbar[k] = s[2 + o.cand[j]] * o.jet[o.cand[j]][k];
  }
  raw_t RW; raw_setup(&RW, c.lp, c.b, c.lm, c.bbar, M[0], M[1], P->m_top, P->m_w);
  Q u[4] = {nu[0], nu[1], nu[2], nubar_z};
  int it = raw_newton(&RW, u);
  if (it < 0) return -1;
  Q qx = (Q)M[0] - u[0], qy = (Q)M[1] - u[1];
  Q ptn = sqrtq(u[0] * u[0] + u[1] * u[1]), ptb = sqrtq(qx * qx + qy * qy);
  out7[0] = (double)u[0]; out7[1] = (double)u[1]; out7[2] = (double)u[2];
  out7[3] = (double)qx; out7[4] = (double)qy; out7[5] = (double)u[3];
  out7[6] = (double)(logq(ptn * ptb) - (ptn + ptb) / (Q)P->lambda_nu);
  return it;
}

/* a pairing from explicit FP64 four-vectors (worked example, hand-built cases): same outputs as ref_cell */
int ref_pairing(const double lp[4], const double b[4], const double lm[4], const double bbar[4], const double met[2],
                const ref_params_t* P, ref_cell_t* out) {
  if (!out || !P) return -1;
  memset(out, 0, sizeof(*out));
  out->min_abs_p_rel = 1.0;
  memcpy(out->lp, lp, 32); memcpy(out->b, b, 32); memcpy(out->lm, lm, 32); memcpy(out->bbar, bbar, 32);
  out->met[0] = met[0]; out->met[1] = met[1];
  return solve_core(out, P);
}

/* real roots and tangency measure of a monic quartic given in FP64 (hand-built near-tangent pins) */
int ref_quartic(const double g_in[4], double roots[4], double* min_abs_p_rel) {
  Q g[5] = {g_in[0], g_in[1], g_in[2], g_in[3], 1};
  Q R = 1; for (int k = 0; k < 4; k++) if (1 + fabsq(g[k]) > R) R = 1 + fabsq(g[k]);
  Q P1[4] = {g[1], 2 * g[2], 3 * g[3], 4}, P2[3] = {2 * g[2], 6 * g[3], 12};
  Q c2[2]; int n2 = 0;
  Q disc = P2[1] * P2[1] - 4 * P2[2] * P2[0];
  if (disc > 0) { Q sq = sqrtq(disc); c2[0] = (-P2[1] - sq) / 24; c2[1] = (-P2[1] + sq) / 24; n2 = 2; }
  Q c1[3]; int n1 = roots_between(P1, 3, c2, n2, R, c1);
  Q xr[4]; int n = roots_between(g, 4, c1, n1, R, xr);
  double m = 1.0;
  for (int k = 0; k < n1; k++) {
    Q sum = 0, xp = 1; for (int q = 0; q <= 4; q++) { sum += fabsq(g[q] * xp); xp *= c1[k]; }
    double rel = (double)(fabsq(polyv(g, 4, c1[k])) / sum);
    if (rel < m) m = rel;
  }
  for (int k = 0; k < n; k++) roots[k] = (double)xr[k];
  if (min_abs_p_rel) *min_abs_p_rel = m;
  return n;
}
