// hepf_reco.cu — hepf_reconstruct_tth: smear -> leg conics -> quartic -> score -> argmax.
//
// Paper: PAPER.md:134-138 (§4) — the neutrino four-momenta are reconstructed analytically from energy-momentum
// conservation and the m_W = 80.4 / m_t = 172.5 constraints on both legs ("quadratic forms", several solutions or
// none), every b-jet/lepton pairing is tried, two of the remaining b-jets should give m_bb = 125 GeV and the most
// probable solution wins; PAPER.md:145 — the measured momenta are varied V times within the resolution.  The
// equations themselves are in DESIGN.md "Method" (the paper defers them to its ref. [27]).
//
// B200 mapping (v1): one thread owns one (event, variation).  It draws the ten normals in registers (Philox4x32-10
// + Box-Muller, bit-identical to the specified operation sequence), smears the objects, builds the n_b leg-2 conics
// once (kept in a per-thread, bank-conflict-free column of shared memory), then walks the ordered pairings (i, j):
// leg-1 conic in registers, resultant -> monic quartic -> Ferrari closed form -> two Newton steps per root ->
// neutrino pT score.  The thread keeps its best candidate; a shared-memory atomicMax/atomicMin pair reduces the
// threads of one event with the total order (loglik, then lowest (variation, pairing)); the winning thread
// re-derives the full solution and writes the 128-byte record.  No tensor cores: nothing here is a contraction.
#include <math_constants.h>

#include "hepf_common.cuh"

namespace hepf {

constexpr int RECO_THREADS = 128;
constexpr int NB_MAX = HEPF_MAX_B;
constexpr int TH_CONIC2 = 0;                      // per-thread shared layout, in doubles
constexpr int TH_SCALE = TH_CONIC2 + 6 * NB_MAX;  // scales of the b candidates
constexpr int TH_HT = TH_SCALE + NB_MAX;          // Higgs term of every unordered candidate pair
constexpr int TH_DOUBLES = TH_HT + 15;

struct RecoCols {
  const double *lep_px, *lep_py, *lep_pz, *lep_e, *jet_px, *jet_py, *jet_pz, *jet_e, *met_x, *met_y;
  const uint32_t* flags;
  int64_t n, stride, event_base;
};

struct V4 { double x, y, z, e; };
struct Conic { double a, b, c, d, e, f; };

#define SM(k) sm[(k) * RECO_THREADS + threadIdx.x]

__device__ __forceinline__ int tri(int k, int l) { return (k * (11 - k)) / 2 + (l - k - 1); }  // k < l < 6

__device__ __forceinline__ V4 load_v4(const double* px, const double* py, const double* pz, const double* e, int64_t at) {
  return V4{__ldg(px + at), __ldg(py + at), __ldg(pz + at), __ldg(e + at)};
}
__device__ __forceinline__ V4 scale_v4(const V4& p, double s) {
  return V4{__dmul_rn(s, p.x), __dmul_rn(s, p.y), __dmul_rn(s, p.z), __dmul_rn(s, p.e)};
}
__device__ __forceinline__ double mass_of(double e, double x, double y, double z) {
  const double m2 = e * e - (x * x + y * y + z * z);
  return sqrt(m2 > 0.0 ? m2 : 0.0);
}

// Leg conic of (lepton l, b-jet b): neutrino p_z = c0 + c1 p_x + c2 p_y and the conic in (p_x, p_y).
__device__ __forceinline__ bool leg_conic(const V4& l, const V4& b, double mt2, double mw2, Conic& q, double& c0,
                                          double& c1, double& c2) {
  const double ml2 = l.e * l.e - (l.x * l.x + l.y * l.y + l.z * l.z);
  const double mb2 = b.e * b.e - (b.x * b.x + b.y * b.y + b.z * b.z);
  const double bl = b.e * l.e - (b.x * l.x + b.y * l.y + b.z * l.z);
  const double A = 0.5 * (mw2 - ml2);
  const double B = 0.5 * (mt2 - mw2 - mb2) - bl;
  const double nx = b.e * l.x - l.e * b.x, ny = b.e * l.y - l.e * b.y, nz = b.e * l.z - l.e * b.z;
  const double k = l.e * B - b.e * A;
  const bool ok = fabs(nz) > 1e-12 * b.e * l.e;
  const double inz = 1.0 / nz, ile = 1.0 / l.e;
  c0 = k * inz; c1 = -nx * inz; c2 = -ny * inz;
  const double d0 = (A + l.z * c0) * ile, d1 = (l.x + l.z * c1) * ile, d2 = (l.y + l.z * c2) * ile;
  q.a = d1 * d1 - 1.0 - c1 * c1;
  q.b = 2.0 * (d1 * d2 - c1 * c2);
  q.c = d2 * d2 - 1.0 - c2 * c2;
  q.d = 2.0 * (d0 * d1 - c0 * c1);
  q.e = 2.0 * (d0 * d2 - c0 * c2);
  q.f = d0 * d0 - c0 * c0;
  return ok;
}

__device__ __forceinline__ Conic shift_conic(const Conic& q, double Mx, double My) {
  Conic s;
  s.a = q.a; s.b = q.b; s.c = q.c;
  s.d = -2.0 * q.a * Mx - q.b * My - q.d;
  s.e = -2.0 * q.c * My - q.b * Mx - q.e;
  s.f = q.a * Mx * Mx + q.b * Mx * My + q.c * My * My + q.d * Mx + q.e * My + q.f;
  return s;
}

struct Resultant { double p0, p1, p2, q0, q1, g0, g1, g2, g3; };

// resultant of the two conics in x (y eliminated) as a MONIC quartic g, plus D1 = p0+p1x+p2x^2, D2 = q0+q1x
__device__ __forceinline__ Resultant resultant(const Conic& k1, const Conic& k2) {
  Resultant R;
  R.p0 = k1.c * k2.f - k2.c * k1.f; R.p1 = k1.c * k2.d - k2.c * k1.d; R.p2 = k1.c * k2.a - k2.c * k1.a;
  R.q0 = k1.c * k2.e - k2.c * k1.e; R.q1 = k1.c * k2.b - k2.c * k1.b;
  const double r0 = k1.e * k2.f - k2.e * k1.f;
  const double r1 = k1.e * k2.d + k1.b * k2.f - k2.e * k1.d - k2.b * k1.f;
  const double r2 = k1.e * k2.a + k1.b * k2.d - k2.e * k1.a - k2.b * k1.d;
  const double r3 = k1.b * k2.a - k2.b * k1.a;
  const double h0 = R.p0 * R.p0 - R.q0 * r0;
  const double h1 = 2.0 * R.p0 * R.p1 - (R.q0 * r1 + R.q1 * r0);
  const double h2 = 2.0 * R.p0 * R.p2 + R.p1 * R.p1 - (R.q0 * r2 + R.q1 * r1);
  const double h3 = 2.0 * R.p1 * R.p2 - (R.q0 * r3 + R.q1 * r2);
  const double h4 = R.p2 * R.p2 - R.q1 * r3;
  const double ih4 = 1.0 / h4;   // h4 == 0 -> inf/NaN coefficients -> every discriminant test below is false
  R.g0 = h0 * ih4; R.g1 = h1 * ih4; R.g2 = h2 * ih4; R.g3 = h3 * ih4;
  return R;
}

// Real roots of x^4 + g3 x^3 + g2 x^2 + g1 x + g0 by Ferrari's closed form (the Newton polish happens in
// refine_xy, on the pair of conics).  Roots come out as (pair A: x[0], x[1]) then (pair B), unsorted.  Returns 0, 2 or 4.
__device__ __forceinline__ int solve_quartic(double g3, double g2, double g1, double g0, double (&x)[4]) {
  const double aq = 0.25 * g3, aq2 = aq * aq;
  const double p = g2 - 6.0 * aq2;
  const double q = g1 - 2.0 * aq * g2 + 8.0 * aq2 * aq;
  const double r = g0 - aq * g1 + aq2 * g2 - 3.0 * aq2 * aq2;
  // resolvent cubic m^3 + p m^2 + (p^2/4 - r) m - q^2/8 = 0, largest real root (>= 0)
  const double c1 = 0.25 * p * p - r, c0 = -0.125 * q * q;
  const double p3 = p * (1.0 / 3.0);
  const double P = c1 - p * p3;
  const double Q = 2.0 * p3 * p3 * p3 - p3 * c1 + c0;
  const double u = -0.5 * Q, P3 = P * (1.0 / 3.0);
  const double D = u * u + P3 * P3 * P3;
  double w;
  if (D > 0.0) {
    const double sD = sqrt(D);
    const double A = (u >= 0.0) ? cbrt(u + sD) : -cbrt(sD - u);
    w = (A != 0.0) ? A - P3 / A : 0.0;
  } else {
    const double rho = sqrt(-P3);
    double ct = u / (rho * rho * rho);
    ct = fmin(1.0, fmax(-1.0, ct));
    w = (rho > 0.0) ? 2.0 * rho * cos(acos(ct) * (1.0 / 3.0)) : 0.0;
  }
  double m = w - p3;
#pragma unroll
  for (int it = 0; it < 2; it++) {   // Newton on the resolvent: removes the closed form's cancellation error
    const double f = ((m + p) * m + c1) * m + c0, df = (3.0 * m + 2.0 * p) * m + c1;
    const double step = f / df;
    if (isfinite(step)) m -= step;
  }
  int n = 0;
  double t[4];
  if (m > 0.0) {
    const double s = sqrt(2.0 * m), qs = q / (2.0 * s);
    const double base = -2.0 * (m + p);
    const double dA = base - 4.0 * qs, dB = base + 4.0 * qs;
    if (dA >= 0.0) { const double sq = sqrt(dA); t[n++] = 0.5 * (s + sq); t[n++] = 0.5 * (s - sq); }
    if (dB >= 0.0) { const double sq = sqrt(dB); t[n++] = 0.5 * (-s + sq); t[n++] = 0.5 * (-s - sq); }
  } else if (m == m) {               // q == 0 up to rounding: biquadratic t^4 + p t^2 + r
    const double dz = p * p - 4.0 * r;
    if (dz >= 0.0) {
      const double sq = sqrt(dz), z1 = 0.5 * (-p + sq), z2 = 0.5 * (-p - sq);
      if (z1 >= 0.0) { const double st = sqrt(z1); t[n++] = st; t[n++] = -st; }
      if (z2 >= 0.0) { const double st = sqrt(z2); t[n++] = st; t[n++] = -st; }
    }
  }
  for (int k = 0; k < n; k++) x[k] = t[k] - aq;
  return n;
}

// y of a root x: y = -D1(x)/D2(x); when the conics share the y direction at x, solve conic 1 and keep the
// y closer to conic 2 (step 3).
__device__ __forceinline__ double root_y(const Resultant& R, const Conic& k1, const Conic& k2, double x) {
  const double D1 = R.p0 + x * (R.p1 + x * R.p2), D2 = R.q0 + R.q1 * x;
  if (fabs(D2) > 1e-12 * (fabs(R.q0) + fabs(R.q1 * x))) return -D1 / D2;
  const double qa = k1.c, qb = k1.b * x + k1.e, qc = (k1.a * x + k1.d) * x + k1.f;
  const double dd = qb * qb - 4.0 * qa * qc;
  if (!(dd >= 0.0) || qa == 0.0) return CUDART_NAN;
  const double sq = sqrt(dd), y1 = (-qb - sq) / (2.0 * qa), y2 = (-qb + sq) / (2.0 * qa);
  const double r1 = fabs(k2.a * x * x + k2.b * x * y1 + k2.c * y1 * y1 + k2.d * x + k2.e * y1 + k2.f);
  const double r2 = fabs(k2.a * x * x + k2.b * x * y2 + k2.c * y2 * y2 + k2.d * x + k2.e * y2 + k2.f);
  return r1 <= r2 ? y1 : y2;
}

// Newton polish of one intersection: start from the Ferrari root x and y = -D1/D2, then two Newton steps on the
// pair of conics in (x, y).  The quotient alone cancels when D2(x) is small; the 2x2 system is conditioned like
// the intersection itself (R11a).
__device__ __forceinline__ void refine_xy(const Resultant& R, const Conic& A, const Conic& B, double& x, double& y) {
  y = root_y(R, A, B, x);
#pragma unroll
  for (int it = 0; it < 2; it++) {
    const double F1 = (A.a * x + A.b * y + A.d) * x + (A.c * y + A.e) * y + A.f;
    const double F2 = (B.a * x + B.b * y + B.d) * x + (B.c * y + B.e) * y + B.f;
    const double F1x = 2.0 * A.a * x + A.b * y + A.d, F1y = A.b * x + 2.0 * A.c * y + A.e;
    const double F2x = 2.0 * B.a * x + B.b * y + B.d, F2y = B.b * x + 2.0 * B.c * y + B.e;
    const double idet = 1.0 / (F1x * F2y - F1y * F2x);
    const double dx = (F1 * F2y - F2 * F1y) * idet, dy = (F1x * F2 - F2x * F1) * idet;
    if (isfinite(dx) && isfinite(dy)) { x -= dx; y -= dy; }
  }
}

struct EventHead {   // what a thread needs to know about its event (uniform over the event's threads)
  int64_t e;         // index inside the view
  uint64_t gidx;     // global index (keys the smearing stream)
  uint32_t status;
  int n_jet, n_b, lp_slot;
  uint32_t cand;     // candidate jet slots, one nibble each
  uint32_t pos;      // for each jet slot: its candidate position (nibble), 15 = not a candidate
  bool applicable;
};

__device__ __forceinline__ EventHead load_head(const RecoCols& ev, int64_t e) {
  EventHead h;
  h.e = e; h.gidx = (uint64_t)(ev.event_base + e);
  const uint32_t f = __ldg(ev.flags + e);
  const int n_lep = f & 15u;
  h.n_jet = min(8u, (f >> 8) & 15u);
  const bool q0 = (f >> 4) & 1u, q1 = (f >> 5) & 1u;
  h.cand = 0; h.pos = 0xffffffffu; h.n_b = 0; h.status = 0;
  int n_tag = 0;
#pragma unroll
  for (int s = 0; s < HEPF_N_JET; s++) {
    if (s < h.n_jet && ((f >> (16 + s)) & 1u)) {
      if (h.n_b < NB_MAX) {
        h.cand |= (uint32_t)s << (4 * h.n_b);
        h.pos = (h.pos & ~(15u << (4 * s))) | ((uint32_t)h.n_b << (4 * s));
        h.n_b++;
      }
      n_tag++;
    }
  }
  if (n_tag > NB_MAX) h.status |= 4u;
  h.applicable = (n_lep == 2) && (q0 != q1) && (h.n_b >= 4);
  if (!h.applicable) h.status |= 2u;
  h.lp_slot = q0 ? 0 : 1;
  return h;
}

struct Smeared { V4 lp, lm; double Mx, My; };

// Normals, scales, MET' of one (event, variation); candidate scales go to the thread's shared column.
__device__ __forceinline__ Smeared smear_variation(const RecoCols& ev, const EventHead& h, int v, uint32_t k0, uint32_t k1,
                                                  const hepf_tth_params_t& P, double* sm) {
  double z[10];
#pragma unroll
  for (int blk = 0; blk < 5; blk++) {
    uint32_t x[4];
    philox4x32_10((uint32_t)h.gidx, (uint32_t)(h.gidx >> 32), (uint32_t)v, 0x54544800u + blk, k0, k1, x);
    block_normals(x, z[2 * blk], z[2 * blk + 1]);
  }
  const int64_t S = ev.stride, e = h.e;
  double dx = 0.0, dy = 0.0, sl[2];
  V4 lep[2];
#pragma unroll
  for (int t = 0; t < 2; t++) {
    lep[t] = load_v4(ev.lep_px, ev.lep_py, ev.lep_pz, ev.lep_e, t * S + e);
    const double sc = __fma_rn(__dmul_rn(P.sigma_scale, P.lep_sigma), z[t], 1.0);
    sl[t] = sc > P.s_min ? sc : P.s_min;
    const double d = __dadd_rn(sl[t], -1.0);
    dx = __dadd_rn(dx, __dmul_rn(d, lep[t].x)); dy = __dadd_rn(dy, __dmul_rn(d, lep[t].y));
  }
#pragma unroll
  for (int t = 0; t < HEPF_N_JET; t++) {
    if (t < h.n_jet) {
      const double E = __ldg(ev.jet_e + t * S + e), px = __ldg(ev.jet_px + t * S + e), py = __ldg(ev.jet_py + t * S + e);
      const double sigma = __dadd_rn(__ddiv_rn(P.jet_stoch, __dsqrt_rn(E)), P.jet_const);
      const double sc = __fma_rn(__dmul_rn(P.sigma_scale, sigma), z[2 + t], 1.0);
      const double s = sc > P.s_min ? sc : P.s_min;
      const double d = __dadd_rn(s, -1.0);
      dx = __dadd_rn(dx, __dmul_rn(d, px)); dy = __dadd_rn(dy, __dmul_rn(d, py));
      const int pos = (h.pos >> (4 * t)) & 15;
      if (pos < NB_MAX) SM(TH_SCALE + pos) = s;
    }
  }
  Smeared o;
  o.Mx = __dadd_rn(__ldg(ev.met_x + e), -dx); o.My = __dadd_rn(__ldg(ev.met_y + e), -dy);
  o.lp = scale_v4(lep[h.lp_slot], sl[h.lp_slot]);
  o.lm = scale_v4(lep[1 - h.lp_slot], sl[1 - h.lp_slot]);
  return o;
}

__device__ __forceinline__ V4 smeared_cand(const RecoCols& ev, const EventHead& h, int c, const double* sm) {
  const int slot = (h.cand >> (4 * c)) & 15;
  const V4 nom = load_v4(ev.jet_px, ev.jet_py, ev.jet_pz, ev.jet_e, slot * ev.stride + h.e);
  return scale_v4(nom, SM(TH_SCALE + c));
}

struct Cand { double ll; double x; int v, a, h; };

__device__ __forceinline__ unsigned long long ordered_key(double v) {   // monotone map double -> uint64
  const long long b = __double_as_longlong(v);
  return (b < 0) ? ~(unsigned long long)b : ((unsigned long long)b | 0x8000000000000000ull);
}

__global__ void __launch_bounds__(RECO_THREADS)
reco_kernel(RecoCols ev, const uint32_t* __restrict__ idx, int64_t n_idx, int V, uint32_t k0, uint32_t k1,
            hepf_tth_params_t P, hepf_best_t* __restrict__ out) {
  extern __shared__ double sm[];
  __shared__ unsigned long long s_key[RECO_THREADS];
  __shared__ unsigned long long s_flat[RECO_THREADS];
  const int tid = threadIdx.x;
  const int lpe = V < RECO_THREADS ? V : RECO_THREADS;   // lanes per event
  const int epb = RECO_THREADS / lpe;                    // events per block
  const int slot = tid / lpe, v_first = tid - slot * lpe;
  const int64_t k = (int64_t)blockIdx.x * epb + slot;    // position in idx
  const bool live = slot < epb && k < n_idx;
  if (tid < epb) { s_key[tid] = 0ull; s_flat[tid] = ~0ull; }
  __syncthreads();

  EventHead h{};
  Cand best{-CUDART_INF, 0.0, -1, -1, -1};
  const double mt2 = P.m_top * P.m_top, mw2 = P.m_w * P.m_w, inv_lambda = 1.0 / P.lambda_nu, inv_sh = 1.0 / P.sigma_higgs;
  if (live) {
    h = load_head(ev, (int64_t)__ldg(idx + k));
    if (h.applicable) {
      const int nb = h.n_b;
      for (int v = v_first; v < V; v += RECO_THREADS) {
        const Smeared S = smear_variation(ev, h, v, k0, k1, P, sm);
        // ---- per-variation tables: leg-2 conics (shifted by MET') and Higgs terms of all candidate pairs --------
        for (int j = 0; j < nb; j++) {
          const V4 bj = smeared_cand(ev, h, j, sm);
          Conic q; double c0, c1, c2;
          const bool ok = leg_conic(S.lm, bj, mt2, mw2, q, c0, c1, c2);
          const Conic s2 = shift_conic(q, S.Mx, S.My);
          SM(TH_CONIC2 + 6 * j + 0) = ok ? s2.a : CUDART_NAN;   // NaN conic -> no roots for this pairing
          SM(TH_CONIC2 + 6 * j + 1) = s2.b; SM(TH_CONIC2 + 6 * j + 2) = s2.c;
          SM(TH_CONIC2 + 6 * j + 3) = s2.d; SM(TH_CONIC2 + 6 * j + 4) = s2.e; SM(TH_CONIC2 + 6 * j + 5) = s2.f;
          for (int l = j + 1; l < nb; l++) {
            const V4 bl = smeared_cand(ev, h, l, sm);
            const double mbb = mass_of(bj.e + bl.e, bj.x + bl.x, bj.y + bl.y, bj.z + bl.z);
            const double t = (mbb - P.m_higgs) * inv_sh;
            SM(TH_HT + tri(j, l)) = -0.5 * (t * t);
          }
        }
        // ---- ordered pairings ---------------------------------------------------------------------------------------
        for (int i = 0; i < nb; i++) {
          const V4 bi = smeared_cand(ev, h, i, sm);
          Conic k1c; double c0, c1, c2;
          const bool ok1 = leg_conic(S.lp, bi, mt2, mw2, k1c, c0, c1, c2);
          if (!ok1) k1c.a = CUDART_NAN;
          for (int j = 0; j < nb; j++) {
            if (j == i) continue;
            const Conic k2c{SM(TH_CONIC2 + 6 * j + 0), SM(TH_CONIC2 + 6 * j + 1), SM(TH_CONIC2 + 6 * j + 2),
                            SM(TH_CONIC2 + 6 * j + 3), SM(TH_CONIC2 + 6 * j + 4), SM(TH_CONIC2 + 6 * j + 5)};
            const Resultant R = resultant(k1c, k2c);
            double x[4];
            const int nr = solve_quartic(R.g3, R.g2, R.g1, R.g0, x);
            if (nr == 0) continue;
            // best Higgs pair among the candidates not used by (i, j), lexicographic order, first maximum
            double ht = -CUDART_INF; int hbest = 0, hcount = 0;
            for (int kk = 0; kk < nb; kk++) for (int l = kk + 1; l < nb; l++) {
              if (kk == i || kk == j || l == i || l == j) continue;
              const double t = SM(TH_HT + tri(kk, l));
              if (t > ht) { ht = t; hbest = hcount; }
              hcount++;
            }
            for (int rr = 0; rr < nr; rr++) {
              double xx = x[rr], yy; refine_xy(R, k1c, k2c, xx, yy);
              const double qx = S.Mx - xx, qy = S.My - yy;
              const double ptn = sqrt(xx * xx + yy * yy), ptb = sqrt(qx * qx + qy * qy);
              const double ll = ht + (log(ptn * ptb) - (ptn + ptb) * inv_lambda);
              if (ll > best.ll) { best.ll = ll; best.x = xx; best.v = v; best.a = i * nb + j; best.h = hbest; }
            }
          }
        }
      }
    }
  }
  // ---- argmax over the threads of one event: max loglik, then lowest (variation, pairing) ----------------------
  const bool have = live && best.v >= 0;
  const unsigned long long key = have ? ordered_key(best.ll) : 0ull;
  const unsigned long long flat = have ? (((unsigned long long)best.v << 8) | (unsigned long long)best.a) : ~0ull;
  if (have) atomicMax(&s_key[slot], key);
  __syncthreads();
  if (have && key == s_key[slot]) atomicMin(&s_flat[slot], flat);
  __syncthreads();
  if (!live) return;
  hepf_best_t* o = out + k;
  if (s_key[slot] == 0ull) {                     // no thread of this event found a solution
    if (v_first == 0) {
      const double n = CUDART_NAN;
      o->nu[0] = o->nu[1] = o->nu[2] = o->nubar[0] = o->nubar[1] = o->nubar[2] = n;
      o->m_top = o->m_antitop = o->m_wplus = o->m_wminus = o->m_higgs = o->loglik = n;
      o->variation = o->jet_b = o->jet_bbar = o->jet_h1 = o->jet_h2 = o->root = -1;
      o->status = h.status; o->event = (uint32_t)h.e;
    }
    return;
  }
  if (!(have && key == s_key[slot] && flat == s_flat[slot])) return;
  // ---- the winner re-derives its solution in full and writes the record ---------------------------------------------
  {
    const int nb = h.n_b, i = best.a / nb, j = best.a - i * nb;
    const Smeared S = smear_variation(ev, h, best.v, k0, k1, P, sm);
    const V4 bi = smeared_cand(ev, h, i, sm), bj = smeared_cand(ev, h, j, sm);
    Conic k1c, q2; double c0, c1, c2, e0, e1, e2;
    leg_conic(S.lp, bi, mt2, mw2, k1c, c0, c1, c2);
    leg_conic(S.lm, bj, mt2, mw2, q2, e0, e1, e2);
    const Conic k2c = shift_conic(q2, S.Mx, S.My);
    const Resultant R = resultant(k1c, k2c);
    double x[4];
    const int nr = solve_quartic(R.g3, R.g2, R.g1, R.g0, x);
    // polish every root as the hot loop did; the winner is the recomputed root closest to the remembered one,
    // its rank is its position among the real roots in ascending order
    double ys[4];
    for (int r = 0; r < nr; r++) refine_xy(R, k1c, k2c, x[r], ys[r]);
    int rsel = 0; double dmin = CUDART_INF;
    for (int r = 0; r < nr; r++) { const double d = fabs(x[r] - best.x); if (d < dmin) { dmin = d; rsel = r; } }
    const double xx = (nr > 0) ? x[rsel] : best.x;
    const double yy = (nr > 0) ? ys[rsel] : CUDART_NAN;
    int rank = 0;
    for (int r = 0; r < nr; r++) rank += (x[r] < xx) || (x[r] == xx && r < rsel);
    const double pz = c0 + c1 * xx + c2 * yy;
    const double qx = S.Mx - xx, qy = S.My - yy, qz = e0 + e1 * qx + e2 * qy;
    const double en = sqrt(xx * xx + yy * yy + pz * pz), eb = sqrt(qx * qx + qy * qy + qz * qz);
    // Higgs pair index -> candidate positions
    int hk = -1, hl = -1, hcount = 0;
    for (int kk = 0; kk < nb; kk++) for (int l = kk + 1; l < nb; l++) {
      if (kk == i || kk == j || l == i || l == j) continue;
      if (hcount == best.h) { hk = kk; hl = l; }
      hcount++;
    }
    const V4 h1 = smeared_cand(ev, h, hk, sm), h2 = smeared_cand(ev, h, hl, sm);
    const double mbb = mass_of(h1.e + h2.e, h1.x + h2.x, h1.y + h2.y, h1.z + h2.z);
    const double ptn = sqrt(xx * xx + yy * yy), ptb = sqrt(qx * qx + qy * qy);
    const double t = (mbb - P.m_higgs) * inv_sh;
    o->nu[0] = xx; o->nu[1] = yy; o->nu[2] = pz;
    o->nubar[0] = qx; o->nubar[1] = qy; o->nubar[2] = qz;
    o->m_wplus = mass_of(S.lp.e + en, S.lp.x + xx, S.lp.y + yy, S.lp.z + pz);
    o->m_top = mass_of(S.lp.e + en + bi.e, S.lp.x + xx + bi.x, S.lp.y + yy + bi.y, S.lp.z + pz + bi.z);
    o->m_wminus = mass_of(S.lm.e + eb, S.lm.x + qx, S.lm.y + qy, S.lm.z + qz);
    o->m_antitop = mass_of(S.lm.e + eb + bj.e, S.lm.x + qx + bj.x, S.lm.y + qy + bj.y, S.lm.z + qz + bj.z);
    o->m_higgs = mbb;
    o->loglik = -0.5 * (t * t) + (log(ptn * ptb) - (ptn + ptb) * inv_lambda);
    o->variation = best.v;
    o->jet_b = (h.cand >> (4 * i)) & 15; o->jet_bbar = (h.cand >> (4 * j)) & 15;
    o->jet_h1 = (h.cand >> (4 * hk)) & 15; o->jet_h2 = (h.cand >> (4 * hl)) & 15;
    o->root = rank;
    o->status = h.status | 1u; o->event = (uint32_t)h.e;
  }
}

}  // namespace hepf

using namespace hepf;

extern "C" size_t hepf_reconstruct_workspace_bytes(int64_t n_idx, int32_t n_variations) {
  (void)n_idx; (void)n_variations;
  return 0;   // all intermediate state lives in registers and shared memory
}

extern "C" int hepf_reconstruct_tth(const hepf_events_t* events, const uint32_t* idx, int64_t n_idx, int32_t n_variations,
                                    uint64_t seed, const hepf_tth_params_t* host_params, hepf_best_t* out_best, void* ws,
                                    size_t ws_bytes, void* stream_) {
  (void)ws; (void)ws_bytes;
  cudaStream_t stream = (cudaStream_t)stream_;
  int rc = check_events(events);
  if (rc != HEPF_OK) return rc;
  if (n_idx < 0 || n_variations < 1 || n_variations > (1 << 23)) {
    set_error("hepf_reconstruct_tth: need n_idx >= 0 and 1 <= n_variations <= 2^23"); return HEPF_ERR_ARG;
  }
  if (n_idx == 0) return HEPF_OK;
  if (!idx || !aligned(idx, 4) || !out_best || !aligned(out_best, 16)) {
    set_error("hepf_reconstruct_tth: idx/out_best NULL or misaligned"); return HEPF_ERR_ARG;
  }
  hepf_tth_params_t P;
  if (host_params) P = *host_params; else hepf_default_params(&P);
  RecoCols cols{events->lep_px, events->lep_py, events->lep_pz, events->lep_e, events->jet_px, events->jet_py,
                events->jet_pz, events->jet_e, events->met_x, events->met_y, events->flags,
                events->n_events, events->stride, events->event_base};
  const int lpe = n_variations < RECO_THREADS ? n_variations : RECO_THREADS;
  const int epb = RECO_THREADS / lpe;
  const int64_t blocks = (n_idx + epb - 1) / epb;
  if (blocks > 0x7fffffffll) { set_error("hepf_reconstruct_tth: too many blocks"); return HEPF_ERR_ARG; }
  const size_t smem = (size_t)TH_DOUBLES * RECO_THREADS * sizeof(double);
  static thread_local bool attr_set = false;
  if (!attr_set) {
    HEPF_CUDA_TRY(cudaFuncSetAttribute(reco_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    attr_set = true;
  }
  reco_kernel<<<(unsigned)blocks, RECO_THREADS, smem, stream>>>(cols, idx, n_idx, n_variations, (uint32_t)seed,
                                                               (uint32_t)(seed >> 32), P, out_best);
  count_launch();
  HEPF_CUDA_TRY(cudaGetLastError());
  return HEPF_OK;
}
