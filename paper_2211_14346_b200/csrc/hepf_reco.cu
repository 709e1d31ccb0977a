// hepf_reco.cu — hepf_reconstruct_tth: smear -> leg conics -> quartic -> score -> argmax.
//
// Paper: PAPER.md:134-138 (§4) — the neutrino four-momenta are reconstructed analytically from energy-momentum
// conservation and the m_W = 80.4 / m_t = 172.5 constraints on both legs ("quadratic forms", several solutions or
// none), every b-jet/lepton pairing is tried, two of the remaining b-jets should give m_bb = 125 GeV and the most
// probable solution wins; PAPER.md:145 — the measured momenta are varied V times within the resolution.  The
// equations themselves are in DESIGN.md "Method" (the paper defers them to its ref. [27]).
//
// B200 mapping.  The work is FP64-pipe bound (no bytes to speak of), so the design goal is: every FP64
// instruction issued with 32 useful lanes, from a code body small enough to live in the instruction cache.
//   reco_search_kernel   persistent warps draw groups of list entries from a global counter; one WARP reconstructs one
//                        event at a time.  Once per event: nominal objects, conic frames (the variation-independent
//                        part of every leg conic) and pairing constants.  The V variations are processed in chunks of VC;
//                        each chunk runs a pipeline of short, convergent stages whose work items are spread over the lanes:
//       A  (variation, Philox block)      -> 2 normals (in-register Philox4x32-10 + Box-Muller) -> 2 scales
//       M  (variation, x|y)               -> MET' (slot-ordered sum, bit-identical to the definition)
//       B  (variation, leg, b candidate)  -> (d, e, f) of the leg conic from its frame (leg 2 shifted by MET') -> shared memory
//       H  (variation, candidate pair)    -> Higgs mass term
//       C  (variation, ordered pairing)   -> resultant -> monic quartic -> Ferrari (FP32 seed for the resolvent cubic,
//                                            FP64 Newton) -> 0/2/4 real roots PUSHED on a per-warp shared-memory stack
//       D  (one root per lane, popped 32 at a time) -> y, 2 Newton steps on the pair of conics, neutrino-pT score,
//                                            lane-local best with the total order (loglik, then lowest (v, a, h, root))
//     Stage D is where SIMT divergence would hurt (62 % / 34 % / 4 % of the wrong pairings have 0 / 2 / 4 roots); the
//     stack compacts the roots so that D always runs with full warps.  A warp-shuffle argmax ends the event and lane 0
//     writes an 8-byte winner key to the workspace.  No block-level barrier anywhere: warps drift apart freely, which
//     keeps the FP64 pipe fed while other warps sit in integer (Philox) or load phases.
//   reco_finalize_kernel one THREAD per selected event: re-derives the winning (variation, pairing, root) with the same
//                        device functions (this translation unit is compiled with -fmad=false and spells every fused
//                        operation, so both kernels produce the same bits) and writes the 128-byte hepf_best_t record.
// No tensor cores: nothing here is a contraction.
#include <math_constants.h>

#include "hepf_common.cuh"

// Checked build (build.py checked=True; tests/test_checked_build.py): every index into the per-warp queues and tables and into
// the workspace is tested against its bound and the kernel traps on a violation.  compute-sanitizer is not available on the
// pool this library is developed on; this is the stand-in for its memcheck on the one kernel that stages data by hand.
#ifdef HEPF_CHECKED
#define HEPF_CHECK(cond) do { if (!(cond)) __trap(); } while (0)
#else
#define HEPF_CHECK(cond) do { } while (0)
#endif

namespace hepf {

constexpr int NBM = HEPF_MAX_B;   // candidate slots in the tables
constexpr int QCAP = 160;          // root stack: <= 31 left over + 4 new roots per lane of a C2 pass (the pass is cut short if it would not fit)
constexpr int NOMINAL_ROWS = 42;   // workspace copy of an event's nominal objects: 10 x (px, py, pz, E) + MET x, y
constexpr int SCAP = 64;          // solve queue: <= 31 left over + 32 new quartics
constexpr uint32_t TAG_MASK = (1u << 20) - 1u;   // root-stack tag: vv 5 | i 3 | j 3 | h 3 | pair 4 | slot 2
constexpr uint32_t STAG_MASK = (1u << 11) - 1u;  // solve-queue tag: vv 5 | i 3 | j 3

struct RecoCols {
  const double *lep_px, *lep_py, *lep_pz, *lep_e, *jet_px, *jet_py, *jet_pz, *jet_e, *met_x, *met_y;
  const uint32_t* flags;
  int64_t n, stride, event_base;
  int64_t out_off;   // added to the `event` field of the records (hepf_tth_host reconstructs chunk views of one sample)
};

struct V4 { double x, y, z, e; };
struct Conic { double a, b, c, d, e, f; };

// nibble-packed lexicographic lists of the unordered candidate pairs (k < l) for n_b = 4, 5, 6
__device__ __forceinline__ uint64_t pair_k_list(int nb) {
  return nb == 4 ? 0x211000ull : (nb == 5 ? 0x3221110000ull : 0x433222111100000ull);
}
__device__ __forceinline__ uint64_t pair_l_list(int nb) {
  return nb == 4 ? 0x332321ull : (nb == 5 ? 0x4434324321ull : 0x554543543254321ull);
}
// position of the pair (k, l), k < l < NBT, in the lexicographic list of pairs
template <int NBT> __device__ __forceinline__ int pair_index(int k, int l) { return (k * (2 * NBT - 1 - k)) / 2 + (l - k - 1); }

// (rcp_fast / sqrt_fast: hepf_common.cuh)
// ln(a), a > 0 normal: a = m 2^e with m in (sqrt(1/2), sqrt(2)], ln m = 2 atanh(s), s = (m-1)/(m+1); error < 3e-16 relative
__device__ __forceinline__ double ln_fast(double a) {
  int hi = __double2hiint(a);
  int e = ((hi >> 20) & 0x7ff) - 1023;
  double m = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, __double2loint(a));
  if (m > 0x1.6a09e667f3bcdp+0) { m *= 0.5; e += 1; }
  const double f = m - 1.0, s = f * rcp_fast(2.0 + f), z = s * s;
  double p = kLogC[0];
#pragma unroll
  for (int k = 1; k < 9; k++) p = fma(p, z, kLogC[k]);
  const double lm = fma(s, p * z, 2.0 * s), ed = (double)e;
  const double r = fma(ed, 0x1.62e42fee00000p-1, fma(ed, 0x1.a39ef35793c76p-33, lm));
  return a > 0.0 ? r : (a == 0.0 ? -CUDART_INF : CUDART_NAN);
}

__device__ __forceinline__ V4 scale_v4(const double* p, double s) {
  return V4{__dmul_rn(s, p[0]), __dmul_rn(s, p[1]), __dmul_rn(s, p[2]), __dmul_rn(s, p[3])};
}
__device__ __forceinline__ double mass_of(double e, double x, double y, double z) {
  const double m2 = fma(e, e, -fma(x, x, fma(y, y, z * z)));
  return sqrt_fast(m2 > 0.0 ? m2 : 0.0);
}

// ---- variation-independent part of a leg conic ("frame") -------------------------------------------------------------
// Smearing multiplies the lepton by s_l and the b-jet by s_b.  Then n = E_b l - E_l b scales by s_l s_b, so c1 = -n_x/n_z,
// c2 = -n_y/n_z, d1, d2 and with them the quadratic part (a, b, c) of the conic do not depend on the variation at all;
// only c0, d0 and hence (d, e, f) do.  The frame is computed once per event from the nominal four-vectors; per variation
//   A = (m_W^2 - s_l^2 m_l^2)/2,  B = (m_t^2 - m_W^2 - s_b^2 m_b^2)/2 - s_l s_b (b.l),
//   c0 = g1 B / s_b - g2 A / s_l  (g1 = E_l / n_z, g2 = E_b / n_z),  d0 = (A / s_l) / E_l + (l_z / E_l) c0.
struct Frame { double a, b, c, c1, c2, d1, d2, g1, g2, h1, ile, hml2, hmb2, bln; };
constexpr int FRN = 14;
__device__ __forceinline__ Frame make_frame(const double* l, const double* b) {   // nominal (px, py, pz, E)
  Frame F;
  const double ml2 = fma(l[3], l[3], -fma(l[0], l[0], fma(l[1], l[1], l[2] * l[2])));
  const double mb2 = fma(b[3], b[3], -fma(b[0], b[0], fma(b[1], b[1], b[2] * b[2])));
  F.bln = fma(b[3], l[3], -fma(b[0], l[0], fma(b[1], l[1], b[2] * l[2])));
  const double nx = fma(b[3], l[0], -(l[3] * b[0])), ny = fma(b[3], l[1], -(l[3] * b[1])), nz = fma(b[3], l[2], -(l[3] * b[2]));
  const bool ok = fabs(nz) > 1e-12 * b[3] * l[3];
  const double inz = rcp_fast(nz);
  F.ile = rcp_fast(l[3]);
  F.c1 = -nx * inz; F.c2 = -ny * inz;
  F.d1 = fma(l[2], F.c1, l[0]) * F.ile; F.d2 = fma(l[2], F.c2, l[1]) * F.ile;
  F.a = ok ? fma(F.d1, F.d1, -fma(F.c1, F.c1, 1.0)) : CUDART_NAN;   // NaN conic -> no roots for any pairing using it
  F.b = 2.0 * fma(F.d1, F.d2, -(F.c1 * F.c2));
  F.c = fma(F.d2, F.d2, -fma(F.c2, F.c2, 1.0));
  F.g1 = l[3] * inz; F.g2 = b[3] * inz; F.h1 = l[2] * F.ile;
  F.hml2 = -0.5 * ml2; F.hmb2 = -0.5 * mb2;
  return F;
}
// (d, e, f) of the conic and c0 of p_z = c0 + c1 p_x + c2 p_y for scales s_l, s_b (rsl = 1/s_l, rsb = 1/s_b);
// hmw2 = m_W^2 / 2, hcm = (m_t^2 - m_W^2) / 2
__device__ __forceinline__ void conic_def(const Frame& F, double sl, double sb, double rsl, double rsb, double hmw2, double hcm,
                                          double& c0, double& d, double& e, double& f) {
  const double A = fma(F.hml2, sl * sl, hmw2);
  const double B = fma(-F.bln, sl * sb, fma(F.hmb2, sb * sb, hcm));
  const double Ar = A * rsl;
  c0 = fma(F.g1, B * rsb, -(F.g2 * Ar));
  const double d0 = fma(F.h1, c0, Ar * F.ile);
  d = 2.0 * fma(d0, F.d1, -(c0 * F.c1));
  e = 2.0 * fma(d0, F.d2, -(c0 * F.c2));
  f = fma(d0, d0, -(c0 * c0));
}

// the conic of leg 2 is in q = MET' - p; rewrite it in p
__device__ __forceinline__ Conic shift_conic(const Conic& q, double Mx, double My) {
  Conic s;
  s.a = q.a; s.b = q.b; s.c = q.c;
  const double tx = fma(q.a, Mx, fma(q.b, My, q.d)), ty = fma(q.c, My, q.e);
  s.d = -fma(q.a, Mx, tx);                 // -(2 a Mx + b My + d)
  s.e = -fma(q.b, Mx, fma(q.c, My, ty));   // -(2 c My + b Mx + e)
  s.f = fma(tx, Mx, fma(ty, My, q.f));
  return s;
}

struct Lines { double p0, p1, p2, q0, q1; };   // D1(x) = p0 + p1 x + p2 x^2, D2(x) = q0 + q1 x
__device__ __forceinline__ Lines lines_of(const Conic& k1, const Conic& k2) {
  Lines L;
  L.p0 = fma(k1.c, k2.f, -(k2.c * k1.f)); L.p1 = fma(k1.c, k2.d, -(k2.c * k1.d)); L.p2 = fma(k1.c, k2.a, -(k2.c * k1.a));
  L.q0 = fma(k1.c, k2.e, -(k2.c * k1.e)); L.q1 = fma(k1.c, k2.b, -(k2.c * k1.b));
  return L;
}

// The part of the resultant that only depends on the quadratic coefficients of the two conics, i.e. (frames) on the
// event and the pairing but not on the variation: p2, q1, r3 and 1 / h4.  Computed once per event and pairing; it also
// takes the reciprocal off the critical path of stage C.
struct PairConst { double p2, q1, r3, ih4; };
__device__ __forceinline__ PairConst pair_consts(double a1, double b1, double c1, double a2, double b2, double c2) {
  PairConst K;
  K.p2 = fma(c1, a2, -(c2 * a1)); K.q1 = fma(c1, b2, -(c2 * b1)); K.r3 = fma(b1, a2, -(b2 * a1));
  K.ih4 = rcp_fast(fma(K.p2, K.p2, -(K.q1 * K.r3)));   // h4 == 0 -> NaN coefficients -> no roots
  return K;
}
// resultant of the two conics in x (y eliminated) as a MONIC quartic x^4 + g3 x^3 + g2 x^2 + g1 x + g0
__device__ __forceinline__ void resultant(const Conic& k1, const Conic& k2, const PairConst& K, double& g3, double& g2,
                                          double& g1, double& g0) {
  const double p0 = fma(k1.c, k2.f, -(k2.c * k1.f)), p1 = fma(k1.c, k2.d, -(k2.c * k1.d));
  const double q0 = fma(k1.c, k2.e, -(k2.c * k1.e));
  const double r0 = fma(k1.e, k2.f, -(k2.e * k1.f));
  const double r1 = fma(k1.e, k2.d, fma(k1.b, k2.f, -fma(k2.e, k1.d, k2.b * k1.f)));
  const double r2 = fma(k1.e, k2.a, fma(k1.b, k2.d, -fma(k2.e, k1.a, k2.b * k1.d)));
  const double tp0 = 2.0 * p0, tp1 = 2.0 * p1;
  const double h0 = fma(p0, p0, -(q0 * r0));
  const double h1 = fma(tp0, p1, -fma(q0, r1, K.q1 * r0));
  const double h2 = fma(tp0, K.p2, fma(p1, p1, -fma(q0, r2, K.q1 * r1)));
  const double h3 = fma(tp1, K.p2, -fma(q0, K.r3, K.q1 * r2));
  g0 = h0 * K.ih4; g1 = h1 * K.ih4; g2 = h2 * K.ih4; g3 = h3 * K.ih4;
}

__device__ __forceinline__ int exp_of(double v) { return ((__double2hiint(v) >> 20) & 0x7ff) - 1023; }
__device__ __forceinline__ double pow2(int e) { return __hiloint2double((1023 + e) << 20, 0); }   // -1022 <= e <= 1023

// cos(acos(c) / 3) for c in [-1, 1], FP32, ~1e-6: acos(|c|) = sqrt(1 - |c|) * poly(|c|) (Abramowitz & Stegun 4.4.46,
// |error| <= 2e-8), reflected for c < 0; then the cosine series on [0, pi/3].  No libm call: only a seed is needed.
__device__ __forceinline__ float cos_third_acos(float c) {
  const float a = fabsf(c);
  float p = -0.0012624911f;
  p = fmaf(p, a, 0.0066700901f); p = fmaf(p, a, -0.0170881256f); p = fmaf(p, a, 0.0308918810f);
  p = fmaf(p, a, -0.0501743046f); p = fmaf(p, a, 0.0889789874f); p = fmaf(p, a, -0.2145988016f);
  p = fmaf(p, a, 1.5707963050f);
  const float om = fmaxf(1.0f - a, 1e-30f);
  float phi = om * rsqrtf(om) * p;
  phi = (c < 0.0f) ? 3.14159265f - phi : phi;
  const float t = phi * (1.0f / 3.0f), z = t * t;
  float q = -1.0f / 3628800.0f;
  q = fmaf(q, z, 1.0f / 40320.0f); q = fmaf(q, z, -1.0f / 720.0f); q = fmaf(q, z, 1.0f / 24.0f); q = fmaf(q, z, -0.5f);
  return fmaf(q, z, 1.0f);
}

// Seed for the largest real root of the resolvent cubic m^3 + p m^2 + (p^2/4 - r) m - q^2/8 = 0: the closed form
// (Cardano / trigonometric) evaluated in FP32 on the FP32 pipe, after an exact power-of-two rescaling t = 2^E tau that
// brings the depressed quartic's coefficients to O(1).  2^E is the scale of the problem, taken from the imposed top mass
// (the roots are neutrino momenta of that order); a quartic far off that scale over- or underflows FP32, the seed is
// then useless and the rescue path below takes over, at a cost in speed only.  A starting point: FP64 Newton steps follow.
__device__ __forceinline__ double resolvent_seed(double p, double q, double r, int E) {
  const float pf = (float)(p * pow2(-2 * E)), qf = (float)(q * pow2(-3 * E)), rf = (float)(r * pow2(-4 * E));
  const float c1 = fmaf(0.25f * pf, pf, -rf), c0 = -0.125f * qf * qf;
  const float p3 = pf * (1.0f / 3.0f);
  const float P3 = (c1 - pf * p3) * (1.0f / 3.0f);
  const float u = -0.5f * fmaf(2.0f * p3 * p3, p3, fmaf(-p3, c1, c0));
  const float D = fmaf(u, u, P3 * P3 * P3);
  float w;                           // MUFU-grade arithmetic is enough for a seed: rsqrt / rcp / lg2 / ex2 approximations
  if (D > 0.0f) {
    const float t = fabsf(u) + D * rsqrtf(D);
    float A = exp2f(__log2f(t) * (1.0f / 3.0f));                     // cbrt(t), then one Newton step
    A = A - __fdividef(fmaf(A * A, A, -t), 3.0f * A * A);
    A = copysignf(A, u);
    w = A - __fdividef(P3, A);
  } else {
    const float rr = rsqrtf(fmaxf(-P3, 1e-30f)), rho = -P3 * rr;    // rho = sqrt(-P3), rr = 1 / rho
    const float ct = fminf(1.0f, fmaxf(-1.0f, u * rr * rr * rr));
    w = 2.0f * rho * cos_third_acos(ct);
  }
  return (double)(w - p3) * pow2(2 * E);
}

// exponent of the FP32 seed's scale: 2^E <= m_top < 2^(E+1), clamped so that 2^(+-4E) stays a normal double
__device__ __forceinline__ int seed_scale(const hepf_tth_params_t& P) { return min(250, max(-250, exp_of(P.m_top))); }

// Largest real root of m^3 + p m^2 + c1 m + c0 (c0 <= 0, so it is >= 0) by Newton from an upper bound of all roots: the
// iterates decrease monotonically onto it.  Slow path of solve_quartic; NaN coefficients fall through and return NaN.
__device__ __noinline__ double resolvent_root_from_above(double p, double tp, double c1, double c0) {
  const int E = max(max(exp_of(p) + 1, (exp_of(c1) + 2) >> 1), (exp_of(c0) + 3) / 3) + 1;   // 2 max(|p|, |c1|^1/2, |c0|^1/3) <= 2^E
  double m = pow2(min(1000, max(-1000, E)));
#pragma unroll 1
  for (int it = 0; it < 200; it++) {
    const double f = fma(fma(m + p, m, c1), m, c0), df = fma(fma(3.0, m, tp), m, c1);
    const double step = f / df;
    if (!(step > 0.0)) break;              // at the root (f <= 0 by rounding), or NaN
    m -= step;
    if (step <= 1e-15 * m) break;
  }
  return m;
}

// The FP32-seeded iterate has not converged onto a positive root yet: a few more Newton steps from where it stands
// (the usual case: the seed lost digits to cancellation), and only then the monotone route from above.
__device__ __noinline__ double resolvent_rescue(double m, double p, double tp, double c1, double c0) {
#pragma unroll 1
  for (int it = 0; it < 5; it++) {
    const double f = fma(fma(m + p, m, c1), m, c0), df = fma(fma(3.0, m, tp), m, c1);
    const double step = f * rcp_fast(df);
    m -= step;
    if (fabs(step) <= 1e-8 * m) return m;
  }
  return resolvent_root_from_above(p, tp, c1, c0);
}

struct Biquad { double x[4]; int mask; };
__device__ __noinline__ Biquad biquadratic_roots(double p, double r, double aq) {
  Biquad b; b.mask = 0; b.x[0] = b.x[1] = b.x[2] = b.x[3] = 0.0;
  const double dz = fma(p, p, -4.0 * r);
  if (dz >= 0.0) {
    const double sq = sqrt(dz), z1 = 0.5 * (sq - p), z2 = -0.5 * (p + sq);
    if (z1 >= 0.0) { const double st = sqrt(z1); b.x[0] = st - aq; b.x[1] = -st - aq; b.mask |= 1; }
    if (z2 >= 0.0) { const double st = sqrt(z2); b.x[2] = st - aq; b.x[3] = -st - aq; b.mask |= 2; }
  }
  return b;
}

// x^4 + g3 x^3 + g2 x^2 + g1 x + g0 with x = t - aq: the depressed quartic t^4 + p t^2 + q t + r
__device__ __forceinline__ void depress(double g3, double g2, double g1, double g0, double& aq, double& p, double& q, double& r) {
  aq = 0.25 * g3;
  const double aq2 = aq * aq;
  p = fma(-6.0, aq2, g2);
  q = fma(aq, fma(8.0, aq2, -2.0 * g2), g1);
  r = fma(aq2, fma(-3.0, aq2, g2), fma(-aq, g1, g0));
}

// Does t^4 + p t^2 + q t + r CERTAINLY have no real root?  Its discriminant, written so that it costs a dozen operations,
//   Delta = 16 r (4 r - p^2)^2 + q^2 (144 p r - 4 p^3 - 27 q^2),
// is positive for 0 or 4 real roots and then (p > 0 or 4 r > p^2) means 0.  About 60 % of the solves have no root (wrong
// pairings mostly): they stop here, and only the others are queued for the closed form (stage C2), which then runs with
// full warps.  "Certainly": Delta must exceed the rounding of its own evaluation a thousandfold; everything else — small
// or negative Delta, NaN, overflow of an absurdly scaled quartic — goes on to the solver, whose answer is the one that
// counts.  The result of the search therefore does not depend on this test, only its speed does.
__device__ __forceinline__ bool certainly_no_real_root(double p, double q, double r) {
  const double p2 = p * p, q2 = q * q, w = fma(4.0, r, -p2);
  const double t1 = (16.0 * r) * (w * w);
  const double u1 = (144.0 * p) * r, u2 = (4.0 * p) * p2, u3 = 27.0 * q2;
  const double u = (u1 - u2) - u3;
  const double delta = fma(q2, u, t1);
  const double mag = fma(q2, (fabs(u1) + fabs(u2)) + u3, fabs(t1));
  return delta > 1e-12 * mag && (p > 0.0 || w > 1e-12 * p2);
}

// Near-double pair of Q(t) = t^4 + p t^2 + q t + r next to t0 (Ferrari's pair discriminant vanished within rounding): the
// critical point t* of Q there by Newton on Q', then the pair t* +- sqrt(-Q(t*) / (Q''(t*) / 2)) if Q(t*) and Q''(t*) have
// opposite signs (the FP64 evaluation of Q resolves a tangency down to a few 1e-15 of sum |terms|; the closed form only to
// about 1e-9 of its discriminant's terms).  Returns (larger, smaller), or NaNs if there is no real pair — an exact double root
// included: the method skips those (R11c).
__device__ __noinline__ double2 near_double_pair(double p, double q, double r, double t0) {
  double t = t0;
#pragma unroll 1
  for (int it = 0; it < 4; it++) {
    const double t2 = t * t, d1 = fma(fma(4.0, t2, 2.0 * p), t, q), d2 = fma(12.0, t2, 2.0 * p);
    t -= d1 / d2;
  }
  const double t2 = t * t, Q = fma(t2, t2 + p, fma(q, t, r)), h = fma(6.0, t2, p);
  const double ratio = -Q / h;
  if (!(ratio > 0.0) || !(ratio < CUDART_INF)) return make_double2(CUDART_NAN, CUDART_NAN);
  const double dl = sqrt(ratio);
  return make_double2(t + dl, t - dl);
}

// Real roots of the depressed quartic by Ferrari's closed form, shifted back to x = t - aq; the polish happens later, on
// the pair of conics.  Roots come out as pair A (xa[0], xa[1]) and pair B (xb[0], xb[1]).  Returns bit 0 = pair A real,
// bit 1 = B.
__device__ __forceinline__ int ferrari(double p, double q, double r, double aq, int seedE, double (&xa)[2], double (&xb)[2]) {
  const double c1 = fma(0.25 * p, p, -r), c0 = -0.125 * q * q, tp = 2.0 * p;
  double m = resolvent_seed(p, q, r, seedE), step = 0.0;
#pragma unroll
  for (int it = 0; it < 2; it++) {   // FP64 Newton on the resolvent cubic
    const double f = fma(fma(m + p, m, c1), m, c0), df = fma(fma(3.0, m, tp), m, c1);
    step = f * rcp_fast(df);
    m -= step;
  }
  // The seed is only FP32: accept the iterate if the last step was a converged one onto a positive root (any positive
  // root of the resolvent gives a real factorisation); otherwise take the slow, monotone route (rare).
  if (!(fabs(step) <= 1e-8 * m)) m = resolvent_rescue(m, p, tp, c1, c0);
  int mask = 0;
  if (m > 0.0) {
    double is_; const double s = sqrt_rcp_fast(2.0 * m, is_), qs = q * is_;   // 2 qs' with qs' = q / (2 s); 1 / s comes with the root
    const double base = -2.0 * (m + p);
    const double dA = fma(-2.0, qs, base), dB = fma(2.0, qs, base);
    // A discriminant that vanishes within the rounding of its own terms is a near-double pair (almost tangent conics) whose
    // existence the closed form cannot decide either way: the quartic itself can (out of line, a few solves per million)
    const double marg = 0x1p-30 * fabs(base);      // base and 2 qs cancel in the vanishing discriminant, so |base| is the size of its terms
    if (fabs(dA) < marg) { const double2 t = near_double_pair(p, q, r, 0.5 * s); if (t.x == t.x) { xa[0] = t.x - aq; xa[1] = t.y - aq; mask |= 1; } }
    else if (dA >= 0.0) { const double sq = sqrt_fast(dA); xa[0] = fma(0.5, s + sq, -aq); xa[1] = fma(0.5, s - sq, -aq); mask |= 1; }
    if (fabs(dB) < marg) { const double2 t = near_double_pair(p, q, r, -0.5 * s); if (t.x == t.x) { xb[0] = t.x - aq; xb[1] = t.y - aq; mask |= 2; } }
    else if (dB >= 0.0) { const double sq = sqrt_fast(dB); xb[0] = fma(0.5, sq - s, -aq); xb[1] = fma(-0.5, s + sq, -aq); mask |= 2; }
  } else if (m == m) {               // q == 0 up to rounding: biquadratic t^4 + p t^2 + r (rare, out of line)
    const Biquad b = biquadratic_roots(p, r, aq);
    xa[0] = b.x[0]; xa[1] = b.x[1]; xb[0] = b.x[2]; xb[1] = b.x[3]; mask = b.mask;
  }
  return mask;
}
__device__ __forceinline__ int solve_quartic(double g3, double g2, double g1, double g0, int seedE, double (&xa)[2], double (&xb)[2]) {
  double aq, p, q, r;
  depress(g3, g2, g1, g0, aq, p, q, r);
  return ferrari(p, q, r, aq, seedE, xa, xb);
}

__device__ __forceinline__ double conic_at(const Conic& k, double x, double y) {
  return fma(fma(k.a, x, fma(k.b, y, k.d)), x, fma(fma(k.c, y, k.e), y, k.f));
}

// one Newton step on the pair of conics in (x, y); mv = |dx| + |dy| (left unchanged, and the point kept, if the
// Jacobian is singular)
template <bool GUARD>
__device__ __forceinline__ void newton_xy(const Conic& A, const Conic& B, double& x, double& y, double& mv) {
  const double t1 = fma(A.a, x, fma(A.b, y, A.d)), t2 = fma(A.c, y, A.e);
  const double F1 = fma(t1, x, fma(t2, y, A.f)), F1x = fma(A.a, x, t1), F1y = fma(A.b, x, fma(A.c, y, t2));
  const double u1 = fma(B.a, x, fma(B.b, y, B.d)), u2 = fma(B.c, y, B.e);
  const double F2 = fma(u1, x, fma(u2, y, B.f)), F2x = fma(B.a, x, u1), F2y = fma(B.b, x, fma(B.c, y, u2));
  const double idet = rcp_fast(fma(F1x, F2y, -(F1y * F2x)));
  const double dx = fma(F1, F2y, -(F2 * F1y)) * idet, dy = fma(F1x, F2, -(F2x * F1)) * idet;
  const double m = fabs(dx) + fabs(dy);
  if (GUARD) {
    const bool fin = m <= CUDART_MAX_NORMAL_F;
    x = fin ? x - dx : x; y = fin ? y - dy : y; mv = fin ? m : 0.0;
  } else {                           // hot path: a singular Jacobian turns the point into NaN, which never wins the argmax
    x -= dx; y -= dy; mv = m;
  }
}
// reject: a point that has not settled after these steps (the last one still moved it by more than 1e-6) is not a solution —
// at an exactly tangent pair of conics Newton wanders instead of converging and the likelihood of where it happens to stand
// means nothing — and is returned as NaN, which never wins the argmax.  The search rejects; the finalize kernel, which only
// re-derives a winner the search has accepted, does not.
__device__ __noinline__ double2 refine_more(const Conic A, const Conic B, double x, double y, bool reject) {
  double mv = 0.0;
#pragma unroll 1
  for (int it = 0; it < 6; it++) {
    mv = 0.0;
    newton_xy<true>(A, B, x, y, mv);
    if (mv <= 1e-10 * (fabs(x) + fabs(y))) break;
  }
  if (reject && !(mv <= 1e-6 * (fabs(x) + fabs(y)))) return make_double2(CUDART_NAN, CUDART_NAN);
  return make_double2(x, y);
}

// One intersection: start from the Ferrari root x and y = -D1/D2, then two Newton steps on the pair of conics in
// (x, y).  The quotient alone cancels when D2(x) is small; the 2x2 system is conditioned like the intersection
// itself (R11a).
template <bool REJECT>
__device__ __forceinline__ void refine_xy(const Conic& A, const Conic& B, double& x, double& y) {
  const Lines L = lines_of(A, B);
  // D2(x) = 0 means the two conics share both y at this x: a double root in x, which the method skips (R11c);
  // the quotient is then non-finite, so is the refined point, and a NaN never wins the argmax
  const double D1 = fma(fma(L.p2, x, L.p1), x, L.p0), D2 = fma(L.q1, x, L.q0);
  y = -D1 * rcp_fast(D2);
  double mv = 0.0;
  newton_xy<false>(A, B, x, y, mv);
  // quadratic convergence: a first step below 1e-6 (relative) leaves an error of order 1e-12 of the step scale; the
  // second step is taken by the lanes that moved more (a per-lane decision: the result depends on the root alone)
  if (mv > 1e-6 * (fabs(x) + fabs(y))) newton_xy<false>(A, B, x, y, mv); else mv = 0.0;
  // a second step that still moved the point by more than 1e-10 (relative) means near-tangent conics (linear
  // convergence): keep polishing out of line, up to six more steps
  if (mv > 1e-10 * (fabs(x) + fabs(y))) { const double2 r = refine_more(A, B, x, y, REJECT); x = r.x; y = r.y; }
}

// log-likelihood of one refined root (Higgs term ht already chosen)
__device__ __forceinline__ double loglik_of(double x, double y, double Mx, double My, double ht, double inv_lambda) {
  const double qx = Mx - x, qy = My - y;
  const double ptn = sqrt_fast(fma(x, x, y * y)), ptb = sqrt_fast(fma(qx, qx, qy * qy));
  return ht + fma(-(ptn + ptb), inv_lambda, ln_fast(ptn * ptb));
}


// ---- winner polish in double-double (finalize kernel only) ---------------------------------------------------------------
// The search compares candidates in plain FP64, which is all a ranking needs.  The reported solution, however, should
// be the solution of the DEFINITION (the four mass constraints on the smeared FP64 four-vectors plus
// the MET' balance) to the 1e-9 that north_star asks, also where the intersection of the two conics is ill-conditioned
// (near-tangent conics, small n_z: an FP64 evaluation loses cond x 2^-53, R11).  So the one winner per event is
// polished by Newton on the RAW constraints in (p_x, p_y, p_z, q_z), residuals evaluated in double-double arithmetic
// (error-free sums and products, ~106 bits) from the exact inputs, the Jacobian in FP64: every step gains about
// -log10(cond x 2^-53) digits, and the result is rounded once at the end.  About 1 % of the search's time in total.
struct DD { double hi, lo; };
__device__ __forceinline__ DD dd_fast2sum(double a, double b) { const double s = a + b; return DD{s, b - (s - a)}; }
__device__ __forceinline__ DD dd_2sum(double a, double b) { const double s = a + b, v = s - a; return DD{s, (a - (s - v)) + (b - v)}; }
__device__ __forceinline__ DD dd_2prod(double a, double b) { const double p = a * b; return DD{p, fma(a, b, -p)}; }
// double-double sum: the high parts exactly, the low parts in plain FP64 (error <= 2^-105 (|a| + |b|): the residuals below
// are needed to about 2^-80 of their largest term)
__device__ __forceinline__ DD dd_add(DD a, DD b) {
  const DD s = dd_2sum(a.hi, b.hi);
  return dd_fast2sum(s.hi, s.lo + (a.lo + b.lo));
}
__device__ __forceinline__ DD dd_neg(DD a) { return DD{-a.hi, -a.lo}; }
__device__ __forceinline__ DD dd_sub(DD a, DD b) { return dd_add(a, dd_neg(b)); }
__device__ __forceinline__ DD dd_mul(DD a, DD b) { DD p = dd_2prod(a.hi, b.hi); p.lo += a.hi * b.lo + a.lo * b.hi; return dd_fast2sum(p.hi, p.lo); }
__device__ __forceinline__ DD dd_muld(DD a, double b) { DD p = dd_2prod(a.hi, b); p.lo += a.lo * b; return dd_fast2sum(p.hi, p.lo); }
__device__ __forceinline__ DD dd_sqrt(DD a) {
  const double s = sqrt(a.hi);
  const DD r = dd_sub(a, dd_2prod(s, s));
  return dd_fast2sum(s, r.hi / (2.0 * s));
}
// Minkowski product of two FP64 four-vectors (x, y, z, e), exact products, double-double sums
__device__ __forceinline__ DD dd_dot4(const V4& u, const V4& v) {
  return dd_sub(dd_2prod(u.e, v.e), dd_add(dd_add(dd_2prod(u.x, v.x), dd_2prod(u.y, v.y)), dd_2prod(u.z, v.z)));
}
// residuals of one leg: (l + n)^2 - m_W^2 and (l + n + b)^2 - m_t^2 for the massless n = (p, |p|).  w0 = m_l^2 - m_W^2 and
// t0 = (l + b)^2 - m_t^2 do not depend on n: they are formed once per polish.
__device__ __forceinline__ void dd_leg_consts(const V4& l, const V4& b, DD mw2, DD mt2, DD& w0, DD& t0) {
  const DD ml2 = dd_dot4(l, l), mb2 = dd_dot4(b, b), lb = dd_dot4(l, b);
  w0 = dd_sub(ml2, mw2);
  t0 = dd_sub(dd_add(dd_add(ml2, mb2), dd_add(lb, lb)), mt2);
}
__device__ __forceinline__ void dd_leg_residuals(const V4& l, const V4& b, const DD p[3], DD E, DD w0, DD t0, double& fw, double& ft) {
  const DD lp = dd_sub(dd_muld(E, l.e), dd_add(dd_add(dd_muld(p[0], l.x), dd_muld(p[1], l.y)), dd_muld(p[2], l.z)));
  const DD bp = dd_sub(dd_muld(E, b.e), dd_add(dd_add(dd_muld(p[0], b.x), dd_muld(p[1], b.y)), dd_muld(p[2], b.z)));
  const DD w = dd_add(w0, dd_add(lp, lp));                                    // m_l^2 + 2 l.n - m_W^2
  const DD t = dd_add(t0, dd_add(dd_add(lp, lp), dd_add(bp, bp)));            // (l + b)^2 + 2 (l + b).n - m_t^2
  fw = w.hi + w.lo; ft = t.hi + t.lo;
}
// Returns false (and leaves the point alone) if the iteration does not settle next to where it started.
__device__ __noinline__ bool polish_raw(const V4 lp, const V4 bi, const V4 lm, const V4 bj, double Mx, double My, double m_top,
                                        double m_w, double& x, double& y, double& pz, double& qx, double& qy, double& qz) {
  const DD mw2 = dd_2prod(m_w, m_w), mt2 = dd_2prod(m_top, m_top);
  DD w01, t01, w02, t02;
  dd_leg_consts(lp, bi, mw2, mt2, w01, t01); dd_leg_consts(lm, bj, mw2, mt2, w02, t02);
  DD u[4] = {DD{x, 0.0}, DD{y, 0.0}, DD{pz, 0.0}, DD{qz, 0.0}};
  const double scale = fabs(x) + fabs(y) + fabs(pz) + fabs(qz);
  double mv = CUDART_INF, total = 0.0;
  // A step of size mv leaves an error of about C mv^2 + (rounding of the FP64 Jacobian, 1e-15) mv: once a step is below
  // 1e-10 of the scale the point is converged far beyond the 1e-9 the record is compared at, and no further residual
  // evaluation is spent on confirming it.  The usual case is ONE step (the search's FP64 point is 1e-12 .. 1e-15 away).
#pragma unroll 1
  for (int it = 0; it < 6 && mv > 1e-10 * scale; it++) {
    const DD q[3] = {dd_sub(DD{Mx, 0.0}, u[0]), dd_sub(DD{My, 0.0}, u[1]), u[3]};
    const DD p[3] = {u[0], u[1], u[2]};
    const DD E = dd_sqrt(dd_add(dd_add(dd_mul(p[0], p[0]), dd_mul(p[1], p[1])), dd_mul(p[2], p[2])));
    const DD Eq = dd_sqrt(dd_add(dd_add(dd_mul(q[0], q[0]), dd_mul(q[1], q[1])), dd_mul(q[2], q[2])));
    double A[4][5];
    dd_leg_residuals(lp, bi, p, E, w01, t01, A[0][4], A[1][4]);
    dd_leg_residuals(lm, bj, q, Eq, w02, t02, A[2][4], A[3][4]);
    const double ie = rcp_fast(E.hi), iq = rcp_fast(Eq.hi);
    const double ux = p[0].hi * ie, uy = p[1].hi * ie, uz = p[2].hi * ie, vx = q[0].hi * iq, vy = q[1].hi * iq, vz = q[2].hi * iq;
    const double s1 = lp.e, s2 = lp.e + bi.e, t1 = lm.e, t2 = lm.e + bj.e;
    A[0][0] = 2.0 * (s1 * ux - lp.x); A[0][1] = 2.0 * (s1 * uy - lp.y); A[0][2] = 2.0 * (s1 * uz - lp.z); A[0][3] = 0.0;
    A[1][0] = 2.0 * (s2 * ux - (lp.x + bi.x)); A[1][1] = 2.0 * (s2 * uy - (lp.y + bi.y)); A[1][2] = 2.0 * (s2 * uz - (lp.z + bi.z)); A[1][3] = 0.0;
    A[2][0] = -2.0 * (t1 * vx - lm.x); A[2][1] = -2.0 * (t1 * vy - lm.y); A[2][2] = 0.0; A[2][3] = 2.0 * (t1 * vz - lm.z);
    A[3][0] = -2.0 * (t2 * vx - (lm.x + bj.x)); A[3][1] = -2.0 * (t2 * vy - (lm.y + bj.y)); A[3][2] = 0.0; A[3][3] = 2.0 * (t2 * vz - (lm.z + bj.z));
    // Gaussian elimination with partial pivoting; the step only has to be good to a few digits.  Every index is a compile-time
    // constant (the pivot row is brought up by conditional swaps of whole rows), so the matrix stays in registers.
    double ipv[4];
#pragma unroll
    for (int c = 0; c < 4; c++) {
#pragma unroll
      for (int r = c + 1; r < 4; r++) {
        const bool sw = fabs(A[r][c]) > fabs(A[c][c]);
#pragma unroll
        for (int k = c; k < 5; k++) { const double t = A[c][k]; A[c][k] = sw ? A[r][k] : t; A[r][k] = sw ? t : A[r][k]; }
      }
      ipv[c] = rcp_fast(A[c][c]);
#pragma unroll
      for (int r = c + 1; r < 4; r++) {
        const double m = A[r][c] * ipv[c];
#pragma unroll
        for (int k = c + 1; k < 5; k++) A[r][k] -= m * A[c][k];
      }
    }
    double d[4];
#pragma unroll
    for (int c = 3; c >= 0; c--) {
      double sacc = A[c][4];
#pragma unroll
      for (int k = c + 1; k < 4; k++) sacc -= A[c][k] * d[k];
      d[c] = sacc * ipv[c];
    }
    mv = fabs(d[0]) + fabs(d[1]) + fabs(d[2]) + fabs(d[3]);
    total += mv;
    if (!(total <= 1e-3 * scale)) return false;     // NaN, or wandering off to another intersection
#pragma unroll
    for (int c = 0; c < 4; c++) u[c] = dd_sub(u[c], DD{d[c], 0.0});
  }
  if (!(mv <= 1e-10 * scale)) return false;
  const DD fqx = dd_sub(DD{Mx, 0.0}, u[0]), fqy = dd_sub(DD{My, 0.0}, u[1]);
  x = u[0].hi; y = u[1].hi; pz = u[2].hi; qz = u[3].hi; qx = fqx.hi; qy = fqy.hi;
  return true;
}

struct EventHead {   // what a warp / thread needs to know about its event
  int64_t e;         // index inside the view
  uint64_t gidx;     // global index (keys the smearing stream)
  uint32_t status;
  int n_jet, n_b, lp_slot, nblk;
  uint32_t cand;     // candidate jet slots, one nibble each
  bool applicable;
};

__device__ __forceinline__ EventHead load_head(const RecoCols& ev, int64_t e) {
  EventHead h;
  h.e = e; h.gidx = (uint64_t)(ev.event_base + e);
  const bool in_range = (uint64_t)e < (uint64_t)ev.n;       // idx[k] >= n_events: flags 0 -> not applicable, status 2 | 8
  const uint32_t f = in_range ? __ldg(ev.flags + e) : 0u;
  const int n_lep = f & 15u;
  h.n_jet = min(8u, (f >> 8) & 15u);
  const bool q0 = (f >> 4) & 1u, q1 = (f >> 5) & 1u;
  h.cand = 0; h.n_b = 0; h.status = 0;
  uint32_t tags = (f >> 16) & ((1u << h.n_jet) - 1u);
  const int n_tag = __popc(tags);
  for (int c = 0; c < NBM && tags; c++) {
    const int s = __ffs(tags) - 1; tags &= tags - 1;
    h.cand |= (uint32_t)s << (4 * c); h.n_b++;
  }
  if (n_tag > NBM) h.status |= 4u;
  if (!in_range) h.status |= 8u;
  h.applicable = (n_lep == 2) && (q0 != q1) && (h.n_b >= 4);
  if (!h.applicable) h.status |= 2u;
  h.lp_slot = q0 ? 0 : 1;
  h.nblk = (2 + h.n_jet + 1) >> 1;   // Philox blocks whose normals are used (objects 0 .. 1 + n_jet)
  return h;
}

// nominal object t (0,1 leptons; 2+j jet slot j) and its kappa*sigma (step 2)
__device__ __forceinline__ void load_object(const RecoCols& ev, int64_t e, int t, const hepf_tth_params_t& P, double* obj4,
                                            double& ks) {
  const int64_t at = (t < 2 ? t : t - 2) * ev.stride + e;
  const double *px = t < 2 ? ev.lep_px : ev.jet_px, *py = t < 2 ? ev.lep_py : ev.jet_py;
  const double *pz = t < 2 ? ev.lep_pz : ev.jet_pz, *pe = t < 2 ? ev.lep_e : ev.jet_e;
  obj4[0] = __ldg(px + at); obj4[1] = __ldg(py + at); obj4[2] = __ldg(pz + at); obj4[3] = __ldg(pe + at);
  const double sigma = t < 2 ? P.lep_sigma : __dadd_rn(__ddiv_rn(P.jet_stoch, __dsqrt_rn(obj4[3])), P.jet_const);
  ks = __dmul_rn(P.sigma_scale, sigma);
}
__device__ __forceinline__ double scale_of(double ks, double z, double s_min) {
  const double sc = __fma_rn(ks, z, 1.0);
  return sc > s_min ? sc : s_min;
}

// winner key: (variation, pairing i*6+j, Higgs pair, Ferrari slot) in enumeration order; smaller = earlier
__device__ __forceinline__ uint32_t make_key(int v, int i, int j, int h, int k) {
  return ((uint32_t)v << 11) | ((uint32_t)(i * 6 + j) << 5) | ((uint32_t)h << 2) | (uint32_t)k;
}

// best Higgs pair for the pairing (i, j): candidates not in {i, j}, lexicographic order, first maximum of the term
template <int NBT, int VC>
__device__ __forceinline__ void best_higgs(const double* ht15, int nb, int i, int j, double& ht, int& h, int& kk, int& ll) {
  uint32_t rem = ((1u << nb) - 1u) & ~(1u << i) & ~(1u << j);
  if (NBT == 4) {                    // exactly one pair is left
    kk = __ffs(rem) - 1; ll = 31 - __clz(rem); h = 0;
    ht = ht15[pair_index<NBT>(kk, ll) * VC];
    return;
  }
  int r[4], nr = 0;
#pragma unroll
  for (int c = 0; c < 4; c++) { r[c] = __ffs(rem) - 1; nr += rem != 0; rem &= rem - 1; }
  ht = -CUDART_INF; h = 0; kk = r[0]; ll = r[1];
  int hc = 0;
#pragma unroll
  for (int a = 0; a < 3; a++)
#pragma unroll
    for (int b = a + 1; b < 4; b++) {
      if (b < nr) {
        const double t = ht15[pair_index<NBT>(r[a], r[b]) * VC];
        if (t > ht) { ht = t; h = hc; kk = r[a]; ll = r[b]; }
        hc++;
      }
    }
}

template <int VC, int NBT>
struct __align__(16) WarpMem {
  static constexpr int NP = NBT * (NBT - 1) / 2;
  double def[3][2 * NBT * VC];   // (d, e, f) of the conic of (leg, candidate, variation); lanes of a pass differ in the variation
  double cc[2 * NBT];            // per event: c of the frame of (leg, candidate)
  double2 pcv[NBT * (NBT - 1)][2];  // per event: pair constants (p2, q1), (r3, 1/h4) of every ordered pairing (128-bit loads)
  double2 ab[2 * NBT];              // per event: (a, b) of the frame of (leg, candidate), read with one 128-bit load
  double ht[VC * NP];            // Higgs term of candidate pair (k, l), k < l
  double hm2[NBT];               // per event: nominal m^2 of candidate c
  double hdot[NP];               // per event: 2 (b_k . b_l) of the nominal candidates k < l (Minkowski product)
  uint32_t hp[NP + (NP & 1)];    // per event: the p-th pair as k | l << 4 | object of k << 8 | object of l << 12 | table row << 16
  double M[VC * 2];              // MET'
  double obj[10 * 4];            // nominal (px, py, pz, E)
  double ks[10];                 // kappa * sigma
  double met[2];
  // Both queues are empty while a chunk's tables are built, and what only the table-building stages (A, M, B, H) read is
  // dead once they are: the scales of the ten objects and the part of the frames that only stage B uses (c1, c2, d1, d2,
  // g1, g2, h1, ile, hml2, hmb2, bln; rebuilt at the top of every chunk from the nominal objects — 8 or 12 lanes' work)
  // live in the queues' bytes.  This is what lets a chunk of 32 variations fit 18 warps on an SM.
  union {
    struct {
      // solve queue (stage C1 -> C2): depressed quartics that may have real roots, (p, q), (r, aq).  The (variation, i, j)
      // tag of the entry rides in the low 11 bits of aq: aq only shifts the roots (x = t - aq), so this moves the Ferrari
      // roots by |aq| 2^-41 before they are refined on the conics (the finalize kernel solves the winner's quartic from
      // unpacked values).  It saves a third array and a load/store per solve.
      double2 s_pq[SCAP], s_ra[SCAP];
      // root stack (stage C2 -> D): the Ferrari root x with the 20-bit tag of its cell in the low mantissa bits, one 8-byte
      // entry per root (x is a starting point: 32 mantissa bits, 2e-10 relative, is finer than the closed form's own
      // error, and stage D refines it by Newton on the conics).
      unsigned long long q[QCAP];
    };
    struct { double sc_[VC * 10]; double frb[FRN - 3][2 * NBT]; };
  };
  __device__ __forceinline__ double* sc() { return sc_; }
  __device__ __forceinline__ void push(int at, double x, uint32_t tag) {
    HEPF_CHECK(at >= 0 && at < QCAP && tag <= TAG_MASK);
    q[at] = ((unsigned long long)__double_as_longlong(x) & ~(unsigned long long)TAG_MASK) | tag;
  }
  __device__ __forceinline__ void pop(int at, double& x, uint32_t& tag) const {
    HEPF_CHECK(at >= 0 && at < QCAP);
    const unsigned long long en = q[at];
    x = __longlong_as_double((long long)(en & ~(unsigned long long)TAG_MASK)); tag = (uint32_t)en & TAG_MASK;   // tag bits cleared: x does not depend on its cell
  }
};

template <int VC, int NBT>
__device__ __forceinline__ void score_entry(const WarpMem<VC, NBT>& W, double x, uint32_t tag, int v0, double inv_lambda,
                                            double& best_ll, uint32_t& best_key) {
  const int vv = tag & 31, i = (tag >> 5) & 7, j = (tag >> 8) & 7, h = (tag >> 11) & 7, t = (tag >> 14) & 15, k = (tag >> 18) & 3;
  const int a1 = i * VC + vv, a2 = (NBT + j) * VC + vv;
  HEPF_CHECK(vv < VC && i < NBT && j < NBT && i != j && t < (WarpMem<VC, NBT>::NP));
  const double2 abA = W.ab[i], abB = W.ab[NBT + j];
  const Conic A{abA.x, abA.y, W.cc[i], W.def[0][a1], W.def[1][a1], W.def[2][a1]};
  const Conic B{abB.x, abB.y, W.cc[NBT + j], W.def[0][a2], W.def[1][a2], W.def[2][a2]};
  double y;
  refine_xy<true>(A, B, x, y);
  const double ll = loglik_of(x, y, W.M[vv], W.M[VC + vv], W.ht[t * VC + vv], inv_lambda);
  if (ll >= best_ll) {               // the key is only needed by a candidate that can replace the incumbent (rare per lane)
    const uint32_t key = make_key(v0 + vv, i, j, h, k);
    if (ll > best_ll || key < best_key) { best_ll = ll; best_key = key; }
  }
}

// One event, all variations, by one warp (see the header of this file).  Returns the winner key in every lane.
template <int VC, int NBT>
__device__ __forceinline__ uint32_t search_event(WarpMem<VC, NBT>& W, const RecoCols& ev, const EventHead& h, int V, uint32_t k0,
                                                 uint32_t k1, const hepf_tth_params_t& P, int lane) {
  constexpr int LPB = 32 / VC;     // item sub-groups per warp pass
  constexpr bool FUSE_M = (LPB == 1);   // a lane owns a variation: MET' is accumulated in stage A
  const int vv = lane & (VC - 1), sub = lane / VC;
  // ---- prologue: nominal objects, kappa*sigma, MET ------------------------------------------------------------------
  if (lane < 10) {
    if (lane < 2 + h.n_jet) load_object(ev, h.e, lane, P, &W.obj[lane * 4], W.ks[lane]);
    else { W.obj[lane * 4] = W.obj[lane * 4 + 1] = W.obj[lane * 4 + 2] = W.obj[lane * 4 + 3] = 0.0; W.ks[lane] = 0.0; }
  } else if (lane < 12) {
    W.met[lane - 10] = __ldg((lane == 10 ? ev.met_x : ev.met_y) + h.e);
  }
  __syncwarp();
  // the n_b = 4 instantiation only ever sees events with four candidates: a compile-time constant there
  const int nb = (NBT == 4) ? 4 : h.n_b, n_pair = nb * (nb - 1) / 2, n_ord = nb * (nb - 1);
  const uint64_t PK = pair_k_list(nb), PL = pair_l_list(nb);
  // ap / (nb - 1) for ap < nb (nb - 1) as a multiply-shift: /3 -> *11 >> 5 (ap < 12), /4 -> >> 2, /5 -> *13 >> 6 (ap < 30)
  const int dmul = nb == 4 ? 11 : (nb == 5 ? 1 : 13), dsh = nb == 4 ? 5 : (nb == 5 ? 2 : 6);
  // Higgs-pair constants: (s_k b_k + s_l b_l)^2 = s_k^2 m_k^2 + s_l^2 m_l^2 + s_k s_l 2 (b_k . b_l), so a variation costs
  // three products and three fused operations per pair instead of two scaled four-vectors, their sum and its square
  if (lane < n_pair) {
    const int kk = (int)(PK >> (4 * lane)) & 15, ll = (int)(PL >> (4 * lane)) & 15;
    const double* bk = &W.obj[(2 + ((h.cand >> (4 * kk)) & 15)) * 4];
    const double* bl = &W.obj[(2 + ((h.cand >> (4 * ll)) & 15)) * 4];
    W.hdot[pair_index<NBT>(kk, ll)] = 2.0 * fma(bk[3], bl[3], -fma(bk[0], bl[0], fma(bk[1], bl[1], bk[2] * bl[2])));
    W.hp[lane] = (uint32_t)kk | ((uint32_t)ll << 4) | ((2u + ((h.cand >> (4 * kk)) & 15u)) << 8) | ((2u + ((h.cand >> (4 * ll)) & 15u)) << 12) |
                 ((uint32_t)pair_index<NBT>(kk, ll) << 16);
  } else if (lane >= 16 && lane < 16 + nb) {
    const double* b = &W.obj[(2 + ((h.cand >> (4 * (lane - 16))) & 15)) * 4];
    W.hm2[lane - 16] = fma(b[3], b[3], -fma(b[0], b[0], fma(b[1], b[1], b[2] * b[2])));
  }
  const double mt2 = P.m_top * P.m_top, mw2 = P.m_w * P.m_w, hmw2 = 0.5 * mw2, hcm = 0.5 * (mt2 - mw2), inv_lambda = rcp_fast(P.lambda_nu), inv_sh = rcp_fast(P.sigma_higgs);
  const unsigned lt = (1u << lane) - 1u;
  const int seedE = seed_scale(P);
  // a candidate must beat the most negative finite double: a loglik of -inf (p_T = 0) or NaN is not a solution, exactly
  // as the definition's strict '>' against an initial -inf
  double best_ll = -1.7976931348623157e308;
  uint32_t best_key = 0xffffffffu;
  int qn = 0, sn = 0;                              // heights of the root stack and of the solve queue (warp-uniform)

#pragma unroll 1
  for (int v0 = 0; v0 < V; v0 += VC) {
    const int nv = min(VC, V - v0);
    const bool vok = vv < nv;
    // ---- F: frames of (leg, candidate).  (a, b, c) are kept for the whole event, the rest only until stage B has run.
    if (lane < 2 * nb) {
      const int leg = lane >= nb, c = lane - leg * nb;
      const int ls = leg ? 1 - h.lp_slot : h.lp_slot, js = 2 + ((h.cand >> (4 * c)) & 15);
      const Frame F = make_frame(&W.obj[ls * 4], &W.obj[js * 4]);
      const int fi = leg * NBT + c;
      W.ab[fi] = make_double2(F.a, F.b); W.cc[fi] = F.c;
      W.frb[0][fi] = F.c1; W.frb[1][fi] = F.c2; W.frb[2][fi] = F.d1; W.frb[3][fi] = F.d2; W.frb[4][fi] = F.g1; W.frb[5][fi] = F.g2;
      W.frb[6][fi] = F.h1; W.frb[7][fi] = F.ile; W.frb[8][fi] = F.hml2; W.frb[9][fi] = F.hmb2; W.frb[10][fi] = F.bln;
    }
    // ---- A: normals -> scales.  With 32 variations per chunk a lane owns a variation and walks its blocks, i.e. its objects,
    //      in slot order: MET' = MET - sum_t (s_t - 1) pT_t is then accumulated on the way (the objects past 2 + n_jet have a
    //      zero four-vector and s = 1: they add +0, which leaves the sum's bits alone) and stage M is not needed.
    double ax = 0.0, ay = 0.0;
    for (int b0 = 0; b0 < h.nblk; b0 += LPB) {
      const int blk = b0 + sub;
      if (vok && blk < h.nblk) {
        uint32_t x[4];
        philox4x32_10((uint32_t)h.gidx, (uint32_t)(h.gidx >> 32), (uint32_t)(v0 + vv), 0x54544800u + blk, k0, k1, x);
        double ze, zo; block_normals(x, ze, zo);
        const double s0 = scale_of(W.ks[2 * blk], ze, P.s_min), s1 = scale_of(W.ks[2 * blk + 1], zo, P.s_min);
        W.sc()[(2 * blk) * VC + vv] = s0; W.sc()[(2 * blk + 1) * VC + vv] = s1;
        if (FUSE_M) {
          const double d0 = __dadd_rn(s0, -1.0), d1 = __dadd_rn(s1, -1.0);
          ax = __dadd_rn(ax, __dmul_rn(d0, W.obj[8 * blk])); ay = __dadd_rn(ay, __dmul_rn(d0, W.obj[8 * blk + 1]));
          ax = __dadd_rn(ax, __dmul_rn(d1, W.obj[8 * blk + 4])); ay = __dadd_rn(ay, __dmul_rn(d1, W.obj[8 * blk + 5]));
        }
      }
    }
    const double Mx_own = __dadd_rn(W.met[0], -ax), My_own = __dadd_rn(W.met[1], -ay);   // (only meaningful with FUSE_M)
    if (FUSE_M && vok) { W.M[vv] = Mx_own; W.M[VC + vv] = My_own; }
    __syncwarp();
    if (v0 == 0 && lane < n_ord) {     // pair constants of every ordered pairing: once per event
      const int i = (lane * dmul) >> dsh; int j = lane - i * (nb - 1); j += (j >= i);
      const PairConst K = pair_consts(W.ab[i].x, W.ab[i].y, W.cc[i], W.ab[NBT + j].x, W.ab[NBT + j].y, W.cc[NBT + j]);
      W.pcv[lane][0] = make_double2(K.p2, K.q1); W.pcv[lane][1] = make_double2(K.r3, K.ih4);
    }
    // ---- M: MET' = MET - sum_t (s_t - 1) pT_t, summed in slot order ----------------------------------------------------
#pragma unroll 1
    for (int c0 = 0; c0 < (FUSE_M ? 0 : 2); c0 += LPB) {
      const int comp = c0 + sub;
      if (vok && comp < 2) {
        double acc = 0.0;
        for (int t = 0; t < 2 + h.n_jet; t++)
          acc = __dadd_rn(acc, __dmul_rn(__dadd_rn(W.sc()[t * VC + vv], -1.0), W.obj[t * 4 + comp]));
        W.M[comp * VC + vv] = __dadd_rn(W.met[comp], -acc);
      }
    }
    if (!FUSE_M) __syncwarp();
    // ---- B: leg conics (leg 0: l+ with candidate c; leg 1: l- with candidate c, shifted by MET').  With 32-variation chunks a
    //      lane owns a variation: its scales and their reciprocals are loaded once (6 reciprocals instead of 16), the eight
    //      conics are unrolled with compile-time table offsets, and MET' is the lane's own from stage A.
    double sv[4] = {1.0, 1.0, 1.0, 1.0};        // the lane's scales of the four candidates (32-variation chunks: a lane owns a variation)
    if (NBT == 4 && LPB == 1) {
      if (vok) {
        double rv[4];
#pragma unroll
        for (int c = 0; c < 4; c++) { sv[c] = W.sc()[(2 + ((h.cand >> (4 * c)) & 15)) * VC + vv]; rv[c] = rcp_fast(sv[c]); }
#pragma unroll
        for (int leg = 0; leg < 2; leg++) {
          const int ls = leg ? 1 - h.lp_slot : h.lp_slot;
          const double sl = W.sc()[ls * VC + vv], rl = rcp_fast(sl);
#pragma unroll
          for (int c = 0; c < 4; c++) {
            const int fi = leg * NBT + c;
            Frame F;
            F.a = W.ab[fi].x; F.b = W.ab[fi].y; F.c = W.cc[fi]; F.c1 = W.frb[0][fi]; F.c2 = W.frb[1][fi];
            F.d1 = W.frb[2][fi]; F.d2 = W.frb[3][fi]; F.g1 = W.frb[4][fi]; F.g2 = W.frb[5][fi]; F.h1 = W.frb[6][fi];
            F.ile = W.frb[7][fi]; F.hml2 = W.frb[8][fi]; F.hmb2 = W.frb[9][fi]; F.bln = W.frb[10][fi];
            Conic q; double c0_;
            q.a = F.a; q.b = F.b; q.c = F.c;
            conic_def(F, sl, sv[c], rl, rv[c], hmw2, hcm, c0_, q.d, q.e, q.f);
            if (leg) q = shift_conic(q, Mx_own, My_own);
            const int at = fi * VC + vv;
            W.def[0][at] = q.d; W.def[1][at] = q.e; W.def[2][at] = q.f;
          }
        }
      }
    } else
    if (NBT == 4 && LPB == 2) {         // 16-variation chunks: a lane owns a (variation, leg): one lepton scale and reciprocal, the four
                                        // candidates unrolled (for n_b = 6 the rolled loop below is the faster one: measured)
      if (vok) {
        const int leg = sub;
        const int ls = leg ? 1 - h.lp_slot : h.lp_slot;
        const double sl = W.sc()[ls * VC + vv], rl = rcp_fast(sl);
        const double Mx = W.M[vv], My = W.M[VC + vv];
#pragma unroll
        for (int c = 0; c < NBT; c++) {
          if (c < nb) {
            const int fi = leg * NBT + c;
            const double sb = W.sc()[(2 + ((h.cand >> (4 * c)) & 15)) * VC + vv];
            Frame F;
            F.a = W.ab[fi].x; F.b = W.ab[fi].y; F.c = W.cc[fi]; F.c1 = W.frb[0][fi]; F.c2 = W.frb[1][fi];
            F.d1 = W.frb[2][fi]; F.d2 = W.frb[3][fi]; F.g1 = W.frb[4][fi]; F.g2 = W.frb[5][fi]; F.h1 = W.frb[6][fi];
            F.ile = W.frb[7][fi]; F.hml2 = W.frb[8][fi]; F.hmb2 = W.frb[9][fi]; F.bln = W.frb[10][fi];
            Conic q; double c0_;
            q.a = F.a; q.b = F.b; q.c = F.c;
            conic_def(F, sl, sb, rl, rcp_fast(sb), hmw2, hcm, c0_, q.d, q.e, q.f);
            if (leg) q = shift_conic(q, Mx, My);
            const int at = fi * VC + vv;
            W.def[0][at] = q.d; W.def[1][at] = q.e; W.def[2][at] = q.f;
          }
        }
      }
    } else
    if (NBT == 6 && LPB == 2) {         // a lane owns a (variation, leg): lepton scale and reciprocal hoisted, candidates in a rolled loop
      if (vok) {
        const int leg = sub;
        const int ls = leg ? 1 - h.lp_slot : h.lp_slot;
        const double sl = W.sc()[ls * VC + vv], rl = rcp_fast(sl);
        const double Mx = W.M[vv], My = W.M[VC + vv];
#pragma unroll 1
        for (int c = 0; c < nb; c++) {
          const int fi = leg * NBT + c;
          const double sb = W.sc()[(2 + ((h.cand >> (4 * c)) & 15)) * VC + vv];
          Frame F;
          F.a = W.ab[fi].x; F.b = W.ab[fi].y; F.c = W.cc[fi]; F.c1 = W.frb[0][fi]; F.c2 = W.frb[1][fi];
          F.d1 = W.frb[2][fi]; F.d2 = W.frb[3][fi]; F.g1 = W.frb[4][fi]; F.g2 = W.frb[5][fi]; F.h1 = W.frb[6][fi];
          F.ile = W.frb[7][fi]; F.hml2 = W.frb[8][fi]; F.hmb2 = W.frb[9][fi]; F.bln = W.frb[10][fi];
          Conic q; double c0_;
          q.a = F.a; q.b = F.b; q.c = F.c;
          conic_def(F, sl, sb, rl, rcp_fast(sb), hmw2, hcm, c0_, q.d, q.e, q.f);
          if (leg) q = shift_conic(q, Mx, My);
          const int at = fi * VC + vv;
          W.def[0][at] = q.d; W.def[1][at] = q.e; W.def[2][at] = q.f;
        }
      }
    } else
#pragma unroll 1
    for (int c0 = 0; c0 < 2 * nb; c0 += LPB) {
      const int comb = c0 + sub;
      if (vok && comb < 2 * nb) {
        const int leg = comb >= nb, c = comb - leg * nb;
        const int ls = leg ? 1 - h.lp_slot : h.lp_slot, js = 2 + ((h.cand >> (4 * c)) & 15);
        const int fi = leg * NBT + c;
        Frame F;
        F.a = W.ab[fi].x; F.b = W.ab[fi].y; F.c = W.cc[fi]; F.c1 = W.frb[0][fi]; F.c2 = W.frb[1][fi];
        F.d1 = W.frb[2][fi]; F.d2 = W.frb[3][fi]; F.g1 = W.frb[4][fi]; F.g2 = W.frb[5][fi]; F.h1 = W.frb[6][fi];
        F.ile = W.frb[7][fi]; F.hml2 = W.frb[8][fi]; F.hmb2 = W.frb[9][fi]; F.bln = W.frb[10][fi];
        Conic q; double c0_;
        q.a = F.a; q.b = F.b; q.c = F.c;
        const double sl = W.sc()[ls * VC + vv], sb = W.sc()[js * VC + vv];
        conic_def(F, sl, sb, rcp_fast(sl), rcp_fast(sb), hmw2, hcm, c0_, q.d, q.e, q.f);
        if (leg) q = shift_conic(q, W.M[vv], W.M[VC + vv]);
        const int at = (leg * NBT + c) * VC + vv;
        W.def[0][at] = q.d; W.def[1][at] = q.e; W.def[2][at] = q.f;
      }
    }
    // ---- H: Higgs term of every unordered candidate pair ---------------------------------------------------------------
    if (NBT == 4 && LPB == 1) {         // a lane owns a variation: the six pairs unrolled, on the scales stage B loaded
      if (vok) {
        double sq[4];
#pragma unroll
        for (int c = 0; c < 4; c++) sq[c] = sv[c] * sv[c];
        int pi = 0;
#pragma unroll
        for (int kk = 0; kk < 4; kk++)
#pragma unroll
          for (int ll = kk + 1; ll < 4; ll++, pi++) {
            const double m2 = fma(sq[kk], W.hm2[kk], fma(sq[ll], W.hm2[ll], (sv[kk] * sv[ll]) * W.hdot[pi]));
            const double t = (sqrt_fast(m2 < 0.0 ? 0.0 : m2) - P.m_higgs) * inv_sh;
            W.ht[pi * VC + vv] = -0.5 * (t * t);
          }
      }
    } else
#pragma unroll 1
    for (int p0 = 0; p0 < n_pair; p0 += LPB) {
      const int p = p0 + sub;
      if (vok && p < n_pair) {
        const uint32_t hd = W.hp[p];
        const int kk = hd & 15, ll = (hd >> 4) & 15, j1 = (hd >> 8) & 15, j2 = (hd >> 12) & 15, pi = hd >> 16;
        const double sk = W.sc()[j1 * VC + vv], sl = W.sc()[j2 * VC + vv];
        const double m2 = fma(sk * sk, W.hm2[kk], fma(sl * sl, W.hm2[ll], (sk * sl) * W.hdot[pi]));
        // a NaN (garbage inputs: inf - inf) stays a NaN, so that such a pair never wins here while the finalize kernel, which
        // adds the four-vectors, finds no finite mass for it
        const double t = (sqrt_fast(m2 < 0.0 ? 0.0 : m2) - P.m_higgs) * inv_sh;
        W.ht[pi * VC + vv] = -0.5 * (t * t);
      }
    }
    __syncwarp();
    // ---- C1: ordered pairings -> resultant -> depressed quartic -> "may have real roots?" -> solve queue
    //      C2: pop 32 queued quartics -> Ferrari -> 0/2/4 real roots pushed on the root stack
    //      D : pop 32 roots -> refine on the conics, score
    // One more trip of the loop (last) drains what is left of both queues with partial warps: the tables of this chunk
    // are about to be overwritten.
#pragma unroll 1
    for (int a0 = 0;; a0 += LPB) {
      const bool last = a0 >= n_ord;
      if (!last) {
        const int ap = a0 + sub;
        // Every lane computes (no branch, no default values): a lane without an item (variation past V, or pairing past the last
        // one when the sub-groups do not divide their number) works on whatever its table slot holds — the indices stay inside
        // the warp's tables — and is not kept.
        const int i = (ap * dmul) >> dsh; int j = ap - i * (nb - 1); j += (j >= i);   // i = ap / (nb - 1)
        const int a1 = i * VC + vv, a2 = (NBT + j) * VC + vv;
        const double2 abA = W.ab[i], abB = W.ab[NBT + j], k01 = W.pcv[ap][0], k23 = W.pcv[ap][1];
        const Conic A{abA.x, abA.y, W.cc[i], W.def[0][a1], W.def[1][a1], W.def[2][a1]};
        const Conic B{abB.x, abB.y, W.cc[NBT + j], W.def[0][a2], W.def[1][a2], W.def[2][a2]};
        const PairConst K{k01.x, k01.y, k23.x, k23.y};
        double g3, g2, g1, g0, qp, qq, qr, qaq;
        resultant(A, B, K, g3, g2, g1, g0);
        depress(g3, g2, g1, g0, qaq, qp, qq, qr);
        const bool keep = !certainly_no_real_root(qp, qq, qr) && vok && ap < n_ord;
        const uint32_t stag = (uint32_t)vv | (i << 5) | (j << 8);
        const unsigned bk = __ballot_sync(0xffffffffu, keep);
        if (keep) {
          const int at = sn + __popc(bk & lt);
          const double aqt = __hiloint2double(__double2hiint(qaq), (int)(((uint32_t)__double2loint(qaq) & ~STAG_MASK) | stag));
          HEPF_CHECK(at >= 0 && at < SCAP && a1 < 2 * NBT * VC && a2 < 2 * NBT * VC && ap < NBT * (NBT - 1));
          W.s_pq[at] = make_double2(qp, qq); W.s_ra[at] = make_double2(qr, aqt);
        }
        sn += __popc(bk);
        __syncwarp();
      }
      while (sn >= 32 || (last && (sn | qn) != 0)) {
        const int take = min(min(32, sn), (QCAP - qn) >> 2);   // every lane may push four roots
        if (take > 0) {                                        // (warp-uniform; 0 only while draining the root stack at the end)
          sn -= take;
          int mask = 0; uint32_t tag = 0;
          double xa[2], xb[2];
          if (lane < take) {
            HEPF_CHECK(sn >= 0 && sn + lane < SCAP);
            const double2 pq = W.s_pq[sn + lane], ra = W.s_ra[sn + lane];
            const uint32_t st = (uint32_t)__double2loint(ra.y) & STAG_MASK;
            const double aq = __hiloint2double(__double2hiint(ra.y), (int)((uint32_t)__double2loint(ra.y) & ~STAG_MASK));   // tag bits cleared
            mask = ferrari(pq.x, pq.y, ra.x, aq, seedE, xa, xb);
            if (mask) {
              double ht; int hh, kk, ll;
              best_higgs<NBT, VC>(&W.ht[st & 31], nb, (st >> 5) & 7, (st >> 8) & 7, ht, hh, kk, ll);
              tag = st | (hh << 11) | (pair_index<NBT>(kk, ll) << 14);
            }
          }
          // push: Ferrari slots are numbered over the real pairs in the order A+, A-, B+, B-
          const unsigned bA = __ballot_sync(0xffffffffu, mask & 1), bB = __ballot_sync(0xffffffffu, mask & 2);
          int at = qn + 2 * (__popc(bA & lt) + __popc(bB & lt));
          if (mask & 1) {
            W.push(at, xa[0], tag); W.push(at + 1, xa[1], tag | (1u << 18)); at += 2;
          }
          if (mask & 2) {
            const uint32_t s0 = (mask & 1) ? 2u : 0u;
            W.push(at, xb[0], tag | (s0 << 18)); W.push(at + 1, xb[1], tag | ((s0 + 1u) << 18));
          }
          qn += 2 * (__popc(bA) + __popc(bB));
          __syncwarp();
        }
        while (qn >= 32 || (last && sn == 0 && qn > 0)) {
          const int tk = min(32, qn);
          qn -= tk;
          if (lane < tk) {
            double ex; uint32_t et; W.pop(qn + lane, ex, et);
            score_entry<VC, NBT>(W, ex, et, v0, inv_lambda, best_ll, best_key);
          }
          __syncwarp();
        }
      }
      if (last) break;
    }
    __syncwarp();
  }
  // ---- argmax over the lanes: max loglik, then the earliest key ---------------------------------------------------------
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const double oll = __shfl_xor_sync(0xffffffffu, best_ll, o);
    const uint32_t okey = __shfl_xor_sync(0xffffffffu, best_key, o);
    if (oll > best_ll || (oll == best_ll && okey < best_key)) { best_ll = oll; best_key = okey; }
  }
  return best_key;
}

// length of the list: a host value (n_dev == NULL), or read from device memory and clamped to the capacity
__device__ __forceinline__ int64_t list_length(const int64_t* n_dev, int64_t n_cap) {
  if (!n_dev) return n_cap;
  const int64_t n = __ldg(n_dev);
  return n < 0 ? 0 : (n < n_cap ? n : n_cap);
}

// Persistent warps: each warp draws the next group of `epc` consecutive list entries from a global counter; its
// lanes look at one entry each (index, flags), the entries this instantiation owns are then reconstructed one after the
// other by the whole warp.  NBT = 4 owns the events with exactly four b candidates (and writes the "nothing to do" key
// of the non-applicable ones); NBT = 6 owns those with five or six: two launches, each with shared-memory tables sized
// for its class.
template <int VC, int NBT, int RW, int MINB>
__global__ void __launch_bounds__(32 * RW, MINB)
reco_search_kernel(RecoCols ev, const uint32_t* __restrict__ idx, const int64_t* __restrict__ n_dev, int64_t n_cap, int epc, int V,
                   uint32_t k0, uint32_t k1, hepf_tth_params_t P, uint2* __restrict__ winners, double* __restrict__ nominal,
                   unsigned long long* __restrict__ next_group) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  WarpMem<VC, NBT>& W = reinterpret_cast<WarpMem<VC, NBT>*>(smem_raw)[threadIdx.x >> 5];
  const int lane = threadIdx.x & 31;
  const int64_t n_idx = list_length(n_dev, n_cap);
  const int64_t n_groups = (n_idx + epc - 1) / epc;
  for (;;) {
    unsigned long long gq = 0;
    if (lane == 0) gq = atomicAdd(next_group, 1ull);
    const int64_t g = (int64_t)__shfl_sync(0xffffffffu, gq, 0);
    if (g >= n_groups) break;
    const int64_t kl = g * epc + lane;
    bool mine = false;
    if (lane < epc && kl < n_idx) {
      const EventHead hl = load_head(ev, (int64_t)__ldg(idx + kl));
      if (!hl.applicable) { if (NBT == 4) winners[kl] = make_uint2(0xffffffffu, 0u); }
      else mine = (NBT == 4) ? (hl.n_b == 4) : (hl.n_b > 4);
    }
    unsigned todo = __ballot_sync(0xffffffffu, mine);
    while (todo) {
      const int src = __ffs(todo) - 1; todo &= todo - 1;
      const int64_t k = g * epc + src;
      const EventHead h = load_head(ev, (int64_t)__ldg(idx + k));
      const uint32_t key = search_event<VC, NBT>(W, ev, h, V, k0, k1, P, lane);
      HEPF_CHECK(k >= 0 && k < n_cap);
      if (lane == 0) winners[k] = make_uint2(key, key != 0xffffffffu ? 1u : 0u);
      // The nominal objects and the MET of the event, as this warp gathered them, go to the workspace as 42 columns of
      // n_cap doubles: the finalize kernel then reads them coalesced instead of gathering 40 scattered 64-byte DRAM atoms per
      // event a second time (the selected events are a few per cent of the store).
      for (int it = lane; it < NOMINAL_ROWS; it += 32) nominal[(int64_t)it * n_cap + k] = it < 40 ? W.obj[it] : W.met[it - 40];
      __syncwarp();
    }
  }
}

constexpr int FIN_THREADS = 128;
__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gmem_src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// One selected event: re-derive the winner in full, polish it and write the record.
__device__ __forceinline__ void finalize_event(const RecoCols& ev, const uint32_t* __restrict__ idx, int64_t k, int64_t n_cap, uint32_t k0,
                                               uint32_t k1, const hepf_tth_params_t& P, const uint2* __restrict__ winners,
                                               const double* __restrict__ nominal, hepf_best_t* __restrict__ out,
                                               double (*__restrict__ s_obj)[FIN_THREADS]) {
  const EventHead h = load_head(ev, (int64_t)__ldg(idx + k));
  const uint2 w = winners[k];
  hepf_best_t* o = out + k;
  const int tid = threadIdx.x;
  if (!h.applicable || !w.y) {
    const double n = CUDART_NAN;
    o->nu[0] = o->nu[1] = o->nu[2] = o->nubar[0] = o->nubar[1] = o->nubar[2] = n;
    o->m_top = o->m_antitop = o->m_wplus = o->m_wminus = o->m_higgs = o->loglik = n;
    o->variation = o->jet_b = o->jet_bbar = o->jet_h1 = o->jet_h2 = o->root = -1;
    o->status = h.status; o->event = (uint32_t)(h.e + ev.out_off);
    return;
  }
  const int v = (int)(w.x >> 11), a6 = (w.x >> 5) & 63, i = a6 / 6, j = a6 - 6 * i, hsel = (w.x >> 2) & 7, ksel = w.x & 3;
  const int nb = h.n_b;
  const double mt2 = P.m_top * P.m_top, mw2 = P.m_w * P.m_w, inv_lambda = rcp_fast(P.lambda_nu), inv_sh = rcp_fast(P.sigma_higgs);
  // Nominal objects and MET from the workspace copy the search kernel left (42 columns of n_cap doubles: consecutive
  // threads read consecutive addresses), not from the store, where every value of a selected event is its own DRAM atom.
  // The 40 object components go straight into this thread's column of the block's shared array (cp.async: all in flight
  // together, no register in between): they are indexed by jet slot further down, and as a thread-local array they were
  // 0.9 KB of local memory per thread that left L2 (0.57 GB of DRAM writes per launch on cfg4).
#pragma unroll
  for (int it = 0; it < 40; it++) cp_async8(&s_obj[it][tid], nominal + (int64_t)it * n_cap + k);
  const double met_x = __ldcs(nominal + 40 * n_cap + k), met_y = __ldcs(nominal + 41 * n_cap + k);
  const int lps = h.lp_slot, lms = 1 - h.lp_slot;
  const int si = (h.cand >> (4 * i)) & 15, sj = (h.cand >> (4 * j)) & 15;
  // Higgs pair hsel among the candidates not used by (i, j)
  int hk = 0, hl = 1, hc = 0;
  for (int kk = 0; kk < nb; kk++) for (int l = kk + 1; l < nb; l++) {
    if (kk == i || kk == j || l == i || l == j) continue;
    if (hc == hsel) { hk = kk; hl = l; }
    hc++;
  }
  const int sh1 = (h.cand >> (4 * hk)) & 15, sh2 = (h.cand >> (4 * hl)) & 15;
  cp_async_wait_all();
  auto obj4 = [&](int t, double (&p)[4]) {
#pragma unroll
    for (int c = 0; c < 4; c++) p[c] = s_obj[4 * t + c][tid];
  };
  // smear this variation: every scale enters the MET, six of them (the two leptons, b, bbar and the Higgs pair) are kept
  double ax = 0.0, ay = 0.0;
  double sc_lp = 1.0, sc_lm = 1.0, sc_bi = 1.0, sc_bj = 1.0, sc_h1 = 1.0, sc_h2 = 1.0;
  for (int blk = 0; blk < h.nblk; blk++) {
    uint32_t x[4];
    philox4x32_10((uint32_t)h.gidx, (uint32_t)(h.gidx >> 32), (uint32_t)v, 0x54544800u + blk, k0, k1, x);
    double z[2]; block_normals(x, z[0], z[1]);
#pragma unroll
    for (int u = 0; u < 2; u++) {
      const int t = 2 * blk + u;
      // kappa * sigma as load_object computes it (step 2)
      const double sigma = t < 2 ? P.lep_sigma : __dadd_rn(__ddiv_rn(P.jet_stoch, __dsqrt_rn(s_obj[4 * t + 3][tid])), P.jet_const);
      const double ks = t < 2 + h.n_jet ? __dmul_rn(P.sigma_scale, sigma) : 0.0;
      const double sct = scale_of(ks, z[u], P.s_min);
      if (t < 2 + h.n_jet) {
        const double d = __dadd_rn(sct, -1.0);
        ax = __dadd_rn(ax, __dmul_rn(d, s_obj[4 * t][tid])); ay = __dadd_rn(ay, __dmul_rn(d, s_obj[4 * t + 1][tid]));
      }
      sc_lp = t == lps ? sct : sc_lp; sc_lm = t == lms ? sct : sc_lm;
      sc_bi = t == 2 + si ? sct : sc_bi; sc_bj = t == 2 + sj ? sct : sc_bj;
      sc_h1 = t == 2 + sh1 ? sct : sc_h1; sc_h2 = t == 2 + sh2 ? sct : sc_h2;
    }
  }
  const double Mx = __dadd_rn(met_x, -ax), My = __dadd_rn(met_y, -ay);
  double o_lp[4], o_lm[4], o_bi[4], o_bj[4];
  obj4(lps, o_lp); obj4(lms, o_lm); obj4(2 + si, o_bi); obj4(2 + sj, o_bj);
  const V4 lp = scale_v4(o_lp, sc_lp), lm = scale_v4(o_lm, sc_lm);
  const V4 bi = scale_v4(o_bi, sc_bi), bj = scale_v4(o_bj, sc_bj);
  // same frame-based construction as the search kernel (identical bits)
  const double hmw2 = 0.5 * mw2, hcm = 0.5 * (mt2 - mw2);
  const Frame F1 = make_frame(o_lp, o_bi), F2 = make_frame(o_lm, o_bj);
  Conic A, q2; double c0, e0;
  A.a = F1.a; A.b = F1.b; A.c = F1.c; q2.a = F2.a; q2.b = F2.b; q2.c = F2.c;
  conic_def(F1, sc_lp, sc_bi, rcp_fast(sc_lp), rcp_fast(sc_bi), hmw2, hcm, c0, A.d, A.e, A.f);
  conic_def(F2, sc_lm, sc_bj, rcp_fast(sc_lm), rcp_fast(sc_bj), hmw2, hcm, e0, q2.d, q2.e, q2.f);
  const double c1 = F1.c1, c2 = F1.c2, e1 = F2.c1, e2 = F2.c2;
  const Conic B = shift_conic(q2, Mx, My);
  double g3, g2, g1, g0, xa[2] = {0, 0}, xb[2] = {0, 0};
  resultant(A, B, pair_consts(A.a, A.b, A.c, B.a, B.b, B.c), g3, g2, g1, g0);
  const int mask = solve_quartic(g3, g2, g1, g0, seed_scale(P), xa, xb);
  // the <= 4 roots: x in registers (static indices), refined one by one; the selected one is kept on the way
  const bool ma = mask & 1, mb = mask & 2;
  const int nr = (ma ? 2 : 0) + (mb ? 2 : 0);
  const double xs[4] = {ma ? xa[0] : xb[0], ma ? xa[1] : xb[1], xb[0], xb[1]};
  const int rs = ksel < nr ? ksel : 0;
  double xx = CUDART_NAN, yy = CUDART_NAN;
  double xr[4];
#pragma unroll 1
  for (int r = 0; r < nr; r++) {
    double x = r == 0 ? xs[0] : r == 1 ? xs[1] : r == 2 ? xs[2] : xs[3], y;
    refine_xy<false>(A, B, x, y);
    if (r == rs) { xx = x; yy = y; }
    if (r == 0) xr[0] = x; else if (r == 1) xr[1] = x; else if (r == 2) xr[2] = x; else xr[3] = x;
  }
  int rank = 0;
#pragma unroll
  for (int r = 0; r < 4; r++) if (r < nr) rank += (xr[r] < xx) || (xr[r] == xx && r < rs);
  double o_h1[4], o_h2[4];
  obj4(2 + sh1, o_h1); obj4(2 + sh2, o_h2);
  const V4 h1 = scale_v4(o_h1, sc_h1), h2 = scale_v4(o_h2, sc_h2);
  const double mbb = mass_of(h1.e + h2.e, h1.x + h2.x, h1.y + h2.y, h1.z + h2.z);
  const double t = (mbb - P.m_higgs) * inv_sh, ht = -0.5 * (t * t);
  double pz = fma(c2, yy, fma(c1, xx, c0));
  double qx = Mx - xx, qy = My - yy, qz = fma(e2, qy, fma(e1, qx, e0));
  double xx_ = xx, yy_ = yy;
  if (nr) polish_raw(lp, bi, lm, bj, Mx, My, P.m_top, P.m_w, xx_, yy_, pz, qx, qy, qz);
  const double en = sqrt_fast(fma(xx_, xx_, fma(yy_, yy_, pz * pz))), eb = sqrt_fast(fma(qx, qx, fma(qy, qy, qz * qz)));
  o->nu[0] = xx_; o->nu[1] = yy_; o->nu[2] = pz;
  o->nubar[0] = qx; o->nubar[1] = qy; o->nubar[2] = qz;
  o->m_wplus = mass_of(lp.e + en, lp.x + xx_, lp.y + yy_, lp.z + pz);
  o->m_top = mass_of(lp.e + en + bi.e, lp.x + xx_ + bi.x, lp.y + yy_ + bi.y, lp.z + pz + bi.z);
  o->m_wminus = mass_of(lm.e + eb, lm.x + qx, lm.y + qy, lm.z + qz);
  o->m_antitop = mass_of(lm.e + eb + bj.e, lm.x + qx + bj.x, lm.y + qy + bj.y, lm.z + qz + bj.z);
  o->m_higgs = mbb;
  o->loglik = loglik_of(xx_, yy_, Mx, My, ht, inv_lambda);
  o->variation = v;
  o->jet_b = si; o->jet_bbar = sj; o->jet_h1 = sh1; o->jet_h2 = sh2;
  o->root = rank;
  o->status = h.status | 1u; o->event = (uint32_t)(h.e + ev.out_off);
}

// One thread per listed event (grid-stride: the grid is sized from the capacity, the length may live on the device).
__global__ void __launch_bounds__(FIN_THREADS, 4)   // 128 registers: the kernel is a chain of dependent FP64 operations, more resident warps hide it
reco_finalize_kernel(RecoCols ev, const uint32_t* __restrict__ idx, const int64_t* __restrict__ n_dev, int64_t n_cap, uint32_t k0,
                     uint32_t k1, hepf_tth_params_t P, const uint2* __restrict__ winners, const double* __restrict__ nominal,
                     hepf_best_t* __restrict__ out) {
  __shared__ double s_obj[40][FIN_THREADS];   // a column per thread: the nominal objects of its event (40 KB per block)
  const int64_t n_idx = list_length(n_dev, n_cap);
  for (int64_t k = (int64_t)blockIdx.x * FIN_THREADS + threadIdx.x; k < n_idx; k += (int64_t)gridDim.x * FIN_THREADS)
    finalize_event(ev, idx, k, n_cap, k0, k1, P, winners, nominal, out, s_obj);
}

// hepf_tth_system: invariant mass and transverse momentum of the reconstructed ttH system of each record (PAPER.md:410-442,
// App. 8.2: "TLorentzVector ttH = Top + Tbar + Higgs; mTTH = ttH.M(); ptTTH = ttH.Pt();").  One thread per record: the
// scales of the record's variation are drawn again (same Philox keys), the eight four-vectors l+, l-, nu, nubar, b, bbar,
// h1, h2 are added in that order, every operation one IEEE operation in a fixed order (bit-identical to the definition).
__global__ void __launch_bounds__(128)
tth_system_kernel(RecoCols ev, const hepf_best_t* __restrict__ best, int64_t n, uint32_t k0, uint32_t k1, hepf_tth_params_t P,
                  double2* __restrict__ out) {
  for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) {
    const hepf_best_t* b = best + k;
    double2 r = make_double2(CUDART_NAN, CUDART_NAN);
    const int64_t e = (int64_t)b->event - ev.out_off;
    if ((b->status & 1u) && e >= 0 && e < ev.n) {
      const EventHead h = load_head(ev, e);
      const int slots[6] = {h.lp_slot, 1 - h.lp_slot, 2 + b->jet_b, 2 + b->jet_bbar, 2 + b->jet_h1, 2 + b->jet_h2};
      const double nx = b->nu[0], ny = b->nu[1], nz = b->nu[2], qx = b->nubar[0], qy = b->nubar[1], qz = b->nubar[2];
      const double en = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(nx, nx), __dmul_rn(ny, ny)), __dmul_rn(nz, nz)));
      const double eq = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(qx, qx), __dmul_rn(qy, qy)), __dmul_rn(qz, qz)));
      double sx = 0.0, sy = 0.0, sz = 0.0, se = 0.0;
#pragma unroll 1
      for (int i = 0; i < 8; i++) {        // order: l+, l-, nu, nubar, b, bbar, h1, h2
        double px, py, pz, pe;
        if (i == 2) { px = nx; py = ny; pz = nz; pe = en; }
        else if (i == 3) { px = qx; py = qy; pz = qz; pe = eq; }
        else {
          const int t = slots[i < 2 ? i : i - 2];
          double obj[4], ks; load_object(ev, e, t, P, obj, ks);
          uint32_t x[4];
          philox4x32_10((uint32_t)h.gidx, (uint32_t)(h.gidx >> 32), (uint32_t)b->variation, 0x54544800u + (t >> 1), k0, k1, x);
          double z[2]; block_normals(x, z[0], z[1]);
          const double sc = scale_of(ks, z[t & 1], P.s_min);
          px = __dmul_rn(sc, obj[0]); py = __dmul_rn(sc, obj[1]); pz = __dmul_rn(sc, obj[2]); pe = __dmul_rn(sc, obj[3]);
        }
        if (i == 0) { sx = px; sy = py; sz = pz; se = pe; }
        else { sx = __dadd_rn(sx, px); sy = __dadd_rn(sy, py); sz = __dadd_rn(sz, pz); se = __dadd_rn(se, pe); }
      }
      const double p2 = __dadd_rn(__dadd_rn(__dmul_rn(sx, sx), __dmul_rn(sy, sy)), __dmul_rn(sz, sz));
      const double m2 = __dadd_rn(__dmul_rn(se, se), -p2);
      r.x = __dsqrt_rn(m2 > 0.0 ? m2 : 0.0);
      r.y = __dsqrt_rn(__dadd_rn(__dmul_rn(sx, sx), __dmul_rn(sy, sy)));
    }
    out[k] = r;
  }
}

template <int VC, int NBT, int RW, int MINB>
static int launch_search(const RecoCols& cols, const uint32_t* idx, const int64_t* n_dev, int64_t n_idx, int V, uint64_t seed,
                         const hepf_tth_params_t& P, uint2* winners, double* nominal, unsigned long long* counter, cudaStream_t stream) {
  const size_t smem = sizeof(WarpMem<VC, NBT>) * RW;
  auto kern = reco_search_kernel<VC, NBT, RW, MINB>;
  static thread_local int blocks_per_sm = 0, sms = 0, cached_dev = -1;   // per instantiation (smem is a constant of it) and device
  int dev = 0;
  HEPF_CUDA_TRY(cudaGetDevice(&dev));
  if (dev != cached_dev) {
    blocks_per_sm = 0;
    HEPF_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    HEPF_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    HEPF_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
    HEPF_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&blocks_per_sm, kern, 32 * RW, smem));
    if (blocks_per_sm < 1) { set_error("hepf_reconstruct_tth: search kernel does not fit on an SM"); return HEPF_ERR_CUDA; }
    cached_dev = dev;
  }
  // persistent grid; groups of up to 8 list entries, fewer when the list is short
  const int64_t max_warps = (int64_t)sms * blocks_per_sm * RW;
  int epc = 8;
  while (epc > 1 && (n_idx + epc - 1) / epc < 8 * max_warps) epc >>= 1;
  const int64_t n_groups = (n_idx + epc - 1) / epc;
  const int64_t want = (n_groups + RW - 1) / RW, cap = (int64_t)sms * blocks_per_sm;
  const unsigned grid = (unsigned)(want < cap ? want : cap);
  kern<<<grid, 32 * RW, smem, stream>>>(cols, idx, n_dev, n_idx, epc, V, (uint32_t)seed, (uint32_t)(seed >> 32), P, winners, nominal, counter);
  count_launch();
  HEPF_CUDA_TRY(cudaGetLastError());
  return HEPF_OK;
}

// both candidate-count classes: n_b = 4 (tables for 4 candidates, more warps per SM) and n_b = 5, 6
template <int VC4, int VC6, int RW4, int RW6, int MINB4, int MINB6>
static int launch_search_both(const RecoCols& cols, const uint32_t* idx, const int64_t* n_dev, int64_t n_idx, int V, uint64_t seed,
                              const hepf_tth_params_t& P, uint2* winners, double* nominal, cudaStream_t stream) {
  unsigned long long* counters = reinterpret_cast<unsigned long long*>(winners + n_idx);   // two group counters
  HEPF_CUDA_TRY(cudaMemsetAsync(counters, 0, 2 * sizeof(unsigned long long), stream));
  timing_mark(T_RECO0, stream);
  int rc = launch_search<VC4, 4, RW4, MINB4>(cols, idx, n_dev, n_idx, V, seed, P, winners, nominal, counters, stream);
  timing_mark(T_RECO1, stream);
  if (rc != HEPF_OK) return rc;
  rc = launch_search<VC6, 6, RW6, MINB6>(cols, idx, n_dev, n_idx, V, seed, P, winners, nominal, counters + 1, stream);
  timing_mark(T_RECO2, stream);
  return rc;
}

}  // namespace hepf

using namespace hepf;

static size_t nominal_offset(int64_t n_idx) {
  const size_t n = (size_t)(n_idx > 0 ? n_idx : 1);
  return (n * sizeof(uint2) + 16 + 15) / 16 * 16;
}

extern "C" size_t hepf_reconstruct_workspace_bytes(int64_t n_idx, int32_t n_variations) {
  (void)n_variations;
  if (n_idx < 0) return 0;
  // one winner key per listed event + two work counters, then the nominal objects of the searched events (42 columns)
  const size_t n = (size_t)(n_idx > 0 ? n_idx : 1);
  return nominal_offset(n_idx) + (size_t)NOMINAL_ROWS * n * sizeof(double);
}

extern "C" int hepf_reconstruct_tth(const hepf_events_t* events, const uint32_t* idx, int64_t n_idx, int32_t n_variations,
                                    uint64_t seed, const hepf_tth_params_t* host_params, hepf_best_t* out_best, void* ws,
                                    size_t ws_bytes, void* stream_) {
  return hepf::reconstruct_impl(events, idx, nullptr, n_idx, n_variations, seed, host_params, out_best, ws, ws_bytes,
                                (cudaStream_t)stream_, 0);
}

extern "C" int hepf_reconstruct_tth_n(const hepf_events_t* events, const uint32_t* idx, const int64_t* n_idx_device, int64_t n_idx_cap,
                                      int32_t n_variations, uint64_t seed, const hepf_tth_params_t* host_params,
                                      hepf_best_t* out_best, void* ws, size_t ws_bytes, void* stream_) {
  if (!n_idx_device || !aligned(n_idx_device, 8)) { set_error("hepf_reconstruct_tth_n: n_idx_device NULL or misaligned"); return HEPF_ERR_ARG; }
  return hepf::reconstruct_impl(events, idx, n_idx_device, n_idx_cap, n_variations, seed, host_params, out_best, ws, ws_bytes,
                                (cudaStream_t)stream_, 0);
}

int hepf::reconstruct_impl(const hepf_events_t* events, const uint32_t* idx, const int64_t* n_dev, int64_t n_idx, int32_t n_variations, uint64_t seed,
                           const hepf_tth_params_t* host_params, hepf_best_t* out_best, void* ws, size_t ws_bytes,
                           cudaStream_t stream, int64_t event_out_offset) {
  int rc = check_events(events);
  if (rc != HEPF_OK) return rc;
  if (n_idx < 0 || n_variations < 1 || n_variations > (1 << 21)) {
    set_error("hepf_reconstruct_tth: need n_idx >= 0 and 1 <= n_variations <= 2^21"); return HEPF_ERR_ARG;
  }
  if (n_idx == 0) return HEPF_OK;
  if (!idx || !aligned(idx, 4) || !out_best || !aligned(out_best, 16)) {
    set_error("hepf_reconstruct_tth: idx/out_best NULL or misaligned"); return HEPF_ERR_ARG;
  }
  if (!ws || !aligned(ws, 8) || ws_bytes < hepf_reconstruct_workspace_bytes(n_idx, n_variations)) {
    set_error("hepf_reconstruct_tth: workspace too small or misaligned (%zu < %zu)", ws_bytes,
              hepf_reconstruct_workspace_bytes(n_idx, n_variations));
    return HEPF_ERR_CAPACITY;
  }
  hepf_tth_params_t P;
  if (host_params) P = *host_params; else hepf_default_params(&P);
  const RecoCols cols{events->lep_px, events->lep_py, events->lep_pz, events->lep_e, events->jet_px, events->jet_py,
                      events->jet_pz, events->jet_e, events->met_x, events->met_y, events->flags,
                      events->n_events, events->stride, events->event_base, event_out_offset};
  uint2* winners = reinterpret_cast<uint2*>(ws);
  double* nominal = reinterpret_cast<double*>(static_cast<char*>(ws) + nominal_offset(n_idx));
  // chunk of variations per pass of the pipeline: 32 when that wastes at most an eighth of the lanes of the last chunk,
  // else 16 or 8.  32 (16 for n_b = 6) needs so much shared memory per warp that one block of 18 (19) warps fills an SM.
  const int waste32 = ((n_variations + 31) & ~31) - n_variations;
  if (n_variations <= 2) rc = launch_search_both<1, 1, 2, 2, 16, 16>(cols, idx, n_dev, n_idx, n_variations, seed, P, winners, nominal, stream);   // lanes = pairings
  else if (n_variations <= 8) rc = launch_search_both<8, 8, 2, 2, 12, 10>(cols, idx, n_dev, n_idx, n_variations, seed, P, winners, nominal, stream);
  else if (8 * waste32 > n_variations) rc = launch_search_both<16, 8, 3, 2, 7, 9>(cols, idx, n_dev, n_idx, n_variations, seed, P, winners, nominal, stream);
  else rc = launch_search_both<32, 16, 18, 19, 1, 1>(cols, idx, n_dev, n_idx, n_variations, seed, P, winners, nominal, stream);
  if (rc != HEPF_OK) return rc;
  int dev = 0, sms = 148;
  HEPF_CUDA_TRY(cudaGetDevice(&dev));
  HEPF_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int64_t want = (n_idx + 127) / 128, cap = (int64_t)sms * 32;
  reco_finalize_kernel<<<(unsigned)(want < cap ? want : cap), FIN_THREADS, 0, stream>>>(cols, idx, n_dev, n_idx, (uint32_t)seed,
                                                                             (uint32_t)(seed >> 32), P, winners, nominal, out_best);
  count_launch();
  timing_mark(T_RECO3, stream);
  HEPF_CUDA_TRY(cudaGetLastError());
  return HEPF_OK;
}

extern "C" int hepf_tth_system(const hepf_events_t* events, const hepf_best_t* best, int64_t n, uint64_t seed,
                               const hepf_tth_params_t* host_params, double* out, void* stream_) {
  int rc = check_events(events);
  if (rc != HEPF_OK) return rc;
  if (n < 0) { set_error("hepf_tth_system: n < 0"); return HEPF_ERR_ARG; }
  if (n == 0) return HEPF_OK;
  if (!best || !aligned(best, 16) || !out || !aligned(out, 16)) { set_error("hepf_tth_system: best/out NULL or misaligned"); return HEPF_ERR_ARG; }
  hepf_tth_params_t P;
  if (host_params) P = *host_params; else hepf_default_params(&P);
  const RecoCols cols{events->lep_px, events->lep_py, events->lep_pz, events->lep_e, events->jet_px, events->jet_py,
                      events->jet_pz, events->jet_e, events->met_x, events->met_y, events->flags,
                      events->n_events, events->stride, events->event_base, 0};
  int dev = 0, sms = 148;
  HEPF_CUDA_TRY(cudaGetDevice(&dev));
  HEPF_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int64_t want = (n + 127) / 128, cap = (int64_t)sms * 16;
  tth_system_kernel<<<(unsigned)(want < cap ? want : cap), 128, 0, (cudaStream_t)stream_>>>(
      cols, best, n, (uint32_t)seed, (uint32_t)(seed >> 32), P, reinterpret_cast<double2*>(out));
  count_launch();
  HEPF_CUDA_TRY(cudaGetLastError());
  return HEPF_OK;
}
