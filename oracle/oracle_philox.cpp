// oracle/oracle_philox.cpp — CPU ORACLE (test infrastructure).  O1 Philox4x32-10, O2 uniforms + normals.
//
// Follows SURVEY.md §8(c) O1-O2 line by line (north_star: "draw Gaussian resolution smearings from a
// counter-based PRNG"; the paper itself offloaded a Mersenne Twister, §5.3).
// Compile with -ffp-contract=off: every + - * / sqrt below is one IEEE-754 round-to-nearest operation and
// std::fma is the only fused operation, exactly where O2 writes "fma".
#include <cmath>
#include <cstdint>
#include <cstring>

#include "hepf_oracle.h"

// ---- O1: Philox4x32-10 (Salmon et al., "Parallel random numbers: as easy as 1, 2, 3") ----------------
// ten rounds; key bumped by the Weyl constants before every round except the first.
extern "C" void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; round++) {
    if (round > 0) { k0 += W0; k1 += W1; }
    uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// ---- O2: L(u) = ln u, deterministic operation sequence ------------------------------------------------
extern "C" double orc_det_log(double u) {
  const double SQRT2 = 0x1.6a09e667f3bcdp+0, LN2_HI = 0x1.62e42fee00000p-1, LN2_LO = 0x1.a39ef35793c76p-33;
  uint64_t bits; std::memcpy(&bits, &u, 8);
  int e = (int)((bits >> 52) & 0x7ff) - 1023;                 // u is always a normal number in (0, 1]
  bits = (bits & 0x000fffffffffffffULL) | 0x3ff0000000000000ULL;
  double m; std::memcpy(&m, &bits, 8);                        // m in [1, 2)
  if (m > SQRT2) { m = m * 0.5; e = e + 1; }                  // exact
  double f = m - 1.0;                                         // exact
  double s = f / (2.0 + f);
  double z = s * s;
  double p = 2.0 / 19.0;                                      // c_9
  for (int k = 8; k >= 1; k--) p = std::fma(p, z, 2.0 / (double)(2 * k + 1));
  p = p * z;
  double lm = std::fma(s, p, 2.0 * s);
  double ed = (double)e;
  return std::fma(ed, LN2_HI, std::fma(ed, LN2_LO, lm));
}

// ---- O2: SC(u) = (sin 2 pi u, cos 2 pi u) ---------------------------------------------------------------
extern "C" void orc_det_sincos2pi(double u, double* sn, double* cs) {
  const double PIO2_HI = 0x1.921fb54442d18p+0, PIO2_LO = 0x1.1a62633145c07p-54;
  double t = 4.0 * u;                                         // exact
  double n = std::floor(t + 0.5);
  double r = t - n;                                           // exact, |r| <= 1/2
  double th = std::fma(r, PIO2_HI, r * PIO2_LO);
  double z = th * th;
  // S_k = (-1)^k / (2k+1)!, C_k = (-1)^k / (2k)!  (factorials up to 17! are exact doubles)
  double fact[18]; fact[0] = 1.0;
  for (int i = 1; i < 18; i++) fact[i] = fact[i - 1] * (double)i;
  auto S = [&](int k) { return ((k & 1) ? -1.0 : 1.0) / fact[2 * k + 1]; };
  auto C = [&](int k) { return ((k & 1) ? -1.0 : 1.0) / fact[2 * k]; };
  double ps = S(8);
  for (int k = 7; k >= 1; k--) ps = std::fma(ps, z, S(k));
  double s = std::fma(th * z, ps, th);
  double pc = C(8);
  for (int k = 7; k >= 1; k--) pc = std::fma(pc, z, C(k));
  double c = std::fma(z, pc, 1.0);
  int q = ((int)n) & 3;
  switch (q) {
    case 0: *sn = s; *cs = c; break;
    case 1: *sn = c; *cs = -s; break;
    case 2: *sn = -s; *cs = -c; break;
    default: *sn = -c; *cs = s; break;
  }
}

// one Philox block -> (Z_even, Z_odd)
static void block_normals(const uint32_t x[4], double* z_even, double* z_odd) {
  uint64_t w0 = ((uint64_t)x[1] << 32) | x[0], w1 = ((uint64_t)x[3] << 32) | x[2];
  double u1 = (double)((w0 >> 11) + 1) * 0x1p-53;             // (0, 1], exact
  double u2 = (double)(w1 >> 11) * 0x1p-53;                   // [0, 1), exact
  double rho = std::sqrt(-2.0 * orc_det_log(u1));
  double sn, cs; orc_det_sincos2pi(u2, &sn, &cs);
  *z_even = rho * cs; *z_odd = rho * sn;
}

// normals of an arbitrary Philox (ctr, key) — used by the reconstruction's smearing domain
void orc_block_normals(const uint32_t ctr[4], const uint32_t key[2], double* z_even, double* z_odd) {
  uint32_t x[4]; orc_philox4x32_10(ctr, key, x); block_normals(x, z_even, z_odd);
}

// the single infinite stream Z[g]: block b = g >> 1, ctr = (b lo, b hi, 0, 0), key = (seed lo, seed hi)
extern "C" void orc_philox_normal(uint64_t seed, uint64_t counter, uint64_t n, double* out) {
  const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  for (uint64_t i = 0; i < n; i++) {
    uint64_t g = counter + i, b = g >> 1;
    uint32_t ctr[4] = {(uint32_t)b, (uint32_t)(b >> 32), 0u, 0u};
    double ze, zo; orc_block_normals(ctr, key, &ze, &zo);
    out[i] = (g & 1) ? zo : ze;
  }
}
