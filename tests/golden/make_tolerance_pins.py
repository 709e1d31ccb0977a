#!/usr/bin/env python
"""Writes tests/golden/tolerance_pins.txt: 50-digit values of the DIAGNOSTICS the oracle emits next to a solution
(kappa, the p_z term sums, the tangency measure) for the worked example of tests/golden/worked_example.txt, and of a
hand-built near-tangent quartic.  mpmath at 60 digits, written from the definitions in DESIGN.md section 2 / R11
(conics, resultant, kappa = 2^-53 sum|h_i x^i| / |x P'(x)|, tangency = min over critical points of |P| / sum|g_i x^i|).
It calls neither oracle/ nor the CUDA package.   Usage: python tests/golden/make_tolerance_pins.py
"""
import os

from mpmath import mp, mpf, polyroots, sqrt

mp.dps = 60
HERE = os.path.dirname(os.path.abspath(__file__))
MT, MW = mpf("172.5"), mpf("80.4")


def v4(p, m):
    # inputs of the worked example are FP64 numbers: E = sqrt(|p|^2 + m^2) rounded to double, as the tests build them
    import math
    e = math.sqrt(sum(float(c) ** 2 for c in p) + float(m) ** 2)
    return [mpf(c) for c in p] + [mpf(e)]


def leg(l, b):
    ml2 = l[3] ** 2 - sum(c * c for c in l[:3]); mb2 = b[3] ** 2 - sum(c * c for c in b[:3])
    bl = b[3] * l[3] - sum(x * y for x, y in zip(b[:3], l[:3]))
    A = (MW ** 2 - ml2) / 2; B = (MT ** 2 - MW ** 2 - mb2) / 2 - bl
    n = [b[3] * l[i] - l[3] * b[i] for i in range(3)]; k = l[3] * B - b[3] * A
    c0, c1, c2 = k / n[2], -n[0] / n[2], -n[1] / n[2]
    d0, d1, d2 = (A + l[2] * c0) / l[3], (l[0] + l[2] * c1) / l[3], (l[1] + l[2] * c2) / l[3]
    return (d1 * d1 - 1 - c1 * c1, 2 * (d1 * d2 - c1 * c2), d2 * d2 - 1 - c2 * c2, 2 * (d0 * d1 - c0 * c1),
            2 * (d0 * d2 - c0 * c2), d0 * d0 - c0 * c0), (c0, c1, c2)


def tangency(g):          # g[0..4] ascending, any leading coefficient
    crit = [r.real for r in polyroots([4 * g[4], 3 * g[3], 2 * g[2], g[1]], maxsteps=500, extraprec=200) if abs(r.imag) < mpf(10) ** -40]
    best = mpf(1)
    for c in crit:
        val = abs(sum(g[i] * c ** i for i in range(5))) / sum(abs(g[i] * c ** i) for i in range(5))
        best = min(best, val)
    return best


def main():
    lp, b, lm, bb = v4([4, 45, -108], 0), v4([-7, -68, -42], "4.7"), v4([-64, 6, -24], 0), v4([46, -17, -76], "4.7")
    Mx, My = mpf(-10), mpf(-46)
    (a1, b1, c1, d1, e1, f1), z1 = leg(lp, b)
    (qa, qb, qc, qd, qe, qf), z2 = leg(lm, bb)
    a2, b2, c2 = qa, qb, qc
    d2 = -2 * qa * Mx - qb * My - qd; e2 = -2 * qc * My - qb * Mx - qe
    f2 = qa * Mx * Mx + qb * Mx * My + qc * My * My + qd * Mx + qe * My + qf
    p = [c1 * f2 - c2 * f1, c1 * d2 - c2 * d1, c1 * a2 - c2 * a1]
    q = [c1 * e2 - c2 * e1, c1 * b2 - c2 * b1]
    r = [e1 * f2 - e2 * f1, e1 * d2 + b1 * f2 - e2 * d1 - b2 * f1, e1 * a2 + b1 * d2 - e2 * a1 - b2 * d1, b1 * a2 - b2 * a1]
    h = [p[0] ** 2 - q[0] * r[0], 2 * p[0] * p[1] - (q[0] * r[1] + q[1] * r[0]),
         2 * p[0] * p[2] + p[1] ** 2 - (q[0] * r[2] + q[1] * r[1]), 2 * p[1] * p[2] - (q[0] * r[3] + q[1] * r[2]),
         p[2] ** 2 - q[1] * r[3]]
    roots = sorted(x.real for x in polyroots(h[::-1], maxsteps=500, extraprec=200) if abs(x.imag) < mpf(10) ** -40)
    eps = mpf(2) ** -53
    lines = ["# 50-digit diagnostics of the worked example (tests/golden/worked_example.txt) and of a hand-built near-tangent quartic.",
             "# Written by tests/golden/make_tolerance_pins.py (mpmath, 60 digits) from DESIGN.md section 2 / R11; do not edit.",
             "# per root (ascending x): kappa  pz_terms  pzbar_terms"]
    for i, x in enumerate(roots):
        y = -(p[0] + p[1] * x + p[2] * x * x) / (q[0] + q[1] * x)
        kappa = eps * sum(abs(h[k] * x ** k) for k in range(5)) / abs(x * (h[1] + 2 * h[2] * x + 3 * h[3] * x ** 2 + 4 * h[4] * x ** 3))
        sz = abs(z1[0]) + abs(z1[1] * x) + abs(z1[2] * y)
        szb = abs(z2[0]) + abs(z2[1] * (Mx - x)) + abs(z2[2] * (My - y))
        lines.append(f"r{i} {mp.nstr(kappa, 50)} {mp.nstr(sz, 50)} {mp.nstr(szb, 50)}")
    g = [c / h[4] for c in h]
    lines.append("# tangency measure of the worked example: min over critical points of |P| / sum|g_i x^i|")
    lines.append(f"tangency {mp.nstr(tangency(g), 50)}")
    # hand-built near-tangent monic quartic ((x-3)^2 - 2^-26)((x+2)^2 + 5): every coefficient is an exact double,
    # real roots exactly 3 -+ 2^-13, |P(3)| = 30 * 2^-26
    dl = mpf(2) ** -26; c = 9 - dl
    gt = [9 * c, 4 * c - 54, c - 15, mpf(-2), mpf(1)]
    lines.append("# near-tangent quartic x^4 - 2 x^3 + (c-15) x^2 + (4c-54) x + 9c, c = 9 - 2^-26: g0 g1 g2 g3 (exact doubles), roots, tangency")
    lines.append("tq_g " + " ".join(repr(float(v)) for v in gt[:4]))
    lines.append(f"tq_roots {mp.nstr(3 - mpf(2) ** -13, 50)} {mp.nstr(3 + mpf(2) ** -13, 50)}")
    lines.append(f"tq_tangency {mp.nstr(tangency(gt), 50)}")
    with open(os.path.join(HERE, "tolerance_pins.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")
    print("\n".join(lines))


if __name__ == "__main__":
    main()
