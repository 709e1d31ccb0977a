"""Pins for oracle O1/O2 (Philox4x32-10, uniforms, deterministic log/sincos, normal stream).

None of these re-types the oracle's formulae: they use printed known answers (tests/golden), an independent
big-integer restatement of the Philox round, libm, and statistical/structural invariants.
"""
import math
import os

import numpy as np

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _lines(name):
    with open(os.path.join(GOLD, name)) as f:
        return [ln.strip() for ln in f if ln.strip() and not ln.startswith("#")]


def test_philox_known_answer_vectors():
    for ln in _lines("philox_kat.txt"):
        lhs, out = ln.split("->")
        ctr, key = lhs.split("|")
        ctr = [int(x, 16) for x in ctr.split()]
        key = [int(x, 16) for x in key.split()]
        out = [int(x, 16) for x in out.split()]
        assert oracle.philox4x32_10(ctr, key) == out


def test_philox_is_a_bijection_of_the_counter_and_depends_on_every_word():
    base = oracle.philox4x32_10([1, 2, 3, 4], [5, 6])
    seen = {tuple(base)}
    for w in range(4):
        c = [1, 2, 3, 4]; c[w] ^= 1
        o = tuple(oracle.philox4x32_10(c, [5, 6]))
        assert o not in seen; seen.add(o)
    for w in range(2):
        k = [5, 6]; k[w] ^= 1
        o = tuple(oracle.philox4x32_10([1, 2, 3, 4], k))
        assert o not in seen; seen.add(o)


def test_philox_single_round_structure_by_inverse():
    """Philox rounds are invertible: undo ten rounds with modular inverses of the multipliers (an
    independent statement of the round function) and recover the counter."""
    M0, M1, W0, W1 = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85
    inv0, inv1 = pow(M0, -1, 1 << 32), pow(M1, -1, 1 << 32)
    ctr, key = [0xdeadbeef, 0x12345678, 0x0badf00d, 0xcafef00d], [0x11111111, 0x22222222]
    out = oracle.philox4x32_10(ctr, key)
    c = list(out)
    for r in reversed(range(10)):
        k0, k1 = (key[0] + r * W0) & 0xffffffff, (key[1] + r * W1) & 0xffffffff
        # forward: n0 = hi1^c1^k0, n1 = lo1, n2 = hi0^c3^k1, n3 = lo0
        lo1, lo0 = c[1], c[3]
        c2 = (lo1 * inv1) & 0xffffffff; c0 = (lo0 * inv0) & 0xffffffff
        hi1 = (M1 * c2) >> 32; hi0 = (M0 * c0) >> 32
        c1 = c[0] ^ hi1 ^ k0; c3 = c[2] ^ hi0 ^ k1
        c = [c0, c1, c2, c3]
    assert c == ctr


def test_first_six_normals_bit_exact():
    want = [float.fromhex(x) for x in _lines("normals_seed7.txt")]
    got = oracle.philox_normal(7, 0, 6)
    assert [float(x).hex() for x in got] == [w.hex() for w in want]


def test_slice_consistency():
    whole = oracle.philox_normal(7, 0, 4099)
    parts = np.concatenate([oracle.philox_normal(7, 0, 1), oracle.philox_normal(7, 1, 1000),
                            oracle.philox_normal(7, 1001, 3098)])
    assert whole.tobytes() == parts.tobytes()
    # a stream far out (counter beyond 2^33: second counter word in use) is still slice-consistent
    big = (1 << 35) + 3
    a = oracle.philox_normal(9, big, 64)
    b = np.concatenate([oracle.philox_normal(9, big, 31), oracle.philox_normal(9, big + 31, 33)])
    assert a.tobytes() == b.tobytes()
    assert oracle.philox_normal(9, big, 8).tobytes() != oracle.philox_normal(9, 3, 8).tobytes()


def test_moments_of_prefix():
    n = 1 << 20
    z = oracle.philox_normal(7, 0, n)
    assert np.isfinite(z).all()
    # 5 sigma bands: mean ~ N(0,1/n); var ~ N(1, 2/n); kurtosis ~ N(3, 96/n); skew ~ N(0, 6/n)
    assert abs(z.mean()) < 5 / math.sqrt(n)
    assert abs(z.var() - 1) < 5 * math.sqrt(2 / n)
    zs = (z - z.mean()) / z.std()
    assert abs((zs ** 4).mean() - 3) < 5 * math.sqrt(96 / n)
    assert abs((zs ** 3).mean()) < 5 * math.sqrt(6 / n)
    # even / odd members (cos / sin branch) are uncorrelated and each standard normal
    assert abs(np.corrcoef(z[0::2], z[1::2])[0, 1]) < 5 / math.sqrt(n / 2)
    assert abs(z[0::2].var() - 1) < 5 * math.sqrt(4 / n) and abs(z[1::2].var() - 1) < 5 * math.sqrt(4 / n)
    # tail mass beyond 3 sigma: 2.6998e-3
    assert abs((np.abs(z) > 3).mean() - 2.6998e-3) < 5 * math.sqrt(2.7e-3 / n)


def test_det_log_against_libm():
    rng = np.random.default_rng(11)
    us = np.concatenate([rng.random(20000), 2.0 ** -rng.integers(1, 53, 2000) * (1 + rng.random(2000)) / 2,
                         [1.0, 0.5, 2 ** -53, 1 - 2 ** -53, math.sqrt(0.5), 0.7071067811865476, 0.7071067811865475]])
    us = us[(us > 0) & (us <= 1)]
    worst = 0.0
    for u in us:
        got, ref = oracle.det_log(float(u)), math.log(float(u))
        if ref == 0.0:
            assert got == 0.0
            continue
        worst = max(worst, abs(got - ref) / abs(ref))
    assert worst < 4 * 2.0 ** -52, worst


def test_det_sincos_against_libm():
    rng = np.random.default_rng(12)
    us = np.concatenate([rng.random(20000), np.arange(0, 8) / 8.0, np.arange(0, 8) / 8.0 + 2.0 ** -53,
                         [1 - 2.0 ** -53, 0.125 - 2.0 ** -56, 0.375, 0.875 + 2.0 ** -53]])
    worst = 0.0
    for u in us:
        s, c = oracle.det_sincos2pi(float(u))
        # libm of 2*pi*u carries the rounding of the argument: compare against sin/cos of the exactly
        # reduced argument r*(pi/2), r = 4u - round(4u) (exact in binary), rotated by the quadrant
        t = 4.0 * float(u); n = math.floor(t + 0.5); r = t - n
        sr, cr = math.sin(r * (math.pi / 2)), math.cos(r * (math.pi / 2))
        q = int(n) & 3
        rs, rc = [(sr, cr), (cr, -sr), (-sr, -cr), (-cr, sr)][q]
        worst = max(worst, abs(s - rs), abs(c - rc))
        assert abs(s * s + c * c - 1) < 1e-15
    assert worst < 4e-16, worst


def test_normals_match_textbook_box_muller_from_the_same_uniforms():
    """Z_even/Z_odd equal sqrt(-2 ln u1) (cos, sin)(2 pi u2) of the textbook transform, with u1/u2 rebuilt
    here from the raw Philox words by integer arithmetic (the mapping (w>>11 [+1]) / 2^53)."""
    for b in range(50):
        x = oracle.philox4x32_10([b, 0, 0, 0], [7, 0])
        w0, w1 = (x[1] << 32) | x[0], (x[3] << 32) | x[2]
        u1, u2 = ((w0 >> 11) + 1) / 2 ** 53, (w1 >> 11) / 2 ** 53
        assert 0 < u1 <= 1 and 0 <= u2 < 1
        rho = math.sqrt(-2 * math.log(u1))
        z = oracle.philox_normal(7, 2 * b, 2)
        assert abs(z[0] - rho * math.cos(2 * math.pi * u2)) < 1e-14 * max(1, rho)
        assert abs(z[1] - rho * math.sin(2 * math.pi * u2)) < 1e-14 * max(1, rho)
