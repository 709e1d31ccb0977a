"""Pins of the histogram oracle (oracle/oracle_hist.cpp): hand-built edge cases (the definition's boundary rules), a
numpy restatement on values kept away from the bin edges, and conservation of the solved-record count."""
import numpy as np

import oracle


def _records(values, field="m_higgs", status=None):
    b = np.zeros(len(values), dtype=oracle.BEST_DTYPE)
    b[field] = values
    b["status"] = 1 if status is None else status
    return b


def test_edges_underflow_overflow_nan_and_unsolved():
    lo, hi, nb = 100.0, 150.0, 10          # bin width 5
    vals = [100.0, 104.999, 105.0, 149.999, 150.0, 99.999, 1e9, -1e9, np.nan, 125.0]
    h = oracle.histogram(_records(vals), "m_higgs", lo, hi, nb)
    want = np.zeros(nb + 2, dtype=np.uint64)
    want[1] += 2          # 100.0 (lower edge belongs to bin 0), 104.999
    want[2] += 1          # 105.0 starts bin 1
    want[10] += 1         # 149.999 -> last bin
    want[11] += 2         # 150.0 (upper edge is overflow), 1e9
    want[0] += 2          # 99.999, -1e9
    want[6] += 1          # 125.0 -> (25 * 0.2) = 5 -> bin 5
    assert np.array_equal(h, want)         # the NaN is counted nowhere
    st = np.array([1, 0, 1, 2, 3, 0, 1, 1, 1, 4], dtype=np.uint32)   # only odd status (bit 0) is filled
    h2 = oracle.histogram(_records(vals, status=st), "m_higgs", lo, hi, nb)
    filled = [v for v, s in zip(vals, st) if (s & 1) and v == v]
    assert int(h2.sum()) == len(filled)


def test_numpy_restatement_away_from_edges_and_every_field():
    rng = np.random.default_rng(5)
    n, nb, lo, hi = 20000, 64, -3.0, 9.0
    w = (hi - lo) / nb
    centres = lo + (rng.integers(-5, nb + 5, n) + rng.uniform(0.1, 0.9, n)) * w    # never within 0.1 bin of an edge
    for field in ("m_top", "m_antitop", "m_wplus", "m_wminus", "m_higgs", "loglik"):
        h = oracle.histogram(_records(centres, field), field, lo, hi, nb)
        inside, _ = np.histogram(centres, bins=nb, range=(lo, hi))
        assert np.array_equal(h[1:-1], inside.astype(np.uint64))
        assert h[0] == (centres < lo).sum() and h[-1] == (centres >= hi).sum() and h.sum() == n
    # derived fields: pT = sqrt(px^2 + py^2); variation as a number
    b = np.zeros(n, dtype=oracle.BEST_DTYPE); b["status"] = 1
    ang = rng.uniform(0, 2 * np.pi, n); pt = np.abs(centres) + 0.05
    b["nu"][:, 0] = pt * np.cos(ang); b["nu"][:, 1] = pt * np.sin(ang); b["nu"][:, 2] = rng.normal(size=n) * 50
    b["nubar"][:, 0] = 2 * b["nu"][:, 0]; b["nubar"][:, 1] = 2 * b["nu"][:, 1]
    b["variation"] = rng.integers(0, 64, n)
    got = oracle.histogram(b, "nu_pt", 0.0, 12.0, 48)
    ref = np.sqrt(b["nu"][:, 0] * b["nu"][:, 0] + b["nu"][:, 1] * b["nu"][:, 1])
    t = (ref - 0.0) * (48 / 12.0)
    want = np.bincount(np.where(t >= 48, 49, 1 + np.floor(t).astype(int)), minlength=50).astype(np.uint64)
    assert np.array_equal(got, want)
    assert np.array_equal(oracle.histogram(b, "nubar_pt", 0.0, 24.0, 48), want)
    hv = oracle.histogram(b, "variation", 0.0, 64.0, 64)
    assert np.array_equal(hv[1:-1], np.bincount(b["variation"], minlength=64).astype(np.uint64)) and hv[0] == 0 and hv[-1] == 0
