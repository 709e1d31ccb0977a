"""Pins for oracle O3 (cut chain + surviving indices + cutflow).  PAPER.md:96-102, :286-295 (strict cuts)."""
import numpy as np

import hepf_synth as hs
import oracle
from hepf_synth import (INF, LEP_ABSETA_LT, LEP_OS, LEP_PT_GT, MET_GT, MLL_GT, MLL_OUTSIDE, NBJET_GE, NJET_GE,
                        NLEP_EQ, ROW)


def blank(n):
    stride = n + (n & 1)
    return hs.EventStore(n, max(stride, 2), 0, np.zeros((hs.NROW, max(stride, 2))), np.zeros(max(stride, 2), np.uint32))


def flags(n_lep=2, q0=1, q1=0, n_jet=4, tags=0b1111):
    return n_lep | (q0 << 4) | (q1 << 5) | (n_jet << 8) | (tags << 16)


def run(st, chain):
    idx, cf = oracle.select(st, chain)
    return list(idx), list(cf)


def test_each_kind_at_threshold_fails_and_just_above_passes():
    up = np.nextafter
    # (chain, column writes for event 0 (at threshold -> fail), event 1 (just inside -> pass))
    st = blank(2)
    st.flags[:2] = flags()
    # MET_GT 30: 30 fails, nextafter passes ("met <= 30000 -> fail")
    st.cols[ROW["met"], :2] = [30.0, up(30.0, INF)]
    assert run(st, [(MET_GT, 0, 30.0, 0)]) == ([1], [1])
    st.cols[ROW["mll"], :2] = [40.0, up(40.0, INF)]
    assert run(st, [(MLL_GT, 0, 40.0, 0)]) == ([1], [1])
    # LEP_PT_GT needs BOTH leptons above
    st.cols[ROW["lep_pt"], :2] = [25.0, 26.0]; st.cols[ROW["lep_pt"] + 1, :2] = [80.0, up(25.0, INF)]
    assert run(st, [(LEP_PT_GT, 0, 25.0, 0)]) == ([1], [1])
    st.cols[ROW["lep_pt"], :2] = [80.0, 80.0]; st.cols[ROW["lep_pt"] + 1, :2] = [25.0, 80.0]
    assert run(st, [(LEP_PT_GT, 0, 25.0, 0)]) == ([1], [1])
    # LEP_ABSETA_LT 2.5: |eta| = 2.5 fails, negative eta handled by abs
    st.cols[ROW["lep_eta"], :2] = [-2.5, -up(2.5, 0)]; st.cols[ROW["lep_eta"] + 1, :2] = [0.1, 2.4]
    assert run(st, [(LEP_ABSETA_LT, 0, 0, 2.5)]) == ([1], [1])
    # MLL_OUTSIDE (80, 100): 80 and 100 fail, just outside passes
    st3 = blank(4); st3.flags[:4] = flags()
    st3.cols[ROW["mll"], :4] = [80.0, 100.0, up(80.0, 0), up(100.0, INF)]
    assert run(st3, [(MLL_OUTSIDE, 0, 80.0, 100.0)]) == ([2, 3], [2])


def test_lepton_count_and_charge():
    st = blank(5)
    st.flags[:5] = [flags(n_lep=1), flags(n_lep=2, q0=1, q1=1), flags(n_lep=2, q0=0, q1=0), flags(n_lep=3),
                    flags(n_lep=2, q0=0, q1=1)]
    assert run(st, [(NLEP_EQ, 2, 0, 0)]) == ([1, 2, 4], [3])
    assert run(st, [(LEP_OS, 0, 0, 0)])[0] == [0, 3, 4]
    assert run(st, [(NLEP_EQ, 2, 0, 0), (LEP_OS, 0, 0, 0)]) == ([4], [3, 1])


def test_jet_counts_respect_n_jet_threshold_eta_and_tag():
    st = blank(6)
    pt, eta = ROW["jet_pt"], ROW["jet_eta"]
    for s in range(8):
        st.cols[pt + s, :6] = 50.0
    # ev0: 4 jets above -> pass NJET_GE 4
    st.flags[0] = flags(n_jet=4)
    # ev1: 8 good slots stored but n_jet = 3 -> only three counted -> fail
    st.flags[1] = flags(n_jet=3)
    # ev2: 4 jets, one exactly at threshold -> fail
    st.flags[2] = flags(n_jet=4); st.cols[pt + 2, 2] = 25.0
    # ev3: 5 jets, one at |eta| = 2.5 (fails eta), four inside -> pass
    st.flags[3] = flags(n_jet=5); st.cols[eta + 1, 3] = -2.5
    # ev4: 4 jets, only three tagged
    st.flags[4] = flags(n_jet=4, tags=0b0111)
    # ev5: 6 jets, tagged slots 0,2,4,5
    st.flags[5] = flags(n_jet=6, tags=0b110101)
    assert run(st, [(NJET_GE, 4, 25.0, 2.5)])[0] == [0, 3, 4, 5]
    assert run(st, [(NBJET_GE, 4, 25.0, 2.5)])[0] == [0, 5]
    assert run(st, [(NBJET_GE, 4, 25.0, INF)])[0] == [0, 3, 5]
    # tag bit of a slot >= n_jet must not count
    st.flags[4] = flags(n_jet=3, tags=0b1111)
    assert 4 not in run(st, [(NBJET_GE, 4, 25.0, INF)])[0]


def test_nan_fails_every_comparison_cut():
    st = blank(2); st.flags[:2] = flags()
    for name in ("met", "mll"):
        st.cols[ROW[name], :2] = [np.nan, 100.0]
    st.cols[ROW["lep_pt"], :2] = [np.nan, 50]; st.cols[ROW["lep_pt"] + 1, :2] = 50
    assert run(st, [(MET_GT, 0, 30, 0)])[0] == [1]
    assert run(st, [(MLL_OUTSIDE, 0, 80, 100)])[0] == []
    st.cols[ROW["mll"], 0] = np.nan; st.cols[ROW["mll"], 1] = 120
    assert run(st, [(MLL_OUTSIDE, 0, 80, 100)])[0] == [1]
    assert run(st, [(LEP_PT_GT, 0, 25, 0)])[0] == [1]


def test_empty_chain_and_empty_store():
    st = blank(3)
    assert run(st, []) == ([0, 1, 2], [])
    st0 = blank(0)
    st0.n_events = 0
    assert run(st0, hs.CHAIN_BASE)[0] == []


def _numpy_chain(st, chain):
    n = st.n_events
    f = st.flags[:n]
    nj = np.minimum((f >> 8) & 15, 8)
    alive = np.ones(n, bool); flow = []
    for kind, cn, lo, hi in chain:
        if kind == NLEP_EQ: ok = (f & 15) == cn
        elif kind == LEP_OS: ok = ((f >> 4) & 1) != ((f >> 5) & 1)
        elif kind == LEP_PT_GT: ok = (st.col("lep_pt", 0) > lo) & (st.col("lep_pt", 1) > lo)
        elif kind == LEP_ABSETA_LT: ok = (abs(st.col("lep_eta", 0)) < hi) & (abs(st.col("lep_eta", 1)) < hi)
        elif kind in (NJET_GE, NBJET_GE):
            cnt = np.zeros(n, int)
            for s in range(8):
                g = (s < nj) & (st.col("jet_pt", s) > lo) & (abs(st.col("jet_eta", s)) < hi)
                if kind == NBJET_GE: g &= ((f >> (16 + s)) & 1) == 1
                cnt += g
            ok = cnt >= cn
        elif kind == MET_GT: ok = st.col("met") > lo
        elif kind == MLL_GT: ok = st.col("mll") > lo
        alive &= ok; flow.append(int(alive.sum()))
    return np.nonzero(alive)[0], flow


def test_generated_sample_invariants_and_vectorised_restatement():
    for cfg, n in ((hs.CONFIGS[1], 10_000), (hs.CONFIGS[4], 200_000)):
        st = cfg.events(n)
        idx, cf = oracle.select(st, cfg.cuts)
        assert (np.diff(idx.astype(np.int64)) > 0).all()                 # ascending, unique
        assert all(a >= b for a, b in zip([n] + list(cf), cf))           # cutflow non-increasing
        assert cf[-1] == len(idx)
        ref_idx, ref_cf = _numpy_chain(st, cfg.cuts)
        assert np.array_equal(idx, ref_idx) and list(cf) == ref_cf
        # prefix property: the chain truncated after c cuts has cutflow[:c]
        for c in range(1, len(cfg.cuts)):
            assert list(oracle.select(st, cfg.cuts[:c])[1]) == list(cf[:c])


def test_cfg4_chain_passes_about_five_percent():
    cfg = hs.CONFIGS[4]
    st = cfg.events(400_000)
    idx, _ = oracle.select(st, cfg.cuts)
    frac = len(idx) / st.n_events
    assert 0.035 < frac < 0.065, frac
