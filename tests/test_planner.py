"""-m "not gpu": the host logic of the cut-level scheduler analogue: hepf_plan_chain
against a brute force over every assignment of cuts to phases, the oracle's per-cut statistics against single-cut selections."""
import itertools

import numpy as np
import pytest

import hepf_synth as hs
import oracle

GROUP = {hs.LEP_PT_GT: {"lep_pt"}, hs.LEP_ABSETA_LT: {"lep_eta"}, hs.NJET_GE: {"jet_pt", "jet_eta"}, hs.NBJET_GE: {"jet_pt", "jet_eta"},
         hs.MET_GT: {"met"}, hs.MLL_GT: {"mll"}, hs.MLL_OUTSIDE: {"mll"}, hs.NLEP_EQ: set(), hs.LEP_OS: set()}
SIZE = {"lep_pt": 16, "lep_eta": 16, "jet_pt": 64, "jet_eta": 64, "met": 8, "mll": 8}


def _bytes(cuts):
    g = set().union(*[GROUP[c[0]] for c in cuts]) if cuts else set()
    return sum(SIZE[x] for x in g)


def _brute(chain, p, dep):
    """min over ALL dependency-respecting assignments of cuts to two phases of the cost model stated in include/hepf.h."""
    n = len(chain)
    one = 4 + _bytes(chain)
    best = one
    for mask in range(1, (1 << n) - 1):
        s1 = [c for c in range(n) if mask >> c & 1]
        if dep is not None and any((int(dep[c]) & ~mask & 0xffffffff) for c in s1):
            continue
        fam = {}
        for c in s1:
            key = frozenset(GROUP[chain[c][0]])
            fam[key] = min(fam.get(key, 1.0), p[c])          # cuts on the same columns: one family, its smallest pass fraction
        p1 = float(np.prod(list(fam.values())))
        cost = 4 + _bytes([chain[c] for c in s1]) + (1 - (1 - p1) ** 8) * (4 + _bytes([chain[c] for c in range(n) if not mask >> c & 1])) / 0.55 + 8 * p1
        best = min(best, cost)
    return (best if best < 0.9 * one else one), one


@pytest.fixture(scope="module")
def hepf():
    from paper_2211_14346_b200 import build as b
    b.build()
    import paper_2211_14346_b200 as h
    h.load()
    return h


def test_plan_is_the_brute_force_optimum_of_the_stated_cost_model(hepf):
    rng = np.random.default_rng(11)
    kinds = [(hs.NLEP_EQ, 2, 0, 0), (hs.LEP_OS, 0, 0, 0), (hs.LEP_PT_GT, 0, 30.0, 0), (hs.LEP_ABSETA_LT, 0, 0, 2.5), (hs.NJET_GE, 4, 35.0, 2.5),
             (hs.NBJET_GE, 4, 35.0, 2.5), (hs.MET_GT, 0, 55.0, 0), (hs.MLL_GT, 0, 40.0, 0), (hs.MLL_OUTSIDE, 0, 80.0, 100.0)]
    for trial in range(300):
        n = int(rng.integers(1, 9))
        chain = [kinds[i] for i in rng.integers(0, len(kinds), n)]
        p = rng.uniform(0.02, 1.0, n) ** (2 if trial % 2 else 1)
        dep = None
        if trial % 3 == 0:      # random precedence constraints: cut c after some earlier cuts
            dep = np.array([int(rng.integers(0, 1 << c)) if c and rng.random() < 0.5 else 0 for c in range(n)], dtype=np.uint32)
        order, split, planned, one = hepf.plan_chain(chain, p, dep)
        want, one_w = _brute(chain, p, dep)
        assert sorted(order) == list(range(n)) and 0 < split <= n or n == 0
        assert abs(one - one_w) < 1e-12 and abs(planned - want) <= 1e-9 * want, (chain, p, dep, order, split, planned, want)
        # the order keeps the user's order inside each phase, and no cut runs in an earlier phase than a prerequisite
        assert order[:split] == sorted(order[:split]) and order[split:] == sorted(order[split:])
        if dep is not None and split < n:
            s1 = set(order[:split])
            assert all(not (int(dep[c]) >> k & 1) or k in s1 for c in s1 for k in range(n))


def test_plan_for_the_tightened_chain_of_config_4(hepf):
    """BASELINE.json configs[3]: with the measured filter ratios the two jet-count cuts (128 of the 180 bytes) move to phase 2."""
    cfg = hs.CONFIGS[4]
    st = cfg.events(300_000)
    stats = oracle.cut_stats(st, cfg.cuts, 4)
    p = stats[:-1] / stats[-1]
    order, split, planned, one = hepf.plan_chain(cfg.cuts, p)
    assert one == 4 + 16 + 16 + 64 + 64 + 8 + 8
    want, _ = _brute(cfg.cuts, p, None)
    assert abs(planned - want) <= 1e-9 * want
    # measured on B200 (profiles/r02e): at cfg4's filter ratios the cheap cuts pass 13-16 % of the events, most 64-byte atoms of
    # the jet columns still hold a survivor, and the gather loses to the 94 %-of-bandwidth stream: the plan is ONE phase
    assert split == 8 and order == list(range(8)) and planned == one
    # with a lepton-pT cut that passes 2 % the same chain is split: jets (128 of 180 bytes) are fetched for the survivors only
    p_tight = p.copy(); p_tight[2] = 0.02
    order_t, split_t, planned_t, _ = hepf.plan_chain(cfg.cuts, p_tight)
    assert split_t < 8 and {4, 5} <= set(order_t[split_t:]) and 2 in order_t[:split_t] and planned_t < 0.6 * one
    order, split, planned = order_t, split_t, planned_t
    p = p_tight
    # a dependency "the MET cut needs the jet-count cut" keeps MET out of phase 1
    dep = np.zeros(8, dtype=np.uint32); dep[6] = 1 << 4
    order2, split2, planned2, _ = hepf.plan_chain(cfg.cuts, p, dep)
    assert 6 in order2[split2:] and planned2 >= planned
    # nothing to gain: a chain whose cuts all read the same columns stays one phase
    o3, s3, b3, one3 = hepf.plan_chain([(hs.NJET_GE, 4, 35.0, 2.5), (hs.NBJET_GE, 2, 35.0, 2.5)], [0.3, 0.3])
    assert s3 == 2 and b3 == one3


def test_oracle_cut_stats_are_single_cut_selections_of_the_sample():
    st = hs.generate(20_000, 5, bkg_frac=0.4, with_truth=False)
    chain = hs.CHAIN_TIGHT8 + [(hs.MLL_OUTSIDE, 0, 80.0, 100.0)]
    for every in (1, 3, 50):
        stats = oracle.cut_stats(st, chain, every)
        in_sample = (np.arange(st.n_events) // 512) % every == 0
        assert stats[-1] == in_sample.sum()
        for c, cut in enumerate(chain):
            idx, _ = oracle.select(st, [cut])
            assert stats[c] == in_sample[idx].sum()
    assert list(oracle.cut_stats(st, [], 1)) == [st.n_events]
