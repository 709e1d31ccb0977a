"""Pins of the chi^2 oracle (oracle/oracle_chi2.cpp; eq. 1)."""
import itertools

import numpy as np

import hepf_synth as hs
import oracle


def _m(e, x, y, z):
    return np.sqrt(np.maximum(e * e - x * x - y * y - z * z, 0.0))


def test_neutrino_pz_against_a_dense_scan_of_the_w_mass_constraint():
    rng = np.random.default_rng(0)
    n2 = n1 = 0
    for _ in range(300):
        l3 = rng.normal(size=3) * 40; lep = np.array([*l3, np.linalg.norm(l3)])
        nux, nuy = rng.normal(size=2) * rng.choice([20, 60, 150])
        sol = oracle.nu_pz(lep, nux, nuy, 80.4)
        pz = np.linspace(-4000, 4000, 800001)
        mw = _m(lep[3] + np.sqrt(nux**2 + nuy**2 + pz**2), lep[0] + nux, lep[1] + nuy, lep[2] + pz)
        g = mw - 80.4
        crossings = pz[:-1][np.sign(g[:-1]) != np.sign(g[1:])]
        if len(sol) == 2:
            n2 += 1
            assert sol[0] <= sol[1]
            for s in sol:      # each solution satisfies the constraint ...
                assert abs(_m(lep[3] + np.sqrt(nux**2 + nuy**2 + s**2), lep[0] + nux, lep[1] + nuy, lep[2] + s) - 80.4) < 1e-7
            inside = [c for c in crossings]          # ... and the scan sees exactly these crossings (if inside its range)
            assert len(inside) == sum(abs(s) < 3999 for s in sol)
            for c in inside:
                assert min(abs(c - s) for s in sol) < 0.05
        else:
            n1 += 1
            assert len(crossings) == 0               # no real solution: m(l nu) > m_W everywhere
            assert abs(pz[np.argmin(g)] - sol[0]) < 0.05   # the real part is where m(l nu) comes closest to m_W
    assert n2 > 100 and n1 > 20


def test_truth_recovery_in_closure_mode():
    st = hs.generate(3000, 5, semilep=True, closure=True)
    o, second = oracle.chi2_semilep(st, np.arange(st.n_events))
    assert (o["status"] == 1).all()
    assert o["chi2"].max() < 1e-12
    t = st.truth
    assert (o["jet_b_lep"] == t[:, 6]).all() and (o["jet_b_had"] == t[:, 7]).all()
    q = np.sort(t[:, 8:10], axis=1)
    assert (o["jet_q1"] == q[:, 0]).all() and (o["jet_q2"] == q[:, 1]).all()
    assert np.allclose(o["nu_pz"], t[:, 2], rtol=1e-7, atol=1e-6)
    for f, m in (("m_top_lep", 172.5), ("m_top_had", 172.5), ("m_w_lep", 80.4), ("m_w_had", 80.4)):
        assert np.abs(o[f] - m).max() < 1e-7
    assert (second > 1e-3).mean() > 0.95     # the other combinations and the other p_z solution are clearly worse


def test_brute_force_enumeration_in_numpy():
    st = hs.generate(400, 6, semilep=True)
    o, second = oracle.chi2_semilep(st, np.arange(st.n_events))
    S = st.stride
    for e in range(st.n_events):
        f = int(st.flags[e]); nj = min(8, (f >> 8) & 15)
        bt = [s for s in range(nj) if (f >> (16 + s)) & 1][:4]; lt = [s for s in range(nj) if not (f >> (16 + s)) & 1][:4]
        if (f & 15) != 1 or len(bt) < 2 or len(lt) < 2:
            assert o["status"][e] == 2; continue
        lep = np.array([st.col("lep_px")[e], st.col("lep_py")[e], st.col("lep_pz")[e], st.col("lep_e")[e]])
        jets = [np.array([st.col(c, s)[e] for c in ("jet_px", "jet_py", "jet_pz", "jet_e")]) for s in range(nj)]
        nux, nuy = st.col("met_x")[e], st.col("met_y")[e]
        best = (np.inf, None); count = 0
        for i, j in itertools.permutations(range(len(bt)), 2):
            for a, b in itertools.combinations(range(len(lt)), 2):
                wh = jets[lt[a]] + jets[lt[b]]; th = wh + jets[bt[j]]
                for s, pz in enumerate(oracle.nu_pz(lep, nux, nuy)):
                    nu = np.array([nux, nuy, pz, np.sqrt(nux**2 + nuy**2 + pz**2)])
                    wl = lep + nu; tl = wl + jets[bt[i]]
                    mm = lambda v: float(_m(v[3], v[0], v[1], v[2]))
                    c2 = ((mm(tl) - 172.5) / 11.5) ** 2 + ((mm(wl) - 80.4) / 7.5) ** 2 + ((mm(th) - 172.5) / 11.5) ** 2 + ((mm(wh) - 80.4) / 7.5) ** 2
                    count += 1
                    if c2 < best[0]: best = (c2, (bt[i], bt[j], lt[a], lt[b], s))
        assert o["n_comb"][e] == count
        assert abs(o["chi2"][e] - best[0]) <= 1e-10 * max(1.0, best[0])
        if second[e] - o["chi2"][e] > 1e-9 * max(1.0, best[0]):
            assert (o["jet_b_lep"][e], o["jet_b_had"][e], o["jet_q1"][e], o["jet_q2"][e], o["solution"][e]) == best[1]


def test_status_bits_and_rotation_invariance():
    st = hs.generate(500, 7, semilep=True)
    o, _ = oracle.chi2_semilep(st, np.arange(st.n_events))
    dil = hs.generate(50, 7)                                   # two leptons: not applicable
    od, _ = oracle.chi2_semilep(dil, np.arange(50))
    assert (od["status"] == 2).all() and np.isnan(od["chi2"]).all() and (od["jet_b_lep"] == -1).all()
    # rotate everything about z: chi2 and indices unchanged
    th = 0.7; c, s = np.cos(th), np.sin(th)
    r = hs.EventStore(st.n_events, st.stride, st.event_base, st.cols.copy(), st.flags.copy())
    for px, py, n in (("lep_px", "lep_py", 2), ("jet_px", "jet_py", 8), ("met_x", "met_y", 1)):
        X = st.cols[hs.ROW[px]:hs.ROW[px] + n].copy(); Y = st.cols[hs.ROW[py]:hs.ROW[py] + n].copy()
        r.cols[hs.ROW[px]:hs.ROW[px] + n] = c * X - s * Y; r.cols[hs.ROW[py]:hs.ROW[py] + n] = s * X + c * Y
    orr, _ = oracle.chi2_semilep(r, np.arange(st.n_events))
    assert np.allclose(orr["chi2"], o["chi2"], rtol=1e-9, atol=1e-12)
    same = orr["jet_b_lep"] == o["jet_b_lep"]
    assert same.mean() > 0.99


# ------------------------------------------------------------------------------------- single-top variants
def test_single_top_truth_recovery_and_ordering_against_the_ttbar_chi2():
    """Closure sample (semileptonic ttbar, no widths, no smearing): the leptonic top alone (t-channel terms) is exact for the true
    b-jet and neutrino p_z; Wt's three terms vanish for the true leptonic top + hadronic W; and dropping non-negative terms
    can only lower the minimum: chi2(t-channel) <= chi2(ttbar), chi2(Wt) <= chi2(ttbar)."""
    st = hs.generate(3000, 5, semilep=True, closure=True)
    idx = np.arange(st.n_events)
    t = st.truth
    o1, s1 = oracle.chi2_single_top(st, idx, 1)
    assert (o1["status"] == 1).all() and o1["chi2"].max() < 1e-12
    assert (o1["jet_b_lep"] == t[:, 6]).all() and np.allclose(o1["nu_pz"], t[:, 2], rtol=1e-7, atol=1e-6)
    assert (o1["jet_b_had"] == -1).all() and (o1["jet_q1"] == -1).all() and np.isnan(o1["m_top_had"]).all() and np.isnan(o1["m_w_had"]).all()
    o2, s2 = oracle.chi2_single_top(st, idx, 2)
    assert (o2["status"] == 1).all() and o2["chi2"].max() < 1e-12
    q = np.sort(t[:, 8:10], axis=1)
    assert (o2["jet_q1"] == q[:, 0]).all() and (o2["jet_q2"] == q[:, 1]).all()
    # here BOTH hypotheses are exact (the event has two tops): whichever rounding makes smaller wins, with its own true b-jet
    lep_top = o2["jet_b_lep"] >= 0
    assert (o2["jet_b_lep"][lep_top] == t[lep_top, 6]).all() and np.isnan(o2["m_top_had"][lep_top]).all()
    assert (o2["jet_b_had"][~lep_top] == t[~lep_top, 7]).all() and np.isnan(o2["m_top_lep"][~lep_top]).all()
    assert ((o2["jet_b_lep"] >= 0) ^ (o2["jet_b_had"] >= 0)).all()
    # not in closure: ordering of the minima
    st2 = hs.generate(4000, 8, semilep=True)
    idx2 = np.arange(st2.n_events)
    full, _ = oracle.chi2_semilep(st2, idx2)
    a, _ = oracle.chi2_single_top(st2, idx2, 1); b, _ = oracle.chi2_single_top(st2, idx2, 2)
    ok = full["status"] == 1
    assert ok.sum() > 3000 and (a["chi2"][ok] <= full["chi2"][ok] * (1 + 1e-12)).all() and (b["chi2"][ok] <= full["chi2"][ok] * (1 + 1e-12)).all()
    assert (b["jet_b_had"][ok] >= 0).sum() > 100 and (b["jet_b_lep"][ok] >= 0).sum() > 100         # both Wt hypotheses occur


def test_single_top_brute_force_enumeration_in_numpy():
    st = hs.generate(300, 16, semilep=True)
    # make some events single-b / few-jet so that the applicability rules are exercised
    st.flags[:60] &= ~np.uint32(0x00020000)
    for mode in (1, 2):
        o, second = oracle.chi2_single_top(st, np.arange(st.n_events), mode)
        for e in range(st.n_events):
            f = int(st.flags[e]); nj = min(8, (f >> 8) & 15)
            bt = [s for s in range(nj) if (f >> (16 + s)) & 1][:4]; lt = [s for s in range(nj) if not (f >> (16 + s)) & 1][:4]
            if (f & 15) != 1 or len(bt) < 1 or (mode == 2 and len(lt) < 2):
                assert o["status"][e] == 2 and np.isnan(o["chi2"][e]); continue
            lep = np.array([st.col("lep_px")[e], st.col("lep_py")[e], st.col("lep_pz")[e], st.col("lep_e")[e]])
            jets = [np.array([st.col(c, s)[e] for c in ("jet_px", "jet_py", "jet_pz", "jet_e")]) for s in range(nj)]
            nux, nuy = st.col("met_x")[e], st.col("met_y")[e]
            mm = lambda v: float(_m(v[3], v[0], v[1], v[2]))
            cands = []
            for s, pz in enumerate(oracle.nu_pz(lep, nux, nuy)):
                nu = np.array([nux, nuy, pz, np.sqrt(nux**2 + nuy**2 + pz**2)]); wl = lep + nu
                for i in bt:
                    tl = ((mm(wl + jets[i]) - 172.5) / 11.5) ** 2; w = ((mm(wl) - 80.4) / 7.5) ** 2
                    if mode == 1:
                        cands.append((tl + w, (0, i, -1, -1, s)))
                    else:
                        for a, b in itertools.combinations(lt, 2):
                            wh = jets[a] + jets[b]; w2 = ((mm(wh) - 80.4) / 7.5) ** 2
                            cands.append((tl + w + w2, (0, i, a, b, s)))
                            cands.append((((mm(wh + jets[i]) - 172.5) / 11.5) ** 2 + w + w2, (1, i, a, b, s)))
            assert o["n_comb"][e] == len(cands)
            best = min(c[0] for c in cands)
            assert abs(o["chi2"][e] - best) <= 1e-10 * max(1.0, best)
            if second[e] - o["chi2"][e] > 1e-9 * max(1.0, best):
                hyp, i, a, b, s = min(cands, key=lambda c: c[0])[1]
                got = (0 if o["jet_b_lep"][e] >= 0 else 1, max(o["jet_b_lep"][e], o["jet_b_had"][e]), o["jet_q1"][e], o["jet_q2"][e], o["solution"][e])
                assert got == (hyp, i, a, b, s)
