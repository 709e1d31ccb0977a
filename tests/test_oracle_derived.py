"""-m "not gpu": pins of the oracle's derived per-event variables: the recording cut of PAPER.md:278-295
(ETmis = 1.05 met), the ttH-system mass / pT of PAPER.md:410-442, and the histogram of a plain column."""
import numpy as np

import hepf_synth as hs
import oracle

REC = 10   # ORC_MET_GT_RECORD


def _tiny_store(met):
    n = len(met)
    st = hs.generate(max(n, 2), 3, with_truth=False)
    st.n_events = n
    st.cols[hs.ROW["met"], :n] = met
    return st


def test_recording_cut_follows_the_papers_listing():
    """'if (met_met <= 30000.) return false; else { ETmis = met_met; ETmis *= 1.05; return true; }' (GeV here).
    A value exactly at the threshold fails (strict), NaN fails, a failing event keeps the default."""
    st = _tiny_store(np.array([29.0, 30.0, np.nextafter(30.0, 31.0), 31.0, 100.0, np.nan, 1e300]))
    idx, cf, d = oracle.select_record(st, [(REC, 0, 30.0, 1.05)], derived_default=-1.0)
    assert list(idx) == [2, 3, 4, 6] and list(cf) == [4]
    want = [-1.0, -1.0, np.nextafter(30.0, 31.0) * 1.05, 31.0 * 1.05, 100.0 * 1.05, -1.0, 1e300 * 1.05]
    assert d.tobytes() == np.array(want).tobytes()
    # an event dropped BEFORE the recording cut never reaches it; one dropped AFTER it keeps the value it wrote
    st.cols[hs.ROW["mll"], :7] = [50, 50, 50, 10, 50, 50, 50]
    idx, cf, d = oracle.select_record(st, [(hs.MLL_GT, 0, 40.0, 0), (REC, 0, 30.0, 1.05)], derived_default=0.0)
    assert list(idx) == [2, 4, 6] and d[3] == 0.0 and d[4] == 105.0
    idx, cf, d = oracle.select_record(st, [(REC, 0, 30.0, 1.05), (hs.MLL_GT, 0, 40.0, 0)], derived_default=0.0)
    assert list(idx) == [2, 4, 6] and d[3] == 31.0 * 1.05 and list(cf) == [4, 3]


def test_recording_cut_filters_like_met_gt_and_writes_for_exactly_the_events_that_reach_and_pass_it():
    cfg = hs.CONFIGS[4]
    st = cfg.events(200_000)
    chain = list(cfg.cuts)
    k = [c[0] for c in chain].index(hs.MET_GT)
    rec = chain[:k] + [(REC, 0, chain[k][2], 1.05)] + chain[k + 1:]
    idx0, cf0 = oracle.select(st, chain)
    idx1, cf1, d = oracle.select_record(st, rec, derived_default=-7.0)
    assert np.array_equal(idx0, idx1) and np.array_equal(cf0, cf1)
    reached, _ = oracle.select(st, chain[:k + 1])          # events that pass the chain up to and including the MET cut
    want = np.full(st.n_events, -7.0)
    want[reached] = st.col("met")[reached] * 1.05
    assert d.tobytes() == want.tobytes() and len(reached) == cf0[k]


def test_histogram_of_a_plain_column():
    rng = np.random.default_rng(5)
    v = np.concatenate([rng.normal(50, 30, 5000), [0.0, 100.0, np.nextafter(100.0, 0), np.nan, np.inf, -np.inf, -0.0]])
    h = oracle.histogram_values(v, 0.0, 100.0, 40)
    ok = v[~np.isnan(v)]
    t = (ok - 0.0) * (40 / 100.0)            # the rule is stated on t, each operation rounded once: 99.99999999999999 * 0.4 == 40.0
    assert h[0] == (t < 0).sum() and h[41] == (t >= 40).sum() and h.sum() == len(ok)
    assert np.array_equal(h[1:41], np.bincount(t[(t >= 0) & (t < 40)].astype(int), minlength=40))
    assert h[41] == (ok >= 100.0).sum() + 1  # ... so the value one ulp below the upper edge lands in the overflow slot


def _closure_records(n=3000):
    st = hs.generate(n, 77, closure=True, with_truth=True)
    idx = np.arange(n, dtype=np.uint32)
    P0 = oracle.default_params(sigma_scale=0.0)
    best, aux = oracle.reconstruct_tth(st, idx, 1, 9, P0, n_threads=8)
    return st, best, P0


def test_tth_system_equals_the_generated_system_when_the_truth_is_recovered():
    """Closure sample (no widths, no detector smearing) without variations: where the winner is the true pairing with the true
    neutrinos, l+ + l- + nu + nubar + b + bbar + h1 + h2 is the generated ttH system; its mass and pT, summed here in numpy from
    the store and the TRUTH table's neutrinos, must come back."""
    st, best, P0 = _closure_records()
    sysm = oracle.tth_system(st, best, 9, P0)
    n_ok = 0
    for k in range(len(best)):
        b, t = best[k], st.truth[k]
        if not (b["status"] & 1):
            assert np.isnan(sysm[k]).all()
            continue
        if not (np.allclose(b["nu"], t[0:3], rtol=1e-7, atol=1e-7) and np.allclose(b["nubar"], t[3:6], rtol=1e-7, atol=1e-7)):
            continue
        roles = {int(b["jet_b"]), int(b["jet_bbar"]), int(b["jet_h1"]), int(b["jet_h2"])}
        assert len(roles) == 4
        vis = np.zeros(4)
        for s in range(2):
            vis += [st.col("lep_px", s)[k], st.col("lep_py", s)[k], st.col("lep_pz", s)[k], st.col("lep_e", s)[k]]
        for s in roles:
            vis += [st.col("jet_px", s)[k], st.col("jet_py", s)[k], st.col("jet_pz", s)[k], st.col("jet_e", s)[k]]
        for nu in (t[0:3], t[3:6]):
            vis += [nu[0], nu[1], nu[2], np.sqrt(nu @ nu)]
        m = np.sqrt(max(vis[3] ** 2 - vis[:3] @ vis[:3], 0.0)); pt = np.hypot(vis[0], vis[1])
        assert abs(sysm[k, 0] - m) <= 1e-6 * m and abs(sysm[k, 1] - pt) <= 1e-6 * max(pt, 1.0)
        assert sysm[k, 0] >= 172.5 + 172.5 + 125.0 - 1e-3        # the system cannot be lighter than its three resonances
        n_ok += 1
    assert n_ok > 0.3 * len(best)


def test_tth_system_transverse_momentum_needs_no_neutrino_solution():
    """nu_T + nubar_T = MET' exactly, so pT(ttH) = |sum of the six visible objects' p_T + MET'|: a second formula, from the
    smeared objects (oracle.smear) alone; and a rotation of the event about the beam axis changes neither quantity."""
    cfg = hs.CONFIGS[1]
    st = cfg.events(1500)
    idx, _ = oracle.select(st, cfg.cuts)
    best, _ = oracle.reconstruct_tth(st, idx, 8, cfg.reco_seed, n_threads=8)
    sysm = oracle.tth_system(st, best, cfg.reco_seed)
    for k in range(0, len(best), 7):
        b = best[k]
        if not (b["status"] & 1):
            continue
        e = int(b["event"])
        s, metp = oracle.smear(st, e, int(b["variation"]), cfg.reco_seed)
        tx = metp[0] + sum(s[i] * st.col("lep_px", i)[e] for i in range(2)); ty = metp[1] + sum(s[i] * st.col("lep_py", i)[e] for i in range(2))
        for j in (b["jet_b"], b["jet_bbar"], b["jet_h1"], b["jet_h2"]):
            tx += s[2 + j] * st.col("jet_px", int(j))[e]; ty += s[2 + j] * st.col("jet_py", int(j))[e]
        assert abs(sysm[k, 1] - np.hypot(tx, ty)) <= 1e-9 * max(1.0, sysm[k, 1])
    # rotation about z
    c, sn = np.cos(0.7), np.sin(0.7)
    rot = hs.EventStore(st.n_events, st.stride, st.event_base, st.cols.copy(), st.flags.copy())
    for px, py, nrow in (("lep_px", "lep_py", 2), ("jet_px", "jet_py", 8), ("met_x", "met_y", 1)):
        x, y = st.cols[hs.ROW[px]:hs.ROW[px] + nrow], st.cols[hs.ROW[py]:hs.ROW[py] + nrow]
        rot.cols[hs.ROW[px]:hs.ROW[px] + nrow] = c * x - sn * y
        rot.cols[hs.ROW[py]:hs.ROW[py] + nrow] = sn * x + c * y
    best_r, _ = oracle.reconstruct_tth(rot, idx[:300], 8, cfg.reco_seed, n_threads=8)
    sys_r = oracle.tth_system(rot, best_r, cfg.reco_seed)
    same = (best_r["variation"] == best["variation"][:300]) & ((best_r["status"] & 1) == 1) & (best_r["jet_b"] == best["jet_b"][:300]) \
        & (best_r["root"] == best["root"][:300])
    assert same.sum() > 200
    assert np.allclose(sys_r[same], sysm[:300][same], rtol=1e-8, atol=1e-8)
