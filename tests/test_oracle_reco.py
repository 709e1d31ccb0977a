"""Pins for oracle O4 (smearing, conics, quartic, score, argmax).  PAPER.md:134-146 (§4); SURVEY.md §8(c).

The pins never re-type the oracle's conic/resultant algebra: they use the printed worked example, the raw mass
constraints (closure, multi-start Newton on the 4x4 constraint system), numpy's companion-matrix roots, dense
sign-change scans, generator truth, and symmetry/prefix invariants.
"""
import math
import os

import numpy as np
import pytest

import hepf_synth as hs
import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")
MT, MW, MH = 172.5, 80.4, 125.0


def v4(p, m):
    p = list(map(float, p))
    return np.array(p + [math.sqrt(sum(x * x for x in p) + m * m)])


def inv_mass(*vs):
    s = np.sum(vs, axis=0)
    return math.sqrt(max(0.0, s[3] ** 2 - s[0] ** 2 - s[1] ** 2 - s[2] ** 2))


def load_worked():
    d, roots = {}, []
    with open(os.path.join(GOLD, "worked_example.txt")) as f:
        for ln in f:
            if ln.startswith("#") or not ln.strip():
                continue
            k, *vals = ln.split()
            vals = [float(x) for x in vals]
            if k.startswith("r") and len(vals) == 9:
                roots.append(vals)
            else:
                d[k] = vals
    return d, roots


def test_worked_example_matches_printed_values():
    d, roots = load_worked()
    P = oracle.solve_pairing(v4(d["lp"], 0), v4(d["b"], 4.7), v4(d["lm"], 0), v4(d["bbar"], 4.7), d["met"])
    assert P.n_roots == 4
    for k, gi in (("g0", 0), ("g1", 1), ("g2", 2), ("g3", 3)):
        assert P.g[gi] == pytest.approx(d[k][0], rel=1e-11)
    for r, want in enumerate(roots):
        got = list(P.nu[r]) + list(P.nubar[r]) + [P.nterm[r]]
        assert got == pytest.approx(want, rel=2e-13, abs=1e-11)   # printed to 15 significant digits
    assert int(np.argmax([P.nterm[r] for r in range(4)])) == 3    # "r3 wins if m_bb is common"


def test_worked_example_closure_from_raw_four_vectors():
    d, _ = load_worked()
    lp, b, lm, bb = v4(d["lp"], 0), v4(d["b"], 4.7), v4(d["lm"], 0), v4(d["bbar"], 4.7)
    P = oracle.solve_pairing(lp, b, lm, bb, d["met"])
    for r in range(P.n_roots):
        nu, nub = np.array(P.nu[r]), np.array(P.nubar[r])
        assert nu[3] == pytest.approx(np.linalg.norm(nu[:3]), rel=1e-14)
        assert inv_mass(lp, nu) == pytest.approx(MW, rel=1e-10)
        assert inv_mass(lp, nu, b) == pytest.approx(MT, rel=1e-10)
        assert inv_mass(lm, nub) == pytest.approx(MW, rel=1e-10)
        assert inv_mass(lm, nub, bb) == pytest.approx(MT, rel=1e-10)
        assert nu[0] + nub[0] == pytest.approx(d["met"][0], abs=1e-10)
        assert nu[1] + nub[1] == pytest.approx(d["met"][1], abs=1e-10)


def _constraint_system(lp, b, lm, bb, met):
    def F(u):
        a, bq, c, dq = u
        nu = np.array([a, bq, c, math.sqrt(a * a + bq * bq + c * c)])
        qx, qy = met[0] - a, met[1] - bq
        nb = np.array([qx, qy, dq, math.sqrt(qx * qx + qy * qy + dq * dq)])

        def m2(*vs):
            s = np.sum(vs, axis=0)
            return s[3] ** 2 - s[0] ** 2 - s[1] ** 2 - s[2] ** 2
        return np.array([m2(lp, nu) - MW ** 2, m2(lp, nu, b) - MT ** 2, m2(lm, nb) - MW ** 2, m2(lm, nb, bb) - MT ** 2])
    return F


def _multistart_solutions(lp, b, lm, bb, met, n_start=1200, seed=5):
    from scipy.optimize import fsolve
    F = _constraint_system(lp, b, lm, bb, met)
    rng = np.random.default_rng(seed)
    sols = []
    for _ in range(n_start):
        u0 = rng.normal(0, 1, 4) * rng.choice([20.0, 80.0, 250.0])
        u, info, ier, _ = fsolve(F, u0, full_output=True, xtol=1e-13)
        if ier != 1 or np.abs(F(u)).max() > 1e-6:
            continue
        if not any(np.abs(u - s).max() < 1e-5 * (1 + np.abs(s).max()) for s in sols):
            sols.append(u)
    return sorted(sols, key=lambda s: s[0])


def test_brute_force_multistart_newton_on_raw_constraints_finds_the_same_solution_set():
    """Completeness + correctness without the conic/resultant algebra: solve the four mass constraints in
    (nu_x, nu_y, nu_z, nubar_z) from thousands of random starts and compare the solution set."""
    d, _ = load_worked()
    cases = [(v4(d["lp"], 0), v4(d["b"], 4.7), v4(d["lm"], 0), v4(d["bbar"], 4.7), d["met"])]
    st = hs.generate(40, 77, closure=True)
    for e in range(6):   # truth pairings of closure events (>= 2 solutions) and a wrong pairing
        t = st.truth[e]
        lp_slot = int(t[11]); sb, sbb = int(t[6]), int(t[7])
        get = lambda name, s: np.array([st.col(name + "_px", s)[e], st.col(name + "_py", s)[e],
                                        st.col(name + "_pz", s)[e], st.col(name + "_e", s)[e]])
        lp, lm = get("lep", lp_slot), get("lep", 1 - lp_slot)
        met = [st.col("met_x")[e], st.col("met_y")[e]]
        cases.append((lp, get("jet", sb), lm, get("jet", sbb), met))
        if e < 3:
            cases.append((lp, get("jet", sbb), lm, get("jet", sb), met))
    n_total = 0
    for lp, b, lm, bb, met in cases:
        P = oracle.solve_pairing(lp, b, lm, bb, met)
        sols = _multistart_solutions(lp, b, lm, bb, met)
        assert len(sols) == P.n_roots, (len(sols), P.n_roots)
        for r, s in enumerate(sols):
            want = [P.nu[r][0], P.nu[r][1], P.nu[r][2], P.nubar[r][2]]
            assert s == pytest.approx(want, rel=1e-6, abs=1e-6)
        n_total += P.n_roots
    assert n_total >= 16


def _random_cells(n_events=300, seed=123, n_fake_b=0):
    st = hs.generate(n_events, seed, n_fake_b=n_fake_b)
    idx, _ = oracle.select(st, hs.CHAIN_BASE)
    return st, idx


def test_quartic_roots_against_companion_matrix_and_dense_sign_scan():
    st, idx = _random_cells(200, 321)
    n_checked = n_roots = 0
    counts = {0: 0, 2: 0, 4: 0}
    for e in idx[:60]:
        for a in (1, 2, 3, 4, 6, 7):
            P = oracle.eval_cell(st, int(e), 0, a, 99)
            h = np.array(P.h)
            if h[4] == 0:
                continue
            assert P.n_roots in (0, 2, 4)               # odd counts must never occur
            counts[P.n_roots] += 1
            xs = np.array(P.x[: P.n_roots])
            assert (np.diff(xs) > 0).all()
            # (1) numpy companion-matrix eigenvalues: the real ones are the oracle's roots
            if P.min_abs_p_rel > 1e-9:
                ev = np.roots(h[::-1])
                real = np.sort(ev[np.abs(ev.imag) < 1e-7 * (1 + np.abs(ev.real))].real)
                assert len(real) == P.n_roots
                assert xs == pytest.approx(real, rel=1e-7, abs=1e-7)
            # (2) dense sign scan of P on a sinh-spaced grid over the Cauchy bound: a cell has a sign change
            #     iff it holds an odd number of oracle roots
            g = np.array(list(P.g) + [1.0])
            R = 1 + np.abs(g[:4]).max()
            grid = np.sinh(np.linspace(-np.arcsinh(R), np.arcsinh(R), 200001))
            val = np.polyval(g[::-1], grid)
            change = np.signbit(val[:-1]) != np.signbit(val[1:])
            cnt = np.histogram(xs, bins=grid)[0]
            assert np.array_equal(change, (cnt % 2) == 1)
            n_checked += 1; n_roots += P.n_roots
    assert n_checked > 200 and n_roots > 100
    assert counts[0] > 0 and counts[2] > 0


def test_two_dimensional_conic_intersection_scan():
    """Independently of the resultant: scan x, solve conic 1 for y, look for sign changes of conic 2 along
    each branch; every crossing must sit at an oracle root (x, y) and every root must be found."""
    st, idx = _random_cells(100, 555)
    done = 0
    for e, a in [(e, a) for e in idx[:40] for a in (1, 4, 11)]:
        P = oracle.eval_cell(st, int(e), 1, a, 4242)
        if P.n_roots == 0 or P.min_abs_p_rel < 1e-6:
            continue
        a1, b1, c1, d1, e1, f1 = P.conic1
        a2, b2, c2, d2, e2, f2 = P.conic2
        xs = np.array(P.x[: P.n_roots]); ys = np.array([P.nu[r][1] for r in range(P.n_roots)])
        span = 3 * (np.abs(xs).max() + 50)
        grid = np.linspace(-span, span, 400001)
        qb, qc = b1 * grid + e1, a1 * grid ** 2 + d1 * grid + f1
        disc = qb ** 2 - 4 * c1 * qc
        ok = disc >= 0
        found = []
        for sgn in (-1, 1):
            y = np.where(ok, (-qb + sgn * np.sqrt(np.where(ok, disc, 0))) / (2 * c1), np.nan)
            r2 = a2 * grid ** 2 + b2 * grid * y + c2 * y ** 2 + d2 * grid + e2 * y + f2
            both = ok[:-1] & ok[1:]
            ch = both & (np.signbit(r2[:-1]) != np.signbit(r2[1:]))
            for k in np.nonzero(ch)[0]:
                found.append((0.5 * (grid[k] + grid[k + 1]), 0.5 * (y[k] + y[k + 1])))
        inside = [(x, y) for x, y in zip(xs, ys) if abs(x) < span]
        assert len(found) == len(inside), (found, inside)
        for (fx, fy) in found:
            assert min(abs(fx - x) + abs(fy - y) for x, y in inside) < 1e-2 * (1 + abs(fx) + abs(fy))
        done += 1
    assert done >= 10


def _tol(kappa):
    return max(1e-9, 64 * (kappa if np.isfinite(kappa) else 0))


def test_closure_invariant_and_met_balance_on_every_reported_solution():
    st, idx = _random_cells(400, 2024)
    V, seed = 8, 0x5EED0001
    best, aux = oracle.reconstruct_tth(st, idx, V, seed, n_threads=4)
    solved = 0
    for k, e in enumerate(idx):
        bst = best[k]
        assert bst["event"] == e
        if not bst["status"] & 1:
            assert np.isnan(bst["loglik"])
            continue
        solved += 1
        v = int(bst["variation"])
        s, metp = oracle.smear(st, int(e), v, seed)
        f = st.flags[e]; lp_slot = 0 if (f >> 4) & 1 else 1
        obj = lambda name, slot, sc: sc * np.array([st.col(name + "_px", slot)[e], st.col(name + "_py", slot)[e],
                                                    st.col(name + "_pz", slot)[e], st.col(name + "_e", slot)[e]])
        lp, lm = obj("lep", lp_slot, s[lp_slot]), obj("lep", 1 - lp_slot, s[1 - lp_slot])
        jb, jbb = int(bst["jet_b"]), int(bst["jet_bbar"])
        b, bb = obj("jet", jb, s[2 + jb]), obj("jet", jbb, s[2 + jbb])
        nu = np.append(bst["nu"], np.linalg.norm(bst["nu"])); nub = np.append(bst["nubar"], np.linalg.norm(bst["nubar"]))
        tol = _tol(aux[k]["kappa"]) * 10
        assert inv_mass(lp, nu) == pytest.approx(MW, rel=tol)
        assert inv_mass(lm, nub) == pytest.approx(MW, rel=tol)
        assert inv_mass(lp, nu, b) == pytest.approx(MT, rel=tol)
        assert inv_mass(lm, nub, bb) == pytest.approx(MT, rel=tol)
        assert bst["m_wplus"] == pytest.approx(MW, rel=tol) and bst["m_antitop"] == pytest.approx(MT, rel=tol)
        assert nu[0] + nub[0] == pytest.approx(metp[0], abs=1e-9) and nu[1] + nub[1] == pytest.approx(metp[1], abs=1e-9)
        # Higgs pair = two tagged jets that are neither b nor bbar; its mass is the smeared pair mass
        h1, h2 = int(bst["jet_h1"]), int(bst["jet_h2"])
        assert len({jb, jbb, h1, h2}) == 4 and all((f >> (16 + j)) & 1 for j in (jb, jbb, h1, h2))
        assert bst["m_higgs"] == pytest.approx(inv_mass(obj("jet", h1, s[2 + h1]), obj("jet", h2, s[2 + h2])), rel=1e-12)
        # the reported log-likelihood is the stated formula of the reported solution
        ptn, ptb = math.hypot(*bst["nu"][:2]), math.hypot(*bst["nubar"][:2])
        ll = -0.5 * ((bst["m_higgs"] - MH) / 15.0) ** 2 + math.log(ptn * ptb) - (ptn + ptb) / 40.0
        assert bst["loglik"] == pytest.approx(ll, rel=1e-12, abs=1e-12)
        assert aux[k]["loglik2"] <= bst["loglik"]
    assert solved > 0.8 * len(idx)


def test_smearing_scales_follow_the_keyed_philox_stream_and_resolution_model():
    st, idx = _random_cells(50, 31)
    seed = 0xABCDEF0123456789
    e = int(idx[3]); v = 5
    s, metp = oracle.smear(st, e, v, seed)
    key = [seed & 0xffffffff, seed >> 32]
    n_jet = (int(st.flags[e]) >> 8) & 15
    dx = dy = 0.0
    for t in range(10):
        x = oracle.philox4x32_10([e, 0, v, 0x54544800 + (t >> 1)], key)
        w0, w1 = (x[1] << 32) | x[0], (x[3] << 32) | x[2]
        u1, u2 = ((w0 >> 11) + 1) / 2 ** 53, (w1 >> 11) / 2 ** 53
        rho = math.sqrt(-2 * math.log(u1))
        z = rho * (math.sin(2 * math.pi * u2) if t & 1 else math.cos(2 * math.pi * u2))
        if t < 2:
            sigma = 0.01; px, py = st.col("lep_px", t)[e], st.col("lep_py", t)[e]
        else:
            E = st.col("jet_e", t - 2)[e]
            sigma = 0.5 / math.sqrt(E) + 0.03 if E > 0 else float("inf")
            px, py = st.col("jet_px", t - 2)[e], st.col("jet_py", t - 2)[e]
        if t < 2 + n_jet:
            assert s[t] == pytest.approx(max(0.1, 1 + sigma * z), rel=1e-13)
            dx += (s[t] - 1) * px; dy += (s[t] - 1) * py
    assert metp[0] == pytest.approx(st.col("met_x")[e] - dx, abs=1e-10)
    assert metp[1] == pytest.approx(st.col("met_y")[e] - dy, abs=1e-10)
    # event_base shifts the key: a slice starting at e sees the same scales at local index 0
    sl = st.slice(e, e + 2)
    s2, m2 = oracle.smear(sl, 0, v, seed)
    assert s2.tobytes() == s.tobytes() and m2.tobytes() == metp.tobytes()
    # sigma_scale = 0 -> unit scales, MET unchanged
    s0, m0 = oracle.smear(st, e, v, seed, oracle.default_params(sigma_scale=0.0))
    assert (s0[: 2 + n_jet] == 1.0).all() and m0[0] == st.col("met_x")[e] and m0[1] == st.col("met_y")[e]


def test_truth_recovery_in_closure_mode():
    """Generator with zero widths and no detector smearing, sigma_scale = 0: the true neutrinos are a solution
    of the truth pairing (SURVEY.md §8(c) 'Solver vs truth')."""
    st = hs.generate(300, 4321, closure=True)
    P0 = oracle.default_params(sigma_scale=0.0)
    n = 0
    for e in range(st.n_events):
        t = st.truth[e]
        cand = [s for s in range(8) if (st.flags[e] >> (16 + s)) & 1]
        i, j = cand.index(int(t[6])), cand.index(int(t[7]))
        P = oracle.eval_cell(st, e, 0, i * len(cand) + j, 1, P0)
        assert P.n_roots >= 2, e
        errs = []
        for r in range(P.n_roots):
            got = np.array([*P.nu[r][:3], *P.nubar[r][:3]])
            scale = np.abs(t[:6]).max()
            errs.append((np.abs(got - t[:6]).max() / scale, P.kappa[r]))
        err, kap = min(errs)
        assert err < max(1e-7, 1e4 * kap), (e, err, kap)
        n += 1
    assert n == 300
    # and the full reconstruction picks solutions that satisfy closure; most events are solved
    idx = np.arange(st.n_events, dtype=np.uint32)
    best, _ = oracle.reconstruct_tth(st, idx, 1, 1, P0, n_threads=4)
    assert (best["status"] & 1).mean() == 1.0


def test_prefix_property_in_V_and_sigma_scale_zero():
    st, idx = _random_cells(120, 808)
    seed = 0x5EED0002
    b16, _ = oracle.reconstruct_tth(st, idx, 16, seed, n_threads=4)
    b48, _ = oracle.reconstruct_tth(st, idx, 48, seed, n_threads=4)
    for x, y in zip(b16, b48):
        if y["status"] & 1 and y["variation"] < 16:
            assert x.tobytes() == y.tobytes()
        if x["status"] & 1:
            assert y["status"] & 1 and y["loglik"] >= x["loglik"]
    assert (b48["variation"] >= 16).any() and (b48["variation"] < 16).any()
    # sigma_scale = 0: every variation is the nominal event -> first one wins, loglik equals the V=1 value
    P0 = oracle.default_params(sigma_scale=0.0)
    n1, _ = oracle.reconstruct_tth(st, idx, 1, seed, P0)
    n8, a8 = oracle.reconstruct_tth(st, idx, 8, seed, P0, n_threads=4)
    assert n1.tobytes() == n8.tobytes()
    ok = (n8["status"] & 1) == 1
    assert (n8["variation"][ok] == 0).all()
    assert (a8["loglik2"][ok] == n8["loglik"][ok]).all()          # the other 7 variations tie exactly


def test_rotation_about_z_leaves_loglik_and_indices_unchanged():
    st, idx = _random_cells(120, 99)
    seed = 17
    b0, a0 = oracle.reconstruct_tth(st, idx, 4, seed, n_threads=4)
    phi = 0.7345
    c, s = math.cos(phi), math.sin(phi)
    rot = hs.EventStore(st.n_events, st.stride, st.event_base, st.cols.copy(), st.flags.copy())
    R = hs.ROW
    for name, n in (("lep", 2), ("jet", 8)):
        for k in range(n):
            x, y = st.cols[R[name + "_px"] + k], st.cols[R[name + "_py"] + k]
            rot.cols[R[name + "_px"] + k], rot.cols[R[name + "_py"] + k] = c * x - s * y, s * x + c * y
    x, y = st.cols[R["met_x"]], st.cols[R["met_y"]]
    rot.cols[R["met_x"]], rot.cols[R["met_y"]] = c * x - s * y, s * x + c * y
    b1, a1 = oracle.reconstruct_tth(rot, idx, 4, seed, n_threads=4)
    same = 0
    for x, y, ax in zip(b0, b1, a0):
        assert (x["status"] & 1) == (y["status"] & 1) or ax["kappa"] > 1e-10
        if not (x["status"] & 1 and y["status"] & 1):
            continue
        near_tie = abs(ax["loglik"] if False else (x["loglik"] - ax["loglik2"])) < 1e-6 * abs(x["loglik"])
        if near_tie:
            continue
        keys = ("variation", "jet_b", "jet_bbar", "jet_h1", "jet_h2")
        if all(x[k] == y[k] for k in keys):
            tol = max(1e-8, 1e5 * ax["kappa"])
            assert y["loglik"] == pytest.approx(x["loglik"], rel=tol, abs=tol)
            assert y["nu"][2] == pytest.approx(x["nu"][2], rel=tol, abs=tol)
            assert c * x["nu"][0] - s * x["nu"][1] == pytest.approx(y["nu"][0], rel=tol, abs=tol * 100)
            same += 1
    assert same > 0.9 * ((b0["status"] & 1).sum())


def test_jet_slot_permutation_permutes_indices_not_loglik():
    st, idx = _random_cells(400, 4)
    P0 = oracle.default_params(sigma_scale=0.0)
    b0, a0 = oracle.reconstruct_tth(st, idx, 1, 1, P0, n_threads=4)
    perm = hs.EventStore(st.n_events, st.stride, st.event_base, st.cols.copy(), st.flags.copy())
    R = hs.ROW
    for name in ("jet_px", "jet_py", "jet_pz", "jet_e", "jet_pt", "jet_eta"):   # swap slots 0 and 2
        perm.cols[R[name] + 0], perm.cols[R[name] + 2] = st.cols[R[name] + 2].copy(), st.cols[R[name] + 0].copy()
    f = st.flags.copy()
    t0, t2 = (f >> 16) & 1, (f >> 18) & 1
    perm.flags[:] = (f & ~np.uint32((1 << 16) | (1 << 18))) | (t2 << 16) | (t0 << 18)
    b1, _ = oracle.reconstruct_tth(perm, idx, 1, 1, P0, n_threads=4)
    sw = {0: 2, 2: 0}
    n = 0
    for x, y, ax in zip(b0, b1, a0):
        if not x["status"] & 1:
            continue
        n_jet = (int(st.flags[x["event"]]) >> 8) & 15
        if n_jet < 3 or abs(x["loglik"] - ax["loglik2"]) < 1e-9 * abs(x["loglik"]):
            continue
        assert y["loglik"] == pytest.approx(x["loglik"], rel=1e-12)
        for k in ("jet_b", "jet_bbar"):
            assert y[k] == sw.get(int(x[k]), int(x[k]))
        assert {int(y["jet_h1"]), int(y["jet_h2"])} == {sw.get(int(x["jet_h1"]), int(x["jet_h1"])),
                                                       sw.get(int(x["jet_h2"]), int(x["jet_h2"]))}
        n += 1
    assert n > 50


def test_not_applicable_and_truncation_status():
    st = hs.generate(2000, 8, bkg_frac=1.0)          # background only: every topology occurs
    idx = np.arange(st.n_events, dtype=np.uint32)
    best, _ = oracle.reconstruct_tth(st, idx, 2, 3, n_threads=4)
    f = st.flags[: st.n_events]
    n_lep = f & 15; os_ = ((f >> 4) & 1) != ((f >> 5) & 1)
    n_jet = np.minimum((f >> 8) & 15, 8)
    n_tag = np.array([bin((int(x) >> 16) & ((1 << int(nj)) - 1)).count("1") for x, nj in zip(f, n_jet)])
    appl = (n_lep == 2) & os_ & (n_tag >= 4)
    assert np.array_equal((best["status"] & 2) != 0, ~appl)
    assert np.array_equal((best["status"] & 4) != 0, n_tag > 6)
    assert np.isnan(best["loglik"][~appl]).all() and (best["variation"][~appl] == -1).all()
    assert appl.sum() > 10 and (~appl).sum() > 10


def test_six_candidates_enumerate_thirty_pairings_and_six_higgs_pairs():
    st, idx = _random_cells(150, 3, n_fake_b=2)
    best, aux = oracle.reconstruct_tth(st, idx, 2, 0x5EED0003, n_threads=4)
    ok = (best["status"] & 1) == 1
    assert ok.sum() > 30
    assert aux["pairing"][ok].max() > 12 and aux["higgs_pair"][ok].max() >= 3 and aux["higgs_pair"][ok].max() <= 5
    for x, ax in zip(best[ok], aux[ok]):
        f = int(st.flags[x["event"]])
        cand = [s for s in range(8) if (f >> (16 + s)) & 1][:6]
        nb = len(cand)
        i, j = divmod(int(ax["pairing"]), nb)
        assert cand[i] == x["jet_b"] and cand[j] == x["jet_bbar"] and i != j
        rest = [(k, l) for k in range(nb) for l in range(k + 1, nb) if not {k, l} & {i, j}]
        k, l = rest[int(ax["higgs_pair"])]
        assert (cand[k], cand[l]) == (x["jet_h1"], x["jet_h2"])
