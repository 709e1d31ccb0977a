"""oracle — ctypes access to the CPU oracle (TEST INFRASTRUCTURE, not the product).

Only tests/, ``__graft_entry__.smoke()`` and bench.py's cpu_baseline / ``--impl reference`` leg may import
this.  It never imports ``paper_2211_14346_b200`` and the CUDA package never imports it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libhepf_oracle.so")
_SRCS = ["oracle_philox.cpp", "oracle_select.cpp", "oracle_reco.cpp", "oracle_hist.cpp", "oracle_chi2.cpp", "oracle_chi2_dilep.cpp"]


def build(force: bool = False) -> str:
    srcs = [os.path.join(_HERE, s) for s in _SRCS]
    deps = srcs + [os.path.join(_HERE, "hepf_oracle.h")]
    if force or not os.path.exists(_LIB_PATH) or os.path.getmtime(_LIB_PATH) < max(map(os.path.getmtime, deps)):
        subprocess.check_call(["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
                               "-Wall", "-o", _LIB_PATH] + srcs)
    return _LIB_PATH


class Events(C.Structure):
    _fields_ = [("n_events", C.c_int64), ("stride", C.c_int64), ("event_base", C.c_int64)] + \
               [(n, C.c_void_p) for n in ("lep_px", "lep_py", "lep_pz", "lep_e", "lep_pt", "lep_eta",
                                          "jet_px", "jet_py", "jet_pz", "jet_e", "jet_pt", "jet_eta",
                                          "met_x", "met_y", "met", "mll", "flags")]


class Cut(C.Structure):
    _fields_ = [("kind", C.c_uint32), ("n", C.c_uint32), ("lo", C.c_double), ("hi", C.c_double)]


class Params(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("m_top", "m_w", "m_higgs", "sigma_higgs", "lambda_nu", "lep_sigma",
                                          "jet_stoch", "jet_const", "sigma_scale", "s_min")]


BEST_DTYPE = np.dtype([("nu", "f8", 3), ("nubar", "f8", 3), ("m_top", "f8"), ("m_antitop", "f8"),
                       ("m_wplus", "f8"), ("m_wminus", "f8"), ("m_higgs", "f8"), ("loglik", "f8"),
                       ("variation", "i4"), ("jet_b", "i4"), ("jet_bbar", "i4"), ("jet_h1", "i4"),
                       ("jet_h2", "i4"), ("root", "i4"), ("status", "u4"), ("event", "u4")])
AUX_DTYPE = np.dtype([("kappa", "f8"), ("loglik2", "f8"), ("n_cand", "i8"), ("pairing", "i4"),
                      ("higgs_pair", "i4"), ("pz_terms", "f8"), ("pzbar_terms", "f8")])
assert BEST_DTYPE.itemsize == 128 and AUX_DTYPE.itemsize == 48


class Pairing(C.Structure):
    _fields_ = [("n_roots", C.c_int32), ("n_higgs", C.c_int32), ("g", C.c_double * 4), ("h", C.c_double * 5),
                ("conic1", C.c_double * 6), ("conic2", C.c_double * 6), ("x", C.c_double * 4),
                ("kappa", C.c_double * 4), ("nterm", C.c_double * 4), ("nu", (C.c_double * 4) * 4),
                ("nubar", (C.c_double * 4) * 4), ("hterm", C.c_double * 6), ("mbb", C.c_double * 6),
                ("min_abs_p_rel", C.c_double), ("pz_terms", C.c_double * 4), ("pzbar_terms", C.c_double * 4)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_det_log.restype = C.c_double
        L.orc_det_log.argtypes = [C.c_double]
        L.orc_det_sincos2pi.argtypes = [C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.orc_philox_normal.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, C.c_void_p]
        L.orc_philox_normal.restype = None
        L.orc_select.argtypes = [C.POINTER(Events), C.POINTER(Cut), C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_select_record.argtypes = [C.POINTER(Events), C.POINTER(Cut), C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double]
        L.orc_tth_system.argtypes = [C.POINTER(Events), C.c_void_p, C.c_int64, C.c_uint64, C.POINTER(Params), C.c_void_p]
        L.orc_histogram_values.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_double, C.c_double, C.c_int32, C.c_void_p]
        L.orc_cut_stats.argtypes = [C.POINTER(Events), C.POINTER(Cut), C.c_int, C.c_int64, C.c_void_p]
        L.orc_reconstruct_tth.argtypes = [C.POINTER(Events), C.c_void_p, C.c_int64, C.c_int32, C.c_uint64,
                                          C.POINTER(Params), C.c_void_p, C.c_void_p, C.c_int]
        L.orc_solve_pairing.argtypes = [C.c_void_p] * 6 + [C.c_int, C.POINTER(Params), C.POINTER(Pairing)]
        L.orc_eval_cell.argtypes = [C.POINTER(Events), C.c_uint32, C.c_int32, C.c_int32, C.c_uint64,
                                    C.POINTER(Params), C.POINTER(Pairing)]
        L.orc_smear.argtypes = [C.POINTER(Events), C.c_uint32, C.c_int32, C.c_uint64, C.POINTER(Params),
                                C.c_void_p, C.c_void_p]
        L.orc_quartic.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_double)]
        L.orc_nu_pz.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_void_p]
        L.orc_chi2_semilep.argtypes = [C.POINTER(Events), C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_chi2_single_top.argtypes = [C.POINTER(Events), C.c_void_p, C.c_int64, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_histogram.argtypes = [C.c_void_p, C.c_int64, C.c_int, C.c_double, C.c_double, C.c_int32, C.c_void_p]
        _lib = L
    return _lib


def default_params(**over) -> Params:
    p = Params()
    lib().orc_default_params(C.byref(p))
    for k, v in over.items():
        setattr(p, k, v)
    return p


def events_view(store) -> Events:
    """View of a host EventStore (hepf_synth.EventStore: cols[64, stride] float64, flags[stride] uint32)."""
    from hepf_synth import ROW
    ev = Events()
    ev.n_events, ev.stride, ev.event_base = store.n_events, store.stride, store.event_base
    base, rb = store.cols.ctypes.data, store.stride * 8
    for name, row in ROW.items():
        setattr(ev, name, base + row * rb)
    ev.flags = store.flags.ctypes.data
    ev._keep = store
    return ev


def make_cuts(chain):
    arr = (Cut * max(1, len(chain)))()
    for i, (kind, n, lo, hi) in enumerate(chain):
        arr[i] = Cut(kind, n, lo, hi)
    return arr


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr); k = (C.c_uint32 * 2)(*key); o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return list(o)


def det_log(u: float) -> float:
    return lib().orc_det_log(u)


def det_sincos2pi(u: float):
    s, c = C.c_double(), C.c_double()
    lib().orc_det_sincos2pi(u, C.byref(s), C.byref(c))
    return s.value, c.value


def philox_normal(seed: int, counter: int, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.float64)
    lib().orc_philox_normal(seed, counter, n, out.ctypes.data)
    return out


def select(store, chain):
    ev = events_view(store)
    idx = np.empty(store.n_events, dtype=np.uint32)
    count = np.zeros(1, dtype=np.int64)
    cutflow = np.zeros(max(1, len(chain)), dtype=np.int64)
    rc = lib().orc_select(C.byref(ev), make_cuts(chain), len(chain), idx.ctypes.data, count.ctypes.data,
                          cutflow.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"orc_select: {rc}")
    return idx[: int(count[0])].copy(), cutflow[: len(chain)].copy()


def select_record(store, chain, derived_default: float = 0.0):
    """(idx, cutflow, derived column) of a chain that may hold a recording cut (kind 10 = MET_GT_RECORD: met > lo, writes met * hi)."""
    ev = events_view(store)
    idx = np.empty(store.n_events, dtype=np.uint32)
    count = np.zeros(1, dtype=np.int64)
    cutflow = np.zeros(max(1, len(chain)), dtype=np.int64)
    derived = np.empty(store.n_events, dtype=np.float64)
    rc = lib().orc_select_record(C.byref(ev), make_cuts(chain), len(chain), idx.ctypes.data, count.ctypes.data,
                                 cutflow.ctypes.data, derived.ctypes.data, derived_default)
    if rc != 0:
        raise RuntimeError(f"orc_select_record: {rc}")
    return idx[: int(count[0])].copy(), cutflow[: len(chain)].copy(), derived


def cut_stats(store, chain, sample_every: int = 1) -> np.ndarray:
    """int64[n_cuts + 1]: events of the sample passing each cut on its own, and the sample size."""
    ev = events_view(store)
    out = np.zeros(len(chain) + 1, dtype=np.int64)
    rc = lib().orc_cut_stats(C.byref(ev), make_cuts(chain), len(chain), sample_every, out.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"orc_cut_stats: {rc}")
    return out


def tth_system(store, best, seed: int, params: Params | None = None) -> np.ndarray:
    """(n, 2) array: invariant mass and transverse momentum of the reconstructed ttH system of each record (NaN if unsolved)."""
    ev = events_view(store)
    best = np.ascontiguousarray(best)
    out = np.empty((len(best), 2), dtype=np.float64)
    rc = lib().orc_tth_system(C.byref(ev), best.ctypes.data, len(best), seed, C.byref(params) if params is not None else None,
                              out.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"orc_tth_system: {rc}")
    return out


def histogram_values(values: np.ndarray, lo: float, hi: float, nbins: int) -> np.ndarray:
    v = np.ascontiguousarray(values, dtype=np.float64)
    out = np.zeros(nbins + 2, dtype=np.uint64)
    rc = lib().orc_histogram_values(v.ctypes.data, 1, len(v), lo, hi, nbins, out.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"orc_histogram_values: {rc}")
    return out


def reconstruct_tth(store, idx, n_variations: int, seed: int, params: Params | None = None, n_threads: int = 1):
    ev = events_view(store)
    idx = np.ascontiguousarray(idx, dtype=np.uint32)
    best = np.zeros(len(idx), dtype=BEST_DTYPE)
    aux = np.zeros(len(idx), dtype=AUX_DTYPE)
    rc = lib().orc_reconstruct_tth(C.byref(ev), idx.ctypes.data, len(idx), n_variations, seed,
                                   C.byref(params) if params is not None else None, best.ctypes.data,
                                   aux.ctypes.data, n_threads)
    if rc != 0:
        raise RuntimeError(f"orc_reconstruct_tth: {rc}")
    return best, aux


def solve_pairing(lp, b, lm, bbar, met, jets_h=(), params: Params | None = None) -> Pairing:
    arrs = [np.ascontiguousarray(a, dtype=np.float64) for a in (lp, b, lm, bbar, met)]
    jh = np.ascontiguousarray(np.asarray(jets_h, dtype=np.float64).reshape(-1, 4)) if len(jets_h) else np.zeros((0, 4))
    out = Pairing()
    rc = lib().orc_solve_pairing(*[a.ctypes.data for a in arrs], jh.ctypes.data, len(jh),
                                 C.byref(params) if params is not None else None, C.byref(out))
    if rc != 0:
        raise RuntimeError(f"orc_solve_pairing: {rc}")
    return out


def eval_cell(store, e: int, v: int, a: int, seed: int, params: Params | None = None) -> Pairing:
    ev = events_view(store)
    out = Pairing()
    rc = lib().orc_eval_cell(C.byref(ev), e, v, a, seed, C.byref(params) if params is not None else None,
                             C.byref(out))
    if rc < 0:
        raise RuntimeError(f"orc_eval_cell: {rc}")
    return out


def quartic(g):
    """(ascending simple real roots, tangency measure) of the monic quartic x^4 + g[3] x^3 + g[2] x^2 + g[1] x + g[0]."""
    g = np.ascontiguousarray(g, dtype=np.float64)
    roots, m = np.zeros(4), C.c_double()
    n = lib().orc_quartic(g.ctypes.data, roots.ctypes.data, C.byref(m))
    if n < 0:
        raise RuntimeError(f"orc_quartic: {n}")
    return roots[:n].copy(), m.value


def smear(store, e: int, v: int, seed: int, params: Params | None = None):
    ev = events_view(store)
    s = np.zeros(10); m = np.zeros(2)
    rc = lib().orc_smear(C.byref(ev), e, v, seed, C.byref(params) if params is not None else None,
                         s.ctypes.data, m.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"orc_smear: {rc}")
    return s, m


HIST_FIELDS = dict(m_top=0, m_antitop=1, m_wplus=2, m_wminus=3, m_higgs=4, loglik=5, nu_pt=6, nubar_pt=7, variation=8)


def histogram(best: np.ndarray, field: str, lo: float, hi: float, nbins: int) -> np.ndarray:
    """uint64[nbins + 2]: underflow, bins, overflow of the solved records' `field`."""
    best = np.ascontiguousarray(best)
    out = np.zeros(nbins + 2, dtype=np.uint64)
    rc = lib().orc_histogram(best.ctypes.data, len(best), HIST_FIELDS[field], lo, hi, nbins, out.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"orc_histogram: {rc}")
    return out


CHI2_DTYPE = np.dtype([("chi2", "f8"), ("nu_pz", "f8"), ("m_top_lep", "f8"), ("m_top_had", "f8"), ("m_w_lep", "f8"),
                       ("m_w_had", "f8"), ("jet_b_lep", "i4"), ("jet_b_had", "i4"), ("jet_q1", "i4"), ("jet_q2", "i4"),
                       ("solution", "i4"), ("n_comb", "i4"), ("status", "u4"), ("event", "u4")])
assert CHI2_DTYPE.itemsize == 80


def nu_pz(lep, nux: float, nuy: float, m_w: float = 80.4):
    lep = np.ascontiguousarray(lep, dtype=np.float64); pz = np.zeros(2)
    n = lib().orc_nu_pz(lep.ctypes.data, nux, nuy, m_w, pz.ctypes.data)
    return list(pz[:n])


def chi2_semilep(store, idx, params=None):
    """(records CHI2_DTYPE[n], second-best chi2 per event); params = (m_top, m_w, sigma_top, sigma_w) or None."""
    ev = events_view(store)
    idx = np.ascontiguousarray(idx, dtype=np.uint32)
    out = np.zeros(len(idx), dtype=CHI2_DTYPE); second = np.zeros(len(idx))
    par = np.asarray(params, dtype=np.float64) if params is not None else None
    rc = lib().orc_chi2_semilep(C.byref(ev), idx.ctypes.data, len(idx), par.ctypes.data if par is not None else None,
                                out.ctypes.data, second.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"orc_chi2_semilep: {rc}")
    return out, second


def chi2_single_top(store, idx, mode: int, params=None):
    """Single-top chi^2 of eq. (1): mode 1 = t-channel, mode 2 = Wt.  (records CHI2_DTYPE[n], second-best chi2 per event)."""
    ev = events_view(store)
    idx = np.ascontiguousarray(idx, dtype=np.uint32)
    out = np.zeros(len(idx), dtype=CHI2_DTYPE); second = np.zeros(len(idx))
    par = np.asarray(params, dtype=np.float64) if params is not None else None
    rc = lib().orc_chi2_single_top(C.byref(ev), idx.ctypes.data, len(idx), mode, par.ctypes.data if par is not None else None,
                                   out.ctypes.data, second.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"orc_chi2_single_top: {rc}")
    return out, second


CHI2_DILEP_DTYPE = np.dtype([("chi2", "f8"), ("nu", "f8", 3), ("nubar", "f8", 3), ("m_top", "f8"), ("m_antitop", "f8"),
                             ("m_wplus", "f8"), ("m_wminus", "f8"), ("jet_b", "i4"), ("jet_bbar", "i4"), ("grid_x", "i4"),
                             ("grid_y", "i4"), ("sol_nu", "i4"), ("sol_nubar", "i4"), ("n_comb", "i4"), ("status", "u4"),
                             ("event", "u4"), ("pad_", "i4")])
assert CHI2_DILEP_DTYPE.itemsize == 128


class Split(C.Structure):
    _fields_ = [("split_range", C.c_double), ("split_n", C.c_int32), ("pad_", C.c_int32)]


def chi2_dilep(store, idx, params=None, split=None, n_threads: int = 1):
    """Dileptonic chi^2 of eq. (1) (oracle_chi2_dilep.cpp).  split = (split_range, split_n) or None (160 GeV, 32).
    Returns (records CHI2_DILEP_DTYPE[n], second-best chi2 per event)."""
    ev = events_view(store)
    idx = np.ascontiguousarray(idx, dtype=np.uint32)
    out = np.zeros(len(idx), dtype=CHI2_DILEP_DTYPE); second = np.zeros(len(idx))
    par = np.asarray(params, dtype=np.float64) if params is not None else None
    sp = Split(float(split[0]), int(split[1]), 0) if split is not None else None
    L = lib()
    L.orc_chi2_dilep.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
    rc = L.orc_chi2_dilep(C.byref(ev), idx.ctypes.data, len(idx), par.ctypes.data if par is not None else None,
                          C.byref(sp) if sp is not None else None, out.ctypes.data, second.ctypes.data, int(n_threads))
    if rc != 0:
        raise RuntimeError(f"orc_chi2_dilep failed: {rc}")
    return out, second


def chi2_dilep_point(store, e: int, slot_b: int, slot_bbar: int, nux: float, nuy: float, params=None):
    """chi^2 of one hypothesis at one split of the MET: (chi2[2][2] over the p_z solutions, pz_nu[2], pz_nubar[2])."""
    ev = events_view(store)
    par = np.asarray(params, dtype=np.float64) if params is not None else None
    out = np.zeros(4); p1 = np.zeros(2); p2 = np.zeros(2)
    L = lib()
    L.orc_chi2_dilep_point.argtypes = [C.c_void_p, C.c_uint32, C.c_int, C.c_int, C.c_double, C.c_double, C.c_void_p,
                                       C.c_void_p, C.c_void_p, C.c_void_p]
    L.orc_chi2_dilep_point(C.byref(ev), int(e), int(slot_b), int(slot_bbar), float(nux), float(nuy),
                           par.ctypes.data if par is not None else None, out.ctypes.data, p1.ctypes.data, p2.ctypes.data)
    return out.reshape(2, 2), p1, p2
