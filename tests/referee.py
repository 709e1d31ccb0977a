"""referee — ctypes access to tests/referee_q128.c, the TEST-ONLY binary128 referee of the dilepton solve.

It imports neither ``oracle`` nor ``paper_2211_14346_b200``: given an event store (data), a cell (event, variation,
pairing) and the parameters it returns the exact solutions of DESIGN.md section 2, and tells how far a record of
either side is from them (R11).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "referee_q128.c")
_LIB = os.path.join(_HERE, "libreferee.so")

PARAM_NAMES = ("m_top", "m_w", "m_higgs", "sigma_higgs", "lambda_nu", "lep_sigma", "jet_stoch", "jet_const",
               "sigma_scale", "s_min")
DEFAULTS = dict(m_top=172.5, m_w=80.4, m_higgs=125.0, sigma_higgs=15.0, lambda_nu=40.0, lep_sigma=0.01, jet_stoch=0.5,
                jet_const=0.03, sigma_scale=1.0, s_min=0.1)   # PAPER.md:138, :145; BASELINE.json configs[0]; R5, R7

# row offsets of the [64][stride] column block — data layout, restated here on purpose
_ROWS = dict(lep_px=0, lep_py=2, lep_pz=4, lep_e=6, lep_pt=8, lep_eta=10, jet_px=12, jet_py=20, jet_pz=28, jet_e=36,
             jet_pt=44, jet_eta=52, met_x=60, met_y=61, met=62, mll=63)


class Events(C.Structure):
    _fields_ = [("n_events", C.c_int64), ("stride", C.c_int64), ("event_base", C.c_int64)] + \
               [(n, C.c_void_p) for n in ("lep_px", "lep_py", "lep_pz", "lep_e", "lep_pt", "lep_eta", "jet_px", "jet_py",
                                          "jet_pz", "jet_e", "jet_pt", "jet_eta", "met_x", "met_y", "met", "mll", "flags")]


class Params(C.Structure):
    _fields_ = [(n, C.c_double) for n in PARAM_NAMES]


class Cell(C.Structure):
    _fields_ = [("status", C.c_int32), ("n_roots", C.c_int32), ("n_higgs", C.c_int32), ("n_crit", C.c_int32),
                ("lp", C.c_double * 4), ("b", C.c_double * 4), ("lm", C.c_double * 4), ("bbar", C.c_double * 4),
                ("met", C.c_double * 2), ("h", C.c_double * 5), ("g", C.c_double * 4), ("x", C.c_double * 4),
                ("y", C.c_double * 4), ("nu", (C.c_double * 4) * 4), ("nubar", (C.c_double * 4) * 4),
                ("nterm", C.c_double * 4), ("kappa", C.c_double * 4), ("pz_terms", C.c_double * 4),
                ("pzbar_terms", C.c_double * 4), ("newton_shift", C.c_double * 4), ("residual", C.c_double * 4),
                ("crit_x", C.c_double * 3), ("crit_rel", C.c_double * 3), ("min_abs_p_rel", C.c_double),
                ("hterm", C.c_double * 6), ("mbb", C.c_double * 6)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
            subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-Wall", _SRC, "-o", _LIB,
                                   "-lquadmath", "-lm"])
        L = C.CDLL(_LIB)
        L.ref_smear.argtypes = [C.POINTER(Events), C.c_uint32, C.c_int32, C.c_uint64, C.POINTER(Params), C.c_void_p, C.c_void_p]
        L.ref_cell.argtypes = [C.POINTER(Events), C.c_uint32, C.c_int32, C.c_int32, C.c_uint64, C.POINTER(Params), C.POINTER(Cell)]
        L.ref_polish.argtypes = [C.POINTER(Events), C.c_uint32, C.c_int32, C.c_int32, C.c_uint64, C.POINTER(Params),
                                 C.c_void_p, C.c_double, C.c_void_p]
        L.ref_pairing.argtypes = [C.c_void_p] * 5 + [C.POINTER(Params), C.POINTER(Cell)]
        L.ref_quartic.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_double)]
        _lib = L
    return _lib


def params(src=None, **over) -> Params:
    """Referee parameters from defaults, from any object with the ten attributes (e.g. the other sides' structs), or overrides."""
    p = Params(**DEFAULTS)
    if src is not None:
        for n in PARAM_NAMES:
            setattr(p, n, float(getattr(src, n)))
    for k, v in over.items():
        setattr(p, k, float(v))
    return p


def view(store) -> Events:
    ev = Events()
    ev.n_events, ev.stride, ev.event_base = store.n_events, store.stride, store.event_base
    base, rb = store.cols.ctypes.data, store.stride * 8
    for name, row in _ROWS.items():
        setattr(ev, name, base + row * rb)
    ev.flags = store.flags.ctypes.data
    ev._keep = store
    return ev


def smear(store, e: int, v: int, seed: int, p: Params | None = None):
    s, m = np.zeros(10), np.zeros(2)
    if lib().ref_smear(C.byref(view(store)), e, v, seed, C.byref(p or params()), s.ctypes.data, m.ctypes.data) != 0:
        raise ValueError("ref_smear: bad arguments")
    return s, m


def cell(store, e: int, v: int, a: int, seed: int, p: Params | None = None) -> Cell:
    out = Cell()
    if lib().ref_cell(C.byref(view(store)), e, v, a, seed, C.byref(p or params()), C.byref(out)) != 0:
        raise ValueError("ref_cell: bad arguments")
    return out


def pairing(lp, b, lm, bbar, met, p: Params | None = None) -> Cell:
    arrs = [np.ascontiguousarray(x, dtype=np.float64) for x in (lp, b, lm, bbar, met)]
    out = Cell()
    if lib().ref_pairing(*[a.ctypes.data for a in arrs], C.byref(p or params()), C.byref(out)) != 0:
        raise ValueError("ref_pairing: bad arguments")
    return out


def polish(store, e: int, v: int, a: int, seed: int, nu, nubar_z: float, p: Params | None = None):
    """binary128 Newton on the raw constraints from an FP64 point: (nu[3], nubar[3], neutrino term) or None."""
    nu = np.ascontiguousarray(nu, dtype=np.float64)
    out = np.zeros(7)
    it = lib().ref_polish(C.byref(view(store)), e, v, a, seed, C.byref(p or params()), nu.ctypes.data, float(nubar_z), out.ctypes.data)
    return None if it < 0 else (out[:3].copy(), out[3:6].copy(), float(out[6]))


def quartic(g):
    g = np.ascontiguousarray(g, dtype=np.float64)
    roots, m = np.zeros(4), C.c_double()
    n = lib().ref_quartic(g.ctypes.data, roots.ctypes.data, C.byref(m))
    return roots[:n].copy(), m.value


def nearest_root(cl: Cell, nu_xy):
    """Index of the exact root of the cell closest to an FP64 (p_x, p_y), or None."""
    if cl.n_roots == 0:
        return None
    d = [abs(cl.x[r] - nu_xy[0]) + abs(cl.y[r] - nu_xy[1]) for r in range(cl.n_roots)]
    return int(np.argmin(d))


def record_error(cl: Cell, r: int, rec) -> float:
    """max |component difference| of a record's nu / nubar against exact root r, relative to the largest exact component."""
    t = np.array([cl.nu[r][0], cl.nu[r][1], cl.nu[r][2], cl.nubar[r][0], cl.nubar[r][1], cl.nubar[r][2]])
    g = np.concatenate([np.asarray(rec["nu"], float), np.asarray(rec["nubar"], float)])
    return float(np.abs(g - t).max() / max(np.abs(t).max(), 1.0))
