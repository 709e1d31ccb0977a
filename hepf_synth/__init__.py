"""hepf_synth — seeded synthetic inputs shared by the CUDA path and the oracle (data only).

Holds no arithmetic of the method (no Philox, cuts, conics, solver, score): it generates event
columns (``gen.c``), describes the five BASELINE.json configs (cut chains are *data*: descriptor
tuples) and owns the host-side column layout.  Recipe: SURVEY.md §8(d) / DESIGN.md "Inputs".
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libhepf_synth.so")

NROW = 64          # double columns per event (see gen.c header)
NJ = 8             # jet slots
ROW = dict(lep_px=0, lep_py=2, lep_pz=4, lep_e=6, lep_pt=8, lep_eta=10,
           jet_px=12, jet_py=20, jet_pz=28, jet_e=36, jet_pt=44, jet_eta=52,
           met_x=60, met_y=61, met=62, mll=63)

# cut kinds (include/hepf.h)
NLEP_EQ, LEP_OS, LEP_PT_GT, LEP_ABSETA_LT, NJET_GE, NBJET_GE, MET_GT, MLL_GT, MLL_OUTSIDE = range(1, 10)
INF = float("inf")


def build(force: bool = False) -> str:
    src = os.path.join(_HERE, "gen.c")
    if force or not os.path.exists(_LIB_PATH) or os.path.getmtime(_LIB_PATH) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", _LIB_PATH, src, "-lm"])
    return _LIB_PATH


class _GenCfg(ctypes.Structure):
    _fields_ = [("n_events", ctypes.c_int64), ("first_event", ctypes.c_int64), ("stride", ctypes.c_int64),
                ("seed", ctypes.c_uint64), ("n_fake_b", ctypes.c_int32), ("closure", ctypes.c_int32),
                ("bkg_frac", ctypes.c_double), ("semilep", ctypes.c_int32), ("pad_", ctypes.c_int32)]


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.hepf_synth_generate.restype = ctypes.c_int
        _lib.hepf_synth_generate.argtypes = [ctypes.POINTER(_GenCfg), ctypes.c_void_p, ctypes.c_void_p,
                                             ctypes.c_void_p]
    return _lib


@dataclass
class EventStore:
    """Host SoA event store: ``cols[NROW, stride]`` float64 + ``flags[stride]`` uint32."""
    n_events: int
    stride: int
    event_base: int
    cols: np.ndarray
    flags: np.ndarray
    truth: np.ndarray | None = None

    def col(self, name: str, slot: int = 0) -> np.ndarray:
        return self.cols[ROW[name] + slot, : self.n_events]

    def slice(self, lo: int, hi: int) -> "EventStore":
        """Copy of events [lo, hi) as a standalone store whose global indices start at event_base+lo."""
        n = hi - lo
        stride = n + (n & 1)
        cols = np.zeros((NROW, stride), dtype=np.float64)
        cols[:, :n] = self.cols[:, lo:hi]
        flags = np.zeros(stride, dtype=np.uint32)
        flags[:n] = self.flags[lo:hi]
        truth = None if self.truth is None else self.truth[lo:hi].copy()
        return EventStore(n, stride, self.event_base + lo, cols, flags, truth)


def generate(n_events: int, seed: int, *, n_fake_b: int = 0, bkg_frac: float = 0.0, closure: bool = False,
             first_event: int = 0, with_truth: bool = True, semilep: bool = False) -> EventStore:
    lib = _load()
    stride = n_events + (n_events & 1)
    stride = max(stride, 2)
    cols = np.zeros((NROW, stride), dtype=np.float64)
    flags = np.zeros(stride, dtype=np.uint32)
    truth = np.zeros((n_events, 12), dtype=np.float64) if with_truth else None
    cfg = _GenCfg(n_events, first_event, stride, seed, n_fake_b, int(closure), bkg_frac, int(semilep), 0)
    rc = lib.hepf_synth_generate(ctypes.byref(cfg), cols.ctypes.data, flags.ctypes.data,
                                 truth.ctypes.data if truth is not None else None)
    if rc != 0:
        raise RuntimeError(f"hepf_synth_generate failed: {rc}")
    return EventStore(n_events, stride, first_event, cols, flags, truth)


@dataclass
class Config:
    """One BASELINE.json config made concrete."""
    name: str
    n_events: int
    gen_seed: int
    reco_seed: int
    n_variations: int
    cuts: list = field(default_factory=list)     # (kind, n, lo, hi)
    n_fake_b: int = 0
    bkg_frac: float = 0.0

    def events(self, n_events: int | None = None, first_event: int = 0, with_truth: bool = False) -> EventStore:
        return generate(self.n_events if n_events is None else n_events, self.gen_seed, n_fake_b=self.n_fake_b,
                        bkg_frac=self.bkg_frac, first_event=first_event, with_truth=with_truth)


# configs[1] chain (BASELINE.json configs[0]): 2 OS leptons pT>25, >=4 jets pT>25, MET>30
CHAIN_BASE = [(NLEP_EQ, 2, 0.0, 0.0), (LEP_OS, 0, 0.0, 0.0), (LEP_PT_GT, 0, 25.0, 0.0),
              (NJET_GE, 4, 25.0, INF), (MET_GT, 0, 30.0, 0.0)]
# configs[4] tightened 8-cut chain (kinds from PAPER.md:246-262 §6.1); thresholds frozen in BASELINE.md §5
CHAIN_TIGHT8 = [(NLEP_EQ, 2, 0.0, 0.0), (LEP_OS, 0, 0.0, 0.0), (LEP_PT_GT, 0, 30.0, 0.0),
                (LEP_ABSETA_LT, 0, 0.0, 2.5), (NJET_GE, 4, 35.0, 2.5), (NBJET_GE, 4, 35.0, 2.5),
                (MET_GT, 0, 55.0, 0.0), (MLL_GT, 0, 40.0, 0.0)]

CONFIGS = {
    1: Config("cfg1: 1e4 ev, 4b, V=16", 10_000, 1, 0x5EED0001, 16, CHAIN_BASE),
    2: Config("cfg2: 1e6 ev, 4b, V=64", 1_000_000, 2, 0x5EED0002, 64, CHAIN_BASE),
    3: Config("cfg3: 1e6 ev, 6b, V=256", 1_000_000, 3, 0x5EED0003, 256, CHAIN_BASE, n_fake_b=2),
    4: Config("cfg4: 2e7 ev, 30% bkg, 8 cuts, V=16", 20_000_000, 4, 0x5EED0004, 16, CHAIN_TIGHT8, bkg_frac=0.3),
}
PHILOX_CFG5 = dict(seed=7, counter=0, n=1 << 32, prefix=1 << 20)
