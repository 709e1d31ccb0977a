"""ctypes binding of libhepf.so: same names as the C entry points, marshalling only (include/hepf.h)."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = os.path.join(_HERE, "libhepf.so")

# row offsets of the 64-row column block (same layout as the host store the generator writes)
ROW = dict(lep_px=0, lep_py=2, lep_pz=4, lep_e=6, lep_pt=8, lep_eta=10,
           jet_px=12, jet_py=20, jet_pz=28, jet_e=36, jet_pt=44, jet_eta=52,
           met_x=60, met_y=61, met=62, mll=63)
NROW = 64

BEST_DTYPE = np.dtype([("nu", "f8", 3), ("nubar", "f8", 3), ("m_top", "f8"), ("m_antitop", "f8"),
                       ("m_wplus", "f8"), ("m_wminus", "f8"), ("m_higgs", "f8"), ("loglik", "f8"),
                       ("variation", "i4"), ("jet_b", "i4"), ("jet_bbar", "i4"), ("jet_h1", "i4"),
                       ("jet_h2", "i4"), ("root", "i4"), ("status", "u4"), ("event", "u4")])
assert BEST_DTYPE.itemsize == 128


class HepfError(RuntimeError):
    pass


class _Events(C.Structure):
    _fields_ = [("n_events", C.c_int64), ("stride", C.c_int64), ("event_base", C.c_int64)] + \
               [(n, C.c_void_p) for n in ("lep_px", "lep_py", "lep_pz", "lep_e", "lep_pt", "lep_eta",
                                          "jet_px", "jet_py", "jet_pz", "jet_e", "jet_pt", "jet_eta",
                                          "met_x", "met_y", "met", "mll", "flags")]


class _Cut(C.Structure):
    _fields_ = [("kind", C.c_uint32), ("n", C.c_uint32), ("lo", C.c_double), ("hi", C.c_double)]


class Params(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("m_top", "m_w", "m_higgs", "sigma_higgs", "lambda_nu", "lep_sigma",
                                          "jet_stoch", "jet_const", "sigma_scale", "s_min")]


_lib = None


def lib_path() -> str:
    return _LIB


def load():
    """Load libhepf.so (fails loudly if it has not been built: there is no fallback path)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB):
            raise HepfError(f"{_LIB} is missing: run `python -m paper_2211_14346_b200.build` "
                            "(or __graft_entry__.build()) first; there is no CPU fallback")
        L = C.CDLL(_LIB)
        L.hepf_last_error.restype = C.c_char_p
        L.hepf_version.restype = C.c_char_p
        L.hepf_launch_count.restype = C.c_int64
        L.hepf_launch_count.argtypes = [C.c_int]
        L.hepf_select_workspace_bytes.restype = C.c_size_t
        L.hepf_select_workspace_bytes.argtypes = [C.c_int64]
        L.hepf_reconstruct_workspace_bytes.restype = C.c_size_t
        L.hepf_reconstruct_workspace_bytes.argtypes = [C.c_int64, C.c_int32]
        L.hepf_tth_host_arena_bytes.restype = C.c_size_t
        L.hepf_tth_host_arena_bytes.argtypes = [C.c_int64, C.c_int32]
        L.hepf_default_params.argtypes = [C.POINTER(Params)]
        L.hepf_select.argtypes = [C.POINTER(_Events), C.POINTER(_Cut), C.c_int, C.c_void_p, C.c_void_p, C.c_void_p,
                                  C.c_void_p, C.c_size_t, C.c_void_p]
        L.hepf_select_static.argtypes = [C.POINTER(_Events), C.POINTER(_Cut), C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.hepf_reconstruct_tth.argtypes = [C.POINTER(_Events), C.c_void_p, C.c_int64, C.c_int32, C.c_uint64,
                                           C.POINTER(Params), C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
        L.hepf_reconstruct_tth_n.argtypes = [C.POINTER(_Events), C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.c_uint64,
                                             C.POINTER(Params), C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
        L.hepf_philox_normal.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, C.c_void_p, C.c_void_p]
        L.hepf_tth_host.argtypes = [C.POINTER(_Events), C.POINTER(_Cut), C.c_int, C.c_int32, C.c_uint64,
                                    C.POINTER(Params), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                    C.c_size_t, C.c_void_p]
        L.hepf_chi2_semilep.argtypes = [C.POINTER(_Events), C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
        L.hepf_chi2_single_top.argtypes = [C.POINTER(_Events), C.c_void_p, C.c_int64, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.hepf_chi2_dilep.argtypes = [C.POINTER(_Events), C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.hepf_histogram.argtypes = [C.c_void_p, C.c_int64, C.c_int, C.c_double, C.c_double, C.c_int32, C.c_void_p, C.c_void_p]
        L.hepf_select_record.argtypes = [C.POINTER(_Events), C.POINTER(_Cut), C.c_int, C.c_void_p, C.c_void_p, C.c_void_p,
                                         C.c_void_p, C.c_double, C.c_void_p, C.c_size_t, C.c_void_p]
        L.hepf_tth_system.argtypes = [C.POINTER(_Events), C.c_void_p, C.c_int64, C.c_uint64, C.POINTER(Params), C.c_void_p, C.c_void_p]
        L.hepf_histogram_values.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_double, C.c_double, C.c_int32, C.c_void_p, C.c_void_p]
        L.hepf_cut_stats.argtypes = [C.POINTER(_Events), C.POINTER(_Cut), C.c_int, C.c_int64, C.c_void_p, C.c_void_p]
        L.hepf_plan_chain.argtypes = [C.POINTER(_Cut), C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_int), C.c_void_p]
        L.hepf_select_planned.argtypes = [C.POINTER(_Events), C.POINTER(_Cut), C.c_int, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p,
                                          C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
        L.hepf_select_planned_workspace_bytes.restype = C.c_size_t
        L.hepf_select_planned_workspace_bytes.argtypes = [C.c_int64]
        L.hepf_timing_enable.argtypes = [C.c_int]
        L.hepf_timing_ms.restype = C.c_double
        L.hepf_timing_ms.argtypes = [C.c_int, C.c_int]
        L.hepf_fp64_peak_probe.argtypes = [C.c_int, C.c_int, C.c_int64, C.c_void_p, C.c_void_p]
        _lib = L
    return _lib


def last_error() -> str:
    return load().hepf_last_error().decode()


def _check(rc: int, what: str):
    if rc != 0:
        raise HepfError(f"{what} failed ({rc}): {last_error()}")


def launch_count(reset: bool = False) -> int:
    return int(load().hepf_launch_count(int(reset)))


def default_params(**over) -> Params:
    p = Params()
    load().hepf_default_params(C.byref(p))
    for k, v in over.items():
        setattr(p, k, v)
    return p


def make_cuts(chain):
    arr = (_Cut * max(1, len(chain)))()
    for i, (kind, n, lo, hi) in enumerate(chain):
        arr[i] = _Cut(int(kind), int(n), float(lo), float(hi))
    return arr


def _stream_ptr(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _view(base_ptr: int, flags_ptr: int, n_events: int, stride: int, event_base: int) -> _Events:
    ev = _Events()
    ev.n_events, ev.stride, ev.event_base = n_events, stride, event_base
    for name, row in ROW.items():
        setattr(ev, name, base_ptr + row * stride * 8)
    ev.flags = flags_ptr
    return ev


class DeviceEvents:
    """SoA event store resident in HBM: one [64, stride] float64 tensor + one [stride] int32 (uint32 bits) tensor."""

    def __init__(self, cols, flags, n_events: int, event_base: int = 0):
        assert cols.is_cuda and cols.dim() == 2 and cols.shape[0] == NROW and cols.is_contiguous()
        self.cols, self.flags = cols, flags
        self.n_events, self.stride, self.event_base = int(n_events), int(cols.shape[1]), int(event_base)

    @classmethod
    def from_host(cls, store, device="cuda", non_blocking: bool = False):
        """Upload a host store (hepf_synth.EventStore or anything with cols/flags/n_events/event_base)."""
        import torch
        cols = torch.from_numpy(store.cols).to(device, non_blocking=non_blocking)
        flags = torch.from_numpy(store.flags.view(np.int32)).to(device, non_blocking=non_blocking)
        return cls(cols, flags, store.n_events, store.event_base)

    def view(self) -> _Events:
        return _view(self.cols.data_ptr(), self.flags.data_ptr(), self.n_events, self.stride, self.event_base)

    def subview(self, lo: int, hi: int) -> "DeviceEvents":
        """Events [lo, hi) of this store as a pointer-offset view (no copy): same columns, event_base + lo, so the records
        are those of the whole store (the smearing is keyed by the global index).  lo must be a multiple of 4 (16-byte
        alignment of every column, flags included); use sharding.shard_range for rank boundaries."""
        if lo % 4 or not 0 <= lo <= hi <= self.n_events:
            raise HepfError(f"subview [{lo}, {hi}): lo must be a multiple of 4 inside [0, {self.n_events}]")
        sub = object.__new__(DeviceEvents)
        sub.cols, sub.flags = self.cols, self.flags
        sub.n_events, sub.stride, sub.event_base, sub._off = hi - lo, self.stride, self.event_base + lo, getattr(self, "_off", 0) + lo
        sub.view = lambda: _view(self.cols.data_ptr() + 8 * sub._off, self.flags.data_ptr() + 4 * sub._off, sub.n_events,
                                 sub.stride, sub.event_base)
        return sub


def select(events: DeviceEvents, chain, *, with_cutflow: bool = True, out_idx=None, out_count=None, out_cutflow=None,
           ws=None, stream=None):
    """hepf_select: returns (out_idx[int32 tensor, capacity n_events], out_count[int64 tensor(1)], cutflow or None).
    Asynchronous on the stream; read ``out_count.item()`` (a sync) to learn how many entries of out_idx are valid."""
    import torch
    L = load()
    dev = events.cols.device
    n = events.n_events
    if out_idx is None:
        out_idx = torch.empty(max(n, 1), dtype=torch.int32, device=dev)
    if out_count is None:
        out_count = torch.zeros(1, dtype=torch.int64, device=dev)
    if with_cutflow and out_cutflow is None:
        out_cutflow = torch.zeros(max(len(chain), 1), dtype=torch.int64, device=dev)
    need = L.hepf_select_workspace_bytes(n)
    if ws is None or ws.numel() < need:
        ws = torch.empty(max(need, 16), dtype=torch.uint8, device=dev)
    ev = events.view()
    rc = L.hepf_select(C.byref(ev), make_cuts(chain), len(chain), out_idx.data_ptr(), out_count.data_ptr(),
                       out_cutflow.data_ptr() if with_cutflow else None, ws.data_ptr(), ws.numel(), _stream_ptr(stream))
    _check(rc, "hepf_select")
    return out_idx, out_count, (out_cutflow[: len(chain)] if with_cutflow else None)


SELECT_STATIC_MAX_EVENTS = 4194304   # HEPF_SELECT_STATIC_MAX_EVENTS (include/hepf.h)


def select_static(events: DeviceEvents, chain, out_idx, out_count, out_cutflow=None, *, stream=None):
    """hepf_select_static: hepf_select with its scratch in the library's static device array.  The entry point allocates
    nothing, and neither does this wrapper: the caller passes every output (out_idx int32 [>= n_events], out_count int64 [1],
    out_cutflow int64 [>= len(chain)] or None).  At most SELECT_STATIC_MAX_EVENTS events; calls that overlap on the GPU race."""
    ev = events.view()
    rc = load().hepf_select_static(C.byref(ev), make_cuts(chain), len(chain), out_idx.data_ptr(), out_count.data_ptr(),
                                   out_cutflow.data_ptr() if out_cutflow is not None else None, _stream_ptr(stream))
    _check(rc, "hepf_select_static")
    return out_idx, out_count, (out_cutflow[: len(chain)] if out_cutflow is not None else None)


def select_record(events: DeviceEvents, chain, derived_default: float = 0.0, *, with_cutflow: bool = True, ws=None, stream=None):
    """hepf_select_record: (out_idx, out_count, cutflow or None, derived) — derived is the float64 column [n_events] the
    chain's HEPF_CUT_MET_GT_RECORD cut writes (met * hi for the events that pass it, derived_default for the others)."""
    import torch
    L = load()
    dev = events.cols.device
    n = events.n_events
    out_idx = torch.empty(max(n, 1), dtype=torch.int32, device=dev)
    out_count = torch.zeros(1, dtype=torch.int64, device=dev)
    out_cutflow = torch.zeros(max(len(chain), 1), dtype=torch.int64, device=dev) if with_cutflow else None
    derived = torch.empty(max(n, 2), dtype=torch.float64, device=dev)
    need = L.hepf_select_workspace_bytes(n)
    if ws is None or ws.numel() < need:
        ws = torch.empty(max(need, 16), dtype=torch.uint8, device=dev)
    ev = events.view()
    rc = L.hepf_select_record(C.byref(ev), make_cuts(chain), len(chain), out_idx.data_ptr(), out_count.data_ptr(),
                              out_cutflow.data_ptr() if with_cutflow else None, derived.data_ptr(), derived_default,
                              ws.data_ptr(), ws.numel(), _stream_ptr(stream))
    _check(rc, "hepf_select_record")
    return out_idx, out_count, (out_cutflow[: len(chain)] if with_cutflow else None), derived[:n]


def tth_system(events: DeviceEvents, best, n: int, seed: int, params: Params | None = None, *, out=None, stream=None):
    """hepf_tth_system: float64 tensor [n, 2] = (m_ttH, pT_ttH) of each record of `best` (NaN where there is no solution)."""
    import torch
    if out is None:
        out = torch.empty((max(n, 1), 2), dtype=torch.float64, device=best.device)
    ev = events.view()
    rc = load().hepf_tth_system(C.byref(ev), best.data_ptr(), n, seed, C.byref(params) if params is not None else None,
                                out.data_ptr(), _stream_ptr(stream))
    _check(rc, "hepf_tth_system")
    return out[:n]


def histogram_values(values, lo: float, hi: float, nbins: int, *, out=None, stream=None):
    """hepf_histogram_values of a 1-D float64 device tensor (any stride): int64 tensor [nbins + 2]."""
    import torch
    if out is None:
        out = torch.empty(nbins + 2, dtype=torch.int64, device=values.device)
    stride = values.stride(0) if values.numel() > 1 else 1
    rc = load().hepf_histogram_values(values.data_ptr(), stride, values.shape[0], lo, hi, nbins, out.data_ptr(), _stream_ptr(stream))
    _check(rc, "hepf_histogram_values")
    return out


def cut_stats(events: DeviceEvents, chain, sample_every: int = 1, *, stream=None):
    """hepf_cut_stats: int64 device tensor [n_cuts + 1]: per-cut pass counts (each cut on its own) and the number of events looked at."""
    import torch
    out = torch.zeros(len(chain) + 1, dtype=torch.int64, device=events.cols.device)
    ev = events.view()
    rc = load().hepf_cut_stats(C.byref(ev), make_cuts(chain), len(chain), sample_every, out.data_ptr(), _stream_ptr(stream))
    _check(rc, "hepf_cut_stats")
    return out


def plan_chain(chain, pass_frac, dep_mask=None):
    """hepf_plan_chain (host only): (order, split, planned bytes/event, one-phase bytes/event)."""
    n = len(chain)
    pf = np.ascontiguousarray(pass_frac, dtype=np.float64)
    dm = np.ascontiguousarray(dep_mask, dtype=np.uint32) if dep_mask is not None else None
    order = np.zeros(max(n, 1), dtype=np.int32); split = C.c_int(0); by = np.zeros(2)
    rc = load().hepf_plan_chain(make_cuts(chain), n, pf.ctypes.data, dm.ctypes.data if dm is not None else None, order.ctypes.data,
                                C.byref(split), by.ctypes.data)
    _check(rc, "hepf_plan_chain")
    return [int(x) for x in order[:n]], int(split.value), float(by[0]), float(by[1])


def select_planned(events: DeviceEvents, chain, order, split: int, *, with_cutflow: bool = False, out_idx=None, out_count=None, ws=None, stream=None):
    """hepf_select_planned: (out_idx, out_count, cutflow in executed order or None)."""
    import torch
    L = load()
    dev = events.cols.device
    n = events.n_events
    if out_idx is None:
        out_idx = torch.empty(max(n, 1), dtype=torch.int32, device=dev)
    if out_count is None:
        out_count = torch.zeros(1, dtype=torch.int64, device=dev)
    cf = torch.zeros(max(len(chain), 1), dtype=torch.int64, device=dev) if with_cutflow else None
    need = L.hepf_select_planned_workspace_bytes(n)
    if ws is None or ws.numel() < need:
        ws = torch.empty(max(need, 256), dtype=torch.uint8, device=dev)
    ev = events.view()
    od = np.ascontiguousarray(order, dtype=np.int32)
    rc = L.hepf_select_planned(C.byref(ev), make_cuts(chain), len(chain), od.ctypes.data, split, out_idx.data_ptr(), out_count.data_ptr(),
                               cf.data_ptr() if with_cutflow else None, ws.data_ptr(), ws.numel(), _stream_ptr(stream))
    _check(rc, "hepf_select_planned")
    return out_idx, out_count, (cf[: len(chain)] if with_cutflow else None)


def reconstruct_tth(events: DeviceEvents, idx, n_idx: int, n_variations: int, seed: int, params: Params | None = None,
                    *, out_best=None, ws=None, stream=None):
    """hepf_reconstruct_tth: returns a uint8 tensor [n_idx, 128] of hepf_best_t records (see BEST_DTYPE)."""
    import torch
    L = load()
    if out_best is None:
        out_best = torch.empty((max(n_idx, 1), 128), dtype=torch.uint8, device=events.cols.device)
    need = L.hepf_reconstruct_workspace_bytes(max(n_idx, 0), n_variations)
    if ws is None or ws.numel() < need:
        ws = torch.empty(max(need, 16), dtype=torch.uint8, device=events.cols.device)
    ev = events.view()
    rc = L.hepf_reconstruct_tth(C.byref(ev), idx.data_ptr(), n_idx, n_variations, seed,
                                C.byref(params) if params is not None else None, out_best.data_ptr(), ws.data_ptr(),
                                ws.numel(), _stream_ptr(stream))
    _check(rc, "hepf_reconstruct_tth")
    return out_best[:n_idx]


def reconstruct_tth_n(events: DeviceEvents, idx, n_idx_device, n_idx_cap: int, n_variations: int, seed: int,
                      params: Params | None = None, *, out_best=None, ws=None, stream=None):
    """hepf_reconstruct_tth_n: the list length is the int64 device tensor `n_idx_device` (hepf_select's out_count); returns
    the uint8 tensor [n_idx_cap, 128] of which the first n_idx_device records are written.  No host synchronisation."""
    import torch
    L = load()
    if out_best is None:
        out_best = torch.empty((max(n_idx_cap, 1), 128), dtype=torch.uint8, device=events.cols.device)
    need = L.hepf_reconstruct_workspace_bytes(max(n_idx_cap, 0), n_variations)
    if ws is None or ws.numel() < need:
        ws = torch.empty(max(need, 16), dtype=torch.uint8, device=events.cols.device)
    ev = events.view()
    rc = L.hepf_reconstruct_tth_n(C.byref(ev), idx.data_ptr(), n_idx_device.data_ptr(), n_idx_cap, n_variations, seed,
                                  C.byref(params) if params is not None else None, out_best.data_ptr(), ws.data_ptr(),
                                  ws.numel(), _stream_ptr(stream))
    _check(rc, "hepf_reconstruct_tth_n")
    return out_best


def best_to_numpy(out_best) -> np.ndarray:
    return out_best.cpu().numpy().reshape(-1).view(BEST_DTYPE)


def philox_normal(seed: int, counter: int, n: int, *, out=None, device="cuda", stream=None):
    """hepf_philox_normal: out[i] = Z[counter + i] (float64 tensor)."""
    import torch
    L = load()
    if out is None:
        out = torch.empty(n, dtype=torch.float64, device=device)
    rc = L.hepf_philox_normal(seed, counter, n, out.data_ptr(), _stream_ptr(stream))
    _check(rc, "hepf_philox_normal")
    return out


def tth_host_arena_bytes(n_events: int, n_variations: int) -> int:
    return int(load().hepf_tth_host_arena_bytes(n_events, n_variations))


def tth_host(store, chain, n_variations: int, seed: int, params: Params | None = None, *, arena=None, out_best=None,
             out_idx=None, stream=None):
    """hepf_tth_host: whole path from HOST buffers (store.cols / store.flags are numpy arrays or pinned torch CPU
    tensors).  Returns (idx[n_sel] uint32, best[n_sel] BEST_DTYPE, cutflow int64[n_cuts])."""
    import torch
    L = load()
    n = store.n_events
    cols_ptr = store.cols.data_ptr() if hasattr(store.cols, "data_ptr") else store.cols.ctypes.data
    flags_ptr = store.flags.data_ptr() if hasattr(store.flags, "data_ptr") else store.flags.ctypes.data
    ev = _view(cols_ptr, flags_ptr, n, store.stride, store.event_base)
    need = L.hepf_tth_host_arena_bytes(n, n_variations)
    if arena is None or arena.numel() < need:
        arena = torch.empty(need, dtype=torch.uint8, device="cuda")
    if out_best is None:
        out_best = np.empty(max(n, 1), dtype=BEST_DTYPE)
    if out_idx is None:
        out_idx = np.empty(max(n, 1), dtype=np.uint32)
    count = np.zeros(1, dtype=np.int64)
    cutflow = np.zeros(max(len(chain), 1), dtype=np.int64)
    ptr = lambda a: a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data
    rc = L.hepf_tth_host(C.byref(ev), make_cuts(chain), len(chain), n_variations, seed,
                         C.byref(params) if params is not None else None, ptr(out_idx), ptr(out_best),
                         count.ctypes.data, cutflow.ctypes.data, arena.data_ptr(), arena.numel(), _stream_ptr(stream))
    _check(rc, "hepf_tth_host")
    n_sel = int(count[0])
    return out_idx[:n_sel], out_best[:n_sel], cutflow[: len(chain)]


def fp64_peak_probe(blocks: int, threads: int, fma_per_thread: int, sink, stream=None):
    rc = load().hepf_fp64_peak_probe(blocks, threads, fma_per_thread, sink.data_ptr(), _stream_ptr(stream))
    _check(rc, "hepf_fp64_peak_probe")


def timing_enable(on: bool = True):
    load().hepf_timing_enable(int(on))


def timing_ms(from_slot: int, to_slot: int) -> float:
    """Elapsed device milliseconds between two of the library's timing slots (see include/hepf.h)."""
    return float(load().hepf_timing_ms(from_slot, to_slot))


HIST_FIELDS = dict(m_top=0, m_antitop=1, m_wplus=2, m_wminus=3, m_higgs=4, loglik=5, nu_pt=6, nubar_pt=7, variation=8)


def histogram(best, n: int, field: str, lo: float, hi: float, nbins: int, *, out=None, stream=None):
    """hepf_histogram: int64 tensor [nbins + 2] (underflow, bins, overflow) of `field` over the solved records of
    `best` (the uint8 [n, 128] tensor hepf_reconstruct_tth filled)."""
    import torch
    if out is None:
        out = torch.empty(nbins + 2, dtype=torch.int64, device=best.device)
    rc = load().hepf_histogram(best.data_ptr(), n, HIST_FIELDS[field], lo, hi, nbins, out.data_ptr(), _stream_ptr(stream))
    _check(rc, "hepf_histogram")
    return out


CHI2_DTYPE = np.dtype([("chi2", "f8"), ("nu_pz", "f8"), ("m_top_lep", "f8"), ("m_top_had", "f8"), ("m_w_lep", "f8"),
                       ("m_w_had", "f8"), ("jet_b_lep", "i4"), ("jet_b_had", "i4"), ("jet_q1", "i4"), ("jet_q2", "i4"),
                       ("solution", "i4"), ("n_comb", "i4"), ("status", "u4"), ("event", "u4")])
assert CHI2_DTYPE.itemsize == 80


def chi2_semilep(events: DeviceEvents, idx, n_idx: int, params=None, *, out=None, stream=None):
    """hepf_chi2_semilep: uint8 tensor [n_idx, 80] of hepf_chi2_t records (see CHI2_DTYPE); params = (m_top, m_w,
    sigma_top, sigma_w) or None for the paper's values."""
    import torch
    if out is None:
        out = torch.empty((max(n_idx, 1), 80), dtype=torch.uint8, device=events.cols.device)
    ev = events.view()
    par = (C.c_double * 4)(*params) if params is not None else None
    rc = load().hepf_chi2_semilep(C.byref(ev), idx.data_ptr(), n_idx, par, out.data_ptr(), _stream_ptr(stream))
    _check(rc, "hepf_chi2_semilep")
    return out[:n_idx]


def chi2_single_top(events: DeviceEvents, idx, n_idx: int, mode: int, params=None, *, out=None, stream=None):
    """hepf_chi2_single_top: mode 1 = t-channel, mode 2 = Wt; uint8 tensor [n_idx, 80] of hepf_chi2_t records."""
    import torch
    if out is None:
        out = torch.empty((max(n_idx, 1), 80), dtype=torch.uint8, device=events.cols.device)
    ev = events.view()
    par = (C.c_double * 4)(*params) if params is not None else None
    rc = load().hepf_chi2_single_top(C.byref(ev), idx.data_ptr(), n_idx, mode, par, out.data_ptr(), _stream_ptr(stream))
    _check(rc, "hepf_chi2_single_top")
    return out[:n_idx]


CHI2_DILEP_DTYPE = np.dtype([("chi2", "f8"), ("nu", "f8", 3), ("nubar", "f8", 3), ("m_top", "f8"), ("m_antitop", "f8"),
                             ("m_wplus", "f8"), ("m_wminus", "f8"), ("jet_b", "i4"), ("jet_bbar", "i4"), ("grid_x", "i4"),
                             ("grid_y", "i4"), ("sol_nu", "i4"), ("sol_nubar", "i4"), ("n_comb", "i4"), ("status", "u4"),
                             ("event", "u4"), ("pad_", "i4")])
assert CHI2_DILEP_DTYPE.itemsize == 128


class _Split(C.Structure):
    _fields_ = [("split_range", C.c_double), ("split_n", C.c_int32), ("pad_", C.c_int32)]


def chi2_dilep(events: DeviceEvents, idx, n_idx: int, params=None, split=None, *, out=None, stream=None):
    """hepf_chi2_dilep: uint8 tensor [n_idx, 128] of hepf_chi2_dilep_t records (see CHI2_DILEP_DTYPE); params = (m_top, m_w,
    sigma_top, sigma_w) or None; split = (split_range, split_n) or None (160 GeV, 32)."""
    import torch
    ev = events.view()
    if out is None:
        out = torch.empty((max(n_idx, 1), 128), dtype=torch.uint8, device=events.cols.device)
    par = (C.c_double * 4)(*params) if params is not None else None
    sp = _Split(float(split[0]), int(split[1]), 0) if split is not None else None
    rc = load().hepf_chi2_dilep(C.byref(ev), idx.data_ptr(), n_idx, par, C.byref(sp) if sp is not None else None,
                                out.data_ptr(), _stream_ptr(stream))
    _check(rc, "hepf_chi2_dilep")
    return out[:n_idx]
