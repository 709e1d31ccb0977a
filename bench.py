#!/usr/bin/env python
"""bench.py — smeared ttH reconstructions/s on BASELINE.json configs[1] (1e6 events, 4 b-jets, V = 64, FP64).

A step is one pass of the whole hot path over the batch: hepf_select (cut chain + compaction) followed by
hepf_reconstruct_tth_n (Philox/Box-Muller smearing, dilepton solve, score, argmax; the list length stays on the device)
for every surviving event.  `value` counts event x variation x pairing solves per second with the inputs resident in
HBM; `e2e` is the same metric through hepf_tth_host (host buffers in, results out, copies inside the timed region).
The default run also times the other configs of BASELINE.json (cfg3, cfg4, cfg5) and reports them under `configs`.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload cfg1|cfg2|cfg3|cfg4|cfg5|chi2|chi2_dilep]
Under torchrun every rank runs its own shard (events keyed by global index, no data-path collective): weak scaling.
Everything printed is measured in this run, except the per-solve FP64 instruction counts and the DRAM traffic of the
search kernels, which only ncu can count: they are read from profiles/r02_fp64_ops.json and used only if that file's hash
of the kernel sources matches the tree (otherwise the fields say so and the fraction falls back to the frozen round-1 count).
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import hepf_synth as hs  # noqa: E402

METRIC = "smeared ttH reconstructions/sec (event x assignment x variation)"
UNIT = "reconstructions/s"
# FP64 roof of one B200 from the guide's unit counts: 148 SMs x 64 FP64 lanes/clk x clocks.max.sm
FP64_LANES_PER_SM = 64
OPS_FILE = os.path.join(ROOT, "profiles", "r02_fp64_ops.json")
KERNEL_SOURCES = ("paper_2211_14346_b200/csrc/hepf_reco.cu", "paper_2211_14346_b200/csrc/hepf_common.cuh")


def kernel_source_hash() -> str:
    h = hashlib.sha256()
    for rel in KERNEL_SOURCES:
        with open(os.path.join(ROOT, rel), "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def load_profiled_ops() -> dict:
    """ncu-counted FP64 thread instructions per solve of the search kernels (profiles/r02_fp64_ops.json).  `current` is True
    only if the file was written for exactly these kernel sources."""
    try:
        d = json.load(open(OPS_FILE))
    except (OSError, ValueError):
        return {"current": False, "kernels": {}, "algorithmic_fp64_ops_per_solve": {}, "file": None}
    d["current"] = d.get("source_sha256") == kernel_source_hash()
    d["file"] = os.path.relpath(OPS_FILE, ROOT)
    return d


def search_kernel_name(V: int, nb6: bool) -> str:
    """The instantiation hepf_reconstruct_tth launches for V variations (hepf_reco.cu, reconstruct_impl): chunks of 32 variations
    (16 for n_b = 5, 6) unless that wastes more than an eighth of the last chunk's lanes, then 16 (8), and 8 for V <= 8."""
    waste32 = ((V + 31) & ~31) - V
    if V <= 2:
        vc4, vc6 = 1, 1
    elif V <= 8:
        vc4, vc6 = 8, 8
    elif 8 * waste32 > V:
        vc4, vc6 = 16, 8
    else:
        vc4, vc6 = 32, 16
    return f"reco_search_kernel<{vc6},6>" if nb6 else f"reco_search_kernel<{vc4},4>"


def chain_bytes_per_event(chain) -> int:
    """Algorithmic bytes hepf_select must read per event: flags + the columns the chain names."""
    need = set()
    for kind, *_ in chain:
        if kind == hs.LEP_PT_GT: need.add("lep_pt")
        elif kind == hs.LEP_ABSETA_LT: need.add("lep_eta")
        elif kind in (hs.NJET_GE, hs.NBJET_GE): need.update(("jet_pt", "jet_eta"))
        elif kind == hs.MET_GT: need.add("met")
        elif kind in (hs.MLL_GT, hs.MLL_OUTSIDE): need.add("mll")
    size = {"lep_pt": 16, "lep_eta": 16, "jet_pt": 64, "jet_eta": 64, "met": 8, "mll": 8}
    return 4 + sum(size[c] for c in need)


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p)).get("hbm_gbs", 6650.0)), "MEASURED_PEAKS.json hbm_gbs (copy, read+write)"
    return 6650.0, "fallback 6650 GB/s (B200_PROFILING.md)"


def time_philox(hepf, n, steps, warmup):
    import torch
    out = torch.empty(n, dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream()
    for _ in range(warmup):
        hepf.philox_normal(hs.PHILOX_CFG5["seed"], 0, n, out=out, stream=stream)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        hepf.philox_normal(hs.PHILOX_CFG5["seed"], 0, n, out=out, stream=stream)
    e1.record(stream)
    torch.cuda.synchronize()
    del out
    ms = e0.elapsed_time(e1) / steps
    hbm, src = hbm_peak()
    gbs = 8.0 * n / (ms * 1e-3) / 1e9
    return {"ms_per_step": ms, "value": n / (ms * 1e-3), "unit": "normals/s",
            "workload": f"cfg5: {n} normals, seed 7, counter 0",
            "roofline": {"bound": "hbm", "kernel": "philox_normal_pairs_kernel", "achieved": gbs, "peak": hbm, "unit": "GB/s",
                         "frac": gbs / hbm, "traffic": None, "algorithmic_bytes": 8.0 * n, "kernel_ms": ms, "peak_source": src}}


def run_philox(args):
    """--workload cfg5: standalone hepf_philox_normal stream (BASELINE.json configs[4]), normals/s and GB/s written."""
    import torch
    import paper_2211_14346_b200 as hepf
    hepf.load()
    torch.cuda.set_device(0)
    n = args.events or hs.PHILOX_CFG5["n"]
    W = max(3, args.warmup)
    r = time_philox(hepf, n, args.steps, W)
    print(json.dumps({"metric": "standard-normal FP64 draws/sec (Philox4x32-10 + Box-Muller)", "value": r["value"],
                      "unit": "normals/s", "n_gpus": 1, "steps": args.steps, "warmup": W, "ms_per_step": r["ms_per_step"],
                      "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": r["workload"], "l2": "34 GB written per step, far larger than L2"},
                      "gpu_launches": args.steps, "roofline": r["roofline"]}))


def run_chi2(args):
    """--workload chi2: hepf_chi2_semilep (eq. 1) on synthetic semileptonic ttbar events."""
    import torch
    import paper_2211_14346_b200 as hepf
    hepf.load()
    torch.cuda.set_device(0)
    n = args.events or 4_000_000
    st = hs.generate(n, 11, semilep=True, with_truth=False)
    dev = hepf.DeviceEvents.from_host(st)
    idx_t = torch.arange(n, dtype=torch.int32, device="cuda")
    out = torch.empty((n, 80), dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()
    for _ in range(max(3, args.warmup)):
        hepf.chi2_semilep(dev, idx_t, n, out=out, stream=stream)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        hepf.chi2_semilep(dev, idx_t, n, out=out, stream=stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    f = st.flags[:n].astype(np.int64); nj = np.minimum((f >> 8) & 15, 8)
    # algorithmic bytes: idx 4 + flags 4 + lepton 32 + MET 16 + 32 per jet that is a candidate (<= 4 tagged + <= 4 untagged) + 80 out
    by = float((4 + 4 + 32 + 16 + 80) * n + 32 * nj.sum())
    hbm, src = hbm_peak()
    gbs = by / (ms * 1e-3) / 1e9
    print(json.dumps({"metric": "chi2-reconstructed semileptonic ttbar events/sec", "value": n / (ms * 1e-3), "unit": "events/s",
                      "n_gpus": 1, "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": ms, "higher_is_better": True,
                      "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": f"chi2: {n} semileptonic ttbar events (2 b + 2-4 untagged jets)",
                                 "l2": f"{by / 1e6:.0f} MB touched per step, larger than L2"},
                      "gpu_launches": args.steps,
                      "roofline": {"bound": "hbm", "kernel": "chi2_semilep_kernel", "achieved": gbs, "peak": hbm, "unit": "GB/s",
                                   "frac": gbs / hbm, "traffic": None, "algorithmic_bytes": by, "peak_source": src}}))


def run_chi2_dilep(args):
    """--workload chi2_dilep: hepf_chi2_dilep (eq. 1, dileptonic final state; R15) on the cfg2 generator's
    events: a 32 x 32 scan of the MET split per event, 12 ordered b pairs, up to 4 p_z combinations per point."""
    import torch
    import paper_2211_14346_b200 as hepf
    from paper_2211_14346_b200.binding import CHI2_DILEP_DTYPE
    hepf.load()
    torch.cuda.set_device(0)
    n = args.events or 200_000
    st = hs.generate(n, 12, with_truth=False)
    dev = hepf.DeviceEvents.from_host(st)
    idx_t = torch.arange(n, dtype=torch.int32, device="cuda")
    out = torch.empty((n, 128), dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()
    W = max(3, args.warmup)
    for _ in range(W):
        hepf.chi2_dilep(dev, idx_t, n, out=out, stream=stream)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        hepf.chi2_dilep(dev, idx_t, n, out=out, stream=stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    rec = out.cpu().numpy().reshape(-1).view(CHI2_DILEP_DTYPE)
    combos = float(rec["n_comb"].astype(np.int64).sum())
    print(json.dumps({"metric": "chi2-reconstructed dileptonic ttbar events/sec (32 x 32 MET-split scan)", "value": n / (ms * 1e-3),
                      "unit": "events/s", "n_gpus": 1, "steps": args.steps, "warmup": W, "ms_per_step": ms, "higher_is_better": True,
                      "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": f"chi2_dilep: {n} dileptonic events, 4 b-tags, split grid 32 x 32 over +-160 GeV",
                                 "l2": "FP64-bound: one event (about 350 B) per warp and 1024 grid points of arithmetic; nothing to flush"},
                      "gpu_launches": args.steps, "chi2_evaluations_per_s": combos / (ms * 1e-3),
                      "grid_points_per_s": 1024.0 * float((rec["status"] == 1).sum()) / (ms * 1e-3)}))


def solves_of(store, idx, n_variations: int) -> int:
    """event x variation x pairing count of the listed events (A = n_b (n_b - 1) for applicable events)."""
    f = store.flags[idx].astype(np.int64)
    n_jet = np.minimum((f >> 8) & 15, 8)
    tags = (f >> 16) & ((1 << n_jet) - 1)
    n_b = np.minimum(np.array([bin(int(t)).count("1") for t in np.unique(tags)])[np.searchsorted(np.unique(tags), tags)], 6)
    ok = ((f & 15) == 2) & (((f >> 4) & 1) != ((f >> 5) & 1)) & (n_b >= 4)
    return int((n_b * (n_b - 1) * ok).sum()) * n_variations


class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "50"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.rows.append([x.strip() for x in ln.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def cpu_oracle_rate(store, idx, n_variations, seed, n_threads, target_s=10.0):
    """Time the oracle (a non-optimised checker: nested bisection, everything re-enumerated per root), as it stands, on a
    bounded sample of the same workload on the host cores.  A reported baseline; no speed-up claim may be derived from it."""
    import oracle
    probe = idx[:256 * n_threads]
    t0 = time.perf_counter(); oracle.reconstruct_tth(store, probe, n_variations, seed, n_threads=n_threads)
    dt = max(time.perf_counter() - t0, 1e-3)
    m = int(min(len(idx), max(len(probe), len(probe) * target_s / dt)))
    sample = idx[:m]
    t0 = time.perf_counter(); oracle.reconstruct_tth(store, sample, n_variations, seed, n_threads=n_threads)
    dt = time.perf_counter() - t0
    n_solves = solves_of(store, sample, n_variations)
    return {"value": n_solves / dt, "unit": UNIT, "cores": n_threads, "kind": "oracle",
            "note": "the oracle is a non-optimised checker (nested bisection, every Higgs pair re-enumerated per root): a reported baseline, no speed-up claim may be derived from it",
            "sample": f"first {m} selected events of the workload ({n_solves} solves, {dt:.1f} s wall, {n_threads} OpenMP thread(s) over events)"}


def run_reference(args, cfg, name):
    """--impl reference: the oracle is this tier's reference arm (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    cores = os.cpu_count() or 1
    n_ev = min(cfg.n_events, 200_000)
    store = cfg.events(n_ev)
    idx, _ = oracle.select(store, cfg.cuts)
    per_step = min(4000, max(16, len(idx) // 2))
    times, solves = [], 0
    for s in range(args.warmup + args.steps):
        sample = idx[(s * per_step) % max(1, len(idx) - per_step):][:per_step]
        t0 = time.perf_counter()
        oracle.reconstruct_tth(store, sample, cfg.n_variations, cfg.reco_seed, n_threads=cores)
        dt = time.perf_counter() - t0
        if s >= args.warmup:
            times.append(dt); solves += solves_of(store, sample, cfg.n_variations)
    total = sum(times)
    val = solves / total
    sample_txt = f"{per_step} selected events per step of the {name} workload, OpenMP over events on {cores} threads"
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
                      "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / max(1, args.steps),
                      "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": cfg.name, "n_variations": cfg.n_variations, "sample": sample_txt},
                      "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample_txt,
                                       "note": "non-optimised checker: a reported baseline, no speed-up claim may be derived from it"},
                      "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                      "gpu_launches": 0}))


class TthRun:
    """select -> reconstruct on one resident store, device-timed."""

    def __init__(self, hepf, binding, cfg, n_ev, first_event, V, params):
        import torch
        self.hepf, self.binding, self.cfg, self.V, self.params = hepf, binding, cfg, V, params
        self.store = cfg.events(n_ev, first_event=first_event)
        self.dev = hepf.DeviceEvents.from_host(self.store)
        n = self.n = self.store.n_events
        L = hepf.load()
        self.stream = torch.cuda.current_stream()
        self.out_idx = torch.empty(max(n, 1), dtype=torch.int32, device="cuda")
        self.out_count = torch.zeros(1, dtype=torch.int64, device="cuda")
        self.out_cf = torch.zeros(32, dtype=torch.int64, device="cuda")
        self.ws = torch.empty(int(L.hepf_select_workspace_bytes(n)) + 256, dtype=torch.uint8, device="cuda")
        self.out_best = torch.empty((max(n, 1), 128), dtype=torch.uint8, device="cuda")
        self.reco_ws = torch.empty(int(L.hepf_reconstruct_workspace_bytes(n, V)) + 256, dtype=torch.uint8, device="cuda")

    def step(self):
        """One pass of the hot path; nothing comes back to the host between the two calls."""
        h = self.hepf
        h.select(self.dev, self.cfg.cuts, out_idx=self.out_idx, out_count=self.out_count, out_cutflow=self.out_cf, ws=self.ws,
                 stream=self.stream)
        h.reconstruct_tth_n(self.dev, self.out_idx, self.out_count, self.n, self.V, self.cfg.reco_seed, self.params,
                            out_best=self.out_best, ws=self.reco_ws, stream=self.stream)

    def measure(self, steps, warmup, barrier=None):
        import torch
        b = self.binding
        for _ in range(warmup):
            self.step()
        torch.cuda.synchronize()
        self.n_sel = int(self.out_count.item())
        self.idx_host = self.out_idx[:self.n_sel].cpu().numpy().view(np.uint32)
        self.n_solves = solves_of(self.store, self.idx_host, self.V)
        if barrier:
            barrier()
        torch.cuda.synchronize()
        self.hepf.launch_count(reset=True)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        b.timing_enable(True)
        k = {"search4": [], "search6": [], "finalize": [], "select": [], "select_eval": []}
        e0.record(self.stream)
        for _ in range(steps):
            self.step()
            # device time of each kernel of this step, from events the library records on the stream around its launches
            k["search4"].append(b.timing_ms(3, 4)); k["search6"].append(b.timing_ms(4, 5)); k["finalize"].append(b.timing_ms(5, 6))
            k["select"].append(b.timing_ms(0, 2)); k["select_eval"].append(b.timing_ms(0, 1))
        e1.record(self.stream)
        torch.cuda.synchronize()
        b.timing_enable(False)
        self.launches = int(self.hepf.launch_count())
        self.ms_total = e0.elapsed_time(e1)
        self.kernel_ms = {name: float(np.mean(v)) for name, v in k.items()}
        return self.ms_total / steps

    def rooflines(self, ms_per_step, sm_max_mhz, sms, prof):
        """FP64 lane-op roofline of the dominant search kernel + HBM roofline of select_eval."""
        km = self.kernel_ms
        nb6 = km["search6"] > km["search4"]
        name = search_kernel_name(self.V, nb6)
        ms_search = km["search6"] if nb6 else km["search4"]
        lane_peak = sms * FP64_LANES_PER_SM * sm_max_mhz * 1e6
        entry = prof["kernels"].get(name) if prof.get("current") else None
        alg = prof.get("algorithmic_fp64_ops_per_solve", {}).get("nb6" if nb6 else "nb4")
        roof = {"bound": "alu", "kernel": name, "unit": "T FP64 lane-op/s", "peak": lane_peak / 1e12,
                "peak_source": f"{sms} SMs x {FP64_LANES_PER_SM} FP64 lanes x {sm_max_mhz:.0f} MHz (DESIGN.md section 7)",
                "kernel_ms": ms_search, "kernel_share_of_step": ms_search / ms_per_step, "solves_per_launch": self.n_solves,
                "other_kernels_ms": {"reco_search_other_class": km["search4"] if nb6 else km["search6"],
                                     "select_eval+scatter": km["select"], "reco_finalize": km["finalize"]}}
        if entry:     # the kernel's own executed (predicated-on) FP64 thread instructions, counted by ncu on exactly these sources
            ops = entry["dadd"] + entry["dmul"] + entry["dfma"]
            rate = ops * self.n_solves / (ms_search * 1e-3)
            roof.update({"achieved": rate / 1e12, "frac": rate / lane_peak, "fp64_lane_ops_per_solve": ops,
                         "tflops_fma2": (ops + entry["dfma"]) * self.n_solves / (ms_search * 1e-3) / 1e12,
                         "ops_source": f"{prof['file']} ({entry.get('profile')}; kernel sources hash matches this tree)",
                         "traffic": entry.get("dram_bytes_per_launch") if entry.get("workload") == self.cfg.name.split(":")[0] else None,
                         "ncu_sm__pipe_fp64_cycles_active_pct": entry.get("ncu_sm__pipe_fp64_cycles_active_pct")})
        else:
            roof.update({"achieved": None, "frac": None, "traffic": None,
                         "ops_source": "no ncu count for these kernel sources (profiles/r02_fp64_ops.json absent or stale)"})
        if alg:       # the method's FP64 work, frozen: does not shrink when the kernel does
            rate = alg * self.n_solves / (ms_search * 1e-3)
            roof.update({"algorithmic_fp64_ops_per_solve": alg, "algorithmic_achieved": rate / 1e12, "algorithmic_frac": rate / lane_peak})
            if roof["frac"] is None:
                roof.update({"achieved": rate / 1e12, "frac": rate / lane_peak,
                             "ops_source": roof["ops_source"] + "; frac uses the frozen algorithmic count"})
        hbm, src = hbm_peak()
        sel_bytes = chain_bytes_per_event(self.cfg.cuts) * self.n + 4 * self.n_sel
        sel_ms = km["select_eval"]
        select = {"kernel": "select_eval_kernel", "events_per_s": self.n / (sel_ms * 1e-3), "bound": "hbm",
                  "achieved": sel_bytes / (sel_ms * 1e-3) / 1e9, "peak": hbm, "unit": "GB/s", "peak_source": src,
                  "frac": sel_bytes / (sel_ms * 1e-3) / 1e9 / hbm, "algorithmic_bytes": sel_bytes, "kernel_ms": sel_ms,
                  "eval+scatter_ms": km["select"]}
        return roof, select

    def planned_select(self, reps=20):
        """measured filter ratios -> hepf_plan_chain -> hepf_select_planned, timed against hepf_select; the
        same for a variant of the chain whose lepton-pT cut is tight enough for two phases to pay, and a forced split."""
        import torch
        h = self.hepf
        ws = torch.empty(int(h.load().hepf_select_planned_workspace_bytes(self.n)) + 256, dtype=torch.uint8, device="cuda")
        idx2 = torch.empty_like(self.out_idx); cnt2 = torch.zeros_like(self.out_count)

        def timed(f):
            for _ in range(3):
                f()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(self.stream)
            for _ in range(reps):
                f()
            e1.record(self.stream)
            torch.cuda.synchronize()
            return e0.elapsed_time(e1) / reps

        def one_chain(chain, force=None):
            stats = h.cut_stats(self.dev, chain, 16).cpu().numpy()
            p = stats[:-1] / max(1, stats[-1])
            order, split, planned_b, one_b = h.plan_chain(chain, p)
            if force:
                order, split = force
            ms_one = timed(lambda: h.select(self.dev, chain, with_cutflow=False, out_idx=self.out_idx, out_count=self.out_count, ws=self.ws, stream=self.stream))
            ms_two = timed(lambda: h.select_planned(self.dev, chain, order, split, out_idx=idx2, out_count=cnt2, ws=ws, stream=self.stream))
            m = int(cnt2.item())
            same = bool(m == int(self.out_count.item()) and torch.equal(idx2[:m], self.out_idx[:m]))
            return {"measured_pass_fractions": [round(float(x), 4) for x in p], "order": order, "split": split, "phases": 1 if split == len(chain) else 2,
                    "model_bytes_per_event": {"planned": planned_b, "one_phase": one_b}, "survivors": m,
                    "ms_hepf_select_no_cutflow": ms_one, "ms_hepf_select_planned": ms_two, "same_survivors": same}
        chain = list(self.cfg.cuts)
        out = {"planned": one_chain(chain), "note": "phase 1 (cuts order[:split]) over every event, phase 2 over phase 1's survivors only; PAPER.md:192-198"}
        jets = [c for c, cut in enumerate(chain) if cut[0] in (hs.NJET_GE, hs.NBJET_GE)]
        if jets and len(jets) < len(chain):
            rest = [c for c in range(len(chain)) if c not in jets]
            out["forced_jets_in_phase_2"] = one_chain(chain, force=(rest + jets, len(rest)))
        tight = [(k, n, 90.0, hi) if k == hs.LEP_PT_GT else (k, n, lo, hi) for (k, n, lo, hi) in chain]
        if tight != chain:
            out["tight_lepton_pt_90_variant"] = one_chain(tight)
        return out

    def free(self):
        import torch
        for a in ("dev", "out_idx", "out_best", "ws", "reco_ws", "store"):
            setattr(self, a, None)
        torch.cuda.empty_cache()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="hepf", choices=["hepf", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5", "chi2", "chi2_dilep"])
    ap.add_argument("--events", type=int, default=0, help="override the number of events per GPU (debugging)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra-configs", action="store_true", help="skip the cfg3 / cfg4 / cfg5 lines of the default run")
    ap.add_argument("--variations", type=int, default=0, help="override the workload's V (SURVEY 8(f) NEXT-1: 128 = ttH_scinp, 1024 = ttH_sci)")
    ap.add_argument("--sigma-scale", type=float, default=None, help="0 = no smearing, the paper's ttH_as variant")
    args = ap.parse_args()
    if args.workload == "cfg5":
        return run_philox(args)
    if args.workload == "chi2":
        return run_chi2(args)
    if args.workload == "chi2_dilep":
        return run_chi2_dilep(args)
    cfg = hs.CONFIGS[int(args.workload[3])]
    if args.impl == "reference":
        return run_reference(args, cfg, args.workload)

    import torch
    import torch.distributed as dist
    import paper_2211_14346_b200 as hepf
    from paper_2211_14346_b200 import binding

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback for the hepf path")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    hepf.load()
    W = max(3, args.warmup)
    n_ev = args.events or cfg.n_events
    V = args.variations or cfg.n_variations
    params = hepf.default_params(sigma_scale=args.sigma_scale) if args.sigma_scale is not None else None
    # weak scaling: rank r owns global events [r n, (r+1) n); the Philox keys use the global index
    run = TthRun(hepf, binding, cfg, n_ev, rank * n_ev, V, params)
    store, n, seed = run.store, run.n, cfg.reco_seed

    sampler = ClockSampler(local)
    sampler.start()
    ms_local = run.measure(args.steps, W, barrier=(dist.barrier if world > 1 else None))
    clocks = sampler.stop()
    n_sel, n_solves = run.n_sel, run.n_solves
    t = torch.tensor([run.ms_total], dtype=torch.float64, device="cuda")
    tot = torch.tensor([float(n_solves)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.barrier()
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    ms_per_step, all_solves = float(t.item()) / args.steps, float(tot.item())
    value = all_solves / (ms_per_step * 1e-3)

    # ---- end to end through the C ABI with host buffers (pinned), copies inside the timed region --------------
    pin_cols = torch.from_numpy(store.cols).pin_memory()
    pin_flags = torch.from_numpy(store.flags.view(np.int32)).pin_memory()
    hstore = hs.EventStore(n, store.stride, store.event_base, pin_cols, pin_flags)
    arena = torch.empty(binding.tth_host_arena_bytes(n, V) + 512, dtype=torch.uint8, device="cuda")
    hb = torch.empty((max(n, 1), 128), dtype=torch.uint8).pin_memory()
    hi = torch.empty(max(n, 1), dtype=torch.int32).pin_memory()
    stream = run.stream
    for _ in range(2):
        hepf.tth_host(hstore, cfg.cuts, V, seed, params, arena=arena, out_best=hb, out_idx=hi, stream=stream)
    e2e_steps = max(1, min(args.steps, 10))
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        hepf.tth_host(hstore, cfg.cuts, V, seed, params, arena=arena, out_best=hb, out_idx=hi, stream=stream)
    torch.cuda.synchronize()
    te = torch.tensor([(time.perf_counter() - t0) / e2e_steps], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
    e2e = {"value": all_solves / float(te.item()), "unit": UNIT,
           "h2d_bytes_per_step": int(64 * store.stride * 8 + n * 4),
           "d2h_bytes_per_step": int(8 + n_sel * (128 + 4) + 8 * len(cfg.cuts)), "ms_per_step": 1e3 * float(te.item()),
           "steps": e2e_steps}
    del arena, hb, hi, pin_cols, pin_flags, hstore

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    # ---- roofline of the dominant kernel (FP64-ALU bound) and of select (HBM bound) ------------------------------------
    prof = load_profiled_ops()
    sm_max = clocks.get("sm_max_mhz") or 1965.0
    sms = torch.cuda.get_device_properties(local).multi_processor_count
    roofline, select_line = run.rooflines(ms_per_step, sm_max, sms, prof)
    # measured FP64 roof of this box: a register-resident DFMA chain (FMA = 2 flop)
    sink = torch.zeros(1, dtype=torch.float64, device="cuda")
    per_thread = 1 << 20
    binding.fp64_peak_probe(sms * 8, 256, per_thread, sink, stream)
    torch.cuda.synchronize()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record(stream); binding.fp64_peak_probe(sms * 8, 256, per_thread, sink, stream); p1.record(stream)
    torch.cuda.synchronize()
    roofline["dfma_chain_measured_tflops"] = 2.0 * sms * 8 * 256 * per_thread / (p0.elapsed_time(p1) * 1e-3) / 1e12
    roofline["tflops_fma2_peak"] = sms * FP64_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": W,
           "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
           "data": "synthetic",
           "config": {"workload": cfg.name, "events_per_gpu": n, "selected_per_gpu": n_sel,
                      "n_variations": V, "pairings": 12 if cfg.n_fake_b == 0 else 30, "solves_per_step": all_solves,
                      "l2": (f"inputs ({516 * n / 1e6:.0f} MB of columns) larger than the 126 MB L2; no flush needed" if 516 * n > 126e6
                             else f"inputs ({516 * n / 1e6:.1f} MB) fit in L2: parity-test configuration, not a bench line"),
                      "parallelism": f"dp{world} (events sharded by global index, no collective)"},
           "clocks": clocks, "e2e": e2e, "gpu_launches": run.launches, "roofline": roofline, "select": select_line}
    if args.workload == "cfg4" and world == 1:
        out["planned_select"] = run.planned_select()
    idx_host = run.idx_host
    if not args.no_cpu_baseline and world == 1:      # the oracle is timed beside the GPU number on rank 0 at N = 1 only
        cores = os.cpu_count() or 1
        out["cpu_baseline"] = cpu_oracle_rate(store, idx_host, V, seed, cores, target_s=10.0)
        one = cpu_oracle_rate(store, idx_host, V, seed, 1, target_s=6.0)
        out["cpu_baseline"]["single_thread"] = {"value": one["value"], "unit": UNIT, "cores": 1, "sample": one["sample"]}
    # ---- the other configs of BASELINE.json, device-timed in the same run (default workload, one GPU only) ---------------
    if args.workload == "cfg2" and world == 1 and not args.no_extra_configs and not args.events and not args.variations:
        run.free()
        extra = {}
        for cid in (3, 4):
            c = hs.CONFIGS[cid]
            r = TthRun(hepf, binding, c, c.n_events, 0, c.n_variations, None)
            k = max(3, min(args.steps, 10 if cid == 3 else 20))
            ms = r.measure(k, 3)
            roof, sel = r.rooflines(ms, sm_max, sms, prof)
            extra[f"cfg{cid}"] = {"workload": c.name, "ms_per_step": ms, "steps": k, "value": r.n_solves / (ms * 1e-3), "unit": UNIT,
                                  "selected": r.n_sel, "solves_per_step": r.n_solves, "roofline": roof, "select": sel}
            if cid == 4:
                extra["cfg4"]["planned_select"] = r.planned_select()
            r.free()
        free, _ = torch.cuda.mem_get_info()
        n5 = hs.PHILOX_CFG5["n"]
        if free > 8 * n5 + (1 << 30):
            p = time_philox(hepf, n5, max(3, min(args.steps, 10)), 3)
            extra["cfg5"] = {"workload": p["workload"], "ms_per_step": p["ms_per_step"], "value": p["value"], "unit": p["unit"],
                             "roofline": p["roofline"]}
        out["configs"] = extra
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
