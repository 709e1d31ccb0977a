#!/usr/bin/env python
"""bench.py — smeared ttH reconstructions/s on BASELINE.json configs[1] (1e6 events, 4 b-jets, V = 64, FP64).

A step is one pass of the whole hot path over the batch: hepf_select (cut chain + compaction) followed by
hepf_reconstruct_tth (Philox/Box-Muller smearing, dilepton solve, score, argmax) for every surviving event.
`value` counts event x variation x pairing solves per second with the inputs resident in HBM; `e2e` is the same
metric through hepf_tth_host (host buffers in, results out, copies inside the timed region).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload cfg1|cfg2|cfg3|cfg4]
Under torchrun every rank runs its own shard (events keyed by global index, no data-path collective): weak scaling.
"""
from __future__ import annotations

import argparse
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
# FP64 roof of one B200 from the guide's unit counts: 148 SMs x 64 FP64 FMA lanes/clk x 2 flop x clocks.max.sm
FP64_LANES_PER_SM = 64
# Algorithmic FP64 work of one solve: the search kernel's own predicated-on thread-level FP64 instruction counts per
# solve (idle lanes and divergence waste do not count), from the committed ncu capture of this build
# (profiles/r01g_final.md, r01h_final.md): DADD + DMUL + DFMA lane-ops, and flop with FMA = 2.  DESIGN.md section 7.
FP64_OPS_PER_SOLVE = {"dadd": 33.8, "dmul": 75.0, "dfma": 125.9}
FP64_OPS_PER_SOLVE_NB6 = {"dadd": 26.5, "dmul": 60.7, "dfma": 101.9}   # n_b = 6 kernel (cfg3), profiles/r01g
DRAM_BYTES_PER_LAUNCH = 276.3e6   # ncu dram__bytes_read.sum + dram__bytes_write.sum of the search kernel (same profile)


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


def run_philox(args):
    """--workload cfg5: standalone hepf_philox_normal stream (BASELINE.json configs[4]), normals/s and GB/s written."""
    import torch
    import paper_2211_14346_b200 as hepf
    hepf.load()
    torch.cuda.set_device(0)
    n = args.events or hs.PHILOX_CFG5["n"]
    out = torch.empty(n, dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream()
    for _ in range(max(3, args.warmup)):
        hepf.philox_normal(hs.PHILOX_CFG5["seed"], 0, n, out=out, stream=stream)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        hepf.philox_normal(hs.PHILOX_CFG5["seed"], 0, n, out=out, stream=stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))) if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else {}
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    gbs = 8.0 * n / (ms * 1e-3) / 1e9
    print(json.dumps({"metric": "standard-normal FP64 draws/sec (Philox4x32-10 + Box-Muller)", "value": n / (ms * 1e-3),
                      "unit": "normals/s", "n_gpus": 1, "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": ms,
                      "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": f"cfg5: {n} normals, seed 7, counter 0", "l2": "34 GB written per step, far larger than L2"},
                      "gpu_launches": args.steps,
                      "roofline": {"bound": "hbm", "kernel": "philox_normal_kernel<true>", "achieved": gbs, "peak": hbm,
                                   "unit": "GB/s", "frac": gbs / hbm, "traffic": None,
                                   "peak_source": "MEASURED_PEAKS.json hbm_gbs (copy, read+write)" if peaks else "fallback 6650"}}))


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
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    hbm = float(json.load(open(peaks_path)).get("hbm_gbs", 6650.0)) if os.path.exists(peaks_path) else 6650.0
    gbs = by / (ms * 1e-3) / 1e9
    print(json.dumps({"metric": "chi2-reconstructed semileptonic ttbar events/sec", "value": n / (ms * 1e-3), "unit": "events/s",
                      "n_gpus": 1, "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": ms, "higher_is_better": True,
                      "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": f"chi2: {n} semileptonic ttbar events (2 b + 2-4 untagged jets)",
                                 "l2": f"{by / 1e6:.0f} MB touched per step, larger than L2"},
                      "gpu_launches": args.steps,
                      "roofline": {"bound": "hbm", "kernel": "chi2_semilep_kernel", "achieved": gbs, "peak": hbm, "unit": "GB/s",
                                   "frac": gbs / hbm, "traffic": None, "algorithmic_bytes": by}}))


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


def cpu_oracle_rate(store, idx, n_variations, seed, target_s=15.0, chain=hs.CHAIN_BASE):
    """Time the oracle, as it stands, on a bounded sample of the same workload on the host cores."""
    import oracle
    cores = os.cpu_count() or 1
    probe = idx[:2048]
    t0 = time.perf_counter(); oracle.reconstruct_tth(store, probe, n_variations, seed, n_threads=cores)
    dt = max(time.perf_counter() - t0, 1e-3)
    m = int(min(len(idx), max(2048, 2048 * target_s / dt)))
    sample = idx[:m]
    t0 = time.perf_counter()
    oracle.select(store, chain)                    # the oracle's selection of the whole batch is part of a step
    t_sel = time.perf_counter() - t0
    t0 = time.perf_counter(); oracle.reconstruct_tth(store, sample, n_variations, seed, n_threads=cores)
    dt = time.perf_counter() - t0
    n_solves = solves_of(store, sample, n_variations)
    return {"value": n_solves / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"first {m} selected events of the workload ({n_solves} solves, {dt:.1f} s wall, OpenMP over events; "
                      f"oracle select of all {store.n_events} events took {t_sel:.2f} s, not included)"}


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
                      "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample_txt},
                      "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                      "gpu_launches": 0}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="hepf", choices=["hepf", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5", "chi2"])
    ap.add_argument("--events", type=int, default=0, help="override the number of events per GPU (debugging)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--variations", type=int, default=0, help="override the workload's V (SURVEY 8(f) NEXT-1: 128 = ttH_scinp, 1024 = ttH_sci)")
    ap.add_argument("--sigma-scale", type=float, default=None, help="0 = no smearing, the paper's ttH_as variant")
    args = ap.parse_args()
    if args.workload == "cfg5":
        return run_philox(args)
    if args.workload == "chi2":
        return run_chi2(args)
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
    # weak scaling: rank r owns global events [r n, (r+1) n); the Philox keys use the global index
    store = cfg.events(n_ev, first_event=rank * n_ev)
    dev = hepf.DeviceEvents.from_host(store)
    n, V, seed = store.n_events, (args.variations or cfg.n_variations), cfg.reco_seed
    params = hepf.default_params(sigma_scale=args.sigma_scale) if args.sigma_scale is not None else None
    stream = torch.cuda.current_stream()
    out_idx = torch.empty(max(n, 1), dtype=torch.int32, device="cuda")
    out_count = torch.zeros(1, dtype=torch.int64, device="cuda")
    out_cf = torch.zeros(32, dtype=torch.int64, device="cuda")
    ws = torch.empty(int(hepf.load().hepf_select_workspace_bytes(n)) + 256, dtype=torch.uint8, device="cuda")
    out_best = torch.empty((max(n, 1), 128), dtype=torch.uint8, device="cuda")
    reco_ws = torch.empty(int(hepf.load().hepf_reconstruct_workspace_bytes(n, V)) + 256, dtype=torch.uint8, device="cuda")
    count_host = torch.zeros(1, dtype=torch.int64).pin_memory()

    def step(ev_mid=None):
        hepf.select(dev, cfg.cuts, out_idx=out_idx, out_count=out_count, out_cutflow=out_cf, ws=ws, stream=stream)
        count_host.copy_(out_count, non_blocking=True)
        stream.synchronize()                       # hepf_reconstruct_tth takes n_idx as a host value
        n_sel = int(count_host[0])
        if ev_mid is not None:
            ev_mid[0].record(stream)
        hepf.reconstruct_tth(dev, out_idx, n_sel, V, seed, params, out_best=out_best, ws=reco_ws, stream=stream)
        if ev_mid is not None:
            ev_mid[1].record(stream)
        return n_sel

    for _ in range(W):
        n_sel = step()
    torch.cuda.synchronize()
    idx_host = out_idx[:n_sel].cpu().numpy().view(np.uint32)
    n_solves = solves_of(store, idx_host, V)

    sampler = ClockSampler(local)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler.start()
    hepf.launch_count(reset=True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    mids = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    binding.timing_enable(True)
    k_search, k_search6, k_final, k_sel, k_sel_eval = [], [], [], [], []
    e0.record(stream)
    for s in range(args.steps):
        step(mids[s])
        # device time of each kernel of this step, from events the library records on the stream around its launches
        k_search.append(binding.timing_ms(3, 4)); k_search6.append(binding.timing_ms(4, 5)); k_final.append(binding.timing_ms(5, 6)); k_sel.append(binding.timing_ms(0, 2)); k_sel_eval.append(binding.timing_ms(0, 1))
    e1.record(stream)
    torch.cuda.synchronize()
    binding.timing_enable(False)
    launches = hepf.launch_count()
    clocks = sampler.stop()
    ms_total = e0.elapsed_time(e1)
    ms_reco = float(np.mean([a.elapsed_time(b) for a, b in mids]))
    t = torch.tensor([ms_total], dtype=torch.float64, device="cuda")
    tot = torch.tensor([float(n_solves)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.barrier()
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    ms_total, all_solves = float(t.item()), float(tot.item())
    ms_per_step = ms_total / args.steps
    value = all_solves / (ms_per_step * 1e-3)

    # ---- end to end through the C ABI with host buffers (pinned), copies inside the timed region --------------
    pin_cols = torch.from_numpy(store.cols).pin_memory()
    pin_flags = torch.from_numpy(store.flags.view(np.int32)).pin_memory()
    hstore = hs.EventStore(n, store.stride, store.event_base, pin_cols, pin_flags)
    arena = torch.empty(binding.tth_host_arena_bytes(n, V) + 512, dtype=torch.uint8, device="cuda")
    hb = torch.empty((max(n, 1), 128), dtype=torch.uint8).pin_memory()
    hi = torch.empty(max(n, 1), dtype=torch.int32).pin_memory()
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
           "d2h_bytes_per_step": int(8 + n_sel * (128 + 4) + 8 * len(cfg.cuts)), "ms_per_step": 1e3 * float(te.item())}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    # ---- roofline of the dominant kernel (reco_kernel: FP64-ALU bound) -----------------------------------------------
    sm_max = clocks.get("sm_max_mhz") or 1965.0
    sms = torch.cuda.get_device_properties(local).multi_processor_count
    peak_tflops = sms * FP64_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    sink = torch.zeros(1, dtype=torch.float64, device="cuda")
    per_thread = 1 << 20
    binding.fp64_peak_probe(sms * 8, 256, per_thread, sink, stream)
    torch.cuda.synchronize()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record(stream); binding.fp64_peak_probe(sms * 8, 256, per_thread, sink, stream); p1.record(stream)
    torch.cuda.synchronize()
    fma_peak = 2.0 * sms * 8 * 256 * per_thread / (p0.elapsed_time(p1) * 1e-3) / 1e12
    nb6 = float(np.mean(k_search6)) > float(np.mean(k_search))     # which candidate-count class dominates this workload
    ms_search = float(np.mean(k_search6 if nb6 else k_search))
    ops = FP64_OPS_PER_SOLVE_NB6 if nb6 else FP64_OPS_PER_SOLVE
    LANE_OPS_PER_SOLVE = sum(ops.values()); FLOP_PER_SOLVE = ops["dadd"] + ops["dmul"] + 2.0 * ops["dfma"]
    achieved = FLOP_PER_SOLVE * n_solves / (ms_search * 1e-3) / 1e12
    lane_rate = LANE_OPS_PER_SOLVE * n_solves / (ms_search * 1e-3)
    lane_peak = sms * FP64_LANES_PER_SM * sm_max * 1e6
    # ALU-bound: the unit of work is one FP64 pipe instruction per lane (DADD, DMUL or DFMA), the peak is the pipe's issue
    # rate 148 SMs x 64 lanes x clock (DESIGN.md 6.2 / 7); the FMA = 2 flop figures are given beside it
    roofline = {"bound": "alu", "kernel": "reco_search_kernel<16,6>" if nb6 else "reco_search_kernel<16,4>",
                "achieved": lane_rate / 1e12, "peak": lane_peak / 1e12, "unit": "T FP64 lane-op/s",
                "frac": lane_rate / lane_peak, "traffic": DRAM_BYTES_PER_LAUNCH if args.workload == "cfg2" else None,
                "peak_source": f"{sms} SMs x {FP64_LANES_PER_SM} FP64 lanes x {sm_max:.0f} MHz (DESIGN.md section 6.2)",
                "fp64_lane_ops_per_solve": LANE_OPS_PER_SOLVE, "flop_per_solve": FLOP_PER_SOLVE,
                "tflops_fma2": achieved, "tflops_fma2_peak": peak_tflops, "dfma_chain_measured_tflops": fma_peak,
                "ncu_sm__pipe_fp64_cycles_active_pct": None if nb6 or args.workload != "cfg2" else 50.0,
                "kernel_ms": ms_search, "kernel_share_of_step": ms_search / ms_per_step,
                "other_kernels_ms": {"reco_search_other_class": float(np.mean(k_search if nb6 else k_search6)),
                                     "select_eval+scatter": float(np.mean(k_sel)), "reco_finalize": float(np.mean(k_final)),
                                     "hepf_reconstruct_tth_call": ms_reco}}
    sel_bytes = chain_bytes_per_event(cfg.cuts) * n + 4 * n_sel
    sel_ms = float(np.mean(k_sel_eval))
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    hbm_peak = float(json.load(open(peaks_path)).get("hbm_gbs", 6650.0)) if os.path.exists(peaks_path) else 6650.0
    select_line = {"kernel": "select_eval_kernel", "events_per_s": n / (sel_ms * 1e-3), "bound": "hbm",
                   "achieved": sel_bytes / (sel_ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                   "frac": sel_bytes / (sel_ms * 1e-3) / 1e9 / hbm_peak, "algorithmic_bytes": sel_bytes, "kernel_ms": sel_ms,
                   "eval+scatter_ms": float(np.mean(k_sel))}
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": W,
           "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
           "data": "synthetic",
           "config": {"workload": cfg.name, "events_per_gpu": n, "selected_per_gpu": n_sel,
                      "n_variations": V, "pairings": 12 if cfg.n_fake_b == 0 else 30, "variations": V, "solves_per_step": all_solves,
                      "l2": (f"inputs ({516 * n / 1e6:.0f} MB of columns) larger than the 126 MB L2; no flush needed" if 516 * n > 126e6 else f"inputs ({516 * n / 1e6:.1f} MB) fit in L2: parity-test configuration, not a bench line"),
                      "parallelism": f"dp{world} (events sharded by global index, no collective)"},
           "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "select": select_line}
    if not args.no_cpu_baseline and world == 1:      # the oracle is timed beside the GPU number on rank 0 at N = 1 only
        out["cpu_baseline"] = cpu_oracle_rate(store, idx_host, V, seed, chain=cfg.cuts)
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
