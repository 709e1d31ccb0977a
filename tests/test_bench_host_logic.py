"""Host-side logic of bench.py that the reported numbers depend on (no GPU): the solve count of a list of events, the
algorithmic bytes of a cut chain, and the shape of the reference arm's JSON line."""
import json
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402
import hepf_synth as hs  # noqa: E402


def test_solves_of_counts_variations_times_ordered_pairings_of_applicable_events():
    st = hs.generate(3000, 9, n_fake_b=2, bkg_frac=0.4, with_truth=False)
    idx = np.arange(st.n_events)
    want = 0
    for e in idx:
        f = int(st.flags[e]); nj = min(8, (f >> 8) & 15)
        nb = min(6, sum((f >> (16 + s)) & 1 for s in range(nj)))
        if (f & 15) == 2 and ((f >> 4) & 1) != ((f >> 5) & 1) and nb >= 4:
            want += nb * (nb - 1)
    assert bench.solves_of(st, idx, 7) == 7 * want and want > 0
    assert bench.solves_of(st, idx[:0], 7) == 0


def test_chain_bytes_are_the_columns_the_chain_names():
    assert bench.chain_bytes_per_event(hs.CHAIN_BASE) == 4 + 16 + 64 + 64 + 8            # flags, lep_pt, jet_pt, jet_eta, met
    assert bench.chain_bytes_per_event(hs.CHAIN_TIGHT8) == 4 + 16 + 16 + 64 + 64 + 8 + 8  # + lep_eta, mll
    assert bench.chain_bytes_per_event([]) == 4
    assert bench.chain_bytes_per_event([(hs.NLEP_EQ, 2, 0, 0), (hs.LEP_OS, 0, 0, 0)]) == 4


def test_reference_arm_prints_one_json_line_with_the_contract_keys():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "cfg1",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for k in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert k in d, k
    assert d["impl"] == "reference" and d["metric"] == bench.METRIC and d["unit"] == bench.UNIT and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["config"]["workload"] == hs.CONFIGS[1].name


def test_search_kernel_name_follows_the_librarys_dispatch_on_the_number_of_variations():
    """hepf_reco.cu, reconstruct_impl: lanes over pairings for V <= 2, chunks of 8 up to V = 8, chunks of 32 (16 for n_b = 5, 6)
    unless that wastes more than an eighth of the last chunk's lanes, then 16 (8)."""
    name = bench.search_kernel_name
    assert name(1, False) == "reco_search_kernel<1,4>" and name(2, True) == "reco_search_kernel<1,6>"
    assert name(3, False) == "reco_search_kernel<8,4>" and name(8, True) == "reco_search_kernel<8,6>"
    assert name(16, False) == "reco_search_kernel<16,4>" and name(16, True) == "reco_search_kernel<8,6>"     # 16 of 32 lanes wasted
    assert name(33, False) == "reco_search_kernel<16,4>"                                                     # 31 of 64
    assert name(64, False) == "reco_search_kernel<32,4>" and name(256, True) == "reco_search_kernel<16,6>"
    assert name(130, False) == "reco_search_kernel<16,4>" and name(1024, False) == "reco_search_kernel<32,4>"
    assert name(57, False) == "reco_search_kernel<32,4>"                                                     # 7 of 64 <= 57 / 8


def test_ncu_counts_parses_a_per_launch_csv_and_keys_the_file_by_the_kernel_sources(tmp_path, monkeypatch):
    from paper_2211_14346_b200 import ncu_counts
    kern = ("void hepf::reco_search_kernel<(int)32, (int)4, (int)18, (int)1>(hepf::RecoCols, const unsigned int *, const long *, long, "
            "int, int, unsigned int, unsigned int, hepf_tth_params_t, uint2 *, double *, unsigned long long *)")
    rows = ['==PROF== Connected to process 1', '"ID","Process ID","Process Name","Host Name","Kernel Name","Context","Stream","Block Size",'
            '"Grid Size","Device","CC","Section Name","Metric Name","Metric Unit","Metric Value"']
    vals = {"gpu__time_duration.sum": ("ms", "7.0"), "smsp__inst_executed.sum": ("inst", "5,000,000,000"), "sm__cycles_elapsed.avg": ("cycle", "1"),
            "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum": ("inst", "3000000000"), "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum": ("inst", "7000000000"),
            "smsp__sass_thread_inst_executed_op_dfma_pred_on.sum": ("inst", "11000000000"),
            "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active": ("%", "53.5"), "sm__issue_active.avg.pct_of_peak_sustained_elapsed": ("%", "65"),
            "dram__bytes_read.sum": ("Mbyte", "260"), "dram__bytes_write.sum": ("Mbyte", "10"), "launch__registers_per_thread": ("register/thread", "96"),
            "sm__warps_active.avg.per_cycle_active": ("warp", "17.6")}
    for lid, scale in ((0, 1.0), (1, 1.0), (2, 0.01)):          # the third launch is a short end-to-end chunk: not averaged
        for m, (u, v) in vals.items():
            x = v if scale == 1.0 or m != "gpu__time_duration.sum" else "0.07"
            rows.append(f'"{lid}","1","python","h","{kern}","1","7","(576, 1, 1)","(148, 1, 1)","0","10.0","s","{m}","{u}","{x}"')
    csv_path = tmp_path / "ops.csv"; csv_path.write_text("\n".join(rows) + "\n")
    launches = ncu_counts.parse_launches(str(csv_path))
    assert list(launches) == ["reco_search_kernel<32,4>"] and len(launches["reco_search_kernel<32,4>"]) == 3
    assert launches["reco_search_kernel<32,4>"][0]["gpu__time_duration.sum"] == 7.0e-3
    assert launches["reco_search_kernel<32,4>"][0]["dram__bytes_read.sum"] == 260e6
    bench_json = tmp_path / "plain.json"
    bench_json.write_text(json.dumps({"roofline": {"kernel": "reco_search_kernel<32,4>", "solves_per_launch": 100_000_000}}) + "\n")
    ops_file = tmp_path / "ops.json"
    monkeypatch.setattr(ncu_counts, "OPS_FILE", str(ops_file))
    monkeypatch.setattr(sys, "argv", ["ncu_counts", "--csv", str(csv_path), "--bench-json", str(bench_json), "--workload", "cfg2",
                                      "--profile", "profiles/x.md"])
    ncu_counts.main()
    d = json.loads(ops_file.read_text())
    e = d["kernels"]["reco_search_kernel<32,4>"]
    assert d["source_sha256"] == bench.kernel_source_hash() == ncu_counts.source_hash()
    assert (e["dadd"], e["dmul"], e["dfma"]) == (30.0, 70.0, 110.0) and e["launches_averaged"] == 2
    assert e["warp_instructions_per_solve"] == 50.0 and abs(e["ncu_gpu_time_ms"] - 7.0) < 1e-9 and e["dram_bytes_per_launch"] == 270e6
