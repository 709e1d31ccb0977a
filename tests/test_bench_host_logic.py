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
