"""-m gpu: the search kernel stages its data by hand in shared memory (per-warp tables, a solve queue, a root stack, tags packed
into values) and compute-sanitizer is not available on the pool.  This test builds a CHECKED variant of the library
(-DHEPF_CHECKED: every index into those structures and into the workspace is tested against its bound, the kernel traps on a
violation), runs every instantiation of the search kernel on it — all chunk sizes, both candidate classes, ragged variation
counts, background topologies, garbage inputs — and requires (a) no trap and (b) records byte-identical to the product
build's.  It runs in a subprocess: a trap would poison the CUDA context."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_SCRIPT = r"""
import sys, hashlib
sys.path.insert(0, {root!r})
import numpy as np, torch
import hepf_synth as hs
from paper_2211_14346_b200 import binding
if {lib!r}:
    binding._LIB = {lib!r}
import paper_2211_14346_b200 as hepf
hepf.load()
h = hashlib.sha256()
cases = [(1, 4000, 16, 1.0), (2, 3000, 64, 1.0), (2, 2000, 33, 1.0), (2, 1500, 1, 0.0), (2, 1500, 2, 1.0), (2, 1500, 7, 1.0),
         (3, 2500, 256, 1.0), (3, 2000, 16, 1.0), (3, 1500, 5, 1.0), (3, 1500, 2, 1.0), (4, 60000, 16, 1.0), (2, 1200, 130, 3.0)]
for cid, n, V, kappa in cases:
    cfg = hs.CONFIGS[cid]
    st = cfg.events(n)
    if kappa == 3.0:                      # garbage in a third of the events: NaN, inf, zero energies
        rng = np.random.default_rng(n)
        ev = np.arange(0, n, 3); st.cols[rng.integers(0, hs.NROW, len(ev)), ev] = rng.choice([np.nan, np.inf, 0.0, -1e300], len(ev))
    dev = hepf.DeviceEvents.from_host(st)
    idx_t, count, cf = hepf.select(dev, cfg.cuts if cid != 4 else [])
    m = int(count.item())
    out = hepf.reconstruct_tth(dev, idx_t, m, V, cfg.reco_seed, hepf.default_params(sigma_scale=min(kappa, 1.0)))
    torch.cuda.synchronize()
    rec = out.cpu().numpy()
    h.update(rec.tobytes())
    print(cid, n, V, m, flush=True)
print("DIGEST", h.hexdigest())
"""


def _run(lib):
    out = subprocess.run([sys.executable, "-c", _SCRIPT.format(root=ROOT, lib=lib)], capture_output=True, text=True, timeout=900)
    assert out.returncode == 0, (out.stdout[-1500:], out.stderr[-3000:])
    return [ln for ln in out.stdout.splitlines() if ln.startswith("DIGEST")][0]


@pytest.mark.timeout(1500)
def test_checked_build_traps_nowhere_and_gives_the_same_bytes(tmp_path):
    sys.path.insert(0, ROOT)
    from paper_2211_14346_b200 import build
    lib = build.build(checked_out=str(tmp_path / "libhepf_checked.so"))
    assert os.path.exists(lib)
    assert _run(lib) == _run("")
