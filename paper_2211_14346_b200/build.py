"""Build libhepf.so in-tree with nvcc for sm_100a (explicit -gencode, -lineinfo)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libhepf.so")
SOURCES = ["hepf_api.cu", "hepf_philox.cu", "hepf_select.cu", "hepf_reco.cu", "hepf_host.cu", "hepf_hist.cu", "hepf_chi2.cu", "hepf_chi2_dilep.cu"]
# hepf_reco.cu spells every fused multiply-add itself: no contraction, so that the search and the finalize kernel
# (and any two builds) evaluate the shared device functions to the same bits
EXTRA_FLAGS = {"hepf_reco.cu": ["-fmad=false"]}
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(ROOT, "include", "hepf.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, checked_out: str | None = None) -> str:
    """Build libhepf.so in-tree.  checked_out = a path: build instead a CHECKED variant there (-DHEPF_CHECKED: every index into the
    search kernel's hand-staged shared memory and into the workspace is tested and the kernel traps on a violation); used by
    tests/test_checked_build.py, never by the product path."""
    if checked_out is None and not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objs = []
    bdir = os.path.join(HERE, "build") if checked_out is None else os.path.join(os.path.dirname(checked_out), "build_checked")
    lib = LIB if checked_out is None else checked_out
    os.makedirs(bdir, exist_ok=True)
    procs = []
    for s in SOURCES:
        o = os.path.join(bdir, s.replace(".cu", ".o"))
        cmd = [nvcc, "-c", os.path.join(CSRC, s), "-o", o, "-I", os.path.join(ROOT, "include"), "-I", CSRC] + NVCC_FLAGS + EXTRA_FLAGS.get(s, [])
        if checked_out is not None:
            cmd.append("-DHEPF_CHECKED")
        procs.append((s, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(o)
    log = []
    for s, p in procs:
        out, _ = p.communicate()
        log.append(f"== {s}\n{out}")
        if p.returncode != 0:
            sys.stderr.write("\n".join(log))
            raise RuntimeError(f"nvcc failed on {s}")
    subprocess.check_call([nvcc, "-shared", "-o", lib] + objs + ["-gencode", "arch=compute_100a,code=sm_100a",
                                                                 "-cudart", "static"])
    with open(os.path.join(bdir, "ptxas.log"), "w") as f:
        f.write("\n".join(log))
    if verbose:
        print("\n".join(log))
    return lib


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
