"""The C-ABI library loads without a GPU and exports every symbol include/hepf.h declares; argument checks that
need no device behave as documented."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2211_14346_b200 import build as b
    b.build()
    import paper_2211_14346_b200 as h
    return h.load()


def test_every_declared_symbol_is_exported(lib):
    src = open(os.path.join(ROOT, "include", "hepf.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = set(re.findall(r"\b(hepf_[a-z0-9_]+)\s*\(", src))
    assert {"hepf_select", "hepf_reconstruct_tth", "hepf_philox_normal", "hepf_tth_host", "hepf_last_error"} <= names
    for n in names:
        assert hasattr(lib, n), n


def test_struct_sizes_match_the_header():
    from paper_2211_14346_b200 import binding as b
    assert C.sizeof(b._Events) == 3 * 8 + 17 * 8
    assert C.sizeof(b._Cut) == 24 and C.sizeof(b.Params) == 80 and b.BEST_DTYPE.itemsize == 128


def test_workspace_queries_and_defaults(lib):
    import paper_2211_14346_b200 as h
    assert lib.hepf_select_workspace_bytes(0) > 0
    assert lib.hepf_select_workspace_bytes(20_000_000) >= 20_000_000 // 32 * 4
    assert lib.hepf_reconstruct_workspace_bytes(1000, 64) >= 8 * 1000
    assert lib.hepf_tth_host_arena_bytes(1000, 16) >= 1000 * (64 * 8 + 4 + 4 + 128)
    p = h.default_params()
    assert (p.m_top, p.m_w, p.m_higgs, p.lep_sigma, p.jet_stoch, p.jet_const) == (172.5, 80.4, 125.0, 0.01, 0.5, 0.03)


def test_argument_errors_without_a_device(lib):
    import paper_2211_14346_b200 as h
    rc = lib.hepf_philox_normal(1, 0, 10, None, None)
    assert rc == -1 and "out" in h.last_error()
    rc = lib.hepf_philox_normal(1, 2 ** 64 - 5, 10, C.c_void_p(16), None)
    assert rc == -1 and "overflow" in h.last_error()
    assert lib.hepf_philox_normal(1, 0, 0, None, None) == 0
    rc = lib.hepf_select(None, None, 0, None, None, None, None, 0, None)
    assert rc == -1


def test_missing_library_fails_loudly(tmp_path, monkeypatch):
    from paper_2211_14346_b200 import binding as b
    monkeypatch.setattr(b, "_lib", None)
    monkeypatch.setattr(b, "_LIB", str(tmp_path / "nope.so"))
    with pytest.raises(b.HepfError):
        b.load()
