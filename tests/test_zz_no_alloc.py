"""-m gpu, collected last: hepf_select_static, the entry point that allocates nothing (include/hepf.h) — hepf_select with its
scratch in a file-scope device array of the library instead of a caller workspace.  Integer / index work: the bar is bit-exact.

Each case runs the new entry point TWICE in a row on different inputs (the static array keeps the previous call's contents: a
stale mask or block count that leaked into the second call would show), compares survivor list, count and cutflow exactly with
the existing hepf_select path, and checks that the device memory held by the process did not change across the calls.  The
test depends on nothing the other tests leave behind and leaves nothing behind: it passes alone in a fresh process and after
the rest of the suite.
"""
import numpy as np
import pytest

import hepf_synth as hs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hepf():
    import torch
    assert torch.cuda.is_available()
    import paper_2211_14346_b200 as h
    h.load()
    return h


def _outputs(n, n_cuts):
    import torch
    return (torch.full((max(n, 1),), -1, dtype=torch.int32, device="cuda"), torch.full((1,), -7, dtype=torch.int64, device="cuda"),
            torch.full((max(n_cuts, 1),), -7, dtype=torch.int64, device="cuda"))


def _same_as_select(hepf, dev, chain, got):
    import torch
    idx, count, cf = hepf.select(dev, chain)
    torch.cuda.synchronize()
    n = int(count.item())
    assert int(got[1].item()) == n
    assert torch.equal(got[0][:n], idx[:n])
    assert torch.equal(got[2][: len(chain)], cf[: len(chain)])
    return n


def test_select_static_matches_select_on_two_calls_in_a_row(hepf):
    import torch
    cfg = hs.CONFIGS[2]
    big = hepf.DeviceEvents.from_host(hs.generate(300_001, 71, bkg_frac=0.5, with_truth=False))    # ragged tail, 586 tiles
    small = hepf.DeviceEvents.from_host(hs.generate(12_345, 72, bkg_frac=0.3, with_truth=False))   # fewer tiles and blocks than `big`
    loose = [(hs.MET_GT, 0, 20.0, 0)]
    out_big, out_small = _outputs(big.n_events, len(cfg.cuts)), _outputs(small.n_events, len(loose))
    hepf.select_static(small, loose, *_outputs(small.n_events, len(loose)))     # set-up: the per-device address lookup
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    launches0 = hepf.launch_count()
    # two calls in a row, the second on a smaller store whose masks and block counts overwrite only part of the first call's
    a = hepf.select_static(big, cfg.cuts, *out_big)
    b = hepf.select_static(small, loose, *out_small)
    torch.cuda.synchronize()
    assert hepf.launch_count() - launches0 == 4               # select_eval + select_scatter per call, nothing else
    assert torch.cuda.mem_get_info()[0] == free0              # no device allocation by the entry point
    n_big = _same_as_select(hepf, big, cfg.cuts, a)
    n_small = _same_as_select(hepf, small, loose, b)
    assert 0 < n_big < big.n_events and 0 < n_small < small.n_events
    # and the other way round (a larger call after a smaller one), with the cutflow left out and an empty chain
    c = hepf.select_static(small, [], out_small[0], out_small[1], None)
    d = hepf.select_static(big, cfg.cuts, *out_big)
    torch.cuda.synchronize()
    assert int(c[1].item()) == small.n_events and torch.equal(c[0], torch.arange(small.n_events, dtype=torch.int32, device="cuda"))
    assert _same_as_select(hepf, big, cfg.cuts, d) == n_big


def test_select_static_at_the_maximum_size(hepf):
    """Exactly HEPF_SELECT_STATIC_MAX_EVENTS events: the last tile's masks end where the block counts begin."""
    import torch
    cfg = hs.CONFIGS[2]
    full = hepf.DeviceEvents.from_host(hs.generate(hepf.SELECT_STATIC_MAX_EVENTS, 74, bkg_frac=0.5, with_truth=False))
    out = _outputs(full.n_events, len(cfg.cuts))
    for _ in range(2):
        got = hepf.select_static(full, cfg.cuts, *out)
        torch.cuda.synchronize()
        assert 0 < _same_as_select(hepf, full, cfg.cuts, got) < full.n_events
        out[0].fill_(-1); out[1].fill_(-7); out[2].fill_(-7)


def test_select_static_rejects_what_does_not_fit(hepf):
    import torch
    n = hepf.SELECT_STATIC_MAX_EVENTS + 4
    cols = torch.zeros((hs.NROW, 8), dtype=torch.float64, device="cuda")
    flags = torch.zeros(8, dtype=torch.int32, device="cuda")
    too_many = hepf.DeviceEvents(cols, flags, 8, 0)
    too_many.n_events = too_many.stride = n                   # a view only: the size test comes before any access to the columns
    out = _outputs(1, 1)
    with pytest.raises(hepf.HepfError, match="exceed the static scratch"):
        hepf.select_static(too_many, [], *out)
    torch.cuda.synchronize()
    assert int(out[1].item()) == -7                           # nothing was launched
    ok = hepf.DeviceEvents.from_host(hs.generate(1000, 73, with_truth=False))
    with pytest.raises(hepf.HepfError):
        hepf.select_static(ok, [(999, 0, 0.0, 0.0)], *_outputs(1000, 1))
