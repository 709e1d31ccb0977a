"""world_size-2 gloo test (CPU) of the multi-process host logic: contiguous shards keyed by the global event index
give, rank by rank, exactly the slices of the single-process result; survivor offsets and the cutflow combine through
the two tiny collectives of paper_2211_14346_b200.sharding.  The per-rank compute here is the oracle (no GPU in this
test); the same plumbing drives the CUDA path in bench.py under torchrun."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, n_events, tmp):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    import hepf_synth as hs
    import oracle
    from paper_2211_14346_b200 import sharding
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    cfg = hs.CONFIGS[1]
    lo, hi = sharding.shard_range(n_events, rank, world)
    st = cfg.events(hi - lo, first_event=lo)             # generated from the global index: no data exchange
    assert st.event_base == lo
    idx, cf = oracle.select(st, cfg.cuts)
    off, total = sharding.global_survivor_offset(len(idx))
    gcf = sharding.global_cutflow(torch.from_numpy(cf.copy()))
    best, _ = oracle.reconstruct_tth(st, idx[:40], 4, cfg.reco_seed)
    np.savez(os.path.join(tmp, f"r{rank}.npz"), lo=lo, hi=hi, idx=idx.astype(np.int64) + lo, off=off, total=total,
             cutflow=gcf.numpy(), best=best.view(np.uint8).reshape(-1, 128))
    dist.barrier()
    dist.destroy_process_group()


def test_shard_range_covers_everything_with_16_byte_aligned_boundaries():
    from paper_2211_14346_b200.sharding import shard_range
    for n in (0, 1, 2, 7, 10, 1001, 20_000_000):
        for w in (1, 2, 3, 4, 8):
            r = [shard_range(n, k, w) for k in range(w)]
            assert r[0][0] == 0 and r[-1][1] == n
            for a, b in zip(r, r[1:]):
                assert a[1] == b[0] and (b[0] % 4 == 0 or b[0] == n)     # flags column: 4 events = 16 bytes
            assert max(h - l for l, h in r) - min(h - l for l, h in r) <= 7


@pytest.mark.timeout(300)
def test_two_ranks_reproduce_the_single_process_result(tmp_path):
    import torch.multiprocessing as mp
    sys.path.insert(0, ROOT)
    import hepf_synth as hs
    import oracle
    n, world, port = 3001, 2, _free_port()
    mp.spawn(_worker, args=(world, port, n, str(tmp_path)), nprocs=world, join=True)
    cfg = hs.CONFIGS[1]
    st = cfg.events(n)
    idx, cf = oracle.select(st, cfg.cuts)
    parts = [np.load(os.path.join(tmp_path, f"r{r}.npz")) for r in range(world)]
    assert np.array_equal(np.concatenate([p["idx"] for p in parts]), idx.astype(np.int64))
    assert all(int(p["total"]) == len(idx) for p in parts)
    assert int(parts[0]["off"]) == 0 and int(parts[1]["off"]) == len(parts[0]["idx"])
    assert all(np.array_equal(p["cutflow"], cf) for p in parts)
    # reconstruction of a shard equals the single-process records of the same global events (event index is
    # view-local, everything else is bit-identical because the Philox key is the global index)
    for p in parts:
        g = p["idx"][:40]
        want, _ = oracle.reconstruct_tth(st, g.astype(np.uint32), 4, cfg.reco_seed)
        got = p["best"].reshape(-1).view(oracle.BEST_DTYPE).copy()
        got["event"] += np.uint32(int(p["lo"]))
        assert got.tobytes() == want.tobytes()
