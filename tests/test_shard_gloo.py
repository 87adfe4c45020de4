"""N > 1 host logic on CPU (gloo, world_size 2): cells shard into contiguous ranges with no
data-path collective; the only cross-rank datum is the luminosity sum."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, n, ret):
    sys.path.insert(0, ROOT); sys.path.insert(0, os.path.join(ROOT, "tests"))
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle as O
    import common as cm
    from paper_2505_08855_b200 import synth
    desc, data, coul = cm.build_tables([8, 8, 8], nc=[8, 8])
    otab, un = cm.oracle_table(O, desc, data, coul), cm.oracle_units(O, desc)
    f = synth.log_uniform_cells(n, dtype=np.float32, config=2)
    lo, hi = synth.shard_range(n, rank, world)
    sub = {k: v[lo:hi] for k, v in f.items()}
    out = cm.oracle_step(O, otab, un, sub, 5.0, nsub=2, nthreads=1)
    lum = torch.tensor([out["diag"][k] for k in ("lum_total", "n_limited")], dtype=torch.float64)
    dist.all_reduce(lum)                                       # the one cross-rank reduction
    sizes = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(sizes, torch.tensor([hi - lo]))
    if rank == 0:
        ret["lum"] = lum.tolist(); ret["sizes"] = [int(s) for s in sizes]
    ret[f"theta_e_{rank}"] = out["theta_e"]
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_sharding_matches_single_process(oracle):
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import common as cm
    from paper_2505_08855_b200 import synth
    n, world = 10007, 2
    mgr = mp.Manager(); ret = mgr.dict()
    mp.spawn(_worker, args=(world, 29611, n, ret), nprocs=world, join=True)
    desc, data, coul = cm.build_tables([8, 8, 8], nc=[8, 8])
    otab, un = cm.oracle_table(oracle, desc, data, coul), cm.oracle_units(oracle, desc)
    f = synth.log_uniform_cells(n, dtype=np.float32, config=2)
    full = cm.oracle_step(oracle, otab, un, f, 5.0, nsub=2, nthreads=1)
    assert sum(ret["sizes"]) == n and max(ret["sizes"]) - min(ret["sizes"]) <= 1
    cat = np.concatenate([ret[f"theta_e_{k}"] for k in range(world)])
    assert np.array_equal(cat, full["theta_e"])               # cells are independent: sharding changes nothing
    assert ret["lum"][0] == pytest.approx(full["diag"]["lum_total"], rel=1e-12)
    assert int(ret["lum"][1]) == full["diag"]["n_limited"]


def test_shard_ranges_cover_exactly_once():
    from paper_2505_08855_b200 import synth
    for n in (0, 1, 7, 134217728):
        for w in (1, 2, 3, 8):
            r = [synth.shard_range(n, k, w) for k in range(w)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(r[k][1] == r[k + 1][0] for k in range(w - 1))
