"""N > 1 host logic on CPU: position sharding + dose all-reduce over gloo, world_size 2.

The per-position dose here comes from the oracle (tests may use it); the point is the decomposition:
the ranks' partial sums, all-reduced, equal the single-process scan sum."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1811_12391_b200.scan import all_reduce_dose, shard_positions


def test_shard_positions_partition():
    for n_pos in (0, 1, 5, 36):
        for world in (1, 2, 3, 8):
            parts = [shard_positions(n_pos, r, world) for r in range(world)]
            flat = sorted(x for part in parts for x in part)
            assert flat == list(range(n_pos))
            assert max(len(q) for q in parts) - min(len(q) for q in parts) <= 1
    with pytest.raises(ValueError):
        shard_positions(4, 2, 2)


def _worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import oracle
    from paper_1811_12391_b200.inputs import make_problem
    p = make_problem("config4", nx=12, ny=12, nz=4, voxel=3.0, n_group=3, n_iter=2, n_pos=5, sn=4, pl=1)
    part = torch.zeros(p["material"].shape, dtype=torch.float64)
    for s in shard_positions(len(p["sources"]), rank, world):
        part += torch.from_numpy(oracle.run_problem(p, source_index=s)["dose"])
    total = all_reduce_dose(part)
    np.save(os.path.join(out_dir, f"dose_{rank}.npy"), total.numpy())
    dist.destroy_process_group()


def test_two_rank_scan_sum_equals_single_process(tmp_path, orc):
    from paper_1811_12391_b200.inputs import make_problem
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    p = make_problem("config4", nx=12, ny=12, nz=4, voxel=3.0, n_group=3, n_iter=2, n_pos=5, sn=4, pl=1)
    ref = sum(orc.run_problem(p, source_index=s)["dose"] for s in range(5))
    for r in range(2):
        got = np.load(tmp_path / f"dose_{r}.npy")
        assert np.allclose(got, ref, rtol=1e-13, atol=0.0)
