"""Multi-GPU host logic on the CPU: right-hand sides shard over ranks with no data-path collective
(DESIGN.md section 9).  The 2-rank runs use torch.distributed with the gloo backend on 127.0.0.1."""
import os
import socket

import numpy as np
import pytest

from paper_2404_07398_b200.sharding import gather_max, gather_table, partition_rhs, rank_fields


def test_rank_fields_cover_all_fields_once():
    for n in (1, 2, 7, 16):
        for world in (1, 2, 3, 8):
            seen = []
            for r in range(world):
                s = rank_fields(n, world, r)
                seen += list(range(n))[s]
            assert seen == list(range(n))
            sizes = [len(range(n)[rank_fields(n, world, r)]) for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        rank_fields(4, 2, 2)


def test_partition_rhs_is_complete_and_balanced():
    ells = np.geomspace(1.0, 1000.0, 40)
    for order_n in (1, 2):
        for world in (1, 2, 4, 8):
            parts = partition_rhs(ells, 2, order_n, world)
            flat = sorted(p for part in parts for p in part)
            assert flat == [(f, j) for f in range(2) for j in range(40)]
            cost = [sum(ells[j] ** order_n for _, j in part) for part in parts]
            # longest-processing-time first: no rank exceeds the mean by more than the largest single item
            assert max(cost) <= sum(cost) / world + ells[-1] ** order_n + 1e-9


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    import torch.distributed as dist
    import oracle
    from workloads import make_config
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # every rank builds the same mesh and solves only its own fields (what bench.py --gpus N does)
        w = make_config(1, n=16, n_fields=4, n_ells=3, ell_max=4.0)
        mine = rank_fields(w.fields.shape[0], world, rank)
        om = oracle.OracleMesh(w.mesh.coords, w.mesh.tri, w.mesh.period)
        rows = []
        for f in range(w.fields.shape[0])[mine]:
            for j, ell in enumerate(w.ells):
                x, info = om.solve(w.fields[f], float(ell), 1)
                rows.append((f, j, om.energy(x), info["iters"]))
        table = gather_table(rows)
        t_max = gather_max(float(rank + 1))
        if rank == 0:
            np.save(os.path.join(out_dir, "table.npy"), np.array(table, dtype=np.float64))
            np.save(os.path.join(out_dir, "tmax.npy"), np.array([t_max]))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_ranks_shard_fields_and_gather(tmp_path, oracle_mod):
    import torch.multiprocessing as mp
    from workloads import make_config
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    table = np.load(tmp_path / "table.npy")
    assert np.load(tmp_path / "tmax.npy")[0] == 2.0                      # max over ranks
    w = make_config(1, n=16, n_fields=4, n_ells=3, ell_max=4.0)
    assert [(int(r[0]), int(r[1])) for r in table] == [(f, j) for f in range(4) for j in range(3)]
    om = oracle_mod.OracleMesh(w.mesh.coords, w.mesh.tri, w.mesh.period)
    for f, j, e, _ in table:
        x, _ = om.solve(w.fields[int(f)], float(w.ells[int(j)]), 1)
        assert abs(om.energy(x) - e) <= 1e-14 * abs(e)


def test_gather_helpers_without_process_group():
    assert gather_max(3.5) == 3.5
    assert gather_table([(1, 2)]) == [(1, 2)]
