"""The N > 1 path of bench.py is "replicas only": each rank builds its own seeded workload and
the only exchange is a MAX reduction of the timings.  Covered here with world_size 2 on the gloo backend (CPU)."""
import os
import socket

import numpy as np
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    import torch.distributed as dist
    from paper_2110_13481_b200 import inputs, replicas
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = replicas.replica_cfg(inputs.make_config(1), rank)
    X, S, V = inputs.initial_factors(cfg)
    fake_ms = [1.0 + rank, 10.0 - rank]              # rank-dependent "timings"
    red = replicas.max_over_ranks(fake_ms, "cpu", world)
    np.savez(os.path.join(out_dir, f"r{rank}.npz"), seed=cfg["seed"], x_pad=X[:, 1], red=np.array(red))
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_have_own_inputs_and_share_the_max_timing(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    r0, r1 = (np.load(tmp_path / f"r{k}.npz") for k in range(world))
    assert int(r1["seed"]) == int(r0["seed"]) + 1
    assert np.abs(r0["x_pad"] - r1["x_pad"]).max() > 1e-3        # different seeded padding columns
    for r in (r0, r1):
        assert r["red"].tolist() == [2.0, 10.0]                  # max over ranks of [1+rank, 10-rank]


def test_single_rank_needs_no_process_group():
    from paper_2110_13481_b200 import replicas
    assert replicas.max_over_ranks([3.5, 1.25], "cpu", 1) == [3.5, 1.25]
    assert replicas.aggregate_ms_per_step(2.0) == 2.0
