"""N > 1 host logic of bench.py on CPU: two gloo ranks, no GPU.  The path shards by independent
instances: every rank runs its own sweep with its own seeds, there is no
data-path collective, and the job time is the max over ranks."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = bench.make_workload("C1", rank)
    # each rank times its own work; the job time is the max
    t_local = 1.0 + 0.5 * rank
    t = bench.max_over_ranks(t_local, world, device="cpu")
    units = w.batch * w.n * w.nz_per_pass * 7
    value = bench.job_throughput(units, steps=3, world=world, t_total=t)
    np.savez(os.path.join(out_dir, f"r{rank}.npz"), seed=w.seeds[1], pump=w.pump, t=t, value=value)
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_get_distinct_instances_and_max_time(tmp_path):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r0 = np.load(tmp_path / "r0.npz")
    r1 = np.load(tmp_path / "r1.npz")
    assert r0["t"] == r1["t"] == 1.5                                  # max over ranks on both ranks
    assert np.array_equal(r0["pump"], r1["pump"])                     # same physics ...
    assert not np.array_equal(r0["seed"], r1["seed"])                 # ... different noise realisations
    assert np.isclose(np.linalg.norm(r0["seed"]), np.linalg.norm(r1["seed"]), rtol=1e-6)
    # whole-job value: units of ALL ranks over the max time
    w_units = 1 * 16384 * 100 * 7
    assert r0["value"] == r1["value"] == pytest.approx(2 * w_units * 3 / 1.5)


def test_rank0_workload_is_the_config_itself():
    sys.path.insert(0, ROOT)
    import bench
    import opo_workloads as W
    a, b = bench.make_workload("C1", 0), W.config1()
    assert np.array_equal(a.seeds[1], b.seeds[1]) and np.array_equal(a.seeds[2], b.seeds[2])
