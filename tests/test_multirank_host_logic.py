"""CPU test (gloo, world_size 2) of the N > 1 path of bench.py.  The hot path shards by spatial
partition with no data-path collective: every rank assembles its own block,
the job's time is the slowest rank's, the job's value is the points of all ranks over that time."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out_dir):
    import torch.distributed as dist

    import bench

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = bench.rank_workload("slope", rank, world)
        # a stand-in for the device-timed milliseconds of this rank: rank 1 is the slow one
        ms_local = 10.0 + 5.0 * rank
        ms = bench.max_over_ranks(ms_local, world)
        value = bench.job_value(w.Nq, world, ms)
        np.savez(os.path.join(out_dir, f"r{rank}.npz"), nodes=w.nodes[:64], Nq=w.Nq, N=w.N, ms=ms, value=value,
                 bc=w.bc_nodes[:16])
    finally:
        dist.destroy_process_group()


def test_two_ranks_get_their_own_partitions_and_the_slowest_time(tmp_path):
    import torch.multiprocessing as mp

    world, port = 2, 29000 + os.getpid() % 2000
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    r0, r1 = (np.load(tmp_path / f"r{r}.npz") for r in range(world))
    assert int(r0["N"]) == int(r1["N"]) == 62500 and int(r0["Nq"]) == int(r1["Nq"]) == 460992   # weak scaling
    assert not np.array_equal(r0["nodes"], r1["nodes"])          # own jitter stream per rank
    assert np.array_equal(r0["bc"], r1["bc"])                    # same topology and boundary sets
    assert float(r0["ms"]) == float(r1["ms"]) == 15.0            # max over ranks, on every rank
    assert float(r0["value"]) == 2 * 460992 / 15e-3              # whole-job points per second


def test_single_rank_is_the_config_itself():
    import bench
    import workloads

    a, b = bench.rank_workload("slope", 0, 1), workloads.config("slope")
    assert np.array_equal(a.nodes, b.nodes) and np.array_equal(a.qpts, b.qpts)
    assert bench.max_over_ranks(3.5, 1) == 3.5
    assert bench.job_value(1000, 1, 2.0) == 500000.0
