"""The N>1 path of bench.py on CPU: two gloo ranks.  Stars are independent units, so the only
multi-rank logic is the shard assignment and the max/sum aggregation of the per-rank figures."""
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
    ids = bench.shard_star_ids(5, rank)
    ms, e2e, ev, st = bench.aggregate_over_ranks(10.0 + rank, 20.0 - rank, 100 * (rank + 1), 5, world, "cpu")
    np.save(os.path.join(out_dir, f"r{rank}.npy"), np.array([ms, e2e, ev, st, ids[0], ids[-1]], dtype=np.float64))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_shards_and_aggregation(tmp_path):
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    r0, r1 = np.load(tmp_path / "r0.npy"), np.load(tmp_path / "r1.npy")
    # both ranks see the same whole-job figures: time = max over ranks, work = sum over ranks
    assert list(r0[:4]) == list(r1[:4]) == [11.0, 20.0, 300.0, 10.0]
    # disjoint, contiguous shards
    assert (r0[4], r0[5], r1[4], r1[5]) == (0, 4, 5, 9)


def test_shards_reproduce_the_single_rank_stars():
    sys.path.insert(0, ROOT)
    import bench
    from paper_2302_01293_b200 import synth
    whole = synth.make_batch(2, n_stars=4)
    a, b = bench.make_workload(2, 2, 0), bench.make_workload(2, 2, 1)
    assert np.array_equal(np.concatenate([a.t, b.t]), whole.t)
    assert np.array_equal(np.concatenate([a.y, b.y]), whole.y)
    assert np.array_equal(np.concatenate([a.rho, b.rho]), whole.rho)


def test_reference_arm_other_ranks_do_nothing(monkeypatch, capsys):
    sys.path.insert(0, ROOT)
    import bench
    monkeypatch.setenv("RANK", "1")
    bench.run_reference(type("A", (), {"stars": 2, "config": 2, "steps": 1, "warmup": 0, "gpus": 2})())
    assert capsys.readouterr().out == ""


def test_parallel_generation_reproduces_make_batch():
    """bench.py --chunk builds each chunk from blocks of stars made by worker processes; every star has its own seed
    (synth.make_star), so the packed chunk is the batch make_batch gives for the same ids."""
    import multiprocessing
    sys.path.insert(0, ROOT)
    import bench
    from paper_2302_01293_b200 import synth
    with multiprocessing.get_context("fork").Pool(2) as pool:
        got = bench.make_workload_parallel(5, 7, 18, pool, block=4)
    ref = synth.make_batch(5, star_ids=np.arange(7, 18))
    for k in ("row_ptr", "t", "y", "dy", "rho", "rstar", "star_ids"):
        assert np.array_equal(getattr(got, k), getattr(ref, k)), k
    assert got.truth.tobytes() == ref.truth.tobytes()
