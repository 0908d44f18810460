"""The N>1 path on CPU: two gloo ranks.  Stars are independent units, so the multi-rank logic is
the cost-balanced deal of the stars (longest-processing-time greedy on N_pts x n_freq), the max/sum
aggregation of the per-rank figures, and ONE all-gather of the per-star peak table
(paper_2302_01293_b200/shard.py; bench.py uses the same functions over NCCL)."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _fake_peak_table(ids, top_k=3):
    """A stand-in for the search result of the stars `ids`: records that depend on the star id only (the search
    itself needs a GPU; what is tested here is that the plumbing puts every star's own record in its own row)."""
    from paper_2302_01293_b200 import bls
    tab = np.zeros((len(ids), top_k), dtype=bls.PEAK_DTYPE)
    for r in range(top_k):
        tab[:, r]["k"] = np.asarray(ids) * 10 + r
        tab[:, r]["freq"] = 0.25 + np.asarray(ids) * 1e-3 + r
        tab[:, r]["snr"] = np.asarray(ids, dtype=np.float32) - r
        tab[:, r]["m"] = 3 + r
    return tab


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    import bench
    from paper_2302_01293_b200 import shard
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ids = bench.shard_star_ids(5, rank)
    (ms, e2e), (ev, st) = bench.aggregate_over_ranks([10.0 + rank, 20.0 - rank], [100 * (rank + 1), 5], world, "cpu")
    np.save(os.path.join(out_dir, f"r{rank}.npy"), np.array([ms, e2e, ev, st, ids[0], ids[-1]], dtype=np.float64))
    # cost-balanced deal + gather: 37 stars with a heavy tail, every rank computes the same partition
    rng = np.random.default_rng(3)
    cost = np.exp(rng.normal(0.0, 2.0, 37))
    parts = shard.lpt_partition(cost, world)
    mine = parts[rank]
    table = shard.gather_tables(_fake_peak_table(mine), mine, cost.size)
    np.save(os.path.join(out_dir, f"table{rank}.npy"), table)
    # an empty shard is legal (fewer stars than ranks)
    few = shard.lpt_partition(np.array([5.0]), world)
    t1 = shard.gather_tables(_fake_peak_table(few[rank]), few[rank], 1)
    assert t1.shape == (1, 3) and t1[0, 0]["k"] == 0
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_shards_aggregation_and_gather(tmp_path):
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    r0, r1 = np.load(tmp_path / "r0.npy"), np.load(tmp_path / "r1.npy")
    # both ranks see the same whole-job figures: time = max over ranks, work = sum over ranks
    assert list(r0[:4]) == list(r1[:4]) == [11.0, 20.0, 300.0, 10.0]
    # disjoint, contiguous slices for the cost pass
    assert (r0[4], r0[5], r1[4], r1[5]) == (0, 4, 5, 9)
    # the gathered table = the single-rank table, on every rank
    want = _fake_peak_table(np.arange(37))
    t0, t1 = np.load(tmp_path / "table0.npy"), np.load(tmp_path / "table1.npy")
    assert t0.tobytes() == want.tobytes() and t1.tobytes() == want.tobytes()


def test_lpt_partition_properties():
    from paper_2302_01293_b200 import shard
    rng = np.random.default_rng(0)
    cost = np.exp(rng.normal(0.0, 1.5, 500))
    for world in (1, 2, 3, 8):
        parts = shard.lpt_partition(cost, world)
        allv = np.concatenate(parts)
        assert np.array_equal(np.sort(allv), np.arange(500))            # a partition
        assert all(np.all(np.diff(p) > 0) for p in parts)               # sorted ids per rank
        loads = np.array([cost[p].sum() for p in parts])
        assert loads.max() - loads.min() <= cost.max() + 1e-12          # the LPT guarantee
    assert shard.lpt_partition(np.array([]), 2)[0].size == 0
    # ties are broken deterministically (lower index, lower rank)
    parts = shard.lpt_partition(np.ones(4), 2)
    assert [p.tolist() for p in parts] == [[0, 2], [1, 3]]


def test_lpt_balance_on_config5_costs(orc, cfg):
    """the top 1 % of config-5 stars hold ~20 % of the work.  On 2,000 stars dealt to 2 (and 8) ranks
    LPT stays within 5 % of the mean, equal-count contiguous slices do not (costs from the oracle's grid on the
    timestamps alone)."""
    from paper_2302_01293_b200 import shard, synth
    n = 2000
    cost = np.zeros(n)
    for sid in range(n):
        t, rho = synth.star_times(5, sid)
        cost[sid] = float(orc.grid(cfg, t, rho)["n_freq"]) * t.size
    for world in (2, 8):
        parts = shard.lpt_partition(cost, world)
        assert shard.imbalance(cost, parts) <= 1.05
    contiguous = [np.arange(r * n // 8, (r + 1) * n // 8) for r in range(8)]
    assert shard.imbalance(cost, contiguous) > shard.imbalance(cost, shard.lpt_partition(cost, 8))


def test_star_times_match_make_star():
    from paper_2302_01293_b200 import synth
    for config, sid in [(1, 0), (2, 3), (3, 11), (4, 2), (5, 0), (5, 19), (5, 28)]:
        t, rho = synth.star_times(config, sid)
        full = synth.make_star(config, sid)
        assert np.array_equal(t, full[0]) and rho == full[3]


def test_shards_reproduce_the_single_rank_stars():
    import bench
    from paper_2302_01293_b200 import synth
    whole = synth.make_batch(2, n_stars=4)
    a, b = bench.make_workload(2, 2, 0), bench.make_workload(2, 2, 1)
    assert np.array_equal(np.concatenate([a.t, b.t]), whole.t)
    assert np.array_equal(np.concatenate([a.y, b.y]), whole.y)
    assert np.array_equal(np.concatenate([a.rho, b.rho]), whole.rho)


def test_reference_arm_other_ranks_do_nothing(monkeypatch, capsys):
    import bench
    monkeypatch.setenv("RANK", "1")
    bench.run_reference(type("A", (), {"stars": 2, "config": 2, "steps": 1, "warmup": 0, "gpus": 2})())
    assert capsys.readouterr().out == ""


def test_parallel_generation_reproduces_make_batch():
    """bench.py builds a workload from blocks of stars made by worker processes; every star has its own seed
    (synth.make_star), so the packed batch is the one make_batch gives for the same ids, in the same order."""
    import multiprocessing
    import bench
    from paper_2302_01293_b200 import synth
    with multiprocessing.get_context("fork").Pool(2) as pool:
        got = bench.make_workload_parallel(5, 7, 18, pool, block=4)
        ids = np.array([3, 40, 5, 22, 9])
        got2 = bench.make_workload_ids(5, ids, pool, block=2)
        rp, t, rho = bench.make_times_ids(5, ids, pool, block=2)
    ref = synth.make_batch(5, star_ids=np.arange(7, 18))
    for k in ("row_ptr", "t", "y", "dy", "rho", "rstar", "star_ids"):
        assert np.array_equal(getattr(got, k), getattr(ref, k)), k
    assert got.truth.tobytes() == ref.truth.tobytes()
    ref2 = synth.make_batch(5, star_ids=ids)
    for k in ("row_ptr", "t", "y", "dy", "rho"):
        assert np.array_equal(getattr(got2, k), getattr(ref2, k)), k
    assert np.array_equal(rp, ref2.row_ptr) and np.array_equal(t, ref2.t) and np.array_equal(rho, ref2.rho)


def test_gather_without_a_process_group_is_a_reorder():
    """One GPU: no process group; the gathered table is the local one put in global star order."""
    from paper_2302_01293_b200 import shard
    ids = np.array([3, 0, 2, 1])
    got = shard.gather_tables(_fake_peak_table(ids), ids, 4)
    assert got.tobytes() == _fake_peak_table(np.arange(4)).tobytes()
    with pytest.raises(RuntimeError):                       # rows that do not partition the job are refused
        shard.unpack_rows(shard.pack_rows(_fake_peak_table(np.array([0, 0])), np.array([0, 0])), 2,
                          _fake_peak_table(ids).dtype, (3,))


def test_reference_arm_prints_one_json_line(capsys):
    """bench.py --impl reference on rank 0: one JSON line with the contract's keys, timed on a bounded oracle sample."""
    import json
    import bench
    args = type("A", (), {"stars": 12, "config": 2, "steps": 1, "warmup": 0, "gpus": 1, "ref_budget": 0.3})()
    bench.run_reference(args)
    lines = [ln for ln in capsys.readouterr().out.splitlines() if ln.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == bench.METRIC and d["unit"] == bench.UNIT
    assert d["value"] > 0 and d["higher_is_better"] is True and d["vs_baseline"] is None
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"] == {"value": d["value"], "unit": bench.UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert "workload" in d["config"] and d["gpu_launches"] == 0
