"""Multi-process host logic of the "replicas only" multi-GPU path, on CPU with the
gloo backend, world_size 2: sharding of sweep items, max-over-ranks timing, gather on rank 0, and
the aggregation bench.py applies to its per-rank numbers.  No GPU, no kernels."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_1908_05232_b200 import replicas  # noqa: E402


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world_size, port, out_dir):
    import json
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_1908_05232_b200 import replicas as R
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world_size)
    try:
        assert R.world() == (rank, world_size)
        items = R.barrier_sweep_items()                        # the paper's 6 x 6 grid
        ran = []

        def fake_run(i, item):                                 # stands in for a GPU run
            ran.append(i)
            return dict(item, index=i, rank=rank, cost=item["n_layers"] * 10.0)

        recs = R.run_sweep(items, fake_run)
        ms = R.max_over_ranks(100.0 + 50.0 * rank)             # rank 1 is the slow replica
        total = R.sum_over_ranks(len(ran))
        line = bench.aggregate(ms_max=ms, world=world_size, ncell=1000, done=10, active=7)
        with open(os.path.join(out_dir, f"r{rank}.json"), "w") as f:
            json.dump(dict(ran=ran, recs=recs, ms=ms, total=total, line=line), f)
    finally:
        dist.destroy_process_group()


def test_sweep_sharding_timing_and_gather_world_size_2(tmp_path):
    import json
    import torch.multiprocessing as mp
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r0 = json.load(open(tmp_path / "r0.json"))
    r1 = json.load(open(tmp_path / "r1.json"))
    assert sorted(r0["ran"] + r1["ran"]) == list(range(36))            # complete
    assert not set(r0["ran"]) & set(r1["ran"])                          # disjoint
    assert abs(len(r0["ran"]) - len(r1["ran"])) <= 1                    # balanced
    assert r1["recs"] is None and len(r0["recs"]) == 36                 # rank 0 holds everything
    for i, rec in enumerate(r0["recs"]):                                # in item order, run by the owner
        assert rec["index"] == i and rec["rank"] == i % 2
    assert r0["ms"] == r1["ms"] == 150.0                                # max over ranks
    assert r0["total"] == 36.0
    # whole-job throughput: every rank's cells / the slowest rank's time
    assert r0["line"]["value"] == pytest.approx(2 * 1000 * 10 / 0.150)
    assert r0["line"]["agent_updates_per_s"] == pytest.approx(2 * 7 * 10 / 0.150)
    assert r0["line"]["ms_per_step"] == pytest.approx(15.0)


def test_single_process_degenerates_to_one_rank():
    assert replicas.world() == (0, 1)
    assert replicas.shard(5, 0, 1) == [0, 1, 2, 3, 4]
    assert replicas.max_over_ranks(3.5) == 3.5
    out = replicas.run_sweep(["a", "b", "c"], lambda i, it: (i, it))
    assert out == [(0, "a"), (1, "b"), (2, "c")]
    with pytest.raises(ValueError):
        replicas.shard(5, 2, 2)


def test_shards_partition_any_size():
    for n in (0, 1, 7, 36, 37):
        for ws in (1, 2, 3, 8):
            parts = [replicas.shard(n, r, ws) for r in range(ws)]
            assert sorted(sum(parts, [])) == list(range(n))
            assert max(map(len, parts)) - min(map(len, parts)) <= 1


# ---------------------------------------------------------------------------- row slabs

def _slab_worker(rank, world_size, port, out_dir):
    import json
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_1908_05232_b200 import replicas as R
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world_size)
    try:
        ny = 8191                                              # not divisible: the last slab is shorter
        cut = R.slab_cuts(ny, world_size)[rank]
        cuts = [None] * world_size
        dist.all_gather_object(cuts, cut)
        lam = R.global_wave_speed([3.25, 7.5][rank])           # rank 1 holds the fastest cell
        dt = min(0.1, 0.5 / lam)
        with open(os.path.join(out_dir, f"s{rank}.json"), "w") as f:
            json.dump(dict(cut=cut, cuts=cuts, lam=lam, dt=dt), f)
    finally:
        dist.destroy_process_group()


def test_slab_partition_and_global_dt_world_size_2(tmp_path):
    import json
    import torch.multiprocessing as mp
    port = _free_port()
    mp.spawn(_slab_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r0 = json.load(open(tmp_path / "s0.json")); r1 = json.load(open(tmp_path / "s1.json"))
    assert r0["cuts"] == r1["cuts"] == [[0, 4096], [4096, 4095]]   # contiguous, in order, cover the grid
    assert r0["lam"] == r1["lam"] == 7.5 and r0["dt"] == r1["dt"] == 0.5 / 7.5


def test_slab_cuts_cover_any_grid_and_owner_lookup():
    for ny in (1, 2, 7, 64, 8191, 8192):
        for n in (1, 2, 3, 8):
            cuts = replicas.slab_cuts(ny, n)
            assert cuts[0][0] == 0 and sum(c[1] for c in cuts) == ny and len(cuts) <= n
            assert all(cuts[k][0] + cuts[k][1] == cuts[k + 1][0] for k in range(len(cuts) - 1))
            assert all(c[1] == cuts[0][1] for c in cuts[:-1]) and 0 < cuts[-1][1] <= cuts[0][1]
            for row in {0, ny // 2, ny - 1}:
                r = replicas.slab_of_row(row, ny, n)
                assert cuts[r][0] <= row < cuts[r][0] + cuts[r][1]
