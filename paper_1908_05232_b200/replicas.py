"""Independent replicas across processes / GPUs ("replicas only").

The coupled step runs on one GPU (BASELINE.json north_star) and the paper's own workloads are
sweeps of independent runs: 4 hydrographs, with / without the roughness feedback
(P:L186), 36 group-size x layer runs.  So N GPUs run N independent `sim_t` handles, one
process per GPU, and the only traffic between ranks is the bookkeeping here: which rank runs
which item, the max-over-ranks of a time, and the gather of small result records on rank 0.
There is no data-path collective.  Works with any torch.distributed backend (nccl on GPUs, gloo
in the CPU tests); with no process group it degenerates to one rank.
"""
from __future__ import annotations

from typing import Callable, Sequence


def _dist():
    import torch.distributed as dist
    return dist if dist.is_available() and dist.is_initialized() else None


def world() -> tuple[int, int]:
    """(rank, world_size) of the current process group, (0, 1) without one."""
    d = _dist()
    return (d.get_rank(), d.get_world_size()) if d else (0, 1)


def shard(n_items: int, rank: int, world_size: int) -> list[int]:
    """Items of `range(n_items)` that `rank` runs: round-robin, so that a sweep ordered by cost
    (e.g. by number of layers) spreads evenly.  Disjoint over ranks, complete over the group."""
    if not (0 <= rank < world_size):
        raise ValueError("rank out of range")
    return list(range(rank, n_items, world_size))


def max_over_ranks(value: float, device=None) -> float:
    """Max of a per-rank scalar (a device-timed duration) over the group: the job is as slow as
    its slowest replica.  `device`: where the reduction tensor lives (cuda for nccl)."""
    d = _dist()
    if not d:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    d.all_reduce(t, op=d.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    d = _dist()
    if not d:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    d.all_reduce(t, op=d.ReduceOp.SUM)
    return float(t.item())


def gather_records(mine: dict[int, object]) -> dict[int, object] | None:
    """Every rank passes {item index: small picklable record}; rank 0 gets the union (checked to
    be disjoint), the others None."""
    d = _dist()
    if not d:
        return dict(mine)
    rank, ws = d.get_rank(), d.get_world_size()
    out = [None] * ws if rank == 0 else None
    d.gather_object(mine, out, dst=0)
    if rank != 0:
        return None
    merged: dict[int, object] = {}
    for part in out:
        for k, v in part.items():
            if k in merged:
                raise RuntimeError(f"item {k} was run by two ranks")
            merged[k] = v
    return merged


def run_sweep(items: Sequence[object], run_one: Callable[[int, object], object]) -> list[object] | None:
    """Run `run_one(index, item)` for this rank's shard of `items`; rank 0 returns the records in
    item order (None elsewhere).  `run_one` owns its GPU work (one `Sim` handle per item)."""
    rank, ws = world()
    mine = {i: run_one(i, items[i]) for i in shard(len(items), rank, ws)}
    merged = gather_records(mine)
    if merged is None:
        return None
    missing = [i for i in range(len(items)) if i not in merged]
    if missing:
        raise RuntimeError(f"items {missing} were not run")
    return [merged[i] for i in range(len(items))]


# ------------------------------------------------------------------------------------------ 8f-1
def barrier_sweep_items(layers=(1, 2, 3, 4, 5, 6), shares=(0.05, 0.10, 0.20, 0.30, 0.40, 0.50)):
    """The paper's Scenario-2 grid: number of sandbag layers x share of responders."""
    return [dict(n_layers=int(nl), share=float(sh)) for nl in layers for sh in shares]


def run_barrier_item(item: dict, n: int = 128, n_people: int = 400, t_end: float = 600.0, device="cuda:0",
                     t_release: float = 120.0, steps_per_poll: int = 32) -> dict:
    """One run of the pre-flood intervention on the synthetic hall (Config 3 recipe at n x n):
    `share` of the people are responders who build `n_layers` layers of the barrier line, the
    flood is released at `t_release`.  Returns the quantities of the paper's Figs 8-10:
    deployment time, depth downstream of the barrier, maximum hazard rate."""
    import numpy as np
    from . import binding, scenarios as S

    n_resp = max(1, int(round(item["share"] * n_people)))
    sc = S.shopping_centre(n=n, n_evac=n_people - n_resp, n_resp=n_resp, t_release=t_release, t_end=t_end,
                           name="barrier_sweep")
    sc.n_layers = int(item["n_layers"])
    g = binding.Sim(sc, device=device)
    deployed_at = None
    max_hr = 0.0
    while True:
        g.step(steps_per_poll)
        st = g.stats()
        max_hr = max(max_hr, st["max_hr"])
        if deployed_at is None and st["barrier_complete"]:
            deployed_at = st["t"]                       # resolution: one poll interval
        if st["t"] >= t_end:
            break
    fl = g.read_flood(("h",))
    h = fl["h"].reshape(sc.ny, sc.nx)
    line_j = int(sc.line_cells[0] // sc.nx)
    walk = sc.mask.reshape(sc.ny, sc.nx) == 0
    down = walk.copy(); down[:line_j + 1, :] = False      # the exit side of the barrier line
    rec = dict(item, n_responders=n_resp, deployment_time=deployed_at, deposits=int(st["deposits"]),
               depth_downstream=float(h[down].mean()), max_depth_downstream=float(h[down].max()),
               max_hr=float(max_hr), volume=float(st["volume"]), steps=int(st["step"]), t=float(st["t"]))
    g.close()
    return rec


def main(argv=None):
    """`python -m paper_1908_05232_b200.replicas [--n 128] [--people 400] [--t-end 600]` -- the 36-run
    grid on the local GPU, or sharded over ranks under torchrun (one process per GPU, nccl)."""
    import argparse
    import json
    import os
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=128)
    ap.add_argument("--people", type=int, default=400)
    ap.add_argument("--t-end", type=float, default=600.0)
    a = ap.parse_args(argv)
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        import torch
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    recs = run_sweep(barrier_sweep_items(),
                     lambda i, it: run_barrier_item(it, n=a.n, n_people=a.people, t_end=a.t_end, device=f"cuda:{local}"))
    if recs is not None:
        for r in recs:
            print(json.dumps(r))
    if _dist():
        _dist().destroy_process_group()


if __name__ == "__main__":
    main()


# ---------------------------------------------------------------------------- row slabs
# Host logic of the row-slab decomposition (include/floodped.h sim_slab_link): which rows a slab
# holds, which slab holds a row, and the one collective of the data path -- the global time step is
# the minimum over the slabs, i.e. a MAX reduction of the slabs' wave speeds.

def slab_cuts(ny: int, n_slabs: int) -> list[tuple[int, int]]:
    """(first row, number of rows) per slab: equal slabs of ceil(ny / n) rows, the last one shorter;
    fewer slabs than asked when ny is small.  This is the layout sim_slab_link checks."""
    if ny <= 0 or n_slabs <= 0:
        raise ValueError("ny and n_slabs must be positive")
    rows = -(-ny // n_slabs)
    return [(j0, min(rows, ny - j0)) for j0 in range(0, ny, rows)]


def slab_of_row(row: int, ny: int, n_slabs: int) -> int:
    """index of the slab that holds `row` (what the pedestrian kernels compute per agent)"""
    cuts = slab_cuts(ny, n_slabs)
    if not (0 <= row < ny):
        raise ValueError("row outside the grid")
    return min(row // cuts[0][1], len(cuts) - 1)


def global_wave_speed(local_lambda: float, device=None) -> float:
    """max over the slabs of max_cells (|u| + c) / dx: every rank then derives the same
    dt = min(dt_max, CFL / lambda).  One 8-byte all-reduce per step."""
    return max_over_ranks(local_lambda, device)
