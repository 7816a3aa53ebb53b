"""SURVEY 8f-4 with one PROCESS per slab (binding.SlabRank): two processes, both on the one GPU this
box has, their workspaces shared through CUDA IPC, the 8-byte wave-speed reduction through
torch.distributed (gloo here; NCCL refuses two ranks on one device).  No kernel waits on another:
the processes' kernels are ordered by the host-side collective.  The two slabs together must be
bit-identical to the single-handle run, and the pedestrians of rank 0 must walk, count N_p and
sample the water in rank 1's slab."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

pytestmark = pytest.mark.gpu


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir, case):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_1908_05232_b200 import binding, scenarios as S
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        if case == "flood_fp32_tma":
            sc = S.make(2, n=256, n_evac=0); sc.hydro_q = sc.hydro_q * 50.0
            steps = 300
        else:
            sc = S.make(1); sc.couple_roughness = 0
            steps = 100
        g = binding.SlabRank(sc)
        if case == "flood_fp32_tma":
            assert g.sim.flood_variant() == 4
        else:
            assert g.sim.flood_variant() == 0
        g.step(steps)
        c = g.sim.read_conserved()
        st = g.sim.stats()
        occ = g.sim.read_occupancy()
        peds = g.sim.read_peds() if rank == 0 and sc.n_peds else None
        np.savez(os.path.join(out_dir, f"r{rank}.npz"), h=c["h"], qx=c["qx"], qy=c["qy"], occ=occ, t=st["t"], dt=st["dt"],
                 volume=st["volume"], cell=(peds["cell"] if peds else np.zeros(0, np.int32)),
                 active=(peds["active"] if peds else np.zeros(0, np.uint8)))
        g.close()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("case", ["flood_fp32_tma", "config1_fp64_peds"])
def test_two_processes_one_slab_each_bit_identical_to_one_handle(tmp_path, case):
    import torch.multiprocessing as mp
    from paper_1908_05232_b200 import binding, scenarios as S
    try:
        mp.spawn(_worker, args=(2, _free_port(), str(tmp_path), case), nprocs=2, join=True)
    except Exception as e:                              # a box that forbids CUDA IPC between processes cannot run this path
        if any(k in str(e) for k in ("cudaIpc", "IPC", "ipc", "shared memory", "not permitted", "peer access is not supported")):
            pytest.skip(f"CUDA IPC between processes is not available here: {str(e)[-200:]}")
        raise
    r0, r1 = np.load(tmp_path / "r0.npz"), np.load(tmp_path / "r1.npz")
    if case == "flood_fp32_tma":
        sc = S.make(2, n=256, n_evac=0); sc.hydro_q = sc.hydro_q * 50.0
        one = binding.Sim(sc); one.set_flood_variant(4); one.step(300)
    else:
        sc = S.make(1); sc.couple_roughness = 0
        one = binding.Sim(sc); one.set_flood_variant(0); one.step(100)      # the kernel the slabs of a 64-wide grid take
    c, st = one.read_conserved(), one.stats()
    assert (float(r0["t"]), float(r0["dt"])) == (float(r1["t"]), float(r1["dt"])) == (st["t"], st["dt"]), (float(r0["t"]), float(r1["t"]), st["t"])
    for k in ("h", "qx", "qy"):
        both = np.concatenate([r0[k], r1[k]])
        assert np.array_equal(both, c[k]), (k, float(np.max(np.abs(both - c[k]))))
    assert abs(float(r0["volume"]) + float(r1["volume"]) - st["volume"]) <= 1e-12 * st["volume"]
    if case != "flood_fp32_tma":
        # pedestrians (on rank 0) have walked in both slabs and their N_p landed in the slab that holds the cell
        rows = r0["cell"][r0["active"] == 1] // sc.nx
        assert (rows < 32).any() and (rows >= 32).any()
        occ = np.concatenate([r0["occ"], r1["occ"]]).astype(np.int64)
        # N_p of the last step counts the people at level n, r0["active"] is level n+1: somebody may have left since
        n_act = int((r0["active"] == 1).sum())
        assert n_act <= occ.sum() <= n_act + 8 and occ[32 * sc.nx:].sum() > 0 and occ[:32 * sc.nx].sum() > 0
        assert np.abs(occ - one.read_occupancy().astype(np.int64)).sum() <= 4      # pair sums are order-dependent: last-bit positions
