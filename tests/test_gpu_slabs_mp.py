"""SURVEY 8f-4 with one PROCESS per slab (binding.SlabRank): two processes, both on the one GPU this
box has, their workspaces shared through CUDA IPC, the 8-byte wave-speed reduction through
torch.distributed (gloo here; NCCL refuses two ranks on one device).  No kernel waits on another:
the processes' kernels are ordered by the host-side collective.  The two slabs together must be
bit-identical to the single-handle run -- flood state AND pedestrians, with the people -> flow
coupling on (bins in id order, sim_set_deterministic) -- and the pedestrians of rank 0 must walk,
count N_p and sample the water in rank 1's slab."""
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


def _scenario(case):
    from paper_1908_05232_b200 import scenarios as S
    if case == "flood_fp32_tma":
        sc = S.make(2, n=256, n_evac=0); sc.hydro_q = sc.hydro_q * 50.0
        return sc, 300, 4
    if case == "config1_fp64_peds":
        return S.make(1), 100, 0                           # 64 columns: the per-cell kernel
    sc = S.make(3, n=128, n_evac=300, n_resp=60)           # sandbag line on row 20: inside the first slab (see sim_slab_attach)
    return sc, 6000, 0


def _ipc_child(q_in, q_out):
    try:
        t = q_in.get(timeout=120)
        q_out.put(("ok", float(t.sum().item())))
    except Exception as e:                                  # reported to the parent, which names it in the skip reason
        q_out.put(("error", repr(e)[-300:]))


def _cuda_ipc_probe():
    """capability probe: a 4-float CUDA tensor is handed to a second process (cudaIpcGetMemHandle /
    cudaIpcOpenMemHandle under torch.multiprocessing, what binding.SlabRank uses) and summed there"""
    import torch
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q_in, q_out = ctx.Queue(), ctx.Queue()
    p = ctx.Process(target=_ipc_child, args=(q_in, q_out))
    p.start()
    t = torch.full((4,), 1.5, device="cuda:0")
    torch.cuda.synchronize()
    try:
        q_in.put(t)
        kind, val = q_out.get(timeout=180)
    except Exception as e:
        kind, val = "error", repr(e)[-300:]
    p.join(30)
    if p.is_alive():
        p.kill()
    return (kind == "ok" and val == 6.0), val


def _worker(rank, world, port, out_dir, case):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_1908_05232_b200 import binding, scenarios as S
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        sc, steps, variant = _scenario(case)
        g = binding.SlabRank(sc)
        if g.sim.flood_variant() != variant:
            g.sim.set_flood_variant(variant)
        g.set_deterministic(True)
        g.step(steps)
        c = g.sim.read_conserved()
        st = g.sim.stats()
        occ = g.sim.read_occupancy()
        peds = g.sim.read_peds() if rank == 0 and sc.n_peds else None
        np.savez(os.path.join(out_dir, f"r{rank}.npz"), h=c["h"], qx=c["qx"], qy=c["qy"], occ=occ, t=st["t"], dt=st["dt"],
                 volume=st["volume"], deposits=st["deposits"], z=g.sim.read_flood(("z",))["z"],
                 **{k: (peds[k] if peds else np.zeros(0, np.uint8)) for k in ("cell", "active", "x", "y", "vx", "vy", "fsm", "state")})
        g.close()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("case", ["flood_fp32_tma", "config1_fp64_peds", "config3_fp32_barrier"])
def test_two_processes_one_slab_each_bit_identical_to_one_handle(tmp_path, case):
    import torch.multiprocessing as mp
    from paper_1908_05232_b200 import binding
    ok, why = _cuda_ipc_probe()
    if not ok:                                          # a hardware / container capability, probed, not guessed from an error text
        pytest.skip(f"CUDA IPC probe failed (a 4-float CUDA tensor sent to a second process could not be read there): {why}")
    mp.spawn(_worker, args=(2, _free_port(), str(tmp_path), case), nprocs=2, join=True)
    r0, r1 = np.load(tmp_path / "r0.npz"), np.load(tmp_path / "r1.npz")
    sc, steps, variant = _scenario(case)
    one = binding.Sim(sc); one.set_flood_variant(variant); one.set_deterministic(True); one.step(steps)
    c, st = one.read_conserved(), one.stats()
    assert (float(r0["t"]), float(r0["dt"])) == (float(r1["t"]), float(r1["dt"])) == (st["t"], st["dt"]), (float(r0["t"]), float(r1["t"]), st["t"])
    u = {4: np.uint32, 8: np.uint64}
    for k in ("h", "qx", "qy"):
        both = np.concatenate([r0[k], r1[k]])
        assert np.array_equal(both.view(u[both.itemsize]), c[k].view(u[both.itemsize])), (k, float(np.max(np.abs(both - c[k]))))
    assert abs(float(r0["volume"]) + float(r1["volume"]) - st["volume"]) <= 1e-12 * st["volume"]
    if sc.n_peds:
        # pedestrians (on rank 0) have walked in both slabs, their N_p landed in the slab that holds the cell,
        # and every one of them carries the bits of the single-handle run
        half = sc.ny // 2
        occ = np.concatenate([r0["occ"], r1["occ"]])
        if case == "config1_fp64_peds":                 # (by the end of the Config 3 run everybody has left)
            rows = r0["cell"][r0["active"] == 1] // sc.nx
            assert (rows < half).any() and (rows >= half).any()
            assert occ[half * sc.nx:].sum() > 0 and occ[:half * sc.nx].sum() > 0
        assert np.array_equal(occ, one.read_occupancy())
        p = one.read_peds()
        for k in ("x", "y", "vx", "vy"):
            assert np.array_equal(r0[k].view(u[r0[k].itemsize]), p[k].view(u[p[k].itemsize])), k
        for k in ("cell", "active", "fsm", "state"):
            assert np.array_equal(r0[k], p[k]), k
    if case == "config3_fp32_barrier":                  # responders have raised the bed, in the first slab's rows
        assert st["deposits"] > 20 and int(r0["deposits"]) == st["deposits"]
        z = np.concatenate([r0["z"], r1["z"]])
        assert np.array_equal(z, one.read_flood(("z",))["z"]) and (z != np.asarray(sc.z, z.dtype)).any()
