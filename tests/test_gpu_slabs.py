"""the flood grid cut into row slabs, one handle per slab (here all on one GPU, which is
how the path can be exercised without a second device): each slab's flood kernel reads its halo row
from the neighbour slab in place, the wave speeds are max-reduced, the pedestrians of the first
handle sample, count into and raise the bed of whichever slab holds their cell.  The result must be
BIT-IDENTICAL to the single-handle run of the whole grid, and so must agree with the oracle."""
import numpy as np
import pytest

import oracle
from paper_1908_05232_b200 import binding, scenarios as S
from helpers import box
from gpu_common import mixed

pytestmark = pytest.mark.gpu


def _identical(one, slabs, sc, steps, chunks=4):
    for _ in range(chunks):
        one.step(steps); slabs.step(steps)
        a, b = slabs.read_conserved(), one.read_conserved()
        for k in ("h", "qx", "qy"):
            assert np.array_equal(a[k], b[k]), (k, float(np.max(np.abs(a[k] - b[k]))))
        sa, sb = slabs.stats(), one.stats()
        assert sa["t"] == sb["t"] and sa["dt"] == sb["dt"] and sa["step"] == sb["step"]
        assert sa["neg_depth_clamps"] == sb["neg_depth_clamps"]
        assert abs(sa["volume"] - sb["volume"]) <= 1e-13 * sb["volume"]
        assert np.array_equal(slabs.read_occupancy(), one.read_occupancy())
        if sc.n_peds:
            pa, pb = slabs.read_peds(), one.read_peds()
            for k in ("active", "fsm", "state", "cell"):
                assert np.array_equal(pa[k], pb[k]), k
            assert sa["hist"] == sb["hist"] and sa["deposits"] == sb["deposits"]
            assert (sa["cursor"], sa["layer"], sa["barrier_complete"]) == (sb["cursor"], sb["layer"], sb["barrier_complete"])


@pytest.mark.parametrize("n_slabs", [2, 3])
def test_config1_fp64_slabs_bit_identical_per_cell_kernel(n_slabs):
    sc = S.make(1)
    one = binding.Sim(sc); one.set_flood_variant(0)
    slabs = binding.SlabSim(sc, n_slabs)
    assert all(g.flood_variant() == 0 or g.flood_variant() == 4 for g in slabs.sims)
    for g in slabs.sims:
        g.set_flood_variant(0)
    # bins ordered by id (sim_set_deterministic): the pair forces are summed in the same order on the
    # single handle and on the slabs, so with the people -> flow coupling ON the flood state and every
    # pedestrian must agree bit for bit (agents walk across the cuts: Config 1 heads for one exit)
    one.set_deterministic(True); slabs.sims[0].set_deterministic(True)
    for _ in range(4):
        one.step(25); slabs.step(25)
        a, b = slabs.read_conserved(), one.read_conserved()
        for k in ("h", "qx", "qy"):
            assert np.array_equal(a[k].view(np.uint64), b[k].view(np.uint64)), k
        assert slabs.stats()["dt"] == one.stats()["dt"]
        pa, pb = slabs.read_peds(), one.read_peds()
        for k in ("x", "y", "vx", "vy"):
            assert np.array_equal(pa[k].view(np.uint64), pb[k].view(np.uint64)), k
        for k in ("active", "fsm", "state", "cell"):
            assert np.array_equal(pa[k], pb[k]), k
        assert np.array_equal(slabs.read_occupancy(), one.read_occupancy())
    rows = pb["cell"][pb["active"] == 1] // sc.nx
    assert len({int(r) // slabs.cuts[0][1] for r in rows}) >= 2          # people on both sides of a cut
    # ... and against the oracle within the multi-step tolerances
    o = oracle.Oracle(sc)
    o.step(100)
    sa, sb = slabs.stats(), o.stats()
    assert abs(sa["volume"] - sb["volume"]) <= 1e-10 * sb["volume"] and abs(sa["max_h"] - sb["max_h"]) <= 1e-9 * sb["max_h"]
    assert sa["hist"] == sb["hist"]
    assert mixed(slabs.read_conserved()["h"], o.read_conserved()["h"]) <= 1e-9


@pytest.mark.parametrize("n_slabs", [2, 4])
def test_fp32_tma_kernel_slabs_bit_identical_no_peds(n_slabs):
    sc = S.make(2, n=256, n_evac=0)
    sc.hydro_q = sc.hydro_q * 50.0
    one = binding.Sim(sc); one.set_flood_variant(4)
    slabs = binding.SlabSim(sc, n_slabs)
    for g in slabs.sims:
        g.set_flood_variant(4)
    _identical(one, slabs, sc, 150)
    assert slabs.stats()["max_h"] > 0.05


def test_single_step_parity_with_the_oracle_across_the_cut_fp32():
    """one step from identical state: flood 1e-5, every pedestrian integer exact -- agents on both
    sides of the cut, N_p written into the other slab, deposits raising the bed there"""
    sc = S.make(3, n=128, n_evac=400, n_resp=40)
    o = oracle.Oracle(sc)
    slabs = binding.SlabSim(sc, 2)
    o.step(1); slabs.step(1)
    a, b = slabs.read_conserved(), o.read_conserved()
    for k in ("h", "qx", "qy"):
        assert mixed(a[k], b[k]) <= 1e-5
    pa, pb = slabs.read_peds(), o.read_peds()
    for k in ("active", "fsm", "state", "cell"):
        assert np.array_equal(pa[k], pb[k]), k
    assert np.array_equal(slabs.read_occupancy().astype(np.int64), np.minimum(o.read_occupancy(), 255))
    cells = pb["cell"][pb["active"] == 1] // sc.nx
    assert (cells < 64).any() and (cells >= 64).any()


def test_barrier_across_slabs_full_run_matches_single_handle_aggregates():
    sc = S.make(3, n=128, n_evac=300, n_resp=60)
    one = binding.Sim(sc)
    slabs = binding.SlabSim(sc, 3)
    one.step(6000); slabs.step(6000)
    sa, sb = slabs.stats(), one.stats()
    assert sa["step"] == sb["step"]
    assert sb["deposits"] > 20 and abs(sa["deposits"] - sb["deposits"]) <= 2
    za, zb = slabs.read_flood(("z",))["z"], one.read_flood(("z",))["z"]
    assert np.max(np.abs(za - zb)) <= 0.05 + 1e-6               # at most one bag apart
    assert abs(sa["volume"] - sb["volume"]) <= 1e-4 * max(sb["volume"], 1.0)


def test_link_validation():
    sc = S.make(1)
    a = binding.Sim(sc, slab=(0, 32)); b = binding.Sim(sc, slab=(32, 32), with_peds=False)
    with pytest.raises(binding.FloodpedError):
        arr = (binding._vp * 2)(b._h, a._h)
        rc = a._L.sim_slab_link(arr, 2)
        if rc != 0:
            raise binding.FloodpedError(rc, a._L.sim_last_error(b._h).decode())
    g = binding.SlabSim(sc, 2)
    with pytest.raises(binding.FloodpedError):
        g.sims[0].step(1)
    with pytest.raises(binding.FloodpedError):
        g.sims[0].set_flood_variant(4)          # 64 columns: the strip sticks out of the grid, that path reads no halo row


def test_attach_refuses_a_barrier_line_outside_the_first_slab():
    """one process per slab: rank 0's tail kernel raises the bed after the step's only exchange, so a
    deposit into another process's rows would race with that process's next flood kernel"""
    import ctypes as C
    from paper_1908_05232_b200.replicas import slab_cuts
    sc = S.make(3, n=128, n_evac=50, n_resp=10)
    line_rows = np.asarray(sc.line_cells) // sc.nx
    for n_slabs, accepted in ((2, True), (8, False)):
        cuts = slab_cuts(sc.ny, n_slabs)
        assert (line_rows.max() < cuts[0][1]) == accepted
        sims = [binding.Sim(sc, slab=cut, with_peds=(r == 0)) for r, cut in enumerate(cuts)]
        descs = (binding.SlabDesc * n_slabs)()
        for r, g in enumerate(sims):
            g._chk(g._L.sim_slab_describe(g._h, C.byref(descs[r])))
        rc = sims[0]._L.sim_slab_attach(sims[0]._h, 0, n_slabs, descs)
        if accepted:
            assert rc == 0
        else:
            assert rc == binding.SIM_EINVAL and b"first slab" in sims[0]._L.sim_last_error(sims[0]._h)


def test_doors_and_trigger_on_slabs_match_the_oracle_step_by_step():
    """the doors of SURVEY 8f-3 on a grid cut into two slabs: newcomers are placed by the first slab's
    tail kernel, walk across the cut, the trigger comes from the maximum of BOTH slabs' wave speeds"""
    from gpu_common import sync
    sc = S.door_hall(n=64, slots=200, t_pre=20.0, spawn_rate=0.5, t_end=200.0)
    o = oracle.Oracle(sc)
    slabs = binding.SlabSim(sc, 2)
    seen = False
    for k in range(60):
        o.step(1); slabs.step(1)
        sa, sb = slabs.stats(), o.stats()
        assert sa["spawned"] == sb["spawned"] and sa["triggered"] == sb["triggered"], k
        pa, pb = slabs.read_peds(), o.read_peds()
        if not seen:                       # dry phase: dt = dt_max on both sides, everything discrete is exact
            assert np.array_equal(pa["active"], pb["active"]) and np.array_equal(pa["fsm"], pb["fsm"]), k
        seen = seen or bool(sb["triggered"])
    assert seen and sb["spawned"] > 20
    rows = pb["cell"][pb["active"] == 1] // sc.nx
    assert (rows < 32).any() and (rows >= 32).any()
