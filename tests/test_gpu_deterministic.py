"""sim_set_deterministic (include/floodped.h): every sort bin ordered by original agent id, so that
the social-force sum no longer runs in the order warps reached an atomic counter.  The GPU
model "reproduced the same predictions as the sequential counterpart" can only be checked
over many steps if two GPU runs reproduce each other first: these tests pin that, bit for bit."""
import numpy as np
import pytest

import oracle
from paper_1908_05232_b200 import binding, scenarios as S
from gpu_common import make_pair, sync
from test_gpu_parity import _compare_flood, _ped_compare

pytestmark = pytest.mark.gpu


def bits(a):
    """the array as unsigned integers of its own width: -0.0 != +0.0, NaN == the same NaN"""
    a = np.ascontiguousarray(a)
    return a.view({1: np.uint8, 4: np.uint32, 8: np.uint64}[a.dtype.itemsize])


def same_bits(p, q, keys):
    return all(np.array_equal(bits(p[k]), bits(q[k])) for k in keys)


PED_KEYS = ("x", "y", "vx", "vy", "timer", "state", "fsm", "active", "cell")


def _crowd():
    sc = S.make(2)
    sc.hydro_q = sc.hydro_q * 10.0            # the run of test_config2_multi_step_aggregates_fp32
    return sc


def test_two_runs_give_the_same_bits_fp32_crowd():
    sc = _crowd()
    runs = []
    for _ in range(3):
        g = binding.Sim(sc); g.set_deterministic(True)
        assert g.kernels_per_step() == binding.Sim(sc).kernels_per_step() + 2
        g.step(400)
        runs.append((g.read_peds(), g.read_conserved(), g.stats()))
    for p, c, st in runs[1:]:
        assert same_bits(p, runs[0][0], PED_KEYS)
        assert same_bits(c, runs[0][1], ("h", "qx", "qy"))
        assert st["t"] == runs[0][2]["t"] and st["hist"] == runs[0][2]["hist"]
    assert runs[0][2]["hist"][5] > 100          # people have been leaving through the crowded exit


@pytest.mark.parametrize("cfg,kw", [(2, {}), (4, dict(n=256, n_peds=20000))])
def test_bins_are_in_id_order_which_is_the_order_of_the_oracles_cell_lists(cfg, kw):
    sc = S.make(cfg, **kw)
    o, g = make_pair(sc, evolve=25)
    g.set_deterministic(True)
    g.step(3); o.step(3)                       # a few steps so that the slots of A are no longer in id order
    sync(o, g, sc)
    ob, gb = o.binning(), g.bin_peds()
    nb = ob["nbx"] * ob["nby"]
    assert np.array_equal(gb["key"], ob["key"]) and np.array_equal(gb["start"][:nb + 1], ob["start"])
    order, start = gb["order"], gb["start"]
    assert np.array_equal(np.sort(order), np.arange(sc.n_peds))
    # active part of the sorted buffer: (key, id) strictly increasing = a stable sort of the ids by key
    n_act = int(start[nb])
    k = gb["key"][order[:n_act]].astype(np.int64) * sc.n_peds + order[:n_act]
    assert np.all(np.diff(k) > 0)
    assert max(np.diff(start[:nb + 1])) >= 3   # some bins hold several agents: the order inside was tested


def test_results_do_not_depend_on_the_slot_order_the_agents_arrive_in():
    """two handles whose slot order differs (one has been sorting with the atomic ranks for a while)
    are given the same state: from there on they produce the same bits"""
    sc = _crowd()
    o = oracle.Oracle(sc)
    g1 = binding.Sim(sc); g2 = binding.Sim(sc)
    g1.set_deterministic(True)
    g2.step(200)                               # default mode: slots now in some atomic order
    g2.set_deterministic(True)
    o.step(200)
    sync(o, g1, sc); sync(o, g2, sc)
    g1.step(150); g2.step(150)
    assert same_bits(g1.read_peds(), g2.read_peds(), PED_KEYS)
    assert same_bits(g1.read_conserved(), g2.read_conserved(), ("h", "qx", "qy"))
    assert np.array_equal(g1.read_occupancy(), g2.read_occupancy())


@pytest.mark.parametrize("cfg,kw,evolve", [(1, {}, 40), (2, {}, 300), (3, dict(n=128, n_evac=400, n_resp=40), 30),
                                           (4, dict(n=256, n_peds=5000), 150)])
def test_single_step_parity_with_the_oracle_in_deterministic_mode(cfg, kw, evolve):
    sc = S.make(cfg, **kw)
    o, g = make_pair(sc, evolve=evolve)
    g.set_deterministic(True)
    p0 = o.read_peds(); dt = o.stats()["dt"]
    dep = (o.stats()["deposits"], g.stats()["deposits"])
    o.step(1); g.step(1)
    _compare_flood(o, g, sc.real_bits)
    assert np.array_equal(g.read_occupancy().astype(np.int64), np.minimum(o.read_occupancy(), 255))
    _ped_compare(o, g, sc, p0, dt, dep)


def test_switching_modes_between_steps_keeps_the_state():
    sc = S.make(2, n=64, n_evac=300)
    g = binding.Sim(sc)
    g.step(20)
    before = g.read_peds()
    g.set_deterministic(True)
    assert same_bits(g.read_peds(), before, PED_KEYS)
    g.step(20); g.set_deterministic(False); g.step(20)
    st = g.stats()
    assert st["step"] == 60 and sum(st["hist"]) == sc.n_peds
