"""GPU parity of SURVEY 8f-3 (readings D1-D9): open domain edges, doors and
newcomers, wanderers, the evacuation trigger -- the CUDA path through the C ABI against the oracle.
Integers (who is in, which slot, destination, FSM, spawn count, trigger) bit-exact; a newcomer's
position bit-exact (both sides form it in fp64 from the same Philox words); flood fields within
1e-12 / 1e-5."""
import os

import numpy as np
import pytest

import oracle
from paper_1908_05232_b200 import binding, scenarios as S
from helpers import box, doors_box, GOLDEN
from gpu_common import make_pair, sync, mixed, rounded

pytestmark = pytest.mark.gpu

TOL = {64: 1e-12, 32: 1e-5}
W, E, So, N = 1, 2, 4, 8


def test_device_philox_known_answers_and_oracle_agreement():
    g = binding.Sim(S.make(1, n_peds=8))
    rows, want = [], []
    with open(os.path.join(GOLDEN, "philox_kat.txt")) as f:
        for line in f:
            p = line.split("#")[0].split()
            if p and p[0] == "kat":
                v = [int(t, 16) for t in p[1:]]
                rows.append(v[:6]); want.append(v[6:])
    assert np.array_equal(g.philox(rows), np.array(want, np.uint32))
    rng = np.random.default_rng(5)
    r = rng.integers(0, 2 ** 32, size=(500, 6), dtype=np.uint64)
    got = g.philox(r)
    ref = np.array([oracle.philox4x32(row[:4], row[4:]) for row in r], np.uint32)
    assert np.array_equal(got, ref)


@pytest.mark.parametrize("bits", [64, 32])
@pytest.mark.parametrize("order", [1, 2])
def test_open_edges_single_step_parity(bits, order):
    rng = np.random.default_rng(11)
    nx, ny = 45, 23
    z = 0.1 * rng.random((ny, nx))
    h0 = 0.4 + 0.3 * rng.random((ny, nx))
    u0 = 1.0 + rng.random((ny, nx)); v0 = rng.random((ny, nx)) - 0.3
    mask = (rng.random((ny, nx)) < 0.05).astype(np.uint8)
    mask[0, 10:20] = 0                                          # the inflow cells
    sc = box(nx, ny, dx=0.5, real_bits=bits, z=z, h0=h0, u0=u0, v0=v0, mask=mask, manning=0.02,
             open_sides=W | E | N, flood_order=order,
             inflow_cell=np.arange(10, 20, dtype=np.int32), inflow_side=np.full(10, 2, np.uint8),
             hydro_t=np.array([0.0, 100.0]), hydro_q=np.array([3.0, 3.0]))
    for evolve in (0, 12):
        o, g = make_pair(sc, evolve=evolve)
        assert g.flood_variant() == (5 if order == 2 else 0)
        if not evolve:
            sync(o, g, sc)
        out0 = (o.stats()["outflow_volume"], g.stats()["outflow_volume"])
        o.step(1); g.step(1)
        a, b = g.read_conserved(), o.read_conserved()
        for k in ("h", "qx", "qy"):
            assert mixed(a[k], b[k]) <= TOL[bits], (k, mixed(a[k], b[k]))
        sa, sb = g.stats(), o.stats()
        da, db = sa["outflow_volume"] - out0[1], sb["outflow_volume"] - out0[0]
        assert db != 0.0 and abs(da - db) <= 10 * TOL[bits] * max(abs(db), sb["volume"] * 1e-3)
        assert abs(sa["dt"] - sb["dt"]) <= 10 * TOL[bits] * sb["dt"]


@pytest.mark.parametrize("bits", [64, 32])
def test_open_edge_volume_balance_over_a_run(bits):
    n = 40
    h0 = np.where(np.arange(n)[None, :] < 20, 1.0, 0.2) * np.ones((6, 1))
    g = binding.Sim(box(n, 6, dx=1.0, real_bits=bits, h0=h0, manning=0.01, open_sides=E))
    v0 = g.stats()["volume"]
    g.step(300)
    st = g.stats()
    assert st["volume"] < 0.8 * v0
    assert abs(st["volume"] - (v0 - st["outflow_volume"] + st["clamped_volume"])) <= (1e-12 if bits == 64 else 2e-5) * v0


@pytest.mark.parametrize("bits", [64, 32])
def test_newcomers_bit_exact_slots_destinations_positions(bits):
    sc = doors_box(rate=4.0, slots=300, real_bits=bits)         # one newcomer per door and step
    o = oracle.Oracle(sc); g = binding.Sim(sc)
    for step in range(1, 41):
        o.step(1); g.step(1)
        a, b = g.read_peds(), o.read_peds()
        sa, sb = g.stats(), o.stats()
        assert sa["spawned"] == sb["spawned"] == 3 * step and sa["triggered"] == sb["triggered"] == 0
        assert np.array_equal(a["active"], b["active"]) and np.array_equal(a["fsm"], b["fsm"])
        act = b["active"] == 1
        new = act & (np.hypot(b["vx"], b["vy"]) == 0)           # let in this step: still at rest at their door
        assert new.sum() >= 1
        assert np.array_equal(a["x"][new].astype(np.float64), b["x"][new]) and np.array_equal(a["y"][new].astype(np.float64), b["y"][new])
        # everybody else: one step from identical state (re-injected below); the newcomers crowd at the
        # doors, so the bound carries the conditioning of their force sums
        tol = TOL[bits] * sc.nx + 1e3 * TOL[bits]
        assert np.max(np.abs(a["x"][act] - b["x"][act])) <= tol and np.max(np.abs(a["y"][act] - b["y"][act])) <= tol
        sync(o, g, sc)


def test_spawn_cadence_population_cap_and_slot_reuse_match_the_oracle():
    sc = doors_box(rate=0.5, slots=40, target=10, real_bits=32)
    o = oracle.Oracle(sc); g = binding.Sim(sc)
    for _ in range(240):
        # crowds are chaotic (newcomers start a few centimetres apart), so who leaves WHEN is compared one
        # step at a time from identical re-injected state; credit, counter and trigger live on each side
        o.step(1); g.step(1)
        a, b = g.read_peds(), o.read_peds()
        assert g.stats()["spawned"] == o.stats()["spawned"]
        assert np.array_equal(a["active"], b["active"]) and np.array_equal(a["fsm"], b["fsm"])
        assert int(a["active"].sum()) <= 10
        sync(o, g, sc)
    assert g.stats()["spawned"] > 10


def test_wanderer_timeline_on_the_gpu():
    sc = doors_box(rate=0.0, slots=2, real_bits=64)
    o = oracle.Oracle(sc); g = binding.Sim(sc)
    ex, d2 = int(sc.exit_cells[0]), int(sc.door_cells[2])
    x = np.array([ex % 24 + 0.5, d2 % 24 + 1.5]); y = np.array([ex // 24 + 0.5, d2 // 24 + 0.5])
    args = (x, y, np.zeros(2), np.zeros(2), np.array([8 + 1, 8 + 2], np.uint8), np.ones(2, np.uint8), np.zeros(2))
    o.write_peds(*args); g.write_peds(*args)
    o.step(1); g.step(1)
    a, b = g.read_peds(), o.read_peds()
    assert np.array_equal(a["active"], b["active"]) and list(a["active"]) == [1, 0]
    assert abs(a["vx"][0] - b["vx"][0]) <= 1e-12 and a["vx"][0] < 0
    o.step(400); g.step(400)
    assert g.read_peds()["active"][0] == 0 and g.stats()["triggered"] == 0 and g.stats()["hist"] == o.stats()["hist"]


def test_trigger_run_door_hall_fp32():
    """dry pre-flood phase: dt = dt_max on both sides, so entries are bit-exact until the trigger;
    afterwards the aggregates of DESIGN.md 5.4."""
    sc = S.door_hall(n=64, slots=300, t_pre=60.0, spawn_rate=0.2, t_end=900.0)
    o = oracle.Oracle(sc); g = binding.Sim(sc)
    trig = None
    for k in range(200):
        if k:
            sync(o, g, sc)
        o.step(1); g.step(1)
        sa, sb = g.stats(), o.stats()
        assert sa["triggered"] == sb["triggered"] and sa["spawned"] == sb["spawned"]
        a, b = g.read_peds(), o.read_peds()
        assert np.array_equal(a["active"], b["active"]) and np.array_equal(a["fsm"], b["fsm"])
        if sb["triggered"] and trig is None:
            trig = k
        if trig is not None and k >= trig + 3:
            break
    assert trig is not None and sb["spawned"] > 50
    assert not np.any(a["fsm"][a["active"] == 1] >= 8)
    o.step(10 ** 6); g.step(10 ** 6)
    sa, sb = g.stats(), o.stats()
    assert abs(sa["t"] - 900.0) < 1e-6 and abs(sb["t"] - 900.0) < 1e-9
    assert sa["spawned"] == sb["spawned"] and sa["hist"][5] == sb["hist"][5] == 300
    assert abs(sa["volume"] - sb["volume"]) <= 1e-4 * sb["volume"]
    assert abs(sa["max_h"] - sb["max_h"]) <= 1e-3 * sb["max_h"]


def test_initial_water_triggers_and_hooks_are_guarded():
    sc = doors_box(rate=4.0, real_bits=32)
    sc.h0 = np.full(sc.nx * sc.ny, 0.05, np.float32)
    g = binding.Sim(sc)
    assert g.stats()["triggered"] == 1
    g.step(20)
    assert g.stats()["spawned"] == 0
    with pytest.raises(binding.FloodpedError):
        g.set_overlap(True)
    g2 = binding.Sim(box(16, 16, dx=1.0, h0=0.2, open_sides=E))
    assert g2.flood_variant() == 0
    with pytest.raises(binding.FloodpedError):
        g2.set_flood_variant(1)
