"""Pins for the oracle's SURVEY 8f-3 features (readings D1-D9 of DESIGN.md):
open (transmissive) domain edges, entrance doors that let pedestrians in before the flood, their
wandering to a destination door, and the evacuation trigger.  The paper prints no algorithm for
any of this, so the pins are what the mathematics and the generator's publication fix: known-answer
vectors of Philox4x32-10, the exact volume balance with outflow, a uniform stream that an open edge
must leave untouched, supercritical outflow equal to the same flow in a longer channel, spawn counts
in closed form, and scripted timelines."""
import os

import numpy as np
import pytest

import oracle
from paper_1908_05232_b200 import scenarios as S
from helpers import box, GOLDEN, doors_box as _doors_box

G = 9.81
W, E, So, N = 1, 2, 4, 8


# ------------------------------------------------------------------ D5: the generator

def test_philox4x32_10_known_answers():
    n = 0
    with open(os.path.join(GOLDEN, "philox_kat.txt")) as f:
        for line in f:
            p = line.split("#")[0].split()
            if not p or p[0] != "kat":
                continue
            v = [int(t, 16) for t in p[1:]]
            assert oracle.philox4x32(v[0:4], v[4:6]) == v[6:10]
            n += 1
    assert n == 3


def test_philox_counter_streams_are_distinct_and_uniform():
    r = np.array([oracle.philox4x32([k, 0, 0, 0], [0x5eed, 0]) for k in range(4000)], np.float64) / 2.0 ** 32
    assert len({tuple(row) for row in r}) == 4000
    for col in range(4):                                   # mean 1/2 +- 4 sigma, variance 1/12
        assert abs(r[:, col].mean() - 0.5) < 4 * (1 / 12 / 4000) ** 0.5
        assert abs(r[:, col].var() - 1 / 12) < 0.01


# ------------------------------------------------------------------ D1: open edges

def test_uniform_stream_passes_open_edges_unchanged():
    """zero-gradient ghost: a uniform stream through open W and E edges has equal fluxes on both
    faces of every cell, so nothing changes, and what leaves at E equals what enters at W."""
    sc = box(40, 5, dx=1.0, h0=0.8, u0=1.5, manning=0.0, open_sides=W | E, dt_max=0.05)
    o = oracle.Oracle(sc)
    o.step(50)
    c = o.read_conserved()
    assert np.max(np.abs(c["h"] - 0.8)) < 1e-14 and np.max(np.abs(c["qx"] - 1.2)) < 1e-14 and np.all(c["qy"] == 0)
    assert abs(o.stats()["outflow_volume"]) < 1e-11        # +q dy dt at E, -q dy dt at W


def test_volume_balance_with_outflow_and_draining():
    """V(t) = V0 - outflow (+ clamp) exactly; a dam break towards an open edge drains the box while
    the closed box keeps its volume (the invariant of the first-order pins)."""
    n = 40
    h0 = np.where(np.arange(n)[None, :] < 20, 1.0, 0.2) * np.ones((6, 1))
    vols = []
    for sides in (0, E):
        o = oracle.Oracle(box(n, 6, dx=1.0, h0=h0, manning=0.01, open_sides=sides))
        v0 = o.stats()["volume"]
        last = v0
        for _ in range(30):
            o.step(10)
            st = o.stats()
            assert abs(st["volume"] - (v0 - st["outflow_volume"] + st["clamped_volume"])) <= 1e-12 * v0
            assert st["volume"] <= last + 1e-12
            last = st["volume"]
        vols.append((v0, last, st["outflow_volume"]))
    assert abs(vols[0][1] - vols[0][0]) <= 1e-12 * vols[0][0] and vols[0][2] == 0.0
    assert vols[1][1] < 0.8 * vols[1][0] and vols[1][2] > 0.0


@pytest.mark.parametrize("order", [1, 2])
def test_supercritical_outflow_equals_the_longer_channel(order):
    """Froude 2.7: every wave moves downstream, the upwind flux at the open edge is the physical flux
    of the last cell, so cutting the channel there changes nothing upstream of the cut."""
    nl, ns, ny = 80, 50, 3
    x = np.arange(nl) + 0.5
    h = 0.5 + 0.05 * np.exp(-((x - 20.0) ** 2) / 18.0)
    u = np.full(nl, 6.0)
    def run(n, sides):
        sc = box(n, ny, dx=1.0, h0=np.tile(h[:n], (ny, 1)), u0=np.tile(u[:n], (ny, 1)), manning=0.0,
                 open_sides=sides, dt_max=0.02, flood_order=order)
        o = oracle.Oracle(sc)
        o.step(150)                                         # 3 s: the bump travels 18-25 cells
        return {k: v.reshape(ny, n) for k, v in o.read_conserved().items()}
    a, b = run(nl, W | E), run(ns, W | E)
    for k in ("h", "qx", "qy"):
        d = np.abs(a[k][:, :ns] - b[k])
        if order == 1:
            assert d.max() <= 1e-13, k
        else:
            # the slope of the last cell is zero (M1: a domain edge), so the cut is first order in the
            # last cells; the limiter lets that reach a few cells upstream, fading fast
            assert d[:, :ns - 12].max() <= 1e-8 and d.max() <= 2e-2, (k, d.max())   # qx ~ 3: 0.3 %


def test_inflow_faces_stay_inflow_on_an_open_side():
    sc = box(20, 4, dx=1.0, h0=0.0, manning=0.0, open_sides=So,
             inflow_cell=np.arange(5, 10, dtype=np.int32), inflow_side=np.full(5, 2, np.uint8),
             hydro_t=np.array([0.0, 100.0]), hydro_q=np.array([1.0, 1.0]))
    o = oracle.Oracle(sc)
    o.step(5)
    st = o.stats()
    assert abs(st["volume"] - (st["t"] * 1.0 - st["outflow_volume"])) <= 1e-12 and st["volume"] > 0


# ------------------------------------------------------------------ D3, D4: doors

def test_spawn_cadence_closed_form():
    """rate 0.5 /s/door at dt = 0.25 s: the credit grows by exactly 1/8 a step, so every door lets one
    pedestrian in at steps 8, 16, 24, ...  (binary fractions: no rounding anywhere)"""
    sc = _doors_box()
    o = oracle.Oracle(sc)
    for k in range(1, 41):
        o.step(1)
        assert o.stats()["spawned"] == 3 * (k // 8)
    p = o.read_peds()
    # lowest free slot first: a newcomer bound for its own door leaves at once and frees its slot again,
    # so at most 15 slots were ever used and they are the first ones
    act = p["active"] == 1
    assert not np.any(p["fsm"][15:] >= 8) and not np.any(act[15:])
    assert np.all((p["fsm"][act] >= 8) & (p["fsm"][act] < 8 + 3)) and act.sum() >= 5


def test_newcomers_start_inside_their_door_cell_with_a_speed_in_range():
    sc = _doors_box(rate=4.0, slots=600)                              # one per door and step
    o = oracle.Oracle(sc)
    o.step(1)
    p = o.read_peds()
    assert o.stats()["spawned"] == 3
    for k in range(3):                                                # door k -> slot k (doors in index order)
        ci, cj = int(sc.door_cells[k]) % sc.nx, int(sc.door_cells[k]) // sc.nx
        assert ci + 0.1 <= p["x"][k] < ci + 0.9 and cj + 0.1 <= p["y"][k] < cj + 0.9
        assert p["vx"][k] == 0 and p["vy"][k] == 0 and p["active"][k] == 1
    o.step(150)
    # destinations: uniform over the doors ("equal probability"): chi-square, 2 dof, 99.9 % point 13.8
    n = int(o.stats()["spawned"])
    r = np.array([oracle.philox4x32([k, 0, 0, 0], [1234, 0]) for k in range(n)], np.uint64)
    dest = (r[:, 0] * np.uint64(3)) >> np.uint64(32)
    cnt = np.bincount(dest.astype(int), minlength=3)
    assert ((cnt - n / 3) ** 2 / (n / 3)).sum() < 13.8


def test_population_cap_and_slot_reuse():
    sc = _doors_box(rate=4.0, slots=40, target=10)
    o = oracle.Oracle(sc)
    for _ in range(30):
        o.step(1)
        p = o.read_peds()
        assert int(p["active"].sum()) <= 10
    assert o.stats()["spawned"] > 10                                  # those that left were replaced
    # slots are reused lowest first: nobody ever sat beyond the number ever needed at once
    assert not np.any(p["fsm"][20:] >= 8)


def test_wanderer_walks_to_its_door_and_leaves_there_not_at_the_exit():
    sc = _doors_box(rate=0.0, slots=2)
    o = oracle.Oracle(sc)
    ex = int(sc.exit_cells[0])
    # slot 0 stands on the exit cell bound for door 1; slot 1 stands next to door 2 bound for it
    d2 = int(sc.door_cells[2])
    x = np.array([ex % 24 + 0.5, d2 % 24 + 1.5]); y = np.array([ex // 24 + 0.5, d2 // 24 + 0.5])
    o.write_peds(x, y, np.zeros(2), np.zeros(2), np.array([8 + 1, 8 + 2], np.uint8), np.ones(2, np.uint8), np.zeros(2))
    o.step(1)
    p = o.read_peds()
    assert p["active"][0] == 1 and p["active"][1] == 0               # wanderers ignore the exit; arrival within 1 cell
    assert p["vx"][0] < 0                                            # heads west, towards its door
    o.step(400)
    assert o.read_peds()["active"][0] == 0 and o.stats()["triggered"] == 0


# ------------------------------------------------------------------ D7, D8: the trigger

def test_trigger_stops_entries_and_turns_wanderers_into_evacuees():
    sc = S.door_hall(n=64, slots=300, t_pre=60.0, spawn_rate=0.2, t_end=900.0)
    o = oracle.Oracle(sc)
    seen, spawned_at_trigger = False, None
    while o.stats()["t"] < 900.0:
        before = o.stats()
        o.step(1)
        st = o.stats()
        if not seen:
            assert st["triggered"] == (1 if st["max_h"] > sc.h_dry else 0)   # fires on the first wet cell of U^{n+1}
            assert st["t"] <= 60.0 + 40.0
            if st["triggered"]:
                seen, spawned_at_trigger = True, st["spawned"]
                assert before["spawned"] == st["spawned"]              # no entry in the step that saw water
                assert np.any(o.read_peds()["fsm"] >= 8)               # wanderers are still on their way
                o.step(1)
                p = o.read_peds()
                assert not np.any(p["fsm"][p["active"] == 1] >= 8)     # one step later all of them evacuate
        else:
            assert st["spawned"] == spawned_at_trigger
    assert seen and spawned_at_trigger > 50
    st = o.stats()
    assert st["hist"][5] == 300                                        # free slots + everybody who got in has left
    assert abs(st["volume"] - 300.0) <= 0.1                            # the triangle of Q, step quadrature


def test_initial_water_means_triggered_from_the_start():
    sc = _doors_box(rate=4.0)
    sc.h0 = np.full(sc.nx * sc.ny, 0.05)
    o = oracle.Oracle(sc)
    assert o.stats()["triggered"] == 1
    o.step(20)
    assert o.stats()["spawned"] == 0
