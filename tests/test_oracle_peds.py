"""Pins for the pedestrian / coupling half of the CPU oracle.  No GPU."""
import math

import numpy as np
import pytest

import oracle
from paper_1908_05232_b200 import scenarios as S
from helpers import box, golden_rows, compass_scene


# ------------------------------------------------------------------ HR, Table 1, roughness (paper)

def test_hazard_rate_paper_values_and_table1():
    for h, u, v, hr, cls in golden_rows("paper_values.txt", "hr_case"):
        got = oracle.hazard_rate(h, u, v)
        assert abs(got - hr) < 1e-15                       # HR = (V + 0.5) h
        assert abs(got - h * (max(abs(u), abs(v)) + 0.5)) < 1e-15
        assert oracle.risk_state(h, got) == int(cls)
    for hr, cls in golden_rows("paper_values.txt", "hr_edge"):
        assert oracle.risk_state(1.0, hr) == int(cls)
        assert oracle.risk_state(1.0, math.nextafter(hr, 0.0)) == (int(cls) - 1 if hr <= 2.5 else 4)
    assert oracle.risk_state(1e-3, 5.0) == 0 and oracle.risk_state(0.0, 0.0) == 0   # dry class (C17)
    assert oracle.risk_state(math.nextafter(1e-3, 1.0), 0.0) == 1


def test_float_replay_of_integer_decisions():
    """real_bits = 32 evaluates HR in float: pick (h, V) whose float product lands on the 0.75
    edge while the exact product is below it."""
    f = np.float32
    rng = np.random.default_rng(0)
    V = rng.uniform(0.1, 2.0, 400000).astype(f)
    s = (V + f(0.5)).astype(f)
    h = (f(0.75) / s).astype(f)                              # float quotient: product is ~0.75
    flt = (s * h).astype(f)
    exact = (V.astype(np.float64) + 0.5) * h.astype(np.float64)
    hit = np.flatnonzero((flt == f(0.75)) & (exact < 0.75))
    found = 0
    for k in hit[:5]:
        hk, Vk = float(h[k]), float(V[k])
        assert oracle.hazard_rate(hk, Vk, 0.0, real_bits=32) == 0.75
        assert oracle.hazard_rate(hk, -Vk, 0.0, real_bits=64) < 0.75
        assert oracle.risk_state(hk, oracle.hazard_rate(hk, Vk, 0.0, 32), real_bits=32) == 2
        assert oracle.risk_state(hk, oracle.hazard_rate(hk, Vk, 0.0, 64), real_bits=64) == 1
        found += 1
    assert found >= 1


def test_roughness_rule():
    for Np, want in golden_rows("paper_values.txt", "rough"):
        assert abs(oracle.roughness(0.01, int(Np), 20) - want) < 1e-15


def test_walking_speeds_of_table1_are_the_defaults():
    sc = S.make(1, n_peds=1)
    for cls, sp in golden_rows("paper_values.txt", "speed"):
        assert sc.speed_wet[int(cls) - 1] == sp
    assert sc.hr_edges[:3] == (0.75, 1.5, 2.5)


# ------------------------------------------------------------------ occupancy and binning

def _crowd(n, seed, L, clustered=True):
    rng = np.random.default_rng(seed)
    if clustered:
        c = rng.uniform(0.3 * L, 0.7 * L, size=(4, 2))
        p = c[rng.integers(0, 4, n)] + rng.normal(0, 0.8, size=(n, 2))
        p = np.clip(p, 0.01, L - 0.01)
    else:
        p = rng.uniform(0, L, size=(n, 2))
    return p[:, 0], p[:, 1]


def test_occupancy_and_binning_against_brute_force():
    for dx, n in ((1.0, 16), (0.5, 32), (0.25, 64)):
        x, y = _crowd(400, 3, n * dx)
        sc = box(n, n, dx=dx, peds=dict(x=x, y=y), h0=0.0)
        o = oracle.Oracle(sc)
        o.step(1)
        ci = np.floor(x / dx).astype(int); cj = np.floor(y / dx).astype(int)
        assert np.array_equal(o.read_occupancy(), np.bincount(cj * n + ci, minlength=n * n))
        o2 = oracle.Oracle(sc)                          # binning of the initial positions
        b = o2.binning()
        k = b["k"]
        assert k == math.ceil(1.0 / dx) and b["nbx"] == -(-n // k)
        key = (cj // k) * b["nbx"] + ci // k
        assert np.array_equal(b["key"], key)
        cnt = np.bincount(key, minlength=b["nbx"] * b["nby"])
        assert np.array_equal(b["count"], cnt)
        assert np.array_equal(b["start"], np.concatenate([[0], np.cumsum(cnt)]))


def test_roughness_feedback_slows_the_flow_only_where_people_stand():
    n = 16
    h0 = np.full((n, n), 0.5); u0 = np.full((n, n), 1.0)
    xs = np.full(25, 5.5); ys = np.full(25, 7.5)          # 25 people in cell (5,7): capped at 20
    sc = box(n, n, dx=1.0, h0=h0, u0=u0, manning=0.01, peds=dict(x=xs, y=ys), A_s=0.0)
    o = oracle.Oracle(sc); o.step(1)
    ref = oracle.Oracle(box(n, n, dx=1.0, h0=h0, u0=u0, manning=0.01)); ref.step(1)
    off = oracle.Oracle(box(n, n, dx=1.0, h0=h0, u0=u0, manning=0.01, peds=dict(x=xs, y=ys), A_s=0.0,
                            couple_roughness=0)); off.step(1)
    a, b, c = o.read_conserved()["qx"], ref.read_conserved()["qx"], off.read_conserved()["qx"]
    cell = 7 * n + 5
    others = np.arange(n * n) != cell
    assert np.array_equal(a[others], b[others]) and np.array_equal(c, b)
    dt = ref.stats()["t"]
    D0 = 1 + dt * 9.81 * 0.01 ** 2 * 0.5 * 1.0 / 0.5 ** (7 / 3)
    D1 = 1 + dt * 9.81 * 0.21 ** 2 * 0.5 * 1.0 / 0.5 ** (7 / 3)   # n = 0.01 (1 + 20)
    assert abs(a[cell] / b[cell] - D0 / D1) < 1e-12


# ------------------------------------------------------------------ social force

def test_celllist_equals_brute_force_neighbour_search():
    for dx, n in ((1.0, 20), (0.5, 40), (0.25, 80)):
        x, y = _crowd(512, 7, n * dx)
        sc = box(n, n, dx=dx, peds=dict(x=x, y=y))
        o = oracle.Oracle(sc)
        ax, ay = o.social_celllist()
        bx, by = oracle.social_bruteforce(x, y, np.ones(512, np.uint8), sc.A_s, sc.B_s, sc.radius, sc.R_int)
        scale = max(np.abs(bx).max(), np.abs(by).max())
        assert scale > 1.0
        assert np.max(np.abs(ax - bx)) <= 1e-12 * scale and np.max(np.abs(ay - by)) <= 1e-12 * scale


def test_pair_force_value_direction_and_cutoff():
    A, B, r, R = 25.0, 0.08, 0.3, 1.0
    x = np.array([2.0, 2.5, 2.0, 3.2]); y = np.array([2.0, 2.0, 2.0, 2.0])   # agent 2 coincides with 0
    ax, ay = oracle.social_bruteforce(x, y, np.ones(4, np.uint8), A, B, r, R)
    f01 = A * math.exp((0.6 - 0.5) / B)                    # Helbing-type repulsion (C24)
    f13 = A * math.exp((0.6 - 0.7) / B)
    assert abs(ax[0] - (-f01)) < 1e-12 and ay[0] == 0.0     # pushed away from 1; coincident 2 skipped
    assert abs(ax[1] - (2 * f01 - f13)) < 1e-12            # from 0 and 2 (+x), from 3 (-x)
    assert abs(ax[3] - f13) < 1e-12                         # 3 is 1.2 m from 0 and 2: beyond R_int
    ax2, _ = oracle.social_bruteforce(x, y, np.array([1, 0, 1, 1], np.uint8), A, B, r, R)
    assert ax2[0] == 0.0 and ax2[3] == 0.0                  # inactive agents exert nothing


# ------------------------------------------------------------------ kinematics

def test_free_walk_relaxes_geometrically():
    """One agent, no neighbours, dry floor: |v_k - v0| = |v_0 - v0| (1 + dt/tau)^-k (closed form
    of the backward-Euler relaxation)."""
    n = 64
    sc = box(n, 8, dx=1.0, peds=dict(x=[1.5], y=[4.5], vpref=[1.3]), exit_cell=4 * n + n - 1, dt_max=0.2)
    o = oracle.Oracle(sc)
    x_prev, t = 1.5, 0.0
    for k in range(1, 40):
        o.step(1)
        p = o.read_peds()
        want = 1.3 * (1 - (1 + 0.2 / 0.5) ** (-k))
        assert abs(p["vx"][0] - want) < 1e-14 and p["vy"][0] == 0.0
        assert abs(p["x"][0] - (x_prev + 0.2 * want)) < 1e-13
        x_prev = p["x"][0]
        assert p["state"][0] == 0 and p["active"][0] == 1


@pytest.mark.parametrize("code", range(8))
def test_all_eight_navigation_codes_walk_their_compass_direction_at_unit_norm(code):
    """The eight codes of the navigation field (navigation agents hand out the direction to
    the destination) are the compass points E, NE, N, NW, W, SW, S, SE, and the desired direction is a
    UNIT vector: a diagonal walker is no faster than a straight one.  Closed form of the free walk
    (backward-Euler relaxation) along e = (di, dj) / |(di, dj)|:
        v_k = v0 (1 - (1 + dt/tau)^-k) e ,   |v_k| < v0 for every k, -> v0.
    The expected direction is written out here by hand, not taken from any table of the code."""
    r = 1.0 / math.sqrt(2.0)
    compass = {0: (1, 0), 1: (r, r), 2: (0, 1), 3: (-r, r), 4: (-1, 0), 5: (-r, -r), 6: (0, -1), 7: (r, -r)}
    ex, ey = compass[code]
    o = oracle.Oracle(compass_scene(code))
    x, y = 32.5, 32.5
    for k in range(1, 25):
        o.step(1)
        p = o.read_peds()
        s = 1.3 * (1 - (1 + 0.2 / 0.5) ** (-k))
        assert abs(p["vx"][0] - s * ex) < 1e-14 and abs(p["vy"][0] - s * ey) < 1e-14, (code, k)
        assert math.hypot(p["vx"][0], p["vy"][0]) < 1.3
        x += 0.2 * s * ex; y += 0.2 * s * ey
        assert abs(p["x"][0] - x) < 1e-12 and abs(p["y"][0] - y) < 1e-12
    assert math.hypot(p["vx"][0], p["vy"][0]) > 1.3 * (1 - 1e-3)      # 1.4^-24 = 3e-4: at the desired speed, not above
    # a code outside 0..7 (255 = none) gives no direction: the agent stays put
    o = oracle.Oracle(compass_scene(255)); o.step(5)
    p = o.read_peds()
    assert p["vx"][0] == 0.0 and p["vy"][0] == 0.0 and p["x"][0] == 32.5 and p["y"][0] == 32.5


def test_wet_speed_follows_table1_and_trapped_agents_stop():
    n = 32
    for (h, v, speed, cls) in ((1.0, 0.2, 1.8, 1), (1.0, 0.8, 0.9, 2), (1.0, 1.6, 0.45, 3), (1.5, 1.6, 0.0, 4)):
        # frozen water: huge domain-uniform state; flood still evolves but stays uniform away from walls
        sc = box(n, n, dx=1.0, h0=h, v0=v, peds=dict(x=[10.5], y=[16.5], vx=[0.5], vpref=[1.2]),
                 exit_cell=16 * n + n - 1, dt_max=0.05)
        o = oracle.Oracle(sc)
        o.step(1)
        p = o.read_peds()
        assert p["state"][0] == cls
        dt = o.stats()["t"]
        want = (0.5 + dt * speed / 0.5) / (1 + dt / 0.5)
        want = min(want, 1.3 * speed)                       # speed cap; v0 = 0 -> trapped (Table 1)
        assert abs(p["vx"][0] - want) < 1e-14
        if cls == 4:
            assert p["vx"][0] == 0.0 and p["x"][0] == 10.5


def test_walls_reject_moves_and_nobody_enters_a_solid():
    n = 24
    mask = np.zeros((n, n), np.uint8)
    mask[:, 12] = 1
    mask[11:13, 12] = 0                                      # a door
    rng = np.random.default_rng(4)
    x = rng.uniform(1, 11, 150); y = rng.uniform(1, 23, 150)
    sc = box(n, n, dx=1.0, mask=mask, peds=dict(x=x, y=y), exit_cell=12 * n + n - 1, dt_max=0.3)
    o = oracle.Oracle(sc)
    for _ in range(400):
        o.step(1)
        p = o.read_peds()
        act = p["active"] == 1
        ci = np.floor(p["x"][act]).astype(int); cj = np.floor(p["y"][act]).astype(int)
        assert np.all((ci >= 0) & (ci < n) & (cj >= 0) & (cj < n))
        assert np.all(mask[cj, ci] == 0)
    assert o.stats()["hist"][5] >= 140                        # almost everybody got out through the door


def test_exit_removes_agents_within_arrive_cells():
    n = 16
    ex = 8 * n + 15
    sc = box(n, n, dx=1.0, peds=dict(x=[14.5, 13.5, 14.5], y=[8.5, 8.5, 10.5]), exit_cell=ex)
    o = oracle.Oracle(sc); o.step(1)
    p = o.read_peds()
    assert list(p["active"]) == [0, 1, 1]                   # Chebyshev distance 1, 2, 2
    assert p["x"][0] == 14.5                                 # the leaver does not move
    assert o.stats()["hist"][5] == 1


# ------------------------------------------------------------------ responders and the barrier

def _barrier_box(n_resp=1, bags=1, layers=2, line=(5, 6, 7)):
    n = 16
    line_cells = np.array([4 * n + i for i in line], np.int32)
    from paper_1908_05232_b200.scenarios import nav_field
    mask = np.zeros((n, n), np.uint8)
    storage, drop, ex = 12 * n + 2, int(line_cells[0]), 8 * n + 15
    nav = np.stack([nav_field(mask, [c])[0] for c in (ex, storage, drop)])
    xs = np.full(n_resp, 2.5) + 0.01 * np.arange(n_resp); ys = np.full(n_resp, 10.5)
    sc = box(n, n, dx=1.0, peds=dict(x=xs, y=ys, role=np.ones(n_resp)), dt_max=0.25, A_s=0.0)
    sc.nav_dir = nav; sc.exit_cells = np.array([ex], np.int32)
    sc.exit_target, sc.storage_target, sc.drop_target = 0, 1, 2
    sc.storage_cell, sc.drop_cell = storage, drop
    sc.line_cells = line_cells
    sc.bags_per_cell_layer, sc.n_layers, sc.layer_thickness = bags, layers, 0.25
    sc.t_pick = sc.t_drop = 30.0
    return sc


def test_responder_timeline():
    """storage -> wait 30 s -> barrier -> wait 30 s -> deposit -> repeat -> evacuate."""
    sc = _barrier_box(bags=1, layers=1, line=(5,))
    o = oracle.Oracle(sc)
    seen = []
    t_dep = None
    for _ in range(2000):
        o.step(1)
        p = o.read_peds(); st = o.stats()
        if not seen or seen[-1][0] != p["fsm"][0]:
            seen.append((int(p["fsm"][0]), st["t"]))
        if st["deposits"] == 1 and t_dep is None:
            t_dep = st["t"]
        if p["active"][0] == 0:
            break
    fsms = [s for s, _ in seen]
    # starts 2 cells from storage: TO_STORAGE, PICKING, TO_BARRIER, DROPPING, then the barrier is
    # complete only AFTER the deposit step, so one more round trip before EVACUATE (C31, O3.7)
    assert fsms[:4] == [1, 2, 3, 4]
    t = dict((s, tt) for s, tt in reversed(seen))
    assert abs((t[3] - t[2]) - 30.0) <= 0.25 + 1e-9          # picking wait (120 steps of 0.25 s)
    assert st["deposits"] >= 1 and st["barrier_complete"] == 1
    assert abs(o.read_flood()["z"][4 * 16 + 5] - 0.25) < 1e-15
    assert p["active"][0] == 0 and fsms[-1] == 0


def test_barrier_integer_arithmetic():
    """D deposits -> (cursor, layer, bags, z) by integer arithmetic; Config 3 numbers: 40 cells x
    12 layers x 0.05 m = 480 deposits -> 0.6 m everywhere (BASELINE.json configs[2])."""
    sc = _barrier_box(n_resp=7, bags=3, layers=2, line=(5, 6, 7))
    o = oracle.Oracle(sc)
    # put all 7 responders into DROPPING with an expiring timer: 7 deposits in one step
    p0 = o.read_peds()
    o.write_peds(fsm=np.full(7, 4, np.uint8), timer=np.full(7, 0.1))
    o.step(1)
    st = o.stats()
    assert st["deposits"] == 7 and (st["cursor"], st["layer"], st["bags"]) == (2, 0, 1)
    z = o.read_flood()["z"]
    assert z[4 * 16 + 5] == 0.25 and z[4 * 16 + 6] == 0.25 and z[4 * 16 + 7] == 0.0
    assert np.all(o.read_peds()["fsm"] == 1)                # back to storage (barrier not complete)
    # 11 more -> total 18 = 3 bags x 3 cells x 2 layers: complete
    o.write_peds(fsm=np.full(7, 4, np.uint8), timer=np.full(7, 0.1)); o.step(1)
    o.write_peds(fsm=np.full(7, 4, np.uint8), timer=np.full(7, 0.1)); o.step(1)
    st = o.stats()
    assert st["deposits"] == 21 and st["barrier_complete"] == 1 and st["layer"] == 2
    z = o.read_flood()["z"]
    assert np.all(z[[4 * 16 + 5, 4 * 16 + 6, 4 * 16 + 7]] == 0.5)
    assert z.sum() == 1.5                                    # extra deposits after completion are ignored
    # Config 3's own numbers
    sc3 = _barrier_box(n_resp=40, bags=1, layers=12, line=tuple(range(2, 14)))
    sc3.layer_thickness = 0.05
    o3 = oracle.Oracle(sc3)
    total = 0
    while total < 12 * 12:
        o3.write_peds(fsm=np.full(40, 4, np.uint8), timer=np.full(40, 0.1)); o3.step(1)
        total += 40
    z3 = o3.read_flood()["z"][[4 * 16 + i for i in range(2, 14)]]
    assert np.allclose(z3, 0.6, atol=1e-15) and o3.stats()["barrier_complete"] == 1


def test_raising_the_bed_lifts_the_water_and_keeps_volume():
    sc = _barrier_box(n_resp=3, bags=1, layers=1, line=(5, 6, 7))
    sc.h0 = np.full(256, 0.3)
    o = oracle.Oracle(sc)
    v0 = o.stats()["volume"]
    o.write_peds(fsm=np.full(3, 4, np.uint8), timer=np.full(3, 0.01)); o.step(1)
    assert o.stats()["barrier_complete"] == 1
    assert abs(o.stats()["volume"] - v0) <= 1e-13 * v0       # h kept, eta jumps
    o.step(50)
    c = o.read_conserved()
    assert abs(o.stats()["volume"] - v0) <= 1e-12 * v0 and np.abs(c["qy"]).max() > 1e-3


def test_config1_pedestrians_follow_the_papers_rule():
    """in Config 1 the 'dry half' holds 0.1 m so agents start LOW (1.8 m/s), and the
    bore (HR ~ 1.12) turns them MEDIUM."""
    o = oracle.Oracle(S.make(1))
    o.step(1)
    assert np.all(o.read_peds()["state"][o.read_peds()["active"] == 1] == 1)
    o.step(99)
    hist = o.stats()["hist"]
    assert hist[2] > 0 and hist[3] == 0 and hist[4] == 0 and sum(hist) == 256
