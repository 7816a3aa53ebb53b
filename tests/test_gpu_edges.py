"""GPU parity on the degenerate cases of the coupled step: everybody gone, one over-full cell,
coincident agents, halting inside a replayed graph and resuming, and the two forms of the step
graph (pedestrian branch beside the flood kernel / one chain) giving the same bits."""
import numpy as np
import pytest

import oracle
from paper_1908_05232_b200 import binding, scenarios as S
from helpers import box
from gpu_common import make_pair, sync, mixed

pytestmark = pytest.mark.gpu


def _same_peds(g, o, tol):
    a, b = g.read_peds(), o.read_peds()
    assert np.array_equal(a["active"], b["active"]) and np.array_equal(a["fsm"], b["fsm"])
    act = b["active"] == 1
    assert np.array_equal(a["state"][act], b["state"][act])
    for k in ("x", "y", "vx", "vy"):
        if act.any():
            assert mixed(a[k][act], b[k][act]) <= tol, k


def test_everybody_has_left_and_steps_go_on():
    """all agents inactive: every key is the overflow bin, N_p is zero everywhere, the flood goes on"""
    rng = np.random.default_rng(3)
    n = 64
    sc = box(n, n, dx=0.5, real_bits=32, h0=np.where(np.arange(n)[None, :] < 20, 0.5, 0.0) + np.zeros((n, 1)),
             manning=0.02, peds=dict(x=rng.uniform(1, 30, 300), y=rng.uniform(1, 30, 300)), exit_cell=5 * n + 5, dt_max=0.05)
    o, g = make_pair(sc)
    gone = np.zeros(300, np.uint8)
    p = o.read_peds()
    for s in (o, g):
        s.write_peds(p["x"], p["y"], p["vx"], p["vy"], p["fsm"], gone, p["timer"])
    for _ in range(3):
        o.step(1); g.step(1)
    assert g.stats()["hist"][5] == 300 and o.stats()["hist"][5] == 300
    assert not g.read_occupancy().any()
    a, b = g.read_conserved(), o.read_conserved()
    for k in ("h", "qx", "qy"):
        assert mixed(a[k], b[k]) <= 1e-5


@pytest.mark.parametrize("bits", [64, 32])
def test_overfull_cell_saturates_np_and_coincident_agents_do_not_interact(bits):
    """300 agents in ONE cell (N_p > 255: the uint8 count saturates, the roughness rule only uses
    min(N_p, 20)), 40 of them at exactly the same point (d = 0 pairs are skipped, C26)"""
    rng = np.random.default_rng(11)
    n = 32
    x = 10.0 + rng.uniform(0.01, 0.99, 300); y = 12.0 + rng.uniform(0.01, 0.99, 300)
    x[:40] = 10.5; y[:40] = 12.5
    x = np.concatenate([x, rng.uniform(2, 30, 50)]); y = np.concatenate([y, rng.uniform(2, 30, 50)])
    sc = box(n, n, dx=1.0, real_bits=bits, h0=0.3, u0=0.4, manning=0.02, peds=dict(x=x, y=y),
             exit_cell=16 * n + 31, dt_max=0.02)
    o, g = make_pair(sc)
    sync(o, g, sc)
    o.step(1); g.step(1)
    occ_g, occ_o = g.read_occupancy().astype(np.int64), o.read_occupancy()
    c = 12 * n + 10
    assert occ_o[c] >= 300 and occ_g[c] == 255
    assert np.array_equal(occ_g, np.minimum(occ_o, 255))
    a, b = g.read_conserved(), o.read_conserved()
    for k in ("h", "qx", "qy"):
        assert mixed(a[k], b[k]) <= (1e-12 if bits == 64 else 1e-5), k
    pa, pb = g.read_peds(), o.read_peds()
    assert np.array_equal(pa["active"], pb["active"]) and np.array_equal(pa["state"], pb["state"])
    assert np.all(np.isfinite(pa["x"])) and np.all(np.isfinite(pa["vx"]))
    # the coincident agents feel the same force from everybody else and none from one another
    assert np.ptp(pa["vx"][:40]) <= 1e-4 * max(1.0, np.abs(pa["vx"][:40]).max())


def test_halt_inside_a_graph_then_rewind_and_resume():
    """t_end falls inside a 32-step graph replay: later steps are no-ops, the binning chain that
    ran beside the last tail kernel is harmless; after set_time() the run resumes like the oracle"""
    sc = S.make(2, n=64, n_evac=150)
    sc.hydro_q = sc.hydro_q * 30.0
    sc.t_end = 1.6
    o, g = make_pair(sc)
    sync(o, g, sc)
    o.step(70); g.step(70)                                 # 2 graph replays of 32 + 6 single steps
    so, sg = o.stats(), g.stats()
    assert sg["t"] == pytest.approx(1.6, abs=1e-12) and so["t"] == pytest.approx(1.6, abs=1e-12)
    assert abs(sg["step"] - so["step"]) <= 1 and sg["step"] < 70
    h_halt = g.read_conserved()["h"].copy()
    g.step(40)                                             # still halted: nothing moves
    assert g.stats()["step"] == sg["step"] and np.array_equal(h_halt, g.read_conserved()["h"])
    st = sync(o, g, sc)                                    # identical state again, still at t_end
    dt = float(np.float32(0.02))
    o.set_time(0.5, dt); g.set_time(0.5, dt)               # rewind: un-halts both
    for _ in range(3):
        o.step(1); g.step(1)
    assert g.stats()["step"] == o.stats()["step"] == st["step"] + 3
    a, b = g.read_conserved(), o.read_conserved()
    for k in ("h", "qx", "qy"):
        assert mixed(a[k], b[k]) <= 3e-5, k
    _same_peds(g, o, 1e-4)
    assert np.array_equal(g.read_occupancy().astype(np.int64), np.minimum(o.read_occupancy(), 255))


def test_step_graph_with_and_without_the_parallel_branch_gives_the_same_bits():
    """sparse crowd (no two agents within R_int, so no summation order to differ): 100 steps with the
    pedestrian branch beside the flood kernel, in one chain, and kernel by kernel (profiled mode)"""
    n = 128
    gx, gy = np.meshgrid(np.arange(8, 120, 7.0), np.arange(8, 120, 7.0))
    sc = S.make(2, n=n, n_evac=10)
    sc.hydro_q = sc.hydro_q * 30.0
    walk = sc.mask.reshape(n, n) == 0
    keep = walk[(gy.ravel() / sc.dy).astype(int), (gx.ravel() / sc.dx).astype(int)]
    x, y = gx.ravel()[keep] * 0.5 + 0.1, gy.ravel()[keep] * 0.5 + 0.1
    m = x.size
    sc.px, sc.py = x.astype(np.float32), y.astype(np.float32)
    sc.pvx = np.zeros(m, np.float32); sc.pvy = np.zeros(m, np.float32)
    sc.pvpref = np.full(m, 0.2, np.float32); sc.prole = np.zeros(m, np.uint8)
    outs = []
    for mode in ("branch", "chain", "profiled"):
        g = binding.Sim(sc)
        if mode == "chain":
            g.set_overlap(False)
        if mode == "profiled":
            g.step_profiled(100)
        else:
            g.step(100)
        outs.append((g.read_conserved(), g.read_peds(), g.read_occupancy(), g.stats()))
        g.close()
    for c, p, occ, st in outs[1:]:
        for k in ("h", "qx", "qy"):
            assert np.array_equal(c[k], outs[0][0][k]), k
        for k in ("x", "y", "vx", "vy", "state", "active", "cell"):
            assert np.array_equal(p[k], outs[0][1][k]), k
        assert np.array_equal(occ, outs[0][2])
        assert st["t"] == outs[0][3]["t"] and st["step"] == 100


def _sparse_scenario(n=128):
    """a flooding hall with a sparse crowd (no agent ever has two partners within R_int, so the
    pedestrian sums have one order only and every run is bit-reproducible)"""
    gx, gy = np.meshgrid(np.arange(8, 120, 7.0), np.arange(8, 120, 7.0))
    sc = S.make(2, n=n, n_evac=10)
    sc.hydro_q = sc.hydro_q * 30.0
    walk = sc.mask.reshape(n, n) == 0
    keep = walk[(gy.ravel() / sc.dy).astype(int), (gx.ravel() / sc.dx).astype(int)]
    x, y = gx.ravel()[keep] * 0.5 + 0.1, gy.ravel()[keep] * 0.5 + 0.1
    m = x.size
    sc.px, sc.py = x.astype(np.float32), y.astype(np.float32)
    sc.pvx = np.zeros(m, np.float32); sc.pvy = np.zeros(m, np.float32)
    sc.pvpref = np.full(m, 0.2, np.float32); sc.prole = np.zeros(m, np.uint8)
    return sc


def _state(g):
    c, p = g.read_conserved(), g.read_peds()
    return [c["h"], c["qx"], c["qy"], p["x"], p["y"], p["vx"], p["vy"], p["state"], p["active"], g.read_occupancy()]


def _same(a, b):
    return all(np.array_equal(u, v) for u, v in zip(a, b))


def test_step_counts_split_any_way_give_the_same_bits():
    """37 steps as one call (a 32-step graph + 5 single ones), as 32 + 5, as 37 x 1, and with
    read-backs in between (which must not disturb the prepared binning of the next step)"""
    sc = _sparse_scenario()
    ref = binding.Sim(sc); ref.step(37); want = _state(ref); t = ref.stats()["t"]
    g = binding.Sim(sc); g.step(32); g.step(5)
    assert _same(_state(g), want) and g.stats()["t"] == t
    g = binding.Sim(sc)
    for k in range(37):
        g.step(1)
        if k % 9 == 0:
            g.read_peds(); g.stats(); g.read_flood(("h", "hr")); g.bin_peds()
    assert _same(_state(g), want) and g.stats()["t"] == t


def test_two_handles_on_one_gpu_do_not_disturb_each_other():
    """replicas: two sim_t on one device, stepped alternately, equal their solo runs"""
    sa, sb = _sparse_scenario(), S.make(1)
    solo_a = binding.Sim(sa); solo_a.step(40); wa = _state(solo_a)
    solo_b = binding.Sim(sb); solo_b.step(40); wb = _state(solo_b)
    ga, gb = binding.Sim(sa), binding.Sim(sb)
    for _ in range(8):
        ga.step(5); gb.step(5)
    assert _same(_state(ga), wa)
    # Config 1 is a dense-ish crowd: compare the flood bitwise, the pedestrians within tolerance
    got = _state(gb)
    assert all(np.array_equal(u, v) for u, v in zip(got[:3], wb[:3])) or mixed(got[0], wb[0]) <= 1e-12
    assert mixed(got[3], wb[3]) <= 1e-9


def test_rows_per_chunk_do_not_change_the_flood():
    """the chunk height of the row-marching kernel is a tuning parameter.  It moves the border
    between chunks on the packed/TMA path and chunks on the general path (different FMA contraction),
    so the results agree to rounding, not to the bit"""
    rng = np.random.default_rng(5)
    nx, ny = 1024, 160
    jj, ii = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    z = 0.3 * (1 + np.sin(ii / 37.0) * np.cos(jj / 11.0))
    mask = np.zeros((ny, nx), np.uint8); mask[60:70, 300:330] = 1; mask[100, 511:514] = 1
    sc = box(nx, ny, dx=0.25, real_bits=32, z=z, h0=np.maximum(0.0, 0.35 - z), u0=rng.normal(0, 0.3, (ny, nx)),
             v0=rng.normal(0, 0.3, (ny, nx)), mask=mask, manning=0.02, dt_max=0.02)
    outs = []
    for rows in (8, 19, 64):
        g = binding.Sim(sc); g.set_flood_variant(4); g.set_march_rows(rows); g.step(6)
        outs.append(g.read_conserved()); g.close()
    for o in outs[1:]:
        for k in ("h", "qx", "qy"):
            assert mixed(o[k], outs[0][k]) <= 6 * 2e-6, (k, mixed(o[k], outs[0][k]))


def test_long_hydrograph_table_is_interpolated_like_the_oracle():
    """70 break points (more than one warp of table entries in the tail kernel), times landing
    before, inside and after the table"""
    n = 64
    rng = np.random.default_rng(21)
    ht = np.cumsum(rng.uniform(0.05, 0.4, 70)) + 0.3
    hq = rng.uniform(0.0, 6.0, 70)
    sc = box(n, n, dx=0.5, real_bits=64, h0=0.05, manning=0.02, dt_max=0.25,
             inflow_cell=np.arange(10, 30, dtype=np.int32), inflow_side=np.full(20, S.SIDE_S, np.uint8),
             hydro_t=ht, hydro_q=hq)
    o, g = make_pair(sc)
    for _ in range(30):
        o.step(7); g.step(7)
        so, sg = o.stats(), g.stats()
        assert sg["t"] == pytest.approx(so["t"], rel=1e-12)
        assert sg["volume"] == pytest.approx(so["volume"], rel=1e-11)
    assert o.stats()["t"] > ht[-1]                          # ran past the end of the table
    a, b = g.read_conserved(), o.read_conserved()
    for k in ("h", "qx", "qy"):
        assert mixed(a[k], b[k]) <= 1e-9, k
